// ulm_rca_api.cu -- plan construction and the extern "C" boundary declared in include/ulm_rca.h.
//
// Host code here is fp64 table building and launch bookkeeping only; every step of the hot path
// (demodulation, delay, interpolation, apodisation, compounding, projection write) runs in the kernels
// of ulm_rca_device.cuh / ulm_rca_ring.cuh.  There is no CPU fallback.
#include "ulm_rca.h"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "ulm_rca_device.cuh"
#include "ulm_rca_ring_host.cuh"
#include "ulm_rca_stage2_host.cuh"
#include "ulm_rca_clutter_host.cuh"
#include "ulm_rca_motion_host.cuh"
#include "ulm_rca_localize.cuh"

namespace {

thread_local char g_err[512] = "";

ulm_rca_status fail(ulm_rca_status st, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}

#define CUDA_TRY(expr)                                                                          \
    do {                                                                                        \
        cudaError_t e_ = (expr);                                                                \
        if (e_ != cudaSuccess)                                                                  \
            return fail(e_ == cudaErrorMemoryAllocation ? ULM_RCA_ENOMEM : ULM_RCA_ECUDA,       \
                        "%s: %s", #expr, cudaGetErrorString(e_));                              \
    } while (0)

struct DeviceBuf {
    void *p = nullptr;
    ~DeviceBuf() { if (p) cudaFree(p); }
    DeviceBuf() = default;
    DeviceBuf(const DeviceBuf &) = delete;
    DeviceBuf &operator=(const DeviceBuf &) = delete;
    template <class T> T *as() const { return static_cast<T *>(p); }
    template <class T> cudaError_t upload(const std::vector<T> &v) {
        if (p) { cudaFree(p); p = nullptr; }
        if (v.empty()) return cudaSuccess;
        cudaError_t e = cudaMalloc(&p, v.size() * sizeof(T));
        if (e != cudaSuccess) return e;
        return cudaMemcpy(p, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
    }
};

struct Grid {
    int n_lat = 0, n_ax = 0;
    double lat0 = 0, dlat = 0, z0 = 0, dz = 0, ref = 0;
    double lat(int i) const { return lat0 + i * dlat; }
    double z(int i) const { return z0 + i * dz; }
};

// transmit-side tables of one aperture for a list of reference coordinates ("planes")
struct TxTables {
    int n_planes = 0;
    DeviceBuf n0, f0m;
    DeviceBuf tab;      // the same as {bits of f0m, n0}, [plane][iz][k (kpad)] (volume tables only: das_volume_kernel)
    int kpad = 0;
    // mirror form (das_volume_mirror_kernel), built when the planes and the angle set are mirror-symmetric
    DeviceBuf mtab;     // [plane < n_planes / 2][iz][slot (mkpad)]
    int mkpad = 0, n_mpairs = 0, n_msingle = 0;
    short mk[ulm::kVolMirrorMaxAngles] = {};
};

struct Aperture {
    bool row_tx = true;
    int n_tx = 0, n_rx = 0, e0 = 0;
    Grid g;
    std::vector<double> angles, t0;
    // Folded view of the transmit events for the compounded projection (compound = 1): events whose transmit delay
    // U0_k(z) on the reference slice is identical for every depth (mirror angles +-theta about a centred slice with
    // equal t0) have the same sample index, interpolation weight and phase for every (pixel, element), so by
    // linearity their channel data are added in the pre-pass and beamformed as ONE event.  fk[v] = the real event k
    // that represents folded event v, fk2[v] = its partner (-1: none), fe0 = index of the aperture's first folded
    // event among all folded events.  Identity when nothing folds.
    std::vector<int> fk, fk2;
    int fe0 = 0;
    std::vector<double> fangles, ft0;
    DeviceBuf xs, zs, ejs, xm, zm, ejm, win;
    TxTables proj;      // 1 plane: the reference slice; one table row block per FOLDED event
    TxTables vol;       // volume comparator: one plane per pixel of the other lateral axis
    ulm::RingTables ring;
    ulm::RingTables ring2;            // tiles of the two-group work items (ring_plan_dual)
    long long out_base = 0;
};

}  // namespace

struct ulm_rca_plan {
    int n_rows = 0, n_cols = 0;
    double pitch = 0, c = 0, fs = 0, fc = 0, t_start = 0, f_number = 0;
    int input_kind = 0, cpe = 0, n_samples = 0, compound = 1, max_frames = 32, build_volume = 0;
    int n_events = 0, n_rx_max = 0, half_len = 0;
    int device = 0;               // the CUDA device that was current at plan_create: owns every buffer of the plan
    int nv_events = 0;            // folded events of the projection path (= n_events when nothing folds)
    DeviceBuf ev_fold, ev_id;     // short2 per scratch event row: the (first, second or -1) real events it holds
    bool apod = false;
    Aperture ap[2];               // [0] x-z (row-tx), [1] y-z (column-tx)
    int n_lo = 0, l_row = 0;      // IQ scratch origin / entries per row
    int mix_n0 = 0;
    DeviceBuf mixer, iq;
    DeviceBuf vol_rows;           // one frame of fp32 rows for the single-frame volume kernel (build_volume only)
    size_t iq_bytes = 0;
    ulm::DemodConst demod{};
    int kernel = 1;               // 1 generic, 2 ring
    bool d32 = false;             // full (fp32) difference term in the scratch
    bool w2 = false;              // compact entries, interpolation weight carried as two fp16 terms (precision = 3)
    bool quad = false;            // fs = 4 fc exactly, default 17 taps, analytic signal from two real filters
    bool half_band = false;       // every even demodulation tap except the centre is exactly zero (fs = 4 fc)
    bool quarter_band = false;    // every fourth demodulation tap except the centre is exactly zero (fs = 8 fc)
    bool analytic8 = false;       // RF input, fs = 8 fc exactly, 33 taps: analytic signal from two real filters (ga, gb)
    ulm::RingConfig ring{};
    long long out_per_frame = 0, vol_per_frame = 0;
    mutable long long last_launches = 0;
    // host-convenience staging
    // (two slots of h_stage_frames frames each: the upload of chunk i + 1 overlaps the kernels / download of chunk i)
    DeviceBuf h_stage_in, h_stage_out;
    size_t h_stage_frames = 0;
    cudaStream_t h_copy = nullptr, h_compute = nullptr;     // created on the first host call
    static constexpr int kHostSlots = 2;
    cudaEvent_t h_in_done[kHostSlots] = {}, h_slot_free[kHostSlots] = {};
    bool timing = true;           // record CUDA events around the kernels (options.no_timing = 0)
    ulm::Stage2Plan s2;           // Stage 2 + sum-projection tables (options.stage2_block > 0)
    mutable ulm::ClutterPlan cf;  // clutter filter scratch (options.clutter_frames > 0)
    ulm::MotionPlan mo;           // motion estimation scratch (options.motion_frames > 0)
    DeviceBuf loc_frame_max;      // per-frame maximum |V| for ulm_rca_localize (with stage2_block)
    // CUDA events around the kernels of the last kTimedCalls calls (per batch: before demod, after demod,
    // after DAS; the first kTimedBatches batches of a call)
    static constexpr int kTimedCalls = 64, kTimedBatches = 4;
    cudaEvent_t ev[kTimedCalls][kTimedBatches][3] = {};
    mutable int timed_batches[kTimedCalls] = {};
    mutable long long n_calls = 0;
    ~ulm_rca_plan() {
        for (auto &c : ev) for (auto &b : c) for (auto &e : b) if (e) cudaEventDestroy(e);
        for (auto &e : h_in_done) if (e) cudaEventDestroy(e);
        for (auto &e : h_slot_free) if (e) cudaEventDestroy(e);
        if (h_copy) cudaStreamDestroy(h_copy);
        if (h_compute) cudaStreamDestroy(h_compute);
    }
};

namespace {

double elem_pos(int e, int n, double pitch) { return (e - 0.5 * (n - 1)) * pitch; }

// U0 = (t0_k + (z cos th + ref sin th)/c + z/c - t_start) fs
double u0_of(const ulm_rca_plan &P, const Aperture &A, int k, double ref, double z) {
    return (A.t0[k] + (z * std::cos(A.angles[k]) + ref * std::sin(A.angles[k])) / P.c + z / P.c - P.t_start) * P.fs;
}

// largest receive excess H = (sqrt(dx^2 + z^2) - z) fs/c over the lateral grid and elements at depth z
double h_max_at(const ulm_rca_plan &P, const Aperture &A, double z) {
    const double lat_a = A.g.lat(0), lat_b = A.g.lat(A.g.n_lat - 1);
    const double e_a = elem_pos(0, A.n_rx, P.pitch), e_b = elem_pos(A.n_rx - 1, A.n_rx, P.pitch);
    const double d = std::max({std::fabs(lat_a - e_a), std::fabs(lat_a - e_b), std::fabs(lat_b - e_a),
                               std::fabs(lat_b - e_b)});
    return (std::sqrt(d * d + z * z) - z) * P.fs / P.c;
}

void sample_range(const ulm_rca_plan &P, const Aperture &A, const std::vector<double> &refs, double &u_min,
                  double &u_max) {
    for (double ref : refs)
        for (int k = 0; k < A.n_tx; ++k)
            for (int iz = 0; iz < A.g.n_ax; ++iz) {
                const double z = A.g.z(iz);
                const double u0 = u0_of(P, A, k, ref, z);
                u_min = std::min(u_min, u0);
                u_max = std::max(u_max, u0 + h_max_at(P, A, z));
            }
}

// Folding of one aperture's transmit events (host only, fp64): partner[k] = the later event folded into event k
// (-1: none), -2 for an event that is itself the partner of an earlier one.  Two events fold when their transmit
// delay on the reference slice, U0_k(z) = (t0_k + (z cos th_k + ref sin th_k)/c + z/c - t_start) fs, agrees to
// 1e-9 samples on every depth row (far below the fp32 resolution of the delay); greedy, first match wins.
std::vector<int> fold_partners(const std::vector<double> &angles, const std::vector<double> &t0, double c, double fs,
                               double ref, double z0, double dz, int n_ax, bool enable) {
    const int n = (int)angles.size();
    std::vector<int> partner(n, -1);
    auto u0 = [&](int k, double z) { return (t0[k] + (z * std::cos(angles[k]) + ref * std::sin(angles[k])) / c + z / c) * fs; };
    for (int k = 0; k < n && enable; ++k) {
        if (partner[k] == -2) continue;
        for (int k2 = k + 1; k2 < n; ++k2) {
            if (partner[k2] != -1) continue;
            double dmax = 0;
            for (int iz = 0; iz < n_ax; ++iz) dmax = std::max(dmax, std::fabs(u0(k, z0 + iz * dz) - u0(k2, z0 + iz * dz)));
            if (dmax <= 1e-9) { partner[k] = k2; partner[k2] = -2; break; }
        }
    }
    return partner;
}

cudaError_t build_tx_tables(const ulm_rca_plan &P, const Aperture &A, const std::vector<double> &refs,
                            const std::vector<int> &ks, TxTables &T, bool interleaved = false) {
    const size_t n = refs.size() * ks.size() * A.g.n_ax;
    std::vector<int> n0(n);
    std::vector<float> f0m(n);
    size_t i = 0;
    for (double ref : refs)
        for (int k : ks)
            for (int iz = 0; iz < A.g.n_ax; ++iz, ++i) {
                const double u0 = u0_of(P, A, k, ref, A.g.z(iz));
                const double fl = std::floor(u0);
                n0[i] = (int)fl - P.n_lo;
                f0m[i] = (float)(u0 - fl - 0.5);
            }
    T.n_planes = (int)refs.size();
    cudaError_t e;
    if (interleaved) {      // [plane][iz][k], k padded to an even count (das_volume_kernel reads two angles per load)
        const size_t nk = ks.size(), kpad = (nk + 1) / 2 * 2, nz = (size_t)A.g.n_ax;
        std::vector<int2> tab(refs.size() * nz * kpad, make_int2(0, 0));
        for (size_t r = 0; r < refs.size(); ++r)
            for (size_t ki = 0; ki < nk; ++ki)
                for (size_t iz = 0; iz < nz; ++iz) {
                    const size_t q = (r * nk + ki) * nz + iz;
                    int bits;
                    std::memcpy(&bits, &f0m[q], sizeof(bits));
                    tab[(r * nz + iz) * kpad + ki] = make_int2(bits, n0[q]);
                }
        T.kpad = (int)kpad;
        if ((e = T.tab.upload(tab)) != cudaSuccess) return e;
    }
    if ((e = T.n0.upload(n0)) != cudaSuccess) return e;
    return T.f0m.upload(f0m);
}

// Mirror form of the volume tables: possible when the planes come in pairs (p, n - 1 - p) and the angles in pairs (k, kb)
// -- or self-mirrored -- with  U0_k(plane p, z) = U0_kb(plane n - 1 - p, z)  to 1e-5 sample (a centred grid and a
// symmetric angle set with equal start delays; grid parameters that went through fp32 leave ~4e-6 sample on cfg 4, a
// fraction of the fp32 ulp of the delay sum itself).  The shared table entry is the MEAN of the two delays, so each of
// the two terms is off by half that difference.  Leaves T.mtab empty otherwise: the caller keeps das_volume_kernel.
cudaError_t build_mirror_tables(const ulm_rca_plan &P, const Aperture &A, const std::vector<double> &refs, TxTables &T) {
    const int np = (int)refs.size(), nk = A.n_tx, nz = A.g.n_ax;
    if (np < 2 || (np & 1) || nk < 1 || nk > ulm::kVolMirrorMaxAngles || nz < 1) return cudaSuccess;
    std::vector<int> mate(nk, -1);
    const double za = A.g.z(0), zb = A.g.z(nz - 1);
    for (int k = 0; k < nk; ++k) {
        if (mate[k] >= 0) continue;
        for (int k2 = k; k2 < nk; ++k2) {
            if (mate[k2] >= 0) continue;
            double dmax = 0;
            for (int p = 0; p < np; ++p)
                for (double z : {za, zb}) dmax = std::max(dmax, std::fabs(u0_of(P, A, k, refs[p], z) - u0_of(P, A, k2, refs[np - 1 - p], z)));
            if (dmax <= 1e-5) { mate[k] = k2; mate[k2] = k; break; }
        }
        if (mate[k] < 0) return cudaSuccess;          // an angle without a mirror partner
    }
    std::vector<short> mk;
    int n_pairs = 0, n_single = 0;
    for (int k = 0; k < nk; ++k) if (mate[k] > k) { mk.push_back((short)k); mk.push_back((short)mate[k]); ++n_pairs; }
    for (int k = 0; k < nk; ++k) if (mate[k] == k) { mk.push_back((short)k); ++n_single; }
    const size_t kpad = ((size_t)mk.size() + 1) / 2 * 2;
    std::vector<int2> tab((size_t)(np / 2) * nz * kpad, make_int2(0, 0));
    for (int p = 0; p < np / 2; ++p)
        for (int iz = 0; iz < nz; ++iz)
            for (size_t sl = 0; sl < mk.size(); ++sl) {
                const double u0 = 0.5 * (u0_of(P, A, mk[sl], refs[p], A.g.z(iz)) + u0_of(P, A, mate[mk[sl]], refs[np - 1 - p], A.g.z(iz)));
                const double fl = std::floor(u0);
                const float f0m = (float)(u0 - fl - 0.5);
                int bits;
                std::memcpy(&bits, &f0m, sizeof(bits));
                tab[((size_t)p * nz + iz) * kpad + sl] = make_int2(bits, (int)fl - P.n_lo);
            }
    T.mkpad = (int)kpad; T.n_mpairs = n_pairs; T.n_msingle = n_single;
    for (size_t sl = 0; sl < mk.size(); ++sl) T.mk[sl] = mk[sl];
    return T.mtab.upload(tab);
}

ulm_rca_status build_demod(ulm_rca_plan &P, int demod_taps) {
    ulm::DemodConst &D = P.demod;
    if (P.input_kind == 1) {
        P.half_len = D.half_len = 0;
        D.gd[0] = 1.f;
        return ULM_RCA_OK;
    }
    const int L = demod_taps > 0 ? (demod_taps - 1) / 2 : 2 * (int)std::lround(P.fs / P.fc);
    if (2 * L + 1 > ulm::kMaxTaps) return fail(ULM_RCA_EUNSUPPORTED, "demod_taps %d > %d", 2 * L + 1, ulm::kMaxTaps);
    std::vector<double> h(2 * L + 1);
    double sum = 0;
    for (int m = -L; m <= L; ++m) {
        const double x = 2.0 * P.fc * m / P.fs;
        const double sinc = x == 0.0 ? 1.0 : std::sin(M_PI * x) / (M_PI * x);
        const double win = L > 0 ? 0.54 + 0.46 * std::cos(M_PI * m / L) : 1.0;
        h[m + L] = sinc * win;
        sum += h[m + L];
    }
    for (int t = 0; t <= 2 * L; ++t) {
        const double g = 2.0 * h[t] / sum;
        D.gd[t] = std::fabs(g) < 1e-13 ? 0.f : (float)g;     // exact zeros of the sinc (every 2nd tap at fs = 4 fc)
    }
    P.half_len = D.half_len = L;
    P.half_band = P.quarter_band = true;
    for (int t = 0; t <= 2 * L; ++t) {
        if (t != L && ((t - L) & 1) == 0 && D.gd[t] != 0.f) P.half_band = false;
        if (t != L && ((t - L) % 4) == 0 && D.gd[t] != 0.f) P.quarter_band = false;
    }
    // quadrature sampling: fs = 4 fc exactly (the analytic signal needs no mixer, so any t_start qualifies)
    P.quad = P.half_band && L == 8 && P.fs == 4.0 * P.fc;
    if (P.quad) {
        for (int t = 0; t <= 2 * L; ++t) {
            const int m = t - L;
            const int m4 = ((m % 4) + 4) % 4;
            D.qd[t] = (m == 0) ? (float)(h[t] / sum) : (m4 == 1 ? (float)(h[t] / sum) : m4 == 3 ? (float)(-h[t] / sum) : 0.f);
        }
    }
    // analytic variant at fs = 8 fc with the default 33 taps: s[n] = sum_m g[m] rf[n-m] exp(j theta m), theta = pi/4
    P.analytic8 = false;
    if (P.input_kind == 0 && L == 16 && P.quarter_band && P.fs == 8.0 * P.fc) {
        const double oct[8][2] = {{1, 0}, {M_SQRT1_2, M_SQRT1_2}, {0, 1}, {-M_SQRT1_2, M_SQRT1_2},
                                  {-1, 0}, {-M_SQRT1_2, -M_SQRT1_2}, {0, -1}, {M_SQRT1_2, -M_SQRT1_2}};
        bool ok = true;
        for (int t = 0; t <= 2 * L; ++t) {
            const int m = t - L, m8 = ((m % 8) + 8) % 8, m4 = m8 % 4;
            const double g = 2.0 * h[t] / sum;
            D.ga[t] = D.gd[t] == 0.f ? 0.f : (float)(g * oct[m8][0]);
            D.gb[t] = D.gd[t] == 0.f ? 0.f : (float)(g * oct[m8][1]);
            // the zero pattern the kernel skips at compile time
            if (m4 == 0 && m != 0 && (D.ga[t] != 0.f || D.gb[t] != 0.f)) ok = false;
            if (m4 == 2 && D.ga[t] != 0.f) ok = false;
            if (m == 0 && D.gb[t] != 0.f) ok = false;
        }
        D.rot1[0] = (float)M_SQRT1_2;
        D.rot1[1] = (float)M_SQRT1_2;
        P.analytic8 = ok;
    }
    return ULM_RCA_OK;
}

template <class T> bool finite_pos(T v) { return std::isfinite((double)v) && v > 0; }

ulm_rca_status check_grid(const ulm_rca_grid *g, const char *name) {
    if (!g) return fail(ULM_RCA_EINVAL, "%s is NULL", name);
    if (g->n_lat <= 0 || g->n_ax <= 0) return fail(ULM_RCA_EINVAL, "%s: n_lat and n_ax must be positive", name);
    if (!std::isfinite(g->lat0_m) || !std::isfinite(g->dlat_m) || !std::isfinite(g->z0_m) ||
        !std::isfinite(g->dz_m) || !std::isfinite(g->ref_m))
        return fail(ULM_RCA_EINVAL, "%s: non-finite value", name);
    if (g->z0_m < 0 || !(g->dz_m > 0)) return fail(ULM_RCA_EINVAL, "%s: need z0 >= 0 and dz > 0", name);
    if (g->n_lat > 1 && g->dlat_m == 0) return fail(ULM_RCA_EINVAL, "%s: dlat is 0", name);
    if ((long long)g->n_lat * g->n_ax > (1ll << 30)) return fail(ULM_RCA_EINVAL, "%s: too many pixels", name);
    return ULM_RCA_OK;
}

ulm_rca_status upload_aperture(ulm_rca_plan &P, Aperture &A, const float *window) {
    const double k = P.fs / P.c;
    std::vector<float> xs(A.g.n_lat), xm(A.g.n_lat), zs(A.g.n_ax), zm(A.g.n_ax), ejs(A.n_rx), ejm(A.n_rx), win(A.n_rx);
    for (int i = 0; i < A.g.n_lat; ++i) { xs[i] = (float)(A.g.lat(i) * k); xm[i] = (float)A.g.lat(i); }
    for (int i = 0; i < A.g.n_ax; ++i) { zs[i] = (float)(A.g.z(i) * k); zm[i] = (float)A.g.z(i); }
    for (int j = 0; j < A.n_rx; ++j) {
        const double e = elem_pos(j, A.n_rx, P.pitch);
        ejs[j] = (float)(e * k);
        ejm[j] = (float)e;
        win[j] = window ? window[j] : 1.f;
    }
    CUDA_TRY(A.xs.upload(xs)); CUDA_TRY(A.xm.upload(xm)); CUDA_TRY(A.zs.upload(zs)); CUDA_TRY(A.zm.upload(zm));
    CUDA_TRY(A.ejs.upload(ejs)); CUDA_TRY(A.ejm.upload(ejm)); CUDA_TRY(A.win.upload(win));
    return ULM_RCA_OK;
}

// folded = the scratch holds the folded events of the projection path (T = A.proj), else all real events
ulm::DasParams das_params(const ulm_rca_plan &P, const Aperture &A, const TxTables &T, bool folded) {
    ulm::DasParams D{};
    D.iq = P.iq.as<unsigned char>();
    D.l_row = P.l_row; D.n_rx_max = P.n_rx_max; D.n_events = folded ? P.nv_events : P.n_events;
    D.e0 = folded ? A.fe0 : A.e0; D.n_tx = folded ? (int)A.fk.size() : A.n_tx;
    D.n_rx = A.n_rx; D.n_lat = A.g.n_lat; D.n_ax = A.g.n_ax;
    D.xs = A.xs.as<float>(); D.zs = A.zs.as<float>(); D.ejs = A.ejs.as<float>();
    D.xm = A.xm.as<float>(); D.zm = A.zm.as<float>(); D.ejm = A.ejm.as<float>();
    D.win = A.win.as<float>();
    D.two_f = (float)(2.0 * P.f_number);
    D.n0 = T.n0.as<int>(); D.f0m = T.f0m.as<float>();
    D.fcfs = (float)(P.fc / P.fs);
    D.n_planes = T.n_planes;
    D.rows = P.vol_rows.as<float4>(); D.tab = T.tab.as<int2>(); D.tab_kpad = T.kpad;
    D.mtab = T.mtab.as<int2>(); D.mtab_kpad = T.mkpad; D.n_mpairs = T.n_mpairs; D.n_msingle = T.n_msingle;
    for (int i = 0; i < ulm::kVolMirrorMaxAngles; ++i) D.mk[i] = T.mk[i];
    return D;
}

// frames per scratch group for a batch of n_frames
int group_frames(int n_frames) { return n_frames <= 4 ? 4 : 12; }

template <int F>
void launch_generic_f(const ulm_rca_plan &P, const ulm::DasParams &D, int n_frames, cudaStream_t st) {
    const int npix = D.n_lat * D.n_ax;
    dim3 grid((npix + 127) / 128, (n_frames + F - 1) / F, D.n_planes * (D.per_angle ? D.n_tx : 1));
    if (P.d32) {
        if (P.apod) ulm::das_generic_kernel<F, true, true><<<grid, 128, 0, st>>>(D);
        else ulm::das_generic_kernel<F, true, false><<<grid, 128, 0, st>>>(D);
    } else if (P.w2) {
        if (P.apod) ulm::das_generic_kernel<F, false, true, true><<<grid, 128, 0, st>>>(D);
        else ulm::das_generic_kernel<F, false, false, true><<<grid, 128, 0, st>>>(D);
    } else {
        if (P.apod) ulm::das_generic_kernel<F, false, true><<<grid, 128, 0, st>>>(D);
        else ulm::das_generic_kernel<F, false, false><<<grid, 128, 0, st>>>(D);
    }
    ++P.last_launches;
}

void launch_generic(const ulm_rca_plan &P, const ulm::DasParams &D, int n_frames, cudaStream_t st) {
    if (D.n_tx == 0 || D.n_lat * D.n_ax == 0) return;
    if (group_frames(n_frames) == 12) launch_generic_f<12>(P, D, n_frames, st);
    else launch_generic_f<4>(P, D, n_frames, st);
}

// Volume batches of at most kVolFrameKernelMax frames go frame by frame through unpack_frame_kernel +
// das_volume_kernel; larger batches amortise the index arithmetic over the frames of a group in the generic kernel.
constexpr int kVolFrameKernelMax = 2;
constexpr int kVolPlanes = 4;      // planes per thread of das_volume_kernel

void launch_unpack(const ulm_rca_plan &P, int n_frames, int f, cudaStream_t st) {
    const int F = group_frames(n_frames);
    const long long n = (long long)P.n_events * P.n_rx_max * P.l_row;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    const unsigned char *iq = P.iq.as<unsigned char>() + (size_t)(f / F) * n * ulm::entry_bytes(F, P.d32);
    float4 *rows = P.vol_rows.as<float4>();
    if (F == 12) {
        if (P.d32) ulm::unpack_frame_kernel<12, true><<<blocks, 256, 0, st>>>(iq, rows, n, f % F);
        else ulm::unpack_frame_kernel<12, false><<<blocks, 256, 0, st>>>(iq, rows, n, f % F);
    } else {
        if (P.d32) ulm::unpack_frame_kernel<4, true><<<blocks, 256, 0, st>>>(iq, rows, n, f % F);
        else ulm::unpack_frame_kernel<4, false><<<blocks, 256, 0, st>>>(iq, rows, n, f % F);
    }
    ++P.last_launches;
}

constexpr int kVolMirrorPlanes = 3;      // planes of the lower half per thread of das_volume_mirror_kernel (+ their mirrors)

void launch_volume(const ulm_rca_plan &P, const ulm::DasParams &D, cudaStream_t st) {
    if (D.n_tx == 0 || D.n_lat * D.n_ax == 0) return;
    if (D.mtab) {      // mirror-symmetric planes and angles: two gathers per index computation
        const dim3 grid((D.n_lat * D.n_ax + 127) / 128, (D.n_planes / 2 + kVolMirrorPlanes - 1) / kVolMirrorPlanes);
        if (P.apod) ulm::das_volume_mirror_kernel<kVolMirrorPlanes, true><<<grid, 128, 0, st>>>(D);
        else ulm::das_volume_mirror_kernel<kVolMirrorPlanes, false><<<grid, 128, 0, st>>>(D);
        ++P.last_launches;
        return;
    }
    const dim3 grid((D.n_lat * D.n_ax + 127) / 128, (D.n_planes + kVolPlanes - 1) / kVolPlanes);
    if (P.apod) ulm::das_volume_kernel<kVolPlanes, true><<<grid, 128, 0, st>>>(D);
    else ulm::das_volume_kernel<kVolPlanes, false><<<grid, 128, 0, st>>>(D);
    ++P.last_launches;
}

template <int NT, int ZS, bool IQ, int F, bool D32, bool AN = false>
cudaError_t launch_demod_t(const ulm::DemodParams &D, int L, dim3 blocks, cudaStream_t st) {
    const size_t smem = (size_t)ulm::demod_smem_bytes(F, D32, L);
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(ulm::demod_kernel<NT, ZS, IQ, F, D32, AN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    // as in the quadrature kernel: one CTA per scratch row walks its chunks when there are enough rows
    if ((long long)blocks.y * blocks.z >= 2048) blocks.x = 1;
    ulm::demod_kernel<NT, ZS, IQ, F, D32, AN><<<blocks, 256, smem, st>>>(D);
    return cudaSuccess;
}

template <int F, bool D32>
cudaError_t launch_demod_f(const ulm_rca_plan &P, const ulm::DemodParams &D, dim3 blocks, cudaStream_t st) {
    const int L = P.half_len;
    if (P.input_kind == 1) return launch_demod_t<1, 0, true, F, D32>(D, 0, blocks, st);
    if (P.quad) {
        // one CTA per scratch row walks all of its chunks (software-pipelined loads) when there are enough rows to
        // fill the GPU; few rows (single-frame calls) keep one CTA per chunk
        dim3 qb = blocks;
        if ((long long)blocks.y * blocks.z >= 2048) qb.x = 1;
        // aligned int16 pairs when every record starts 4-byte aligned and has an even length
        const bool pair = (D.n_samples & 1) == 0 && (reinterpret_cast<unsigned long long>(D.rf) & 3ull) == 0;
        if (pair) ulm::demod_quad_kernel<F, D32, true><<<qb, 256, ulm::demod_quad_smem_bytes(F, D32), st>>>(D);
        else ulm::demod_quad_kernel<F, D32, false><<<qb, 256, ulm::demod_quad_smem_bytes(F, D32), st>>>(D);
        return cudaSuccess;
    }
    if (L == 8) return P.half_band ? launch_demod_t<17, 2, false, F, D32>(D, L, blocks, st)
                                   : launch_demod_t<17, 0, false, F, D32>(D, L, blocks, st);
    if (L == 16 && P.analytic8) return launch_demod_t<33, 4, false, F, D32, true>(D, L, blocks, st);
    if (L == 16) return P.quarter_band ? launch_demod_t<33, 4, false, F, D32>(D, L, blocks, st)
                                       : launch_demod_t<33, 0, false, F, D32>(D, L, blocks, st);
    return launch_demod_t<0, 0, false, F, D32>(D, L, blocks, st);
}

cudaError_t launch_demod(const ulm_rca_plan &P, const int16_t *d_channel, int n_frames, bool folded, cudaStream_t st) {
    ulm::DemodParams D{};
    D.rf = d_channel; D.iq = P.iq.as<unsigned char>(); D.mixer = P.mixer.as<float2>(); D.mix_n0 = P.mix_n0;
    D.n_frames = n_frames; D.n_events_real = P.n_events; D.channels_per_event = P.cpe; D.n_samples = P.n_samples;
    D.n_events = folded ? P.nv_events : P.n_events;
    D.ev_map = folded ? P.ev_fold.as<short2>() : P.ev_id.as<short2>();
    D.n_row_tx = folded ? (int)P.ap[0].fk.size() : P.ap[0].n_tx;
    D.n_rows = P.n_rows; D.n_cols = P.n_cols; D.n_rx_max = P.n_rx_max;
    D.full_channels = P.cpe == P.n_rows + P.n_cols;
    D.n_lo = P.n_lo; D.l_row = P.l_row;
    D.chunks_per_row = (P.l_row + ulm::kDemodChunk - 1) / ulm::kDemodChunk;
    D.dc = P.demod;
    const int F = group_frames(n_frames);
    const dim3 blocks((unsigned)D.chunks_per_row, (unsigned)P.n_rx_max, (unsigned)(((n_frames + F - 1) / F) * D.n_events));
    ++P.last_launches;
    if (P.d32) return F == 12 ? launch_demod_f<12, true>(P, D, blocks, st) : launch_demod_f<4, true>(P, D, blocks, st);
    return F == 12 ? launch_demod_f<12, false>(P, D, blocks, st) : launch_demod_f<4, false>(P, D, blocks, st);
}

// sample range [s_lo, s_hi) of a record the pre-pass can read (rounded outwards to 16 samples = 32 bytes)
void host_sample_range(const ulm_rca_plan &P, int &s_lo, int &s_hi) {
    const int chunks = (P.l_row + ulm::kDemodChunk - 1) / ulm::kDemodChunk;
    s_lo = std::max(0, P.n_lo - P.half_len) / 16 * 16;
    const long long hi = (long long)P.n_lo + (long long)chunks * ulm::kDemodChunk + P.half_len + 2;
    s_hi = (int)std::min<long long>(P.n_samples, (std::max<long long>(hi, 0) + 15) / 16 * 16);
    if (s_hi < s_lo) s_hi = s_lo;
}

size_t host_upload_bytes_per_frame(const ulm_rca_plan &P) {
    int s_lo = 0, s_hi = 0;
    host_sample_range(P, s_lo, s_hi);
    size_t n = 0;
    for (int a = 0; a < 2; ++a) n += (size_t)P.ap[a].n_tx * P.ap[a].n_rx;
    return n * (size_t)(s_hi - s_lo) * (P.input_kind == 1 ? 4 : 2);
}

// the plan's tables and scratch live on the device that was current at plan_create; a call made with another
// current device would launch there on foreign pointers
ulm_rca_status check_device(const ulm_rca_plan &P) {
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != P.device) return fail(ULM_RCA_EINVAL, "plan belongs to CUDA device %d, the current device is %d", P.device, dev);
    return ULM_RCA_OK;
}

}  // namespace

extern "C" {

const char *ulm_rca_last_error(void) { return g_err; }

void ulm_rca_plan_destroy(ulm_rca_plan *plan) { delete plan; }

ulm_rca_status ulm_rca_plan_create(const ulm_rca_geometry *geo, const float *row_tx, int32_t n_row_tx,
                                   const float *col_tx, int32_t n_col_tx, float c_mps, float fs_hz,
                                   float fc_hz, const ulm_rca_grid *grid_xz, const ulm_rca_grid *grid_yz,
                                   const ulm_rca_options *opt, ulm_rca_plan **out) {
    if (!out) return fail(ULM_RCA_EINVAL, "out is NULL");
    *out = nullptr;
    if (!geo || !opt) return fail(ULM_RCA_EINVAL, "geometry/options is NULL");
    if (geo->n_rows <= 0 || geo->n_cols <= 0 || !finite_pos(geo->pitch_m))
        return fail(ULM_RCA_EINVAL, "geometry: need n_rows, n_cols, pitch > 0");
    if (geo->n_rows > 4096 || geo->n_cols > 4096) return fail(ULM_RCA_EINVAL, "geometry: too many elements");
    if (n_row_tx < 0 || n_col_tx < 0 || n_row_tx + n_col_tx == 0) return fail(ULM_RCA_EINVAL, "need at least one transmit event");
    if ((long long)n_row_tx + n_col_tx > 32767) return fail(ULM_RCA_EINVAL, "too many transmit events");
    if ((n_row_tx > 0 && !row_tx) || (n_col_tx > 0 && !col_tx)) return fail(ULM_RCA_EINVAL, "angle array is NULL");
    if (!finite_pos(c_mps) || !finite_pos(fs_hz) || !finite_pos(fc_hz)) return fail(ULM_RCA_EINVAL, "c, fs, fc must be finite and > 0");
    if (ulm_rca_status s = check_grid(grid_xz, "grid_xz")) return s;
    if (ulm_rca_status s = check_grid(grid_yz, "grid_yz")) return s;
    if (opt->motion_frames < 0 || opt->motion_frames > 65535) return fail(ULM_RCA_EINVAL, "motion_frames must be 0 .. 65535");
    if (opt->clutter_frames != 0 && (opt->clutter_frames < ulm::kCfB || opt->clutter_frames > ulm::kCfMaxFrames))
        return fail(ULM_RCA_EINVAL, "clutter_frames must be 0 or %d .. %d", ulm::kCfB, ulm::kCfMaxFrames);
    if (opt->stage2_block < 0 || opt->stage2_block > 4096) return fail(ULM_RCA_EINVAL, "stage2_block must be 0 .. 4096");
    if (opt->stage2_block && (grid_xz->n_ax != grid_yz->n_ax || grid_xz->z0_m != grid_yz->z0_m || grid_xz->dz_m != grid_yz->dz_m))
        return fail(ULM_RCA_EINVAL, "stage2_block needs identical axial grids");
    if (opt->no_timing != 0 && opt->no_timing != 1) return fail(ULM_RCA_EINVAL, "no_timing must be 0 or 1");
    if (opt->precision < 0 || opt->precision > 3) return fail(ULM_RCA_EINVAL, "precision must be 0, 1, 2 or 3");
    if (opt->input_kind != 0 && opt->input_kind != 1) return fail(ULM_RCA_EINVAL, "input_kind must be 0 or 1");
    if (opt->n_samples < 2) return fail(ULM_RCA_EINVAL, "n_samples must be >= 2");
    if (!std::isfinite(opt->t_start_s) || !std::isfinite(opt->f_number) || opt->f_number < 0)
        return fail(ULM_RCA_EINVAL, "t_start / f_number invalid");
    if (opt->demod_taps < 0 || (opt->demod_taps > 0 && opt->demod_taps % 2 == 0))
        return fail(ULM_RCA_EINVAL, "demod_taps must be odd (or 0)");
    if (opt->compound != 0 && opt->compound != 1) return fail(ULM_RCA_EINVAL, "compound must be 0 or 1");
    if (opt->max_frames < 0 || opt->kernel < 0 || opt->kernel > 2) return fail(ULM_RCA_EINVAL, "max_frames / kernel invalid");
    const int full = geo->n_rows + geo->n_cols;
    int cpe = opt->channels_per_event == 0 ? full : opt->channels_per_event;
    if (cpe != full && !(geo->n_rows == geo->n_cols && cpe == geo->n_rows))
        return fail(ULM_RCA_EINVAL, "channels_per_event must be n_rows+n_cols, or n_rows when n_rows == n_cols");
    for (int i = 0; i < n_row_tx; ++i) if (!std::isfinite(row_tx[i]) || std::fabs(row_tx[i]) >= 1.5) return fail(ULM_RCA_EINVAL, "row_tx angle %d invalid", i);
    for (int i = 0; i < n_col_tx; ++i) if (!std::isfinite(col_tx[i]) || std::fabs(col_tx[i]) >= 1.5) return fail(ULM_RCA_EINVAL, "col_tx angle %d invalid", i);
    if (opt->t0_s) for (int i = 0; i < n_row_tx + n_col_tx; ++i) if (!std::isfinite(opt->t0_s[i])) return fail(ULM_RCA_EINVAL, "t0 %d non-finite", i);
    if (opt->elem_window) for (int i = 0; i < full; ++i) if (!std::isfinite(opt->elem_window[i])) return fail(ULM_RCA_EINVAL, "elem_window %d non-finite", i);
    if (opt->build_volume && (grid_xz->n_ax != grid_yz->n_ax || grid_xz->z0_m != grid_yz->z0_m || grid_xz->dz_m != grid_yz->dz_m))
        return fail(ULM_RCA_EINVAL, "build_volume needs identical axial grids");

    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
        cudaGetLastError();
        return fail(ULM_RCA_ECUDA, "no CUDA device (this library has no CPU fallback)");
    }

    ulm_rca_plan *Pp = new (std::nothrow) ulm_rca_plan;
    if (!Pp) return fail(ULM_RCA_ENOMEM, "host allocation failed");
    struct Guard { ulm_rca_plan *p; ~Guard() { delete p; } } guard{Pp};
    CUDA_TRY(cudaGetDevice(&Pp->device));
    ulm_rca_plan &P = *Pp;
    P.n_rows = geo->n_rows; P.n_cols = geo->n_cols; P.pitch = geo->pitch_m;
    P.c = c_mps; P.fs = fs_hz; P.fc = fc_hz; P.t_start = opt->t_start_s; P.f_number = opt->f_number;
    P.input_kind = opt->input_kind; P.cpe = cpe; P.n_samples = opt->n_samples; P.compound = opt->compound;
    P.max_frames = opt->max_frames > 0 ? opt->max_frames : 32;
    if ((long long)((P.max_frames + 3) / 4) * (n_row_tx + n_col_tx) > 65535)
        return fail(ULM_RCA_EUNSUPPORTED, "max_frames x events too large for one batch: lower max_frames");
    P.build_volume = opt->build_volume;
    P.timing = opt->no_timing == 0;
    P.n_events = n_row_tx + n_col_tx;
    P.n_rx_max = std::max(P.n_rows, P.n_cols);
    P.apod = opt->f_number > 0 || opt->elem_window != nullptr;
    // auto: RF input (band-limited by the library's own low-pass) -> compact entries with the exact weight;
    // IQ input (spectrum unknown) -> full entries
    P.d32 = opt->precision == 2 || (opt->precision == 0 && opt->input_kind == 1);
    P.w2 = !P.d32 && opt->precision != 1;

    for (int a = 0; a < 2; ++a) {
        Aperture &A = P.ap[a];
        const ulm_rca_grid *g = a == 0 ? grid_xz : grid_yz;
        A.row_tx = a == 0;
        A.n_tx = a == 0 ? n_row_tx : n_col_tx;
        A.n_rx = a == 0 ? P.n_cols : P.n_rows;
        A.e0 = a == 0 ? 0 : n_row_tx;
        A.g.n_lat = g->n_lat; A.g.n_ax = g->n_ax; A.g.lat0 = g->lat0_m; A.g.dlat = g->dlat_m;
        A.g.z0 = g->z0_m; A.g.dz = g->dz_m; A.g.ref = g->ref_m;
        for (int k = 0; k < A.n_tx; ++k) {
            A.angles.push_back(a == 0 ? row_tx[k] : col_tx[k]);
            A.t0.push_back(opt->t0_s ? opt->t0_s[A.e0 + k] : 0.0);
        }
    }
    const long long pxz = (long long)P.ap[0].g.n_lat * P.ap[0].g.n_ax, pyz = (long long)P.ap[1].g.n_lat * P.ap[1].g.n_ax;
    if (P.compound) { P.ap[0].out_base = 0; P.ap[1].out_base = pxz; P.out_per_frame = pxz + pyz; }
    else { P.ap[0].out_base = 0; P.ap[1].out_base = n_row_tx * pxz; P.out_per_frame = n_row_tx * pxz + n_col_tx * pyz; }
    P.vol_per_frame = (long long)P.ap[0].g.n_lat * P.ap[1].g.n_lat * P.ap[0].g.n_ax;

    // touched sample range over everything this plan may be asked for
    double u_min = 1e300, u_max = -1e300;
    std::vector<double> vol_refs[2];
    for (int a = 0; a < 2; ++a) {
        sample_range(P, P.ap[a], {P.ap[a].g.ref}, u_min, u_max);
        if (P.build_volume) {
            const Grid &other = P.ap[1 - a].g;      // planes of the x-z kernel are the y pixels and vice versa
            for (int i = 0; i < other.n_lat; ++i) vol_refs[a].push_back(other.lat(i));
            sample_range(P, P.ap[a], vol_refs[a], u_min, u_max);
        }
    }
    if (!(u_max >= u_min) || u_max - u_min > 1e7 || std::fabs(u_min) > 1e9)
        return fail(ULM_RCA_EINVAL, "delay range is empty or absurd (%g .. %g samples)", u_min, u_max);
    P.n_lo = (int)std::floor(u_min) - 4;
    const int n_hi = (int)std::floor(u_max) + 4;
    P.l_row = ((n_hi - P.n_lo + 1) + 7) / 8 * 8;

    if (ulm_rca_status s = build_demod(P, opt->demod_taps)) return s;
    {   // exp(-j 2 pi fc t_n): mixes RF input down; its conjugate rho_n rotates every scratch entry (both input kinds)
        P.mix_n0 = P.n_lo - P.half_len;
        const int n_mix = P.l_row + 2 * P.half_len + 264;
        std::vector<float2> mix(n_mix);
        for (int i = 0; i < n_mix; ++i) {
            const double n = (double)P.mix_n0 + i;
            double cyc = P.fc * P.t_start + (P.fc / P.fs) * n;     // fc * t_n in cycles
            cyc -= std::floor(cyc);
            const double c4 = 4.0 * cyc;
            if (std::fabs(c4 - std::round(c4)) < 1e-12) {       // exact quarter cycles: no 6e-17 residue
                const float tab[4][2] = {{1.f, 0.f}, {0.f, -1.f}, {-1.f, 0.f}, {0.f, 1.f}};
                const int q = (int)std::llround(c4) & 3;
                mix[i] = make_float2(tab[q][0], tab[q][1]);
            } else {
                mix[i] = make_float2((float)std::cos(2 * M_PI * cyc), (float)(-std::sin(2 * M_PI * cyc)));
            }
        }
        CUDA_TRY(P.mixer.upload(mix));
    }

    // fold transmit events with identical reference-slice delays (see Aperture::fk); scratch event maps
    {
        std::vector<short2> map_fold, map_id;
        for (int a = 0; a < 2; ++a) {
            Aperture &A = P.ap[a];
            const std::vector<int> partner = fold_partners(A.angles, A.t0, P.c, P.fs, A.g.ref, A.g.z0, A.g.dz, A.g.n_ax,
                                                           P.compound != 0);
            A.fe0 = (int)map_fold.size();
            for (int k = 0; k < A.n_tx; ++k) {
                map_id.push_back(make_short2((short)(A.e0 + k), (short)-1));
                if (partner[k] == -2) continue;
                A.fk.push_back(k);
                A.fk2.push_back(partner[k]);
                A.fangles.push_back(A.angles[k]);
                A.ft0.push_back(A.t0[k]);
                map_fold.push_back(make_short2((short)(A.e0 + k), (short)(partner[k] >= 0 ? A.e0 + partner[k] : -1)));
            }
        }
        P.nv_events = (int)map_fold.size();
        CUDA_TRY(P.ev_fold.upload(map_fold));
        CUDA_TRY(P.ev_id.upload(map_id));
    }

    for (int a = 0; a < 2; ++a) {
        Aperture &A = P.ap[a];
        const float *win = opt->elem_window ? opt->elem_window + (a == 0 ? 0 : P.n_cols) : nullptr;
        if (ulm_rca_status s = upload_aperture(P, A, win)) return s;
        CUDA_TRY(build_tx_tables(P, A, {A.g.ref}, A.fk, A.proj));
        if (P.build_volume) {
            std::vector<int> all(A.n_tx);
            for (int k = 0; k < A.n_tx; ++k) all[k] = k;
            CUDA_TRY(build_tx_tables(P, A, vol_refs[a], all, A.vol, true));
            CUDA_TRY(build_mirror_tables(P, A, vol_refs[a], A.vol));
        }
    }

    // one scratch row block per event the plan will fill: the folded events of the projection path, or every real
    // event when the volume comparator (which never folds) is prepared as well
    const int scratch_events = P.build_volume ? P.n_events : P.nv_events;
    P.iq_bytes = (size_t)((P.max_frames + 11) / 12) * scratch_events * P.n_rx_max * P.l_row * ulm::entry_bytes(12, P.d32);
    CUDA_TRY(cudaMalloc(&P.iq.p, P.iq_bytes));
    if (P.build_volume) CUDA_TRY(cudaMalloc(&P.vol_rows.p, (size_t)P.n_events * P.n_rx_max * P.l_row * sizeof(float4)));

    // kernel choice: the shared-memory ring kernel covers the projections (compounded, or one slice per event with
    // one work item per angle); the volume and shapes whose window does not fit take the generic kernel.
    P.kernel = 1;
    if (opt->kernel != 1) {
        ulm::RingApertureDesc desc[2];
        for (int a = 0; a < 2; ++a) {
            const Aperture &A = P.ap[a];
            desc[a] = ulm::RingApertureDesc{(int)A.fk.size(), A.n_rx, A.g.n_lat, A.g.n_ax, A.g.lat0, A.g.dlat, A.g.z0, A.g.dz,
                                            A.g.ref, A.fangles.data(), A.ft0.data()};
        }
        const char *why = nullptr;
        const bool ok = ulm::ring_plan(desc, P.pitch, P.c, P.fs, P.t_start, P.l_row, P.ring, P.ap[0].ring,
                                       P.ap[1].ring, &why);
        if (ok) {
            P.kernel = 2;
            if (!P.d32) ulm::ring_plan_dual(desc, P.pitch, P.c, P.fs, P.t_start, P.l_row, P.ring, P.ap[0].ring2, P.ap[1].ring2);
            CUDA_TRY(ulm::ring_set_attributes());       // per-device function attribute, set on the plan's device
        } else if (opt->kernel == 2) return fail(ULM_RCA_EUNSUPPORTED, "ring kernel unavailable: %s", why ? why : "?");
        if (cudaGetLastError() != cudaSuccess) return fail(ULM_RCA_ECUDA, "ring table upload failed");
    }
    if (P.timing) for (auto &c : P.ev) for (auto &b : c) for (auto &e : b) CUDA_TRY(cudaEventCreate(&e));
    if (opt->stage2_block > 0) {
        ulm::Stage2Axis ax[2];
        for (int a = 0; a < 2; ++a) {
            ax[a].n_lat = P.ap[a].g.n_lat; ax[a].lat0 = P.ap[a].g.lat0; ax[a].dlat = P.ap[a].g.dlat; ax[a].ref = P.ap[a].g.ref;
            ax[a].angles = P.ap[a].angles;
        }
        if (const char *why = ulm::stage2_build(P.s2, ax, P.ap[0].g.n_ax, P.ap[0].g.dz, P.c, P.fc, opt->stage2_block,
                                                 P.max_frames, P.timing)) {
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ULM_RCA_ENOMEM : ULM_RCA_ECUDA, "stage 2: %s: %s", why, cudaGetErrorString(e));
            return fail(ULM_RCA_EUNSUPPORTED, "stage 2: %s", why);
        }
    }
    if (P.s2.ready) {
        CUDA_TRY(cudaMalloc(&P.loc_frame_max.p, (size_t)P.max_frames * sizeof(unsigned int)));
        CUDA_TRY(cudaFuncSetAttribute(ulm::localize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ulm::kLoSmem));
    }
    if (opt->clutter_frames > 0) {
        std::vector<long long> off;
        std::vector<int> npix;
        long long o = 0;
        for (int a = 0; a < 2; ++a)
            for (int k = 0; k < P.ap[a].n_tx; ++k) {
                off.push_back(o);
                npix.push_back(P.ap[a].g.n_lat * P.ap[a].g.n_ax);
                o += (long long)P.ap[a].g.n_lat * P.ap[a].g.n_ax;
            }
        if (const char *why = ulm::clutter_build(P.cf, off, npix, o, opt->clutter_frames, P.timing)) {
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ULM_RCA_ENOMEM : ULM_RCA_ECUDA, "clutter filter: %s: %s", why, cudaGetErrorString(e));
            return fail(ULM_RCA_EUNSUPPORTED, "clutter filter: %s", why);
        }
    }
    if (opt->motion_frames > 0) {
        std::vector<long long> off;
        std::vector<int> nl, nz;
        long long o = 0;
        for (int a = 0; a < 2; ++a)
            for (int k = 0; k < P.ap[a].n_tx; ++k) {
                off.push_back(o); nl.push_back(P.ap[a].g.n_lat); nz.push_back(P.ap[a].g.n_ax);
                o += (long long)P.ap[a].g.n_lat * P.ap[a].g.n_ax;
            }
        const float dl[2] = {(float)P.ap[0].g.dlat, (float)P.ap[1].g.dlat}, dzz[2] = {(float)P.ap[0].g.dz, (float)P.ap[1].g.dz};
        if (const char *why = ulm::motion_build(P.mo, off, nl, nz, P.ap[0].n_tx, o, opt->motion_frames, dl, dzz, P.timing)) {
            const cudaError_t e = cudaGetLastError();
            if (e != cudaSuccess) return fail(e == cudaErrorMemoryAllocation ? ULM_RCA_ENOMEM : ULM_RCA_ECUDA, "motion estimation: %s: %s", why, cudaGetErrorString(e));
            return fail(ULM_RCA_EUNSUPPORTED, "motion estimation: %s", why);
        }
    }
    CUDA_TRY(cudaDeviceSynchronize());
    guard.p = nullptr;
    *out = Pp;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_plan_sizes(const ulm_rca_plan *plan, size_t *ch, size_t *outb, size_t *vol) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (ch) *ch = (size_t)plan->n_events * plan->cpe * plan->n_samples * sizeof(int16_t) * (plan->input_kind == 1 ? 2 : 1);
    if (outb) *outb = (size_t)plan->out_per_frame * sizeof(float2);
    if (vol) *vol = (size_t)plan->vol_per_frame * sizeof(float2);
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_plan_info(const ulm_rca_plan *plan, int64_t *v, int32_t n) {
    if (!plan || !v || n < 0) return fail(ULM_RCA_EINVAL, "plan/values is NULL");
    const bool ring = plan->kernel == 2, d32 = plan->d32;
    const bool dual = ring && plan->ring.window2 > 0;
    const bool vmirror = plan->build_volume && ((plan->ap[0].n_tx == 0 || plan->ap[0].vol.mtab.p) && (plan->ap[1].n_tx == 0 || plan->ap[1].vol.mtab.p));
    const int64_t vals[23] = {plan->n_lo, plan->l_row, (int64_t)plan->iq_bytes, plan->kernel, 12,
                              ring ? ulm::kRingConsumers * ulm::kRingPx : 128, ring ? plan->ring.window : 0,
                              ring ? ulm::ring_stages(plan->ring.window, 12, d32) : 0, ring ? plan->ap[0].ring.n_tiles : 0,
                              ring ? ulm::ring_smem_bytes(plan->ring.window, 12, d32) : 0, plan->last_launches,
                              ring ? plan->ap[1].ring.n_tiles : 0, d32 ? 2 : (plan->w2 ? 3 : 1), ulm::entry_bytes(12, d32) / 12,
                              (int64_t)host_upload_bytes_per_frame(*plan), plan->nv_events,
                              plan->s2.ready ? plan->s2.nt : 0, plan->s2.ready ? plan->s2.ncol : 0,
                              dual ? plan->ring.window2 : 0, dual ? ulm::ring_dual_stages(plan->ring.window2) : 0,
                              dual ? plan->ap[0].ring2.n_tiles : 0, dual ? plan->ap[1].ring2.n_tiles : 0, vmirror ? 1 : 0};
    for (int i = 0; i < n && i < 23; ++i) v[i] = vals[i];
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_beamform(const ulm_rca_plan *plan, const void *d_channel, int32_t n_frames, void *d_out,
                                void *cuda_stream) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (n_frames < 0) return fail(ULM_RCA_EINVAL, "n_frames < 0");
    if (n_frames == 0) return ULM_RCA_OK;
    if (!d_channel || !d_out) return fail(ULM_RCA_EINVAL, "device pointer is NULL");
    const ulm_rca_plan &P = *plan;
    if (ulm_rca_status s = check_device(P)) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    size_t ch_bytes = 0;
    ulm_rca_plan_sizes(plan, &ch_bytes, nullptr, nullptr);
    P.last_launches = 0;
    const int slot = (int)(P.n_calls % ulm_rca_plan::kTimedCalls);
    ++P.n_calls;
    P.timed_batches[slot] = 0;
    for (int f0 = 0; f0 < n_frames; f0 += P.max_frames) {
        const int nb = std::min(P.max_frames, n_frames - f0);
        const int16_t *in = reinterpret_cast<const int16_t *>(static_cast<const char *>(d_channel) + (size_t)f0 * ch_bytes);
        float2 *outp = static_cast<float2 *>(d_out) + (long long)f0 * P.out_per_frame;
        const int tb = (P.timing && P.timed_batches[slot] < ulm_rca_plan::kTimedBatches) ? P.timed_batches[slot] : -1;
        if (tb >= 0) CUDA_TRY(cudaEventRecord(P.ev[slot][tb][0], st));
        CUDA_TRY(launch_demod(P, in, nb, true, st));
        if (tb >= 0) CUDA_TRY(cudaEventRecord(P.ev[slot][tb][1], st));
        for (int a = 0; a < 2; ++a) {     // an aperture without transmit events: its image is all zeros
            const Aperture &A = P.ap[a];
            if (A.n_tx == 0 && P.compound)
                CUDA_TRY(cudaMemset2DAsync(outp + A.out_base, (size_t)P.out_per_frame * sizeof(float2), 0,
                                           (size_t)A.g.n_lat * A.g.n_ax * sizeof(float2), nb, st));
        }
        if (P.kernel == 2) {
            ulm::RingLaunch L{};
            L.iq = P.iq.as<unsigned char>(); L.l_row = P.l_row; L.n_rx_max = P.n_rx_max; L.n_events = P.nv_events;
            L.out = outp; L.out_frame_stride = P.out_per_frame; L.n_frames = nb; L.per_angle = P.compound ? 0 : 1;
            L.fcfs = (float)(P.fc / P.fs); L.two_f = (float)(2.0 * P.f_number);
            for (int a = 0; a < 2; ++a) {
                const Aperture &A = P.ap[a];
                ulm::RingApertureArgs &R = L.ap[a];
                R.e0 = A.fe0; R.n_tx = (int)A.fk.size(); R.n_rx = A.n_rx; R.n_lat = A.g.n_lat; R.n_ax = A.g.n_ax;
                R.xs = A.xs.as<float>(); R.zs = A.zs.as<float>(); R.ejs = A.ejs.as<float>();
                R.xm = A.xm.as<float>(); R.zm = A.zm.as<float>(); R.ejm = A.ejm.as<float>(); R.win = A.win.as<float>();
                R.n0 = A.proj.n0.as<int>(); R.f0m = A.proj.f0m.as<float>();
                R.out_base = A.out_base;
            }
            P.last_launches += ulm::ring_launch(P.ring, P.ap[0].ring, P.ap[1].ring, P.ap[0].ring2, P.ap[1].ring2, L, group_frames(nb),
                                                P.d32, P.w2, P.apod, st);
        } else {
            for (int a = 0; a < 2; ++a) {
                const Aperture &A = P.ap[a];
                ulm::DasParams D = das_params(P, A, A.proj, true);
                D.out = outp; D.out_frame_stride = P.out_per_frame; D.out_base = A.out_base;
                D.s_lat = A.g.n_ax; D.s_plane = 0; D.s_k = (long long)A.g.n_lat * A.g.n_ax;
                D.per_angle = P.compound ? 0 : 1; D.accumulate = 0; D.n_frames = nb;
                launch_generic(P, D, nb, st);
            }
        }
        if (tb >= 0) { CUDA_TRY(cudaEventRecord(P.ev[slot][tb][2], st)); P.timed_batches[slot] = tb + 1; }
    }
    CUDA_TRY(cudaGetLastError());
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_plan_timing(const ulm_rca_plan *plan, int32_t n_calls, double *demod_ms, double *das_ms) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->timing) return fail(ULM_RCA_EUNSUPPORTED, "plan was created with no_timing = 1");
    if (n_calls < 1 || n_calls > ulm_rca_plan::kTimedCalls || n_calls > plan->n_calls)
        return fail(ULM_RCA_EINVAL, "n_calls must be 1..min(64, calls made)");
    double d = 0, g = 0;
    for (int c = 1; c <= n_calls; ++c) {
        const int slot = (int)((plan->n_calls - c) % ulm_rca_plan::kTimedCalls);
        for (int b = 0; b < plan->timed_batches[slot]; ++b) {
            float a = 0, e = 0;
            CUDA_TRY(cudaEventSynchronize(plan->ev[slot][b][2]));
            CUDA_TRY(cudaEventElapsedTime(&a, plan->ev[slot][b][0], plan->ev[slot][b][1]));
            CUDA_TRY(cudaEventElapsedTime(&e, plan->ev[slot][b][1], plan->ev[slot][b][2]));
            d += a; g += e;
        }
    }
    if (demod_ms) *demod_ms = d / n_calls;
    if (das_ms) *das_ms = g / n_calls;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_beamform_volume(const ulm_rca_plan *plan, const void *d_channel, int32_t n_frames,
                                       void *d_out_volume, void *cuda_stream) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->build_volume) return fail(ULM_RCA_EUNSUPPORTED, "plan was created without build_volume");
    if (n_frames < 0) return fail(ULM_RCA_EINVAL, "n_frames < 0");
    if (n_frames == 0) return ULM_RCA_OK;
    if (!d_channel || !d_out_volume) return fail(ULM_RCA_EINVAL, "device pointer is NULL");
    const ulm_rca_plan &P = *plan;
    if (ulm_rca_status s = check_device(P)) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    size_t ch_bytes = 0;
    ulm_rca_plan_sizes(plan, &ch_bytes, nullptr, nullptr);
    const int nx = P.ap[0].g.n_lat, ny = P.ap[1].g.n_lat, nz = P.ap[0].g.n_ax;
    P.last_launches = 0;
    for (int f0 = 0; f0 < n_frames; f0 += P.max_frames) {
        const int nb = std::min(P.max_frames, n_frames - f0);
        const int16_t *in = reinterpret_cast<const int16_t *>(static_cast<const char *>(d_channel) + (size_t)f0 * ch_bytes);
        float2 *outp = static_cast<float2 *>(d_out_volume) + (long long)f0 * P.vol_per_frame;
        CUDA_TRY(launch_demod(P, in, nb, false, st));
        const bool by_frame = nb <= kVolFrameKernelMax;
        // V_RC: lateral = x, planes = y; then V_CR accumulated on top: lateral = y, planes = x
        for (int f = 0; f < (by_frame ? nb : 1); ++f) {
            if (by_frame) launch_unpack(P, nb, f, st);
            for (int a = 0; a < 2; ++a) {
                const Aperture &A = P.ap[a];
                ulm::DasParams D = das_params(P, A, A.vol, false);
                D.out = outp; D.out_frame_stride = P.vol_per_frame; D.out_base = (long long)f * P.vol_per_frame;
                D.s_lat = a == 0 ? (long long)ny * nz : nz;
                D.s_plane = a == 0 ? nz : (long long)ny * nz;
                D.s_k = 0; D.per_angle = 0; D.accumulate = a == 1 && P.ap[0].n_tx > 0; D.n_frames = nb;
                if (A.n_tx == 0) {
                    if (a == 0) CUDA_TRY(cudaMemsetAsync(outp + D.out_base, 0, (size_t)(by_frame ? 1 : nb) * P.vol_per_frame * sizeof(float2), st));
                    continue;
                }
                if (by_frame) launch_volume(P, D, st);
                else launch_generic(P, D, nb, st);
            }
        }
    }
    (void)nx;
    CUDA_TRY(cudaGetLastError());
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_beamform_host(ulm_rca_plan *plan, const void *h_channel, int32_t n_frames, void *h_out) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (n_frames < 0) return fail(ULM_RCA_EINVAL, "n_frames < 0");
    if (n_frames == 0) return ULM_RCA_OK;
    if (!h_channel || !h_out) return fail(ULM_RCA_EINVAL, "host pointer is NULL");
    if (ulm_rca_status s = check_device(*plan)) return s;
    size_t ch_bytes = 0, out_bytes = 0;
    ulm_rca_plan_sizes(plan, &ch_bytes, &out_bytes, nullptr);
    // pipeline over chunks of whole 12-frame groups through two staging slots: the upload of chunk i + 1 overlaps the
    // kernels and the download of chunk i (the host buffers should be pinned for the copies to be asynchronous)
    constexpr int kSlots = ulm_rca_plan::kHostSlots;
    const int chunk = n_frames >= 48 ? 24 : 12;
    if (plan->h_stage_frames < (size_t)chunk) {
        if (plan->h_stage_in.p) { cudaFree(plan->h_stage_in.p); plan->h_stage_in.p = nullptr; }
        if (plan->h_stage_out.p) { cudaFree(plan->h_stage_out.p); plan->h_stage_out.p = nullptr; }
        plan->h_stage_frames = 0;
        CUDA_TRY(cudaMalloc(&plan->h_stage_in.p, ch_bytes * chunk * kSlots));
        CUDA_TRY(cudaMalloc(&plan->h_stage_out.p, out_bytes * chunk * kSlots));
        plan->h_stage_frames = chunk;
    }
    if (!plan->h_copy) {
        CUDA_TRY(cudaStreamCreateWithFlags(&plan->h_copy, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&plan->h_compute, cudaStreamNonBlocking));
        for (auto &e : plan->h_in_done) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        for (auto &e : plan->h_slot_free) CUDA_TRY(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    const char *h_in = static_cast<const char *>(h_channel);
    char *h_o = static_cast<char *>(h_out);
    const int eb = plan->input_kind == 1 ? 4 : 2;
    int s_lo = 0, s_hi = 0;
    host_sample_range(*plan, s_lo, s_hi);
    // a failure inside the loop must not return while copies still read / write the caller's buffers
    auto drain = [&](ulm_rca_status s) {
        cudaStreamSynchronize(plan->h_copy);
        cudaStreamSynchronize(plan->h_compute);
        return s;
    };
#define HOST_TRY(expr)                                                                                     \
    do {                                                                                                   \
        cudaError_t e_ = (expr);                                                                           \
        if (e_ != cudaSuccess)                                                                             \
            return drain(fail(e_ == cudaErrorMemoryAllocation ? ULM_RCA_ENOMEM : ULM_RCA_ECUDA, "%s: %s", #expr, \
                              cudaGetErrorString(e_)));                                                    \
    } while (0)
    int i = 0;
    for (int f0 = 0; f0 < n_frames; f0 += chunk, ++i) {
        const int nb = std::min(chunk, n_frames - f0);
        const int slot = i % kSlots;
        char *d_in = plan->h_stage_in.as<char>() + (size_t)slot * chunk * ch_bytes;
        char *d_o = plan->h_stage_out.as<char>() + (size_t)slot * chunk * out_bytes;
        // the slot is free once the kernels and the download of the chunk that used it last have finished
        if (i >= kSlots) HOST_TRY(cudaStreamWaitEvent(plan->h_copy, plan->h_slot_free[slot], 0));
        // upload only what the pre-pass reads: the receive aperture of every event, touched sample range
        for (int f = 0; f < nb; ++f)
            for (int a = 0; a < 2; ++a) {
                const Aperture &A = plan->ap[a];
                if (A.n_tx == 0) continue;
                cudaMemcpy3DParms cp = {};
                const size_t row_pitch = (size_t)plan->n_samples * eb;
                cp.srcPtr = make_cudaPitchedPtr(const_cast<char *>(h_in) + (size_t)(f0 + f) * ch_bytes, row_pitch, row_pitch, plan->cpe);
                cp.dstPtr = make_cudaPitchedPtr(d_in + (size_t)f * ch_bytes, row_pitch, row_pitch, plan->cpe);
                const size_t c0 = (a == 0 && plan->cpe == plan->n_rows + plan->n_cols) ? plan->n_rows : 0;
                cp.srcPos = make_cudaPos((size_t)s_lo * eb, c0, A.e0);
                cp.dstPos = cp.srcPos;
                cp.extent = make_cudaExtent((size_t)(s_hi - s_lo) * eb, A.n_rx, A.n_tx);
                cp.kind = cudaMemcpyHostToDevice;
                HOST_TRY(cudaMemcpy3DAsync(&cp, plan->h_copy));
            }
        HOST_TRY(cudaEventRecord(plan->h_in_done[slot], plan->h_copy));
        HOST_TRY(cudaStreamWaitEvent(plan->h_compute, plan->h_in_done[slot], 0));
        if (ulm_rca_status s = ulm_rca_beamform(plan, d_in, nb, d_o, plan->h_compute)) return drain(s);
        HOST_TRY(cudaMemcpyAsync(h_o + (size_t)f0 * out_bytes, d_o, out_bytes * nb, cudaMemcpyDeviceToHost, plan->h_compute));
        HOST_TRY(cudaEventRecord(plan->h_slot_free[slot], plan->h_compute));
    }
    HOST_TRY(cudaStreamSynchronize(plan->h_compute));
#undef HOST_TRY
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_stage2_sizes(const ulm_rca_plan *plan, size_t *slices_bytes_per_frame, size_t *planes_bytes_per_frame,
                                    int32_t *n_planes_xz, int32_t *n_planes_yz) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->s2.ready) return fail(ULM_RCA_EUNSUPPORTED, "plan was created without stage2_block");
    if (slices_bytes_per_frame) *slices_bytes_per_frame = (size_t)plan->s2.slices_per_frame * sizeof(float2);
    if (planes_bytes_per_frame) *planes_bytes_per_frame = (size_t)plan->s2.planes_per_frame * sizeof(float2);
    if (n_planes_xz) *n_planes_xz = plan->s2.n_g[0];
    if (n_planes_yz) *n_planes_yz = plan->s2.n_g[1];
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_stage2_project(const ulm_rca_plan *plan, const void *d_slices, int32_t n_frames, void *d_planes,
                                      void *cuda_stream) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->s2.ready) return fail(ULM_RCA_EUNSUPPORTED, "plan was created without stage2_block");
    if (n_frames < 0) return fail(ULM_RCA_EINVAL, "n_frames < 0");
    if (n_frames == 0) return ULM_RCA_OK;
    if (!d_slices || !d_planes) return fail(ULM_RCA_EINVAL, "device pointer is NULL");
    if (ulm_rca_status s = check_device(*plan)) return s;
    const ulm::Stage2Plan &S = plan->s2;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int launches = 0;
    for (int f0 = 0; f0 < n_frames; f0 += S.max_frames) {
        const int nb = std::min(S.max_frames, n_frames - f0);
        CUDA_TRY(ulm::stage2_launch(S, static_cast<const float2 *>(d_slices) + (long long)f0 * S.slices_per_frame, nb,
                                    static_cast<float2 *>(d_planes) + (long long)f0 * S.planes_per_frame, st, &launches));
    }
    plan->last_launches = launches;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_stage2_timing(const ulm_rca_plan *plan, double *groupsum_ms, double *project_ms) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->s2.ready || !plan->s2.ev[0]) return fail(ULM_RCA_EUNSUPPORTED, "no Stage-2 timing events on this plan");
    float a = 0, b = 0;
    CUDA_TRY(cudaEventSynchronize(plan->s2.ev[2]));
    CUDA_TRY(cudaEventElapsedTime(&a, plan->s2.ev[0], plan->s2.ev[1]));
    CUDA_TRY(cudaEventElapsedTime(&b, plan->s2.ev[1], plan->s2.ev[2]));
    if (groupsum_ms) *groupsum_ms = a;
    if (project_ms) *project_ms = b;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_clutter_filter(const ulm_rca_plan *plan, const void *d_slices, int32_t n_frames, int32_t clutter_rank,
                                      void *d_filtered, void *d_eigenvalues, void *d_covariance, void *cuda_stream) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->cf.ready) return fail(ULM_RCA_EUNSUPPORTED, "plan was created without clutter_frames");
    if (n_frames < ulm::kCfB || n_frames > plan->cf.max_t)
        return fail(ULM_RCA_EINVAL, "n_frames must be %d .. clutter_frames (%d)", ulm::kCfB, plan->cf.max_t);
    if (clutter_rank < 0 || clutter_rank > ulm::kCfMaxRank) return fail(ULM_RCA_EINVAL, "clutter_rank must be 0 .. %d", ulm::kCfMaxRank);
    if (!d_slices || !d_filtered) return fail(ULM_RCA_EINVAL, "device pointer is NULL");
    if (ulm_rca_status s = check_device(*plan)) return s;
    int launches = 0;
    const char *why = nullptr;
    const cudaError_t e = ulm::clutter_launch(plan->cf, static_cast<const float2 *>(d_slices), n_frames, clutter_rank,
                                              static_cast<float2 *>(d_filtered), static_cast<float *>(d_eigenvalues),
                                              static_cast<float2 *>(d_covariance), (cudaStream_t)cuda_stream, &launches, &why);
    if (e != cudaSuccess) return fail(why ? ULM_RCA_EUNSUPPORTED : ULM_RCA_ECUDA, "clutter filter: %s", why ? why : cudaGetErrorString(e));
    plan->last_launches = launches;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_clutter_timing(const ulm_rca_plan *plan, double *ms4) {
    double *ms5 = ms4;
    if (!plan || !ms5) return fail(ULM_RCA_EINVAL, "plan / ms5 is NULL");
    if (!plan->cf.ready || !plan->cf.ev[0]) return fail(ULM_RCA_EUNSUPPORTED, "no clutter-filter timing events on this plan");
    CUDA_TRY(cudaEventSynchronize(plan->cf.ev[5]));
    for (int i = 0; i < 5; ++i) {
        float v = 0;
        CUDA_TRY(cudaEventElapsedTime(&v, plan->cf.ev[i], plan->cf.ev[i + 1]));
        ms5[i] = v;
    }
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_motion_estimate(const ulm_rca_plan *plan, const void *d_slices, int32_t n_frames, int32_t ref_frame,
                                       void *d_motion, void *d_per_event, void *cuda_stream) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->mo.ready) return fail(ULM_RCA_EUNSUPPORTED, "plan was created without motion_frames");
    if (n_frames < 0 || n_frames > plan->mo.max_frames) return fail(ULM_RCA_EINVAL, "n_frames must be 0 .. motion_frames (%d)", plan->mo.max_frames);
    if (n_frames == 0) return ULM_RCA_OK;
    if (ref_frame < 0 || ref_frame >= n_frames) return fail(ULM_RCA_EINVAL, "ref_frame must be a frame of this call");
    if (!d_slices || !d_motion) return fail(ULM_RCA_EINVAL, "device pointer is NULL");
    if (ulm_rca_status s = check_device(*plan)) return s;
    int launches = 0;
    CUDA_TRY(ulm::motion_launch(plan->mo, static_cast<const float2 *>(d_slices), n_frames, ref_frame, static_cast<float4 *>(d_motion),
                                static_cast<float4 *>(d_per_event), (cudaStream_t)cuda_stream, &launches));
    plan->last_launches = launches;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_motion_timing(const ulm_rca_plan *plan, double *ms) {
    if (!plan || !ms) return fail(ULM_RCA_EINVAL, "plan / ms is NULL");
    if (!plan->mo.ready || !plan->mo.ev[0]) return fail(ULM_RCA_EUNSUPPORTED, "no motion-estimation timing events on this plan");
    float v = 0;
    CUDA_TRY(cudaEventSynchronize(plan->mo.ev[1]));
    CUDA_TRY(cudaEventElapsedTime(&v, plan->mo.ev[0], plan->mo.ev[1]));
    *ms = v;
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_localize(const ulm_rca_plan *plan, const void *d_planes, int32_t n_frames,
                                const ulm_rca_localize_params *prm, void *d_loc, void *d_count, void *cuda_stream) {
    if (!plan) return fail(ULM_RCA_EINVAL, "plan is NULL");
    if (!plan->s2.ready) return fail(ULM_RCA_EUNSUPPORTED, "plan was created without stage2_block (the planes' geometry)");
    if (n_frames < 0) return fail(ULM_RCA_EINVAL, "n_frames < 0");
    if (n_frames == 0) return ULM_RCA_OK;
    if (!d_planes || !prm || !d_loc || !d_count) return fail(ULM_RCA_EINVAL, "pointer is NULL");
    if (!(prm->sigma_lat_px > 0) || !(prm->sigma_ax_px > 0) || !std::isfinite(prm->sigma_lat_px) || !std::isfinite(prm->sigma_ax_px) ||
        !std::isfinite(prm->threshold_rel) || !std::isfinite(prm->ncc_min) || prm->capacity < 1)
        return fail(ULM_RCA_EINVAL, "localize parameters invalid");
    if (ulm_rca_status s = check_device(*plan)) return s;
    const ulm::Stage2Plan &S = plan->s2;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    ulm::LoParams L{};
    L.planes_per_frame = S.planes_per_frame; L.n_z = S.n_z;
    for (int a = 0; a < 2; ++a) { L.n_planes[a] = S.n_g[a]; L.n_lat[a] = S.n_lat[a]; }
    L.set_off[0] = 0; L.set_off[1] = (long long)S.n_g[0] * S.n_lat[0] * S.n_z;
    double gm = 0, g1[ulm::kLoTaps], g2[ulm::kLoTaps];
    for (int k = 0; k < ulm::kLoTaps; ++k) {
        const double a = k - ulm::kLoHalf;
        g1[k] = std::exp(-a * a / (2.0 * prm->sigma_lat_px * prm->sigma_lat_px));
        g2[k] = std::exp(-a * a / (2.0 * prm->sigma_ax_px * prm->sigma_ax_px));
        L.g1[k] = (float)g1[k]; L.g2[k] = (float)g2[k];
    }
    for (int i = 0; i < ulm::kLoTaps; ++i) for (int j = 0; j < ulm::kLoTaps; ++j) gm += g1[i] * g2[j];
    gm /= 121.0;
    double gd = 0;
    for (int i = 0; i < ulm::kLoTaps; ++i) for (int j = 0; j < ulm::kLoTaps; ++j) gd += (g1[i] * g2[j] - gm) * (g1[i] * g2[j] - gm);
    L.g_mean = (float)gm; L.g_den = (float)gd;
    L.threshold_rel = prm->threshold_rel; L.ncc_min = prm->ncc_min; L.capacity = prm->capacity;
    const int n_pl = S.n_g[0] + S.n_g[1];
    int launches = 0;
    for (int f0 = 0; f0 < n_frames; f0 += plan->max_frames) {
        const int nb = std::min(plan->max_frames, n_frames - f0);
        L.planes = static_cast<const float2 *>(d_planes) + (long long)f0 * S.planes_per_frame;
        L.n_frames = nb;
        L.frame_max = plan->loc_frame_max.as<unsigned int>();
        L.loc = static_cast<float4 *>(d_loc) + (long long)f0 * n_pl * prm->capacity;
        L.count = static_cast<int *>(d_count) + (long long)f0 * n_pl;
        CUDA_TRY(cudaMemsetAsync(L.frame_max, 0, (size_t)nb * sizeof(unsigned int), st));
        CUDA_TRY(cudaMemsetAsync(L.count, 0, (size_t)nb * n_pl * sizeof(int), st));
        ulm::localize_max_kernel<<<dim3(64, nb), 256, 0, st>>>(L);
        const int lat_tiles = (std::max(S.n_lat[0], S.n_lat[1]) + ulm::kLoTl - 1) / ulm::kLoTl, z_tiles = (S.n_z + ulm::kLoTa - 1) / ulm::kLoTa;
        ulm::localize_kernel<<<dim3(lat_tiles, z_tiles, nb * n_pl), ulm::kLoThreads, ulm::kLoSmem, st>>>(L);
        CUDA_TRY(cudaGetLastError());
        launches += 2;
    }
    plan->last_launches = launches;
    return ULM_RCA_OK;
}

// ---- ulm_rca_localize_static: the same two kernels, no plan, no allocation ------------------------------------------
// The per-frame maximum (the only scratch of the operation) lives in this file-scope device array.  Its name is a
// host-side stand-in in host code: the device address is looked up once per device (that device current) with
// cudaGetSymbolAddress and handed to the kernels in LoParams::frame_max like the plan-owned buffer of ulm_rca_localize.
static __device__ __align__(256) unsigned int g_lo_static_frame_max[ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES];

namespace {
constexpr int kStaticMaxDevices = 64;
std::mutex g_lo_static_mutex;
unsigned int *g_lo_static_ptr[kStaticMaxDevices] = {};      // device address of g_lo_static_frame_max, per device

// set-up of the current device (once per device): address of the scratch array, shared-memory attribute of the kernel
ulm_rca_status lo_static_setup(unsigned int **out) {
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return fail(ULM_RCA_EUNSUPPORTED, "device index %d beyond %d", dev, kStaticMaxDevices - 1);
    std::lock_guard<std::mutex> lock(g_lo_static_mutex);
    if (!g_lo_static_ptr[dev]) {
        unsigned int *ptr = nullptr;
        CUDA_TRY(cudaGetSymbolAddress((void **)&ptr, g_lo_static_frame_max));
        if (!ptr) return fail(ULM_RCA_ECUDA, "cudaGetSymbolAddress returned a NULL address");
        CUDA_TRY(cudaFuncSetAttribute(ulm::localize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, ulm::kLoSmem));
        g_lo_static_ptr[dev] = ptr;
    }
    *out = g_lo_static_ptr[dev];
    return ULM_RCA_OK;
}
}  // namespace

ulm_rca_status ulm_rca_localize_static(const void *d_planes, int32_t n_frames, int32_t n_z, int32_t n_planes_xz,
                                       int32_t n_lat_xz, int32_t n_planes_yz, int32_t n_lat_yz,
                                       const ulm_rca_localize_params *prm, void *d_loc, void *d_count, void *cuda_stream) {
    if (n_frames < 0) return fail(ULM_RCA_EINVAL, "n_frames < 0");
    if (n_frames > ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES)
        return fail(ULM_RCA_EINVAL, "n_frames %d exceeds the static scratch of %d frames (ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES): split the call",
                    n_frames, ULM_RCA_LOCALIZE_STATIC_MAX_FRAMES);
    if (n_z < 1 || n_planes_xz < 0 || n_planes_yz < 0 || n_planes_xz + n_planes_yz < 1 || (n_planes_xz > 0 && n_lat_xz < 1) ||
        (n_planes_yz > 0 && n_lat_yz < 1))
        return fail(ULM_RCA_EINVAL, "plane geometry invalid");
    if (n_frames == 0) return ULM_RCA_OK;
    if (!d_planes || !prm || !d_loc || !d_count) return fail(ULM_RCA_EINVAL, "pointer is NULL");
    if (!(prm->sigma_lat_px > 0) || !(prm->sigma_ax_px > 0) || !std::isfinite(prm->sigma_lat_px) || !std::isfinite(prm->sigma_ax_px) ||
        !std::isfinite(prm->threshold_rel) || !std::isfinite(prm->ncc_min) || prm->capacity < 1)
        return fail(ULM_RCA_EINVAL, "localize parameters invalid");
    const int n_pl = n_planes_xz + n_planes_yz;
    const int lat_max = std::max(n_planes_xz > 0 ? n_lat_xz : 0, n_planes_yz > 0 ? n_lat_yz : 0);
    const long long lat_tiles = (lat_max + ulm::kLoTl - 1) / ulm::kLoTl, z_tiles = (n_z + ulm::kLoTa - 1) / ulm::kLoTa;
    if (z_tiles > 65535 || n_pl > 65535) return fail(ULM_RCA_EINVAL, "grid too large (planes per frame, or depth tiles, beyond 65535)");
    unsigned int *frame_max = nullptr;
    if (ulm_rca_status s = lo_static_setup(&frame_max)) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    ulm::LoParams L{};
    L.n_z = n_z;
    L.n_planes[0] = n_planes_xz; L.n_lat[0] = n_planes_xz > 0 ? n_lat_xz : 0;
    L.n_planes[1] = n_planes_yz; L.n_lat[1] = n_planes_yz > 0 ? n_lat_yz : 0;
    L.set_off[0] = 0; L.set_off[1] = (long long)n_planes_xz * L.n_lat[0] * n_z;
    L.planes_per_frame = L.set_off[1] + (long long)n_planes_yz * L.n_lat[1] * n_z;
    double gm = 0, g1[ulm::kLoTaps], g2[ulm::kLoTaps];
    for (int k = 0; k < ulm::kLoTaps; ++k) {
        const double a = k - ulm::kLoHalf;
        g1[k] = std::exp(-a * a / (2.0 * prm->sigma_lat_px * prm->sigma_lat_px));
        g2[k] = std::exp(-a * a / (2.0 * prm->sigma_ax_px * prm->sigma_ax_px));
        L.g1[k] = (float)g1[k]; L.g2[k] = (float)g2[k];
    }
    for (int i = 0; i < ulm::kLoTaps; ++i) for (int j = 0; j < ulm::kLoTaps; ++j) gm += g1[i] * g2[j];
    gm /= 121.0;
    double gd = 0;
    for (int i = 0; i < ulm::kLoTaps; ++i) for (int j = 0; j < ulm::kLoTaps; ++j) gd += (g1[i] * g2[j] - gm) * (g1[i] * g2[j] - gm);
    L.g_mean = (float)gm; L.g_den = (float)gd;
    L.threshold_rel = prm->threshold_rel; L.ncc_min = prm->ncc_min; L.capacity = prm->capacity;
    const int batch = std::min(n_frames, 65535 / n_pl);        // grid.z = frames x planes of a launch
    for (int f0 = 0; f0 < n_frames; f0 += batch) {
        const int nb = std::min(batch, n_frames - f0);
        L.planes = static_cast<const float2 *>(d_planes) + (long long)f0 * L.planes_per_frame;
        L.n_frames = nb;
        L.frame_max = frame_max + f0;
        L.loc = static_cast<float4 *>(d_loc) + (long long)f0 * n_pl * prm->capacity;
        L.count = static_cast<int *>(d_count) + (long long)f0 * n_pl;
        // the array keeps the previous call's maxima: the entries of this call start at zero
        CUDA_TRY(cudaMemsetAsync(L.frame_max, 0, (size_t)nb * sizeof(unsigned int), st));
        CUDA_TRY(cudaMemsetAsync(L.count, 0, (size_t)nb * n_pl * sizeof(int), st));
        ulm::localize_max_kernel<<<dim3(64, nb), 256, 0, st>>>(L);
        ulm::localize_kernel<<<dim3((unsigned)lat_tiles, (unsigned)z_tiles, (unsigned)(nb * n_pl)), ulm::kLoThreads, ulm::kLoSmem, st>>>(L);
    }
    CUDA_TRY(cudaGetLastError());
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_ring_probe(int32_t n_rx, float pitch_m, const float *angles_rad, const float *t0_s, int32_t n_tx,
                                  float c_mps, float fs_hz, float t_start_s, const ulm_rca_grid *grid,
                                  int32_t *n_tiles, int32_t *window, int32_t *dj, int32_t *wj) {
    if (!angles_rad || !grid || !n_tiles || !window || n_rx <= 0 || n_tx <= 0) return fail(ULM_RCA_EINVAL, "bad argument");
    if (ulm_rca_status s = check_grid(grid, "grid")) return s;
    std::vector<double> ang(angles_rad, angles_rad + n_tx), t0(n_tx, 0.0);
    if (t0_s) for (int k = 0; k < n_tx; ++k) t0[k] = t0_s[k];
    ulm::RingApertureDesc D{n_tx, n_rx, grid->n_lat, grid->n_ax, grid->lat0_m, grid->dlat_m, grid->z0_m, grid->dz_m,
                            grid->ref_m, ang.data(), t0.data()};
    std::vector<int> tab;
    int nt = 0;
    const char *why = nullptr;
    const int w = ulm::ring_plan_aperture(D, pitch_m, c_mps, fs_hz, t_start_s, tab, nt, &why);
    if (w < 0) return fail(ULM_RCA_EUNSUPPORTED, "ring kernel unavailable: %s", why ? why : "?");
    *n_tiles = nt;
    *window = (w + 7) / 8 * 8;
    const size_t n = (size_t)nt * n_rx;
    if (dj) std::copy(tab.begin(), tab.begin() + n, dj);
    if (wj) std::copy(tab.begin() + n, tab.begin() + 2 * n, wj);
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_fold_probe(const float *angles_rad, const float *t0_s, int32_t n_tx, float c_mps, float fs_hz,
                                  const ulm_rca_grid *grid, int32_t *partner) {
    if (!angles_rad || !grid || !partner || n_tx <= 0) return fail(ULM_RCA_EINVAL, "bad argument");
    if (ulm_rca_status s = check_grid(grid, "grid")) return s;
    if (!finite_pos(c_mps) || !finite_pos(fs_hz)) return fail(ULM_RCA_EINVAL, "c, fs must be finite and > 0");
    std::vector<double> ang(angles_rad, angles_rad + n_tx), t0(n_tx, 0.0);
    if (t0_s) for (int k = 0; k < n_tx; ++k) t0[k] = t0_s[k];
    const std::vector<int> p = fold_partners(ang, t0, c_mps, fs_hz, grid->ref_m, grid->z0_m, grid->dz_m, grid->n_ax, true);
    std::copy(p.begin(), p.end(), partner);
    return ULM_RCA_OK;
}

ulm_rca_status ulm_rca_fp32_peak(double *tflops, void *cuda_stream) {
    if (!tflops) return fail(ULM_RCA_EINVAL, "tflops is NULL");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *sink = nullptr;
    CUDA_TRY(cudaMalloc(&sink, sizeof(float)));
    cudaEvent_t a, b;
    CUDA_TRY(cudaEventCreate(&a));
    CUDA_TRY(cudaEventCreate(&b));
    const int blocks = sms * 8, iters = 4000;
    ulm::fp32_peak_kernel<<<blocks, 256, 0, st>>>(sink, 200, 0.999f, 0.001f);   // warm-up
    double best = 0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(a, st);
        ulm::fp32_peak_kernel<<<blocks, 256, 0, st>>>(sink, iters, 0.999f, 0.001f);
        cudaEventRecord(b, st);
        cudaEventSynchronize(b);
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        const double flop = 2.0 * 128.0 * iters * 256.0 * blocks;
        best = std::max(best, flop / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    cudaFree(sink);
    CUDA_TRY(cudaGetLastError());
    *tflops = best;
    return ULM_RCA_OK;
}

}  // extern "C"
