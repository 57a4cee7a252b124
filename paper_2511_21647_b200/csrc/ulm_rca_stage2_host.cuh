// ulm_rca_stage2_host.cuh -- host side of Stage 2: the complex tap tables of the "own" FIRs and
// of the "cross" two-tap interpolations are built in fp64 from the plan's geometry, uploaded once, and the two kernels
// of ulm_rca_stage2.cuh are launched from here.
#pragma once

#include <algorithm>
#include <cmath>
#include <complex>
#include <vector>

#include "ulm_rca_stage2.cuh"

namespace ulm {

struct Stage2Axis {          // one aperture's slices: lateral grid, reference position along the transmit direction
    int n_lat = 0;
    double lat0 = 0, dlat = 0, ref = 0;
    std::vector<double> angles;
    double lat(int i) const { return lat0 + i * dlat; }
};

struct Stage2Plan {
    bool ready = false;
    int block = 0, nt = 0;               // P; taps per own FIR (template instantiation)
    int n_z = 0, halo_lo = 0, ncol = 0, rs = 0, g_max = 0, n_events = 0, n_row_tx = 0;
    int n_lat[2] = {0, 0}, n_g[2] = {0, 0};
    long long slices_per_frame = 0, planes_per_frame = 0;
    int max_frames = 0;
    void *d_own_o[2] = {nullptr, nullptr}, *d_own_w[2] = {nullptr, nullptr};
    void *d_cross_o[2] = {nullptr, nullptr}, *d_cross_w[2] = {nullptr, nullptr};
    void *d_gsum = nullptr;
    cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
    ~Stage2Plan() {
        for (int a = 0; a < 2; ++a) {
            if (d_own_o[a]) cudaFree(d_own_o[a]);
            if (d_own_w[a]) cudaFree(d_own_w[a]);
            if (d_cross_o[a]) cudaFree(d_cross_o[a]);
            if (d_cross_w[a]) cudaFree(d_cross_w[a]);
        }
        if (d_gsum) cudaFree(d_gsum);
        for (auto &e : ev) if (e) cudaEventDestroy(e);
    }
};

namespace s2host {

template <class T> inline cudaError_t upload(void **dst, const std::vector<T> &v) {
    *dst = nullptr;
    if (v.empty()) return cudaSuccess;
    cudaError_t e = cudaMalloc(dst, v.size() * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice);
}

// shift of event angle th at transmit-direction coordinate w, in depth pixels, split as n + b
inline void shift_of(double w, double ref, double th, double dz, int &n, double &b) {
    const double q = (w - ref) * std::tan(0.5 * th) / dz;
    const double fl = std::floor(q);
    n = (int)fl;
    b = q - fl;
}

}  // namespace s2host

inline int stage2_smem_bytes(const Stage2Plan &S) {
    const int n_tx_max = std::max(S.n_row_tx, S.n_events - S.n_row_tx);
    // tile buffers (kS2Ev events per stage) + the CTA's tap tables (own: [events][8 groups][1 + NT], cross: [events][32 positions][3])
    return (kS2Stages * kS2Ev * (kS2Lat * S.rs + kS2Warps * S.ncol) + n_tx_max * kS2Warps * (1 + S.nt) + n_tx_max * kS2Lat * 3) *
           (int)sizeof(float2);
}

// Builds the tables.  ax[0] = x-z slices (row-tx events, transmit direction y), ax[1] = y-z slices.  Returns nullptr on
// success or a reason; cudaGetLastError() tells allocation failures apart.
inline const char *stage2_build(Stage2Plan &S, const Stage2Axis ax[2], int n_z, double dz, double c, double fc,
                                int block, int max_frames, bool timing) {
    using namespace s2host;
    using cd = std::complex<double>;
    const double two_pi_fc = 2.0 * M_PI * fc;
    S.block = block;
    S.n_z = n_z;
    S.max_frames = max_frames;
    S.n_row_tx = (int)ax[0].angles.size();
    S.n_events = (int)(ax[0].angles.size() + ax[1].angles.size());
    int lo = 0, hi = 1, nt = 2;
    // pass 1: tap ranges
    struct Own { std::vector<int> o; std::vector<std::vector<cd>> w; };
    Own own[2];
    std::vector<int> cross_o[2];
    std::vector<cd> cross_w[2];
    for (int a = 0; a < 2; ++a) {
        const Stage2Axis &A = ax[a], &O = ax[1 - a];      // planes of set a: lateral axis of A, grouped axis = lateral axis of O
        S.n_lat[a] = A.n_lat;
        S.n_g[a] = (O.n_lat + block - 1) / block;
        // own events (slices of A, transmit direction = O's lateral axis, slice position A.ref on it)
        for (size_t k = 0; k < A.angles.size(); ++k) {
            const double th = A.angles[k];
            for (int m = 0; m < S.n_g[a]; ++m) {
                const int l0 = m * block, l1 = std::min(l0 + block, O.n_lat);
                int n_min = 1 << 30, n_max = -(1 << 30);
                for (int l = l0; l < l1; ++l) {
                    int n; double b;
                    shift_of(O.lat(l), A.ref, th, dz, n, b);
                    n_min = std::min(n_min, n);
                    n_max = std::max(n_max, n + 1);
                }
                std::vector<cd> w(n_max - n_min + 1, cd(0, 0));
                for (int l = l0; l < l1; ++l) {
                    int n; double b;
                    shift_of(O.lat(l), A.ref, th, dz, n, b);
                    const cd y = std::polar(1.0, two_pi_fc * (O.lat(l) - A.ref) * std::sin(th) / c);
                    w[n - n_min] += (1.0 - b) * y;
                    w[n + 1 - n_min] += b * y;
                }
                for (size_t t = 0; t < w.size(); ++t)       // T_k(i) conj(T_k(i + s)), s = n_min + t
                    w[t] *= std::polar(1.0, -two_pi_fc * (double)(n_min + (int)t) * dz * (1.0 + std::cos(th)) / c);
                own[a].o.push_back(n_min);
                own[a].w.push_back(w);
                nt = std::max(nt, (int)w.size());
                lo = std::min(lo, n_min);
                hi = std::max(hi, n_max);
            }
        }
        // cross events (slices of O, transmit direction = A's lateral axis, slice position O.ref on it)
        for (size_t k = 0; k < O.angles.size(); ++k) {
            const double th = O.angles[k];
            for (int i = 0; i < A.n_lat; ++i) {
                int n; double b;
                shift_of(A.lat(i), O.ref, th, dz, n, b);
                const cd xph = std::polar(1.0, two_pi_fc * (A.lat(i) - O.ref) * std::sin(th) / c);
                const double slope = two_pi_fc * dz * (1.0 + std::cos(th)) / c;
                cross_o[a].push_back(n);
                cross_w[a].push_back((1.0 - b) * xph * std::polar(1.0, -slope * n));
                cross_w[a].push_back(b * xph * std::polar(1.0, -slope * (n + 1)));
                lo = std::min(lo, n);
                hi = std::max(hi, n + 1);
            }
        }
    }
    if (nt > kS2MaxTaps) return "more than 8 depth taps per block (block too thick for this angle / depth step)";
    S.nt = nt <= 2 ? 2 : nt <= 3 ? 3 : nt <= 4 ? 4 : nt <= 6 ? 6 : 8;
    S.halo_lo = -lo;
    // the widest window read: offsets lo .. max(hi, o + NT - 1) relative to a chunk of 8 depths
    S.ncol = kS2Zt + S.halo_lo + hi + (S.nt - 1);
    if (S.ncol > kS2MaxCol) return "axial shift range too large for the shared-memory tile";
    S.rs = S.ncol | 1;
    S.g_max = std::max(S.n_g[0], S.n_g[1]);
    if (stage2_smem_bytes(S) > 100 * 1024) return "too many transmit events for the shared-memory tap tables";
    S.slices_per_frame = ((long long)ax[0].angles.size() * ax[0].n_lat + (long long)ax[1].angles.size() * ax[1].n_lat) * n_z;
    S.planes_per_frame = ((long long)S.n_g[0] * S.n_lat[0] + (long long)S.n_g[1] * S.n_lat[1]) * n_z;
    for (int a = 0; a < 2; ++a) {
        std::vector<float2> w((size_t)own[a].o.size() * S.nt, make_float2(0.f, 0.f));
        for (size_t q = 0; q < own[a].o.size(); ++q)
            for (size_t t = 0; t < own[a].w[q].size(); ++t)
                w[q * S.nt + t] = make_float2((float)own[a].w[q][t].real(), (float)own[a].w[q][t].imag());
        std::vector<float2> cw(cross_w[a].size());
        for (size_t q = 0; q < cw.size(); ++q) cw[q] = make_float2((float)cross_w[a][q].real(), (float)cross_w[a][q].imag());
        if (upload(&S.d_own_o[a], own[a].o) != cudaSuccess || upload(&S.d_own_w[a], w) != cudaSuccess ||
            upload(&S.d_cross_o[a], cross_o[a]) != cudaSuccess || upload(&S.d_cross_w[a], cw) != cudaSuccess)
            return "table upload failed";
    }
    if (cudaMalloc(&S.d_gsum, (size_t)max_frames * S.n_events * S.g_max * n_z * sizeof(float2)) != cudaSuccess)
        return "group-sum scratch allocation failed";
    if (timing) for (auto &e : S.ev) if (cudaEventCreate(&e) != cudaSuccess) return "event creation failed";
    S.ready = true;
    return nullptr;
}

template <int NT>
inline cudaError_t stage2_launch_t(const Stage2Params &P, dim3 grid, int smem, cudaStream_t st) {
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(stage2_project_kernel<NT>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
    }
    stage2_project_kernel<NT><<<grid, kS2Threads, smem, st>>>(P);
    return cudaGetLastError();
}

// one batch of at most S.max_frames frames; returns the CUDA status, *launches += kernels launched
inline cudaError_t stage2_launch(const Stage2Plan &S, const float2 *slices, int n_frames, float2 *planes, cudaStream_t st,
                                 int *launches) {
    cudaError_t e;
    if (S.ev[0] && (e = cudaEventRecord(S.ev[0], st)) != cudaSuccess) return e;
    GroupSumParams G{};
    G.slices = slices; G.slices_per_frame = S.slices_per_frame; G.gsum = static_cast<float2 *>(S.d_gsum);
    G.n_events = S.n_events; G.g_max = S.g_max; G.n_z = S.n_z; G.block = S.block; G.n_frames = n_frames;
    G.n_row_tx = S.n_row_tx; G.n_lat0 = S.n_lat[0]; G.n_lat1 = S.n_lat[1];
    const long long n = (long long)n_frames * S.n_events * S.g_max * S.n_z;
    stage2_groupsum_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(G);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (S.ev[1] && (e = cudaEventRecord(S.ev[1], st)) != cudaSuccess) return e;

    Stage2Params P{};
    P.slices = slices; P.slices_per_frame = S.slices_per_frame; P.gsum = static_cast<const float2 *>(S.d_gsum);
    P.n_events = S.n_events; P.g_max = S.g_max; P.n_z = S.n_z; P.planes = planes; P.planes_per_frame = S.planes_per_frame;
    P.n_frames = n_frames; P.halo_lo = S.halo_lo; P.ncol = S.ncol; P.rs = S.rs;
    P.z_tiles = (S.n_z + kS2Zt - 1) / kS2Zt;
    const int n_own[2] = {S.n_row_tx, S.n_events - S.n_row_tx};
    for (int a = 0; a < 2; ++a) {
        Stage2Set &T = P.set[a];
        T.n_lat = S.n_lat[a]; T.n_w = S.n_lat[1 - a]; T.n_g = S.n_g[a];
        T.own_n = n_own[a]; T.cross_n = n_own[1 - a];
        T.own_off = a == 0 ? 0 : (long long)S.n_row_tx * S.n_lat[0] * S.n_z;
        T.cross_goff = a == 0 ? S.n_row_tx : 0;
        T.own_o = static_cast<const int *>(S.d_own_o[a]); T.own_w = static_cast<const float2 *>(S.d_own_w[a]);
        T.cross_o = static_cast<const int *>(S.d_cross_o[a]); T.cross_w = static_cast<const float2 *>(S.d_cross_w[a]);
        T.out_off = a == 0 ? 0 : (long long)S.n_g[0] * S.n_lat[0] * S.n_z;
    }
    const int lat_tiles = (std::max(S.n_lat[0], S.n_lat[1]) + kS2Lat - 1) / kS2Lat;
    const int m_blocks = (S.g_max + kS2Warps - 1) / kS2Warps;
    // a CTA walks as many consecutive depth tiles as still leaves ~8 CTAs per SM (measured on cfg 2: one tile per CTA
    // 7.80 ms, three 7.45 ms, all eleven 7.30 ms: the tap tables and the pipeline prologue are paid once per CTA)
    {
        int sms = 148, dev = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        const long long base = (long long)lat_tiles * m_blocks * 2 * n_frames;
        int tpc = P.z_tiles;
        while (tpc > 1 && base * ((P.z_tiles + tpc - 1) / tpc) < 8ll * sms) --tpc;
        P.tiles_per_cta = tpc;
    }
    const int z_runs = (P.z_tiles + P.tiles_per_cta - 1) / P.tiles_per_cta;
    const dim3 grid(lat_tiles, m_blocks * z_runs, 2 * n_frames);
    const int smem = stage2_smem_bytes(S);
    switch (S.nt) {
        case 2: e = stage2_launch_t<2>(P, grid, smem, st); break;
        case 3: e = stage2_launch_t<3>(P, grid, smem, st); break;
        case 4: e = stage2_launch_t<4>(P, grid, smem, st); break;
        case 6: e = stage2_launch_t<6>(P, grid, smem, st); break;
        default: e = stage2_launch_t<8>(P, grid, smem, st); break;
    }
    if (e != cudaSuccess) return e;
    if (S.ev[2] && (e = cudaEventRecord(S.ev[2], st)) != cudaSuccess) return e;
    *launches += 2;
    return cudaSuccess;
}

}  // namespace ulm
