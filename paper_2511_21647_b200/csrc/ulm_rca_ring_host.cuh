// ulm_rca_ring_host.cuh -- host side of the shared-memory ring kernel: tile and window planning (fp64),
// the per-(tile, element) window-offset table, and the templated launch.
#pragma once

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>

#include "ulm_rca_ring.cuh"

namespace ulm {

constexpr int kSmemLimit = 232448;   // 227 KB opt-in dynamic shared memory per CTA on sm_100
constexpr int kRingPx = 4;           // rows per strip = pixels per consumer thread
constexpr int kRingPxDual = 2;       // ... of the two-group work items (2 pixels x 24 frames per thread)
// two table buffers (per-item transmit table + 4 per-element arrays), stage headers, ring and table barriers
constexpr int kRingMisc = 2 * (kRingMaxTab * 8 + 4 * kRingMaxRx * 4) + kRingMaxStages * 4 + 2 * kRingMaxStages * 8 + 4 * 8 + 64;

struct RingConfig {
    int window = 0;      // entries per stage
    int window2 = 0;     // ... of the two-group work items (tiles of kRingPxDual rows); 0: not planned
    int n_sms = 0;
    // tail splitting (RingLaunch::split_s): partial sums of the split work items, kRingSplitCap sub-items at most
    float2 *d_partial = nullptr;
    int partial_cap = 0;
    ~RingConfig() { if (d_partial) cudaFree(d_partial); }
};

constexpr int kRingSplitMax = 16;    // slices per split work item at most

// Slices for the r = n_items mod n_sms work items of the last, partially filled round of a grid of n_sms persistent
// CTAs: s slices each turn that round into ceil(r s / n_sms) rounds of 1/s of the time.  Returns 1 (no split) unless a
// split saves at least 10 % of a round.
inline int ring_split_choice(int r, int n_sms, int n_rx, int cap) {
    if (r <= 0) return 1;
    int best = 1;
    double best_cost = 1.0;
    for (int s = 2; s <= kRingSplitMax && s <= n_rx && (long long)r * s <= cap; ++s) {
        const double cost = (double)(((long long)r * s + n_sms - 1) / n_sms) / s + 0.01 * s;     // + per-slice overhead
        if (cost < best_cost - 1e-9) { best_cost = cost; best = s; }
    }
    return best_cost <= 0.9 ? best : 1;
}

struct RingTables {
    int n_tiles = 0;
    int *d_dj = nullptr;     // [tile][j] floor(min H over the tile) - 2, followed by [tile][j] entries the stage needs
    ~RingTables() { if (d_dj) cudaFree(d_dj); }
};

struct RingApertureDesc {
    int n_tx, n_rx, n_lat, n_ax;
    double lat0, dlat, z0, dz, ref;
    const double *angles, *t0;
};

namespace ringhost {

struct Geo {
    const RingApertureDesc *d;
    double pitch, c, fs, t_start;
    double lat(int i) const { return d->lat0 + i * d->dlat; }
    double z(int i) const { return d->z0 + i * d->dz; }
    double elem(int j) const { return (j - 0.5 * (d->n_rx - 1)) * pitch; }
    double u0(int k, double z) const {
        return (d->t0[k] + (z * std::cos(d->angles[k]) + d->ref * std::sin(d->angles[k])) / c + z / c - t_start) * fs;
    }
    double h(double dx, double z) const { return (std::sqrt(dx * dx + z * z) - z) * fs / c; }
};

// one strip segment of a tile: columns [c0, c1], rows [r0, r1] (image rows)
struct Seg { int c0, c1, r0, r1; };

inline std::vector<Seg> tile_segments(const RingApertureDesc &D, int tile, int px = kRingPx) {
    const int n_pos = D.n_lat * ((D.n_ax + px - 1) / px);
    const int p0 = tile * kRingConsumers, p1 = std::min(p0 + kRingConsumers, n_pos) - 1;
    std::vector<Seg> v;
    for (int s = p0 / D.n_lat; s <= p1 / D.n_lat; ++s) {
        Seg g;
        g.c0 = s == p0 / D.n_lat ? p0 % D.n_lat : 0;
        g.c1 = s == p1 / D.n_lat ? p1 % D.n_lat : D.n_lat - 1;
        g.r0 = s * px;
        g.r1 = std::min(s * px + px - 1, D.n_ax - 1);
        v.push_back(g);
    }
    return v;
}

// receive-excess range [h_lo, h_hi] of element j over a segment: H grows with |dx| and shrinks with z
inline void h_range(const Geo &G, const Seg &s, int j, double &h_lo, double &h_hi) {
    const double la = G.lat(s.c0), lb = G.lat(s.c1), e = G.elem(j);
    const double lo = std::min(la, lb), hi = std::max(la, lb);
    const double dmin = (e >= lo && e <= hi) ? 0.0 : std::min(std::fabs(la - e), std::fabs(lb - e));
    const double dmax = std::max(std::fabs(la - e), std::fabs(lb - e));
    h_lo = G.h(dmin, G.z(s.r1));
    h_hi = G.h(dmax, G.z(s.r0));
}

}  // namespace ringhost

// Plans one aperture: fills dj (host) and returns the window (entries) it needs, or -1 with *why.
inline int ring_plan_aperture(const RingApertureDesc &D, double pitch, double c, double fs, double t_start,
                              std::vector<int> &dj, int &n_tiles, const char **why, int px = kRingPx) {
    using namespace ringhost;
    n_tiles = 0;
    dj.clear();
    if (D.n_tx == 0) return 0;
    if (D.n_rx > kRingMaxRx) { *why = "more than 256 receive elements"; return -1; }
    Geo G{&D, pitch, c, fs, t_start};
    const int n_pos = D.n_lat * ((D.n_ax + px - 1) / px);
    n_tiles = (n_pos + kRingConsumers - 1) / kRingConsumers;
    dj.assign((size_t)2 * n_tiles * D.n_rx, 0);     // dj, then the per-(tile, element) window lengths
    int window = 8;
    for (int t = 0; t < n_tiles; ++t) {
        const std::vector<Seg> segs = tile_segments(D, t, px);
        const int iz0 = segs.front().r0, rows = segs.back().r1 - iz0 + 1;
        if ((long long)rows * D.n_tx > kRingMaxTab) { *why = "tile rows x angles exceed the transmit table"; return -1; }
        for (int j = 0; j < D.n_rx; ++j) {
            double h_min = 1e300;
            for (const Seg &s : segs) {
                double lo, hi;
                h_range(G, s, j, lo, hi);
                h_min = std::min(h_min, lo);
            }
            const int d = (int)std::floor(h_min) - 2;
            dj[(size_t)t * D.n_rx + j] = d;
            int need = 8;
            for (const Seg &s : segs) {
                double lo, hi;
                h_range(G, s, j, lo, hi);
                for (int k = 0; k < D.n_tx; ++k) {
                    // upm = U0_k(z_r) - floor(U0_k(z_iz0)) - 0.5 + H - dj; the entry index is rint(upm)
                    const double top = G.u0(k, G.z(s.r1)) - std::floor(G.u0(k, G.z(iz0))) - 0.5 + hi - d;
                    need = std::max(need, (int)std::floor(top + 0.5) + 4);
                }
            }
            need = (need + 7) / 8 * 8;
            dj[(size_t)(n_tiles + t) * D.n_rx + j] = need;
            window = std::max(window, need);
        }
    }
    return window;
}

inline int ring_stage_stride(int window, int F, bool d32) { return (window * entry_bytes(F, d32) + 127) / 128 * 128; }
inline int ring_stages(int window, int F, bool d32) {
    return std::min(kRingMaxStages, (kSmemLimit - kRingMisc) / ring_stage_stride(window, F, d32));
}
inline int ring_smem_bytes(int window, int F, bool d32) {
    return ring_stages(window, F, d32) * ring_stage_stride(window, F, d32) + kRingMisc;
}
// two-group work items (compact entries, F = 12): a ring slot holds the windows of both frame groups
inline int ring_dual_half(int window2) { return ring_stage_stride(window2, 12, false); }
inline int ring_dual_stages(int window2) { return std::min(kRingMaxStages, (kSmemLimit - kRingMisc) / (2 * ring_dual_half(window2))); }
inline int ring_dual_smem_bytes(int window2) { return ring_dual_stages(window2) * 2 * ring_dual_half(window2) + kRingMisc; }

// Plans both apertures.  Returns false (with *why) when the ring kernel does not cover the shape.
inline bool ring_plan(const RingApertureDesc *desc, double pitch, double c, double fs, double t_start,
                      int l_row, RingConfig &cfg, RingTables &tab0, RingTables &tab1, const char **why) {
    RingTables *tabs[2] = {&tab0, &tab1};
    int window = 8;
    for (int a = 0; a < 2; ++a) {
        std::vector<int> dj;
        const int w = ring_plan_aperture(desc[a], pitch, c, fs, t_start, dj, tabs[a]->n_tiles, why);
        if (w < 0) return false;
        window = std::max(window, w);
        if (dj.empty()) continue;
        if (cudaMalloc(&tabs[a]->d_dj, dj.size() * sizeof(int)) != cudaSuccess) { *why = "table allocation failed"; return false; }
        if (cudaMemcpy(tabs[a]->d_dj, dj.data(), dj.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
            *why = "table upload failed";
            return false;
        }
    }
    window = (window + 7) / 8 * 8;
    if (window > l_row) { *why = "window exceeds the scratch row"; return false; }
    if (ring_stages(window, 12, true) < 2) { *why = "fewer than two ring stages fit in shared memory"; return false; }
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cfg.window = window;
    cfg.n_sms = sms;
    cfg.partial_cap = 4 * sms;
    if (cudaMalloc(&cfg.d_partial, (size_t)cfg.partial_cap * kRingConsumers * kRingPx * 12 * sizeof(float2)) != cudaSuccess) {
        cudaGetLastError();
        cfg.d_partial = nullptr;      // no tail splitting
        cfg.partial_cap = 0;
    }
    return true;
}

// Plans the tiles of the two-group work items (kRingPxDual rows per strip).  On any failure cfg.window2 stays 0 and the
// launches keep to the one-group items.
inline void ring_plan_dual(const RingApertureDesc *desc, double pitch, double c, double fs, double t_start,
                           int l_row, RingConfig &cfg, RingTables &tab0, RingTables &tab1) {
    RingTables *tabs[2] = {&tab0, &tab1};
    const char *why = nullptr;
    int window = 8;
    for (int a = 0; a < 2; ++a) {
        std::vector<int> dj;
        const int w = ring_plan_aperture(desc[a], pitch, c, fs, t_start, dj, tabs[a]->n_tiles, &why, kRingPxDual);
        if (w < 0) return;
        window = std::max(window, w);
        if (dj.empty()) continue;
        if (cudaMalloc(&tabs[a]->d_dj, dj.size() * sizeof(int)) != cudaSuccess ||
            cudaMemcpy(tabs[a]->d_dj, dj.data(), dj.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError();
            return;
        }
    }
    window = (window + 7) / 8 * 8;
    if (window > l_row || ring_dual_stages(window) < 3) return;
    cfg.window2 = window;
}

template <int F, bool D32, bool APOD, bool W2, bool DUAL>
inline int ring_launch_t(const RingConfig &cfg, RingLaunch &L, cudaStream_t st) {
    constexpr int PX = DUAL ? kRingPxDual : kRingPx, FE = DUAL ? 2 * F : F;
    int smem;
    if (DUAL) {
        L.stage_half = ring_dual_half(cfg.window2);
        L.stage_stride = 2 * L.stage_half;
        L.n_stages = ring_dual_stages(cfg.window2);
        smem = ring_dual_smem_bytes(cfg.window2);
    } else {
        L.stage_half = 0;
        L.stage_stride = ring_stage_stride(cfg.window, F, D32);
        L.n_stages = ring_stages(cfg.window, F, D32);
        smem = ring_smem_bytes(cfg.window, F, D32);
    }
    L.n_fgroups = (L.n_frames + F - 1) / F;
    // groups (pairs) of this launch: all of them, or the range the caller set (L.g_first, L.n_groups > 0)
    if (L.n_groups <= 0) { L.g_first = 0; L.n_groups = DUAL ? (L.n_fgroups + 1) / 2 : L.n_fgroups; }
    L.n_items = L.n_groups * (L.ap[0].n_tiles * (L.per_angle ? L.ap[0].n_tx : 1) + L.ap[1].n_tiles * (L.per_angle ? L.ap[1].n_tx : 1));
    if (L.n_items == 0) return 0;
    // tail splitting: the items of the last, partially filled round are cut into slices of the receive elements
    // (a call with fewer items than SMs -- a single frame -- is one partially filled round: n_whole = 0)
    const int rem = L.n_items % cfg.n_sms;
    int n_rx_min = 1 << 30;
    for (int a = 0; a < 2; ++a) if (L.ap[a].n_tiles > 0) n_rx_min = std::min(n_rx_min, L.ap[a].n_rx);
    L.split_s = ring_split_choice(rem, cfg.n_sms, n_rx_min, cfg.partial_cap);
    L.n_whole = L.split_s > 1 ? L.n_items - rem : L.n_items;
    L.n_work = L.n_whole + (L.n_items - L.n_whole) * L.split_s;
    L.partial = cfg.d_partial;
    const int grid = std::min(L.n_work, cfg.n_sms);
    das_ring_kernel<F, PX, D32, APOD, W2, DUAL><<<grid, kRingThreads, smem, st>>>(L);
    if (L.split_s > 1) {
        ring_combine_kernel<FE, PX><<<dim3(L.n_items - L.n_whole, PX), kRingConsumers, 0, st>>>(L);
        return 2;
    }
    return 1;
}

// The opt-in to 227 KB of dynamic shared memory is a per-device function attribute: ulm_rca_plan_create calls this on
// the plan's device for every instantiation a launch can select (no process-wide "already set" flag).
template <int F, bool D32, bool APOD, bool W2 = false, bool DUAL = false>
inline cudaError_t ring_set_attr_one() {
    return cudaFuncSetAttribute(das_ring_kernel<F, DUAL ? kRingPxDual : kRingPx, D32, APOD, W2, DUAL>,
                                cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
}
inline cudaError_t ring_set_attributes() {
    cudaError_t e;
    if ((e = ring_set_attr_one<12, false, false>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, false, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, true, false>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, true, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<4, false, false>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<4, false, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<4, true, false>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<4, true, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, false, false, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, false, true, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<4, false, false, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<4, false, true, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, false, false, false, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, false, true, false, true>()) != cudaSuccess) return e;
    if ((e = ring_set_attr_one<12, false, false, true, true>()) != cudaSuccess) return e;
    return ring_set_attr_one<12, false, true, true, true>();
}

template <int F, bool D32, bool W2, bool DUAL>
inline int ring_launch_a(const RingConfig &cfg, RingLaunch &L, bool apod, cudaStream_t st) {
    return apod ? ring_launch_t<F, D32, true, W2, DUAL>(cfg, L, st) : ring_launch_t<F, D32, false, W2, DUAL>(cfg, L, st);
}

// returns the number of kernels launched; F = frames per group of the scratch (4 or 12), d32 = full entries,
// w2 = compact entries with the two-term interpolation weight.  dtab0 / dtab1 = the tables of the two-group work items,
// used for compact entries when the call has at least two frame groups of 12.
inline int ring_launch(const RingConfig &cfg, const RingTables &tab0, const RingTables &tab1, const RingTables &dtab0,
                       const RingTables &dtab1, const RingLaunch &Lin, int F, bool d32, bool w2, bool apod, cudaStream_t st) {
    RingLaunch L = Lin;
    const bool dual = F == 12 && !d32 && cfg.window2 > 0 && L.n_frames > 12;
    const RingTables *tabs[2] = {dual ? &dtab0 : &tab0, dual ? &dtab1 : &tab1};
    for (int a = 0; a < 2; ++a) {
        L.ap[a].dj = tabs[a]->d_dj;
        L.ap[a].wj = tabs[a]->d_dj ? tabs[a]->d_dj + (size_t)tabs[a]->n_tiles * L.ap[a].n_rx : nullptr;
        L.ap[a].n_tiles = L.ap[a].n_tx > 0 ? tabs[a]->n_tiles : 0;
    }
    L.window = dual ? cfg.window2 : cfg.window;
    L.g_first = 0;
    L.n_groups = 0;
    if (dual) {
        // whole pairs go through the two-group items; an odd last group is a launch of one-group items of its own
        const int n_fg = (L.n_frames + 11) / 12;
        L.n_groups = n_fg / 2;
        int n = w2 ? ring_launch_a<12, false, true, true>(cfg, L, apod, st) : ring_launch_a<12, false, false, true>(cfg, L, apod, st);
        if (n_fg & 1) {
            RingLaunch L1 = Lin;
            const RingTables *t1[2] = {&tab0, &tab1};
            for (int a = 0; a < 2; ++a) {
                L1.ap[a].dj = t1[a]->d_dj;
                L1.ap[a].wj = t1[a]->d_dj ? t1[a]->d_dj + (size_t)t1[a]->n_tiles * L1.ap[a].n_rx : nullptr;
                L1.ap[a].n_tiles = L1.ap[a].n_tx > 0 ? t1[a]->n_tiles : 0;
            }
            L1.window = cfg.window;
            L1.g_first = n_fg - 1;
            L1.n_groups = 1;
            // (the split tail of this launch reuses cfg.d_partial: stream order puts it after the first launch's combine)
            n += w2 ? ring_launch_a<12, false, true, false>(cfg, L1, apod, st) : ring_launch_a<12, false, false, false>(cfg, L1, apod, st);
        }
        return n;
    }
    if (F == 12) return d32 ? ring_launch_a<12, true, false, false>(cfg, L, apod, st)
                            : (w2 ? ring_launch_a<12, false, true, false>(cfg, L, apod, st) : ring_launch_a<12, false, false, false>(cfg, L, apod, st));
    return d32 ? ring_launch_a<4, true, false, false>(cfg, L, apod, st)
               : (w2 ? ring_launch_a<4, false, true, false>(cfg, L, apod, st) : ring_launch_a<4, false, false, false>(cfg, L, apod, st));
}

}  // namespace ulm
