// ulm_rca_ring_host.cuh -- host side of the shared-memory ring kernel: tile shape and window planning
// (fp64), the per-(tile, element, angle) window-start table, and the templated launch.
#pragma once

#include <algorithm>
#include <cmath>
#include <vector>

#include "ulm_rca_ring.cuh"

namespace ulm {

constexpr int kSmemLimit = 232448;   // 227 KB opt-in dynamic shared memory per CTA on sm_100

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
    // delay range [u_lo, u_hi] (samples) of tile x [ix0, ix1] x z [iz0, iz1] for angle k, element j:
    // U0 grows with z, H grows with |dx| and shrinks with z
    void range(int ix0, int ix1, int iz0, int iz1, int k, int j, double &u_lo, double &u_hi) const {
        const double la = lat(ix0), lb = lat(ix1), e = elem(j);
        const double lo = std::min(la, lb), hi = std::max(la, lb);
        const double dmin = (e >= lo && e <= hi) ? 0.0 : std::min(std::fabs(la - e), std::fabs(lb - e));
        const double dmax = std::max(std::fabs(la - e), std::fabs(lb - e));
        u_lo = u0(k, z(iz0)) + h(dmin, z(iz1));
        u_hi = u0(k, z(iz1)) + h(dmax, z(iz0));
    }
};

struct Tiling {
    int tx = 0, tz = 0, tiles_x = 0, tiles_z = 0, window = 0;
    int n_tiles() const { return tiles_x * tiles_z; }
};

inline int window_of(const Geo &G, const Tiling &T) {
    int w = 0;
    const RingApertureDesc &D = *G.d;
    for (int tzi = 0; tzi < T.tiles_z; ++tzi)
        for (int txi = 0; txi < T.tiles_x; ++txi) {
            const int ix0 = txi * T.tx, ix1 = std::min(D.n_lat, ix0 + T.tx) - 1;
            const int iz0 = tzi * T.tz, iz1 = std::min(D.n_ax, iz0 + T.tz) - 1;
            for (int k = 0; k < D.n_tx; ++k)
                for (int j = 0; j < D.n_rx; ++j) {
                    double lo, hi;
                    G.range(ix0, ix1, iz0, iz1, k, j, lo, hi);
                    w = std::max(w, (int)std::floor(hi) - (int)std::floor(lo) + 6);
                }
        }
    return w;
}

// pick the tile shape that minimises  tiles * (pixel capacity + window)  ~ shared-memory traffic
inline bool choose_tiling(const Geo &G, int max_window, Tiling &best) {
    const RingApertureDesc &D = *G.d;
    double best_cost = 1e300;
    bool found = false;
    for (int tiles_x = 1; tiles_x <= std::max(1, D.n_lat / 8); ++tiles_x) {
        Tiling T;
        T.tiles_x = tiles_x;
        T.tx = (D.n_lat + tiles_x - 1) / tiles_x;
        T.tiles_x = (D.n_lat + T.tx - 1) / T.tx;
        int tz = std::min({D.n_ax, kRingTilePixels / T.tx, kRingMaxTz, kRingMaxBt / std::max(1, D.n_tx)});
        if (tz < 1) continue;
        T.tiles_z = (D.n_ax + tz - 1) / tz;
        T.tz = (D.n_ax + T.tiles_z - 1) / T.tiles_z;
        T.window = (window_of(G, T) + 7) / 8 * 8;
        if (T.window > max_window) continue;
        const double cost = (double)T.n_tiles() * (kRingTilePixels + T.window);
        if (cost < best_cost) { best_cost = cost; best = T; found = true; }
    }
    return found;
}

}  // namespace ringhost

// Plans both apertures.  Returns false (with *why) when the ring kernel does not cover the shape.
inline bool ring_plan(const RingApertureDesc *desc, double pitch, double c, double fs, double t_start, int n_lo,
                      int l_row, bool /*apod*/, RingConfig &cfg, RingTables &tab0, RingTables &tab1, const char **why) {
    using namespace ringhost;
    RingTables *tabs[2] = {&tab0, &tab1};
    Tiling til[2];
    int window = 8;
    for (int a = 0; a < 2; ++a) {
        const RingApertureDesc &D = desc[a];
        if (D.n_tx == 0) continue;
        if (D.n_rx > kRingMaxRx) { *why = "more than 256 receive elements"; return false; }
        if (D.n_tx > kRingMaxBt) { *why = "too many angles"; return false; }
        Geo G{&D, pitch, c, fs, t_start};
        if (!choose_tiling(G, 512, til[a])) { *why = "no tile shape whose window fits 512 entries"; return false; }
        window = std::max(window, til[a].window);
    }
    if (window > l_row) { *why = "window exceeds the scratch row"; return false; }
    const int ws_opts[5] = {128, 192, 256, 384, 512};
    int ws = 0;
    for (int o : ws_opts) if (o >= window) { ws = o; break; }
    if (!ws) { *why = "window too large"; return false; }

    for (int a = 0; a < 2; ++a) {
        const RingApertureDesc &D = desc[a];
        RingTables &T = *tabs[a];
        if (D.n_tx == 0) { T.n_tiles = 0; continue; }
        Geo G{&D, pitch, c, fs, t_start};
        const Tiling &L = til[a];
        T.n_tiles = L.n_tiles(); T.tx = L.tx; T.tz = L.tz; T.tiles_x = L.tiles_x; T.tiles_z = L.tiles_z;
        std::vector<int> s0((size_t)T.n_tiles * D.n_rx * D.n_tx);
        size_t i = 0;
        for (int tzi = 0; tzi < L.tiles_z; ++tzi)
            for (int txi = 0; txi < L.tiles_x; ++txi) {
                const int ix0 = txi * L.tx, ix1 = std::min(D.n_lat, ix0 + L.tx) - 1;
                const int iz0 = tzi * L.tz, iz1 = std::min(D.n_ax, iz0 + L.tz) - 1;
                for (int j = 0; j < D.n_rx; ++j)
                    for (int k = 0; k < D.n_tx; ++k, ++i) {
                        double lo, hi;
                        G.range(ix0, ix1, iz0, iz1, k, j, lo, hi);
                        int rel = (int)std::floor(lo) - 2 - n_lo;
                        rel = std::max(0, std::min(rel, l_row - window));
                        s0[i] = rel;
                    }
            }
        if (cudaMalloc(&T.d_s0, s0.size() * sizeof(int)) != cudaSuccess) { *why = "table allocation failed"; return false; }
        if (cudaMemcpy(T.d_s0, s0.data(), s0.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess) {
            *why = "table upload failed";
            return false;
        }
    }
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cfg.frames = 8;
    cfg.tile_pixels = kRingTilePixels;
    cfg.window = window;
    cfg.ws = ws;
    cfg.n_sms = sms;
    const int misc = kRingMaxBt * 4 + 3 * kRingMaxRx * 4 + kRingMaxStages * 16 + 2 * kRingMaxStages * 8 + 64;
    cfg.stages = std::min(kRingMaxStages, (kSmemLimit - misc) / (8 * ws * 16));
    cfg.smem_bytes = cfg.stages * 8 * ws * 16 + misc;
    if (cfg.stages < 2) { *why = "fewer than two ring stages fit in shared memory"; return false; }
    return true;
}

template <int F, int WS, bool APOD>
inline int ring_launch_t(const RingConfig &cfg, RingLaunch &L, cudaStream_t st) {
    const int misc = kRingMaxBt * 4 + 3 * kRingMaxRx * 4 + kRingMaxStages * 16 + 2 * kRingMaxStages * 8 + 64;
    const int stages = std::min(kRingMaxStages, (kSmemLimit - misc) / (F * WS * 16));
    const int smem = stages * F * WS * 16 + misc;
    L.n_stages = stages;
    L.n_groups = (L.n_frames + F - 1) / F;
    L.n_work = L.n_groups * (L.ap[0].n_tiles + L.ap[1].n_tiles);
    if (L.n_work == 0) return 0;
    static bool attr_set = false;
    if (!attr_set) {
        cudaFuncSetAttribute(das_ring_kernel<F, WS, APOD>, cudaFuncAttributeMaxDynamicSharedMemorySize, kSmemLimit);
        attr_set = true;
    }
    const int grid = std::min(L.n_work, cfg.n_sms);
    das_ring_kernel<F, WS, APOD><<<grid, kRingThreads, smem, st>>>(L);
    return 1;
}

template <int F, bool APOD>
inline int ring_launch_ws(const RingConfig &cfg, RingLaunch &L, cudaStream_t st) {
    switch (cfg.ws) {
        case 128: return ring_launch_t<F, 128, APOD>(cfg, L, st);
        case 192: return ring_launch_t<F, 192, APOD>(cfg, L, st);
        case 256: return ring_launch_t<F, 256, APOD>(cfg, L, st);
        case 384: return ring_launch_t<F, 384, APOD>(cfg, L, st);
        default: return ring_launch_t<F, 512, APOD>(cfg, L, st);
    }
}

// returns the number of kernels launched
inline int ring_launch(const RingConfig &cfg, const RingTables &tab0, const RingTables &tab1, const RingLaunch &Lin,
                       bool apod, cudaStream_t st) {
    RingLaunch L = Lin;
    const RingTables *tabs[2] = {&tab0, &tab1};
    for (int a = 0; a < 2; ++a) {
        L.ap[a].s0 = tabs[a]->d_s0;
        L.ap[a].n_tiles = L.ap[a].n_tx > 0 ? tabs[a]->n_tiles : 0;
        L.ap[a].tx = tabs[a]->tx; L.ap[a].tz = tabs[a]->tz; L.ap[a].tiles_x = std::max(1, tabs[a]->tiles_x);
    }
    L.window = cfg.window;
    if (L.n_frames > 2)
        return apod ? ring_launch_ws<8, true>(cfg, L, st) : ring_launch_ws<8, false>(cfg, L, st);
    return apod ? ring_launch_ws<2, true>(cfg, L, st) : ring_launch_ws<2, false>(cfg, L, st);
}

}  // namespace ulm
