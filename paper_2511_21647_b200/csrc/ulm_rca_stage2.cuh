// ulm_rca_stage2.cuh -- Stage-2 beamforming fused with compounding over all 2K events and the P-block
// sum-projection (reading = DESIGN.md section 11) for sm_100a.  The N^3 volume never exists:
// the kernel goes from the per-event slices S_k (the compound = 0 output of Stage 1, or its clutter-filtered
// version) straight to the 2 N/P projected planes.
//
// Definition (restated from DESIGN.md 11): voxel (lat, w, z_i) of event k -- lat = the slice's lateral axis, w = the
// transmit direction, ref = the slice's position along w -- is
//     V_k = T_k(i) Y_k(w) [ (1 - b) B_k(lat, i + n) + b B_k(lat, i + n + 1) ],   B_k(lat, i') = S_k(lat, i') conj(T_k(i')),
//     n + b = (w - ref) tan(th_k / 2) / dz,  Y_k(w) = exp(j 2 pi fc (w - ref) sin(th_k) / c),
//     T_k(i) = exp(j 2 pi fc tau0_k(z_i)),  tau0_k linear in z with slope (1 + cos th_k)/c,  B_k = 0 outside the grid,
// V = sum over all events, XZ_m(x, z) = sum_{y in group m} V, YZ_m(y, z) = sum_{x in group m} V.
//
// Factoring used here (exact regrouping, nothing approximated beyond the definition):
//  * T_k(i) conj(T_k(i + s)) = exp(-j 2 pi fc s dz (1 + cos th_k)/c) depends on the tap offset s only, so the carrier
//    removal / restoration folds into constant complex tap weights and the slices are used as they are;
//  * "own" part of a plane set (XZ planes <- RC slices, YZ planes <- CR slices): the sum over the P transmit-direction
//    positions of a group touches at most NT consecutive depths, so it is ONE complex FIR along z per (event, group),
//    taps W[k][m][t] built in fp64 on the host:  plane_m(lat, i) += sum_t W[k][m][t] S_k(lat, i + o[k][m] + t);
//  * "cross" part (XZ planes <- CR slices, YZ planes <- RC slices): the grouped axis is the slice's own lateral axis, so
//    the slice columns of a group are summed FIRST (stage2_groupsum_kernel, G[k][m][z]) and each plane column is a
//    two-tap interpolation of that sum:  plane_m(lat, i) += c0[k][lat] G_km(i + n[k][lat]) + c1[k][lat] G_km(i + n + 1).
// Per output value that is 3 + 2 complex multiply-adds per event instead of P interpolations + rotations.
//
// Kernel mapping: CTA = (frame, plane set, 32 lateral positions, 24 depths, block of 8 groups); warp = one group m,
// lane = one lateral position, thread = 3 chunks of 8 consecutive depths (a register window of 8 + NT - 1 slice values
// per chunk feeds 8 NT multiply-adds).  The slice tile of event k + 1 (zero-extended halo included) is fetched into
// registers while event k is computed from shared memory (two buffers, one barrier per event); rows are padded to an
// odd stride so the 32 lanes of a warp read 32 different bank pairs.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

constexpr int kS2Lat = 32;        // lateral positions per CTA (= lanes)
constexpr int kS2Chunks = 3;      // chunks of 8 depths per thread
constexpr int kS2Zt = 8 * kS2Chunks;
constexpr int kS2Warps = 8;       // groups per CTA
constexpr int kS2Threads = 32 * kS2Warps;
constexpr int kS2MaxCol = 96;     // tile columns (kS2Zt + halo) at most
constexpr int kS2MaxTaps = 8;

struct Stage2Set {
    int n_lat, n_w, n_g;           // plane width, size of the grouped (summed) axis, number of groups
    int own_n, cross_n;            // events whose slices have this set's lateral axis / the grouped axis as lateral axis
    long long own_off, cross_goff; // float2 offset of own event 0's slice inside a frame of slices; event index of
                                   // cross event 0 in the group-sum array
    const int *own_o;              // [own_n][n_g] first tap offset
    const float2 *own_w;           // [own_n][n_g][NT]
    const int *cross_o;            // [cross_n][n_lat]
    const float2 *cross_w;         // [cross_n][n_lat][2]
    long long out_off;             // float2 offset of the set's planes inside a frame of planes
};

struct Stage2Params {
    const float2 *slices;          // [frame][event][lat][z]
    long long slices_per_frame;
    const float2 *gsum;            // [frame][event][g_max][z]   (stage2_groupsum_kernel)
    int n_events, g_max, n_z;
    float2 *planes;
    long long planes_per_frame;
    int n_frames;
    int halo_lo, ncol, rs;         // tile: columns = depths z0 - halo_lo .. z0 - halo_lo + ncol - 1; row stride (odd)
    int z_tiles;
    Stage2Set set[2];
};

struct GroupSumParams {
    const float2 *slices;
    long long slices_per_frame;
    float2 *gsum;
    int n_events, g_max, n_z, block, n_frames;
    int n_row_tx;                  // events [0, n_row_tx) have n_lat0 lateral positions, the rest n_lat1
    int n_lat0, n_lat1;
};

// G[f][e][g][z] = sum of the slice columns of group g (P consecutive lateral positions) of event e
__global__ void __launch_bounds__(256) stage2_groupsum_kernel(const __grid_constant__ GroupSumParams P) {
    const long long per_event = (long long)P.g_max * P.n_z;
    const long long n = (long long)P.n_frames * P.n_events * per_event;
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    const int z = (int)(i % P.n_z);
    const int g = (int)((i / P.n_z) % P.g_max);
    const int e = (int)((i / per_event) % P.n_events);
    const long long f = i / (per_event * P.n_events);
    const bool first = e < P.n_row_tx;
    const int n_lat = first ? P.n_lat0 : P.n_lat1;
    const long long off = first ? (long long)e * P.n_lat0 * P.n_z
                                : (long long)P.n_row_tx * P.n_lat0 * P.n_z + (long long)(e - P.n_row_tx) * P.n_lat1 * P.n_z;
    const float2 *s = P.slices + f * P.slices_per_frame + off;
    float2 acc = make_float2(0.f, 0.f);
    const int l0 = g * P.block, l1 = min(l0 + P.block, n_lat);
    for (int l = l0; l < l1; ++l) {
        const float2 v = __ldg(s + (long long)l * P.n_z + z);
        acc.x += v.x; acc.y += v.y;
    }
    P.gsum[i] = acc;
}

#define ULM_S2(field) (a ? P.set[1].field : P.set[0].field)

__device__ __forceinline__ void cmac(float2 &acc, const float2 w, const float2 v) {
    acc.x = fmaf(w.x, v.x, acc.x); acc.x = fmaf(-w.y, v.y, acc.x);
    acc.y = fmaf(w.x, v.y, acc.y); acc.y = fmaf(w.y, v.x, acc.y);
}

template <int NT>
__global__ void __launch_bounds__(kS2Threads, 2) stage2_project_kernel(const __grid_constant__ Stage2Params P) {
    extern __shared__ __align__(16) unsigned char s2_smem[];
    const int a = blockIdx.z & 1, f = blockIdx.z >> 1;
    const int n_lat = ULM_S2(n_lat), n_g = ULM_S2(n_g);
    const int lat0 = blockIdx.x * kS2Lat;
    const int zt = blockIdx.y % P.z_tiles, mb = blockIdx.y / P.z_tiles;
    if (lat0 >= n_lat || mb * kS2Warps >= n_g) return;           // block-uniform
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m = mb * kS2Warps + warp;
    const bool m_ok = m < n_g;
    const int lat = min(lat0 + lane, n_lat - 1);
    const int z0 = zt * kS2Zt;
    const int ncol = P.ncol, rs = P.rs, n_z = P.n_z;
    float2 *tile = reinterpret_cast<float2 *>(s2_smem);          // [2][kS2Lat][rs]   own slices
    float2 *gt = tile + 2 * kS2Lat * rs;                          // [2][kS2Warps][ncol] group sums (cross part)

    float2 acc[kS2Chunks][8];
#pragma unroll
    for (int c = 0; c < kS2Chunks; ++c)
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[c][q] = make_float2(0.f, 0.f);

    // ------------------------------ own part: a complex FIR along z per (event, group) ------------------------------
    {
        const int own_n = ULM_S2(own_n);
        const float2 *src0 = P.slices + (long long)f * P.slices_per_frame + ULM_S2(own_off);
        // thread (row = t / 8, column lane = t % 8) fetches columns cl, cl + 8, ... of its row: no index division
        constexpr int PF = kS2MaxCol / 8;                                           // prefetch registers per thread
        const int row = threadIdx.x >> 3, cl = threadIdx.x & 7;
        const bool row_ok = lat0 + row < n_lat;
        float2 pre[PF];
        auto fetch = [&](int k) {
            const float2 *src = src0 + ((long long)k * n_lat + min(lat0 + row, n_lat - 1)) * n_z;
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const int col = cl + 8 * r;
                const int z = z0 - P.halo_lo + col;
                float2 v = make_float2(0.f, 0.f);
                if (col < ncol && row_ok && z >= 0 && z < n_z) v = __ldg(src + z);     // zero extension
                pre[r] = v;
            }
        };
        auto stash = [&](int buf) {
            float2 *dst = tile + buf * kS2Lat * rs + row * rs;
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const int col = cl + 8 * r;
                if (col < ncol) dst[col] = pre[r];
            }
        };
        if (own_n > 0) { fetch(0); stash(0); }
        __syncthreads();
        const int *own_o = ULM_S2(own_o);
        const float2 *own_w = ULM_S2(own_w);
        for (int k = 0; k < own_n; ++k) {
            if (k + 1 < own_n) fetch(k + 1);
            if (m_ok) {
                const int o = __ldg(own_o + k * n_g + m) + P.halo_lo;
                float2 w[NT];
#pragma unroll
                for (int t = 0; t < NT; ++t) w[t] = __ldg(own_w + ((long long)k * n_g + m) * NT + t);
                const float2 *base = tile + (k & 1) * kS2Lat * rs + lane * rs + o;
#pragma unroll
                for (int c = 0; c < kS2Chunks; ++c) {
                    float2 win[8 + NT - 1];
#pragma unroll
                    for (int q = 0; q < 8 + NT - 1; ++q) win[q] = base[c * 8 + q];
#pragma unroll
                    for (int q = 0; q < 8; ++q)
#pragma unroll
                        for (int t = 0; t < NT; ++t) cmac(acc[c][q], w[t], win[q + t]);
                }
            }
            if (k + 1 < own_n) stash((k + 1) & 1);
            __syncthreads();
        }
    }

    // ------------------------------ cross part: two-tap interpolation of the group sums ------------------------------
    {
        const int cross_n = ULM_S2(cross_n);
        // thread (row = warp, column lane) fetches columns lane, lane + 32, ... of the group-sum row of its own group
        constexpr int PF = kS2MaxCol / 32;
        float2 pre[PF];
        const float2 *g0 = P.gsum + ((long long)f * P.n_events + ULM_S2(cross_goff)) * P.g_max * n_z;
        auto fetch = [&](int k) {
            const float2 *src = g0 + ((long long)k * P.g_max + min(m, n_g - 1)) * n_z;
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const int col = lane + 32 * r;
                const int z = z0 - P.halo_lo + col;
                float2 v = make_float2(0.f, 0.f);
                if (col < ncol && m_ok && z >= 0 && z < n_z) v = __ldg(src + z);
                pre[r] = v;
            }
        };
        auto stash = [&](int buf) {
            float2 *dst = gt + buf * kS2Warps * ncol + warp * ncol;
#pragma unroll
            for (int r = 0; r < PF; ++r) {
                const int col = lane + 32 * r;
                if (col < ncol) dst[col] = pre[r];
            }
        };
        if (cross_n > 0) { fetch(0); stash(0); }
        __syncthreads();
        const int *cross_o = ULM_S2(cross_o);
        const float2 *cross_w = ULM_S2(cross_w);
        for (int k = 0; k < cross_n; ++k) {
            if (k + 1 < cross_n) fetch(k + 1);
            if (m_ok) {
                const int o = __ldg(cross_o + k * n_lat + lat) + P.halo_lo;
                const float4 cw = __ldg(reinterpret_cast<const float4 *>(cross_w) + (long long)k * n_lat + lat);
                const float2 c0 = make_float2(cw.x, cw.y), c1 = make_float2(cw.z, cw.w);
                const float2 *base = gt + (k & 1) * kS2Warps * ncol + warp * ncol + o;
#pragma unroll
                for (int c = 0; c < kS2Chunks; ++c) {
                    float2 win[9];
#pragma unroll
                    for (int q = 0; q < 9; ++q) win[q] = base[c * 8 + q];
#pragma unroll
                    for (int q = 0; q < 8; ++q) { cmac(acc[c][q], c0, win[q]); cmac(acc[c][q], c1, win[q + 1]); }
                }
            }
            if (k + 1 < cross_n) stash((k + 1) & 1);
            __syncthreads();
        }
    }

    // ------------------------------ projected planes: [frame][set][m][lat][z], z fastest ------------------------------
    if (m_ok && lat0 + lane < n_lat) {
        float2 *dst = P.planes + (long long)f * P.planes_per_frame + ULM_S2(out_off) + ((long long)m * n_lat + lat) * n_z;
        const bool vec = ((n_z & 1) == 0) && ((ULM_S2(out_off) & 1) == 0) && ((P.planes_per_frame & 1) == 0) &&
                         ((reinterpret_cast<unsigned long long>(P.planes) & 15ull) == 0);
#pragma unroll
        for (int c = 0; c < kS2Chunks; ++c) {
            const int zb = z0 + c * 8;
            if (vec && zb + 8 <= n_z) {
#pragma unroll
                for (int q = 0; q < 8; q += 2)
                    *reinterpret_cast<float4 *>(dst + zb + q) = make_float4(acc[c][q].x, acc[c][q].y, acc[c][q + 1].x, acc[c][q + 1].y);
            } else {
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    if (zb + q < n_z) dst[zb + q] = acc[c][q];
            }
        }
    }
}

#undef ULM_S2

}  // namespace ulm
