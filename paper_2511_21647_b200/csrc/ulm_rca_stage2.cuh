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
// Kernel mapping: CTA = (frame, plane set, 32 lateral positions, block of 8 groups), walking the depth tiles of 16
// depths; warp = one group m, lane = one lateral position, thread = 2 chunks of 8 consecutive depths (a register window
// of 8 + NT - 1 slice values per chunk feeds 8 NT complex multiply-adds as FFMA2).  A stage = the slice tiles of two
// events (zero-extended halo included), brought in with 8-byte LDGSTS two stages ahead through three buffers (one
// barrier per stage); the stage stream runs across depth-tile boundaries; rows are padded to an odd stride so the 32
// lanes of a warp read 32 different bank pairs.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

constexpr int kS2Lat = 32;        // lateral positions per CTA (= lanes)
constexpr int kS2Chunks = 2;      // chunks of 8 depths per thread
constexpr int kS2Stages = 3;      // shared-memory buffers of the asynchronous tile pipeline
constexpr int kS2Ev = 2;          // events per stage (one barrier per stage)
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
    int z_tiles, tiles_per_cta;    // depth tiles of kS2Zt depths; consecutive tiles one CTA walks
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

// packed fp32x2 helpers (FFMA2: two fp32 FMAs per issue slot)
__device__ __forceinline__ unsigned long long s2_pack(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void s2_unpack(unsigned long long v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long s2_ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long s2_lds64(uint32_t addr) {
    unsigned long long v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}
// 8-byte asynchronous copy global -> shared (LDGSTS); ok == false writes zeros (the zero extension of the slices)
__device__ __forceinline__ void s2_cp_async8(uint32_t dst, const void *src, bool ok) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(ok ? 8u : 0u) : "memory");
}
__device__ __forceinline__ void s2_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void s2_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// A complex multiply-accumulate acc += w v needs the swapped pair (v.im, v.re) in the packed form; instead two packed
// accumulators are kept, A += (w.re, w.re) (v.re, v.im) and B += (w.im, w.im) (v.re, v.im), and combined at the very
// end: acc = (A.lo - B.hi, A.hi + B.lo).  Two FFMA2 per complex multiply-add, no data shuffling.
// Per-stage overhead is kept to a few instructions: the tap tables of the CTA's 8 groups / 32 lateral positions are
// copied to shared memory once per CTA, every thread forms its fill pointers and in-range masks once per depth tile, and
// a stage's fill is a handful of predicated 8-byte LDGSTS with immediate offsets (size 0 = zero fill where the depth
// lies outside the grid).
template <int NT>
__global__ void __launch_bounds__(kS2Threads, 2) stage2_project_kernel(const __grid_constant__ Stage2Params P) {
    extern __shared__ __align__(16) unsigned char s2_smem[];
    const int a = blockIdx.z & 1, f = blockIdx.z >> 1;
    const int n_lat = ULM_S2(n_lat), n_g = ULM_S2(n_g);
    const int lat0 = blockIdx.x * kS2Lat;
    // blockIdx.y = (group block, run of tiles_per_cta consecutive depth tiles)
    const int z_runs = (P.z_tiles + P.tiles_per_cta - 1) / P.tiles_per_cta;
    const int mb = blockIdx.y / z_runs;
    const int zt_begin = (blockIdx.y - mb * z_runs) * P.tiles_per_cta, zt_end = min(zt_begin + P.tiles_per_cta, P.z_tiles);
    if (lat0 >= n_lat || mb * kS2Warps >= n_g) return;           // block-uniform
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int m = mb * kS2Warps + warp;
    const bool m_ok = m < n_g;
    const int lat = min(lat0 + lane, n_lat - 1);
    const int ncol = P.ncol, rs = P.rs, n_z = P.n_z;
    const int own_n = ULM_S2(own_n), cross_n = ULM_S2(cross_n);
    // stages of a depth tile: the own events kS2Ev at a time, then the cross events kS2Ev at a time
    const int st_own = (own_n + kS2Ev - 1) / kS2Ev, n_st = st_own + (cross_n + kS2Ev - 1) / kS2Ev;
    // shared memory: kS2Stages buffers of {kS2Ev own slice tiles [kS2Lat][rs], kS2Ev group-sum tiles [kS2Warps][ncol]}, then the tap
    // tables: own [own_n][kS2Warps][1 + NT] float2 ({offset bits, -}, taps), cross [cross_n][kS2Lat][3] float2
    const int own_tile = kS2Lat * rs, gs_tile = kS2Warps * ncol;
    const int buf_elems = kS2Ev * (own_tile + gs_tile);
    float2 *smem = reinterpret_cast<float2 *>(s2_smem);
    float2 *tab_own = smem + kS2Stages * buf_elems;
    float2 *tab_cross = tab_own + own_n * kS2Warps * (1 + NT);
    const uint32_t smem_u = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t smem_end = smem_u + (uint32_t)(kS2Stages * buf_elems) * 8u;
    {
        const int *own_o = ULM_S2(own_o), *cross_o = ULM_S2(cross_o);
        const float2 *own_w = ULM_S2(own_w), *cross_w = ULM_S2(cross_w);
        for (int i = threadIdx.x; i < own_n * kS2Warps; i += kS2Threads) {
            const int k = i / kS2Warps, g = min(mb * kS2Warps + (i - k * kS2Warps), n_g - 1);
            float2 *d = tab_own + i * (1 + NT);
            d[0] = make_float2(__int_as_float(__ldg(own_o + k * n_g + g) + P.halo_lo), 0.f);
            for (int tt = 0; tt < NT; ++tt) d[1 + tt] = __ldg(own_w + ((long long)k * n_g + g) * NT + tt);
        }
        for (int i = threadIdx.x; i < cross_n * kS2Lat; i += kS2Threads) {
            const int k = i / kS2Lat, l = min(lat0 + (i - k * kS2Lat), n_lat - 1);
            float2 *d = tab_cross + i * 3;
            d[0] = make_float2(__int_as_float(__ldg(cross_o + k * n_lat + l) + P.halo_lo), 0.f);
            d[1] = __ldg(cross_w + ((long long)k * n_lat + l) * 2);
            d[2] = __ldg(cross_w + ((long long)k * n_lat + l) * 2 + 1);
        }
    }

    // ---- fill side: a CTA walks all depth tiles of its (frame, plane set, lateral tile, group block); the stage stream
    // (depth tile, stage) is filled kS2Stages - 1 stages ahead of the compute side and runs across tile boundaries.
    // Own tile: thread (row = t / 8, cl = t % 8) copies columns cl + 8 r of its row; group-sum tile: thread (row = warp,
    // lane) copies columns lane + 32 r of its group's row.  Bit r of exist_* = the column exists, bit r of in_* = its
    // depth lies inside the grid (otherwise the copy writes zeros: the zero extension of the slices).
    constexpr int RO = kS2MaxCol / 8, RC = kS2MaxCol / 32;
    const int frow = threadIdx.x >> 3, fcl = threadIdx.x & 7;
    const bool frow_ok = lat0 + frow < n_lat;
    uint32_t exist_o = 0, exist_c = 0, in_o = 0, in_c = 0;
#pragma unroll
    for (int r = 0; r < RO; ++r) if (fcl + 8 * r < ncol) exist_o |= 1u << r;
#pragma unroll
    for (int r = 0; r < RC; ++r) if (lane + 32 * r < ncol) exist_c |= 1u << r;
    const float2 *row_o = P.slices + (long long)f * P.slices_per_frame + ULM_S2(own_off) +
                          (long long)min(lat0 + frow, n_lat - 1) * n_z + fcl;
    const float2 *row_c = P.gsum + ((long long)f * P.n_events + ULM_S2(cross_goff)) * P.g_max * n_z +
                          (long long)min(m, n_g - 1) * n_z + lane;
    const long long step_o = (long long)n_lat * n_z, step_c = (long long)P.g_max * n_z;
    const uint32_t dst_o = (uint32_t)(frow * rs + fcl) * 8u, dst_c = (uint32_t)(kS2Ev * own_tile + warp * ncol + lane) * 8u;
    int zt_issue = zt_begin, s_issue = 0;
    uint32_t buf_issue = smem_u;
    const float2 *src_o = row_o, *src_c = row_c;
    auto start_tile = [&](int zt) {
        const int zb = zt * kS2Zt - P.halo_lo;
        in_o = in_c = 0;
#pragma unroll
        for (int r = 0; r < RO; ++r) { const int z = zb + fcl + 8 * r; if (frow_ok && z >= 0 && z < n_z) in_o |= 1u << r; }
#pragma unroll
        for (int r = 0; r < RC; ++r) { const int z = zb + lane + 32 * r; if (m_ok && z >= 0 && z < n_z) in_c |= 1u << r; }
        in_o &= exist_o;
        in_c &= exist_c;
        src_o = row_o + zb;
        src_c = row_c + zb;
    };
    start_tile(zt_begin);
    // Zero extension: the buffers are cleared once, so columns outside the grid need no work while a CTA stays on its
    // first depth tile; a later tile whose window leaves the grid (only the last ones do) overwrites what earlier tiles
    // left in those columns with explicit zero stores (zero_o / zero_c, normally 0).
    uint32_t zero_o = 0, zero_c = 0;
    auto issue = [&]() {
        if (zt_issue < zt_end) {
            if (s_issue < st_own) {
#pragma unroll
                for (int u = 0; u < kS2Ev; ++u) {
                    if (s_issue * kS2Ev + u < own_n) {
                        const uint32_t d = buf_issue + dst_o + (uint32_t)(u * own_tile) * 8u;
#pragma unroll
                        for (int r = 0; r < RO; ++r)
                            if (in_o & (1u << r)) s2_cp_async8(d + r * 64u, src_o + 8 * r, true);
                        if (zero_o)
                            for (int r = 0; r < RO; ++r)
                                if (zero_o & (1u << r)) smem[(d - smem_u) / 8u + 8 * r] = make_float2(0.f, 0.f);
                        src_o += step_o;
                    }
                }
            } else {
#pragma unroll
                for (int u = 0; u < kS2Ev; ++u) {
                    if ((s_issue - st_own) * kS2Ev + u < cross_n) {
                        const uint32_t d = buf_issue + dst_c + (uint32_t)(u * gs_tile) * 8u;
#pragma unroll
                        for (int r = 0; r < RC; ++r)
                            if (in_c & (1u << r)) s2_cp_async8(d + r * 256u, src_c + 32 * r, true);
                        if (zero_c)
                            for (int r = 0; r < RC; ++r)
                                if (zero_c & (1u << r)) smem[(d - smem_u) / 8u + 32 * r] = make_float2(0.f, 0.f);
                        src_c += step_c;
                    }
                }
            }
            if (++s_issue == n_st) {
                s_issue = 0;
                ++zt_issue;
                start_tile(zt_issue);
                zero_o = exist_o & ~in_o;
                zero_c = exist_c & ~in_c;
            }
        }
        s2_commit();
        buf_issue += (uint32_t)buf_elems * 8u;
        if (buf_issue == smem_end) buf_issue = smem_u;
    };
    for (int i = threadIdx.x; i < kS2Stages * buf_elems; i += kS2Threads) smem[i] = make_float2(0.f, 0.f);
    __syncthreads();                                               // tables in place
#pragma unroll
    for (int s = 0; s < kS2Stages - 1; ++s) issue();

    float2 *out_col = P.planes + (long long)f * P.planes_per_frame + ULM_S2(out_off) + ((long long)min(m, n_g - 1) * n_lat + lat) * n_z;
    const bool store_ok = m_ok && lat0 + lane < n_lat;
    const bool vec = ((n_z & 1) == 0) && ((ULM_S2(out_off) & 1) == 0) && ((P.planes_per_frame & 1) == 0) &&
                     ((reinterpret_cast<unsigned long long>(P.planes) & 15ull) == 0);
    uint32_t buf = smem_u;
    for (int zt = zt_begin; zt < zt_end; ++zt) {
        // A += (w.re, w.re) (v.re, v.im), B += (w.im, w.im) (v.re, v.im); acc = (A.lo - B.hi, A.hi + B.lo) at the end
        unsigned long long accA[kS2Chunks][8], accB[kS2Chunks][8];
#pragma unroll
        for (int c = 0; c < kS2Chunks; ++c)
#pragma unroll
            for (int q = 0; q < 8; ++q) accA[c][q] = accB[c][q] = 0ull;
        for (int s = 0; s < n_st; ++s) {
            s2_wait<kS2Stages - 2>();
            __syncthreads();                       // this stage has landed; every warp is done with the previous one
            issue();                               // refills the buffer the previous stage used
            if (m_ok) {
                if (s < st_own) {
#pragma unroll
                    for (int u = 0; u < kS2Ev; ++u) {
                        const int ev = s * kS2Ev + u;
                        if (ev < own_n) {
                            const float2 *tb = tab_own + (ev * kS2Warps + warp) * (1 + NT);
                            const int o = __float_as_int(tb[0].x);
                            unsigned long long WR[NT], WI[NT];
#pragma unroll
                            for (int t2 = 0; t2 < NT; ++t2) { const float2 w = tb[1 + t2]; WR[t2] = s2_pack(w.x, w.x); WI[t2] = s2_pack(w.y, w.y); }
                            const uint32_t base = buf + (uint32_t)(u * own_tile + lane * rs + o) * 8u;
#pragma unroll
                            for (int c = 0; c < kS2Chunks; ++c) {
                                unsigned long long win[8 + NT - 1];
#pragma unroll
                                for (int q = 0; q < 8 + NT - 1; ++q) win[q] = s2_lds64(base + (c * 8 + q) * 8u);
#pragma unroll
                                for (int q = 0; q < 8; ++q)
#pragma unroll
                                    for (int t2 = 0; t2 < NT; ++t2) {
                                        accA[c][q] = s2_ffma2(WR[t2], win[q + t2], accA[c][q]);
                                        accB[c][q] = s2_ffma2(WI[t2], win[q + t2], accB[c][q]);
                                    }
                            }
                        }
                    }
                } else {
#pragma unroll
                    for (int u = 0; u < kS2Ev; ++u) {
                        const int ev = (s - st_own) * kS2Ev + u;
                        if (ev < cross_n) {
                            const float2 *tb = tab_cross + (ev * kS2Lat + lane) * 3;
                            const int o = __float_as_int(tb[0].x);
                            unsigned long long WR[2], WI[2];
#pragma unroll
                            for (int t2 = 0; t2 < 2; ++t2) { const float2 w = tb[1 + t2]; WR[t2] = s2_pack(w.x, w.x); WI[t2] = s2_pack(w.y, w.y); }
                            const uint32_t base = buf + (uint32_t)(kS2Ev * own_tile + u * gs_tile + warp * ncol + o) * 8u;
#pragma unroll
                            for (int c = 0; c < kS2Chunks; ++c) {
                                unsigned long long win[9];
#pragma unroll
                                for (int q = 0; q < 9; ++q) win[q] = s2_lds64(base + (c * 8 + q) * 8u);
#pragma unroll
                                for (int q = 0; q < 8; ++q)
#pragma unroll
                                    for (int t2 = 0; t2 < 2; ++t2) {
                                        accA[c][q] = s2_ffma2(WR[t2], win[q + t2], accA[c][q]);
                                        accB[c][q] = s2_ffma2(WI[t2], win[q + t2], accB[c][q]);
                                    }
                            }
                        }
                    }
                }
            }
            buf += (uint32_t)buf_elems * 8u;
            if (buf == smem_end) buf = smem_u;
        }
        // projected planes: [frame][set][m][lat][z], z fastest
        if (store_ok) {
            const int z0 = zt * kS2Zt;
#pragma unroll
            for (int c = 0; c < kS2Chunks; ++c) {
                const int zb = z0 + c * 8;
                float2 v[8];
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    float ar, ai, br, bi;
                    s2_unpack(accA[c][q], ar, ai);
                    s2_unpack(accB[c][q], br, bi);
                    v[q] = make_float2(ar - bi, ai + br);
                }
                if (vec && zb + 8 <= n_z) {
#pragma unroll
                    for (int q = 0; q < 8; q += 2)
                        *reinterpret_cast<float4 *>(out_col + zb + q) = make_float4(v[q].x, v[q].y, v[q + 1].x, v[q + 1].y);
                } else {
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        if (zb + q < n_z) out_col[zb + q] = v[q];
                }
            }
        }
    }
    s2_wait<0>();
}

#undef ULM_S2

}  // namespace ulm
