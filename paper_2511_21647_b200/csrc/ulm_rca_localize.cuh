// ulm_rca_localize.cuh -- 2-D NCC microbubble localization on the projected planes (reading =
// DESIGN.md section 14) for sm_100a, evaluated separably as the paper does (Fig. 1g: "conventional 2D NCC is accelerated
// using two 1D separable correlations", 11-tap kernels).
//
//   LO-1  B = |V_p| of one plane (0 outside), template g(a, b) = g1(a) g2(b), 11 x 11 Gaussian
//   LO-2  ncc(p) = sum_W (B - Bm)(g - gm) / sqrt(sum_W (B - Bm)^2 sum_W (g - gm)^2)
//         = (S_g - gm S_1) / sqrt((S_2 - S_1^2 / 121) G),   S_g = sum_W B g, S_1 = sum_W B, S_2 = sum_W B^2:
//         three separable correlations = two 11-tap 1-D passes each (along depth, then along the lateral axis).  The sums
//         are taken on B - c, c = the value at the tile centre: the map does not depend on an offset, and the
//         subtraction S_2 - S_1^2 / 121 then cancels far fewer digits in fp32.
//   LO-3  candidates: interior pixels with B >= threshold_rel * (maximum of B over all planes of the frame) and
//         ncc >= ncc_min that are regional peaks (> the 4 neighbours that follow in row-major order, >= the 4 before)
//   LO-4  3-point parabola along each axis on the NCC map -> (lat + dl, ax + di, ncc, B)
//
// localize_max_kernel: per-frame maximum of |V| (the paper uses a Thrust reduction).  localize_kernel: CTA = one tile of
// 32 x 64 pixels of one plane; tile + halo in shared memory, row pass, column pass, peak test; localizations are appended
// to the plane's list with an atomic counter (their order inside a plane is therefore not fixed; the set is).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

constexpr int kLoHalf = 5, kLoTaps = 11;
constexpr int kLoTl = 32, kLoTa = 64;                 // tile: lateral x axial
constexpr int kLoHalo = kLoHalf + 1;                  // + 1: the NCC map is needed one pixel around the tile
constexpr int kLoBl = kLoTl + 2 * kLoHalo, kLoBa = kLoTa + 2 * kLoHalo;       // B tile 44 x 76
constexpr int kLoRa = kLoTa + 2;                      // after the depth pass: 44 x 66
constexpr int kLoNl = kLoTl + 2;                      // NCC tile 34 x 66
constexpr int kLoBs = kLoBa + 1, kLoRs = kLoRa + 1;   // odd row strides: the lanes of the depth pass walk over rows
constexpr int kLoSeg = 6;                             // depth pass: outputs per thread (66 = 11 segments of 6)
constexpr int kLoBlk = 12;                            // lateral pass: outputs per thread at most (34 = 12 + 11 + 11)
constexpr int kLoThreads = 256;
constexpr int kLoSmem = (kLoBl * kLoBs + 3 * kLoBl * kLoRs) * 4;     // the NCC tile reuses the B tile
static_assert(kLoRa % kLoSeg == 0 && kLoBlk == 2 * kLoSeg && kLoNl <= 3 * kLoBlk && kLoNl * kLoRs <= kLoBl * kLoBs, "localize tiling");

struct LoParams {
    const float2 *planes;            // [frame][x-z planes | y-z planes] (layout of ulm_rca_stage2_project)
    long long planes_per_frame;
    int n_frames, n_z;
    int n_planes[2], n_lat[2];       // per plane set
    long long set_off[2];            // float2 offset of the set inside a frame
    float g1[kLoTaps], g2[kLoTaps];  // template factors along the lateral axis / depth
    float g_mean, g_den;             // mean of g and sum (g - gm)^2
    float threshold_rel, ncc_min;
    unsigned int *frame_max;         // [frame] bits of the maximum |V| (non-negative floats order like their bits)
    float4 *loc;                     // [frame][plane][capacity]
    int *count;                      // [frame][plane] number found (may exceed capacity: the surplus is dropped)
    int capacity;
};

__global__ void __launch_bounds__(256) localize_max_kernel(const __grid_constant__ LoParams P) {
    const int f = blockIdx.y;
    const float2 *v = P.planes + (long long)f * P.planes_per_frame;
    float m = 0.f;                   // maximum of |V|^2: the square root is monotone, so it is taken once at the end
    const long long n = P.planes_per_frame, t0 = (long long)blockIdx.x * 256 + threadIdx.x, step = (long long)gridDim.x * 256;
    if (((reinterpret_cast<unsigned long long>(v) & 15ull) == 0) && (n & 1) == 0) {
        const float4 *v4 = reinterpret_cast<const float4 *>(v);
        const long long n4 = n >> 1;
        long long i = t0;
        for (; i + 3 * step < n4; i += 4 * step) {
            float4 x[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) x[u] = __ldg(v4 + i + u * step);
#pragma unroll
            for (int u = 0; u < 4; ++u) m = fmaxf(m, fmaxf(fmaf(x[u].x, x[u].x, x[u].y * x[u].y), fmaf(x[u].z, x[u].z, x[u].w * x[u].w)));
        }
        for (; i < n4; i += step) {
            const float4 x = __ldg(v4 + i);
            m = fmaxf(m, fmaxf(fmaf(x.x, x.x, x.y * x.y), fmaf(x.z, x.z, x.w * x.w)));
        }
    } else {
        for (long long i = t0; i < n; i += step) {
            const float2 x = __ldg(v + i);
            m = fmaxf(m, fmaf(x.x, x.x, x.y * x.y));
        }
    }
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(P.frame_max + f, __float_as_uint(sqrtf(m)));
}

// the kLoSeg = 6 sums of 11 consecutive values inside a run of 16: the six values common to all windows are added once,
// the rest comes from running sums towards either end (25 additions instead of 60, all terms added directly)
__device__ __forceinline__ void lo_box6(const float *b, float *s) {
    const float core = ((b[5] + b[6]) + (b[7] + b[8])) + (b[9] + b[10]);
    float l[6], r[6];
    l[5] = 0.f; r[0] = 0.f;
#pragma unroll
    for (int k = 4; k >= 0; --k) l[k] = k == 4 ? b[4] : l[k + 1] + b[k];
#pragma unroll
    for (int k = 1; k < 6; ++k) r[k] = k == 1 ? b[11] : r[k - 1] + b[10 + k];
#pragma unroll
    for (int k = 0; k < 6; ++k) s[k] = (core + l[k]) + r[k];
}
__device__ __forceinline__ float lo_abs(float2 x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(fmaf(x.x, x.x, x.y * x.y)));
    return r;
}

// grid = (lateral tiles, depth tiles, frames * planes).  Both passes are register-blocked (a thread loads a run of
// kLoSeg + 10 / kLoBlk + 10 values once and forms all the windows inside it), so the shared-memory pipe carries ~20 words per
// pixel instead of ~60; the Gaussian sums tap by tap, the two box sums by lo_box6.
#ifndef ULM_LO_MINB
#define ULM_LO_MINB 4
#endif
__global__ void __launch_bounds__(kLoThreads, ULM_LO_MINB) localize_kernel(const __grid_constant__ LoParams P) {
    extern __shared__ __align__(16) unsigned char lo_smem[];
    float *sB = reinterpret_cast<float *>(lo_smem);                  // [kLoBl][kLoBs]
    float *sR = sB + kLoBl * kLoBs;                                   // [3][kLoBl][kLoRs]  depth-pass sums (g, 1, squares)
    float *sN = sB;                                                   // [kLoNl][kLoRs]     NCC map of the tile + 1 (the B tile is dead by then)
    const int n_pl = P.n_planes[0] + P.n_planes[1];
    const int f = blockIdx.z / n_pl, pl = blockIdx.z - f * n_pl;
    const int a = pl >= P.n_planes[0] ? 1 : 0, m = a ? pl - P.n_planes[0] : pl;
    const int n_lat = a ? P.n_lat[1] : P.n_lat[0], n_z = P.n_z;
    const int l0 = blockIdx.x * kLoTl, i0 = blockIdx.y * kLoTa;
    if (l0 >= n_lat || i0 >= n_z) return;
    const float2 *v = P.planes + (long long)f * P.planes_per_frame + (a ? P.set_off[1] : P.set_off[0]) + (long long)m * n_lat * n_z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // B tile: a warp per row, the lanes along depth (coalesced); all loads of a thread are issued before the first use
    const float2 xc = __ldg(v + (long long)min(l0 + kLoTl / 2, n_lat - 1) * n_z + min(i0 + kLoTa / 2, n_z - 1));
    constexpr int kRows = (kLoBl + 7) / 8, kCols = (kLoBa + 31) / 32;
    float2 x[kRows][kCols];
    const float2 *rowp = v + (long long)(l0 - kLoHalo + warp) * n_z + (i0 - kLoHalo + lane);      // row `warp` of the tile
    bool col_in[kCols];
#pragma unroll
    for (int q = 0; q < kCols; ++q) {
        const int bi = lane + 32 * q, i = i0 - kLoHalo + bi;
        col_in[q] = bi < kLoBa && i >= 0 && i < n_z;
    }
#pragma unroll
    for (int r = 0; r < kRows; ++r) {
        const int bl = warp + 8 * r, l = l0 - kLoHalo + bl;
        const bool row_in = bl < kLoBl && l >= 0 && l < n_lat;
#pragma unroll
        for (int q = 0; q < kCols; ++q) {
            x[r][q] = make_float2(0.f, 0.f);
            if (row_in && col_in[q]) x[r][q] = __ldg(rowp + 32 * q);
        }
        rowp += 8 * (long long)n_z;
    }
    const float c = lo_abs(xc);                                       // offset of this tile: B at its centre
#pragma unroll
    for (int r = 0; r < kRows; ++r) {
        const int bl = warp + 8 * r;
#pragma unroll
        for (int q = 0; q < kCols; ++q) {
            const int bi = lane + 32 * q;
            if (bl < kLoBl && bi < kLoBa) sB[bl * kLoBs + bi] = lo_abs(x[r][q]) - c;
        }
    }
    __syncthreads();
    // depth pass: a thread forms the three 11-tap sums of kLoSeg consecutive depth positions of one row from the
    // kLoSeg + 10 values they span; the lanes of a warp are consecutive rows (odd stride: conflict-free)
    for (int t = threadIdx.x; t < kLoBl * (kLoRa / kLoSeg); t += kLoThreads) {
        const int seg = t / kLoBl, bl = t - seg * kLoBl;
        const float *row = sB + bl * kLoBs + seg * kLoSeg;            // output r: window r .. r + 10 (centre = i0 - 1 + seg * kLoSeg + r)
        float b[kLoSeg + kLoTaps - 1];
#pragma unroll
        for (int k = 0; k < kLoSeg + kLoTaps - 1; ++k) b[k] = row[k];
        float *dst = sR + bl * kLoRs + seg * kLoSeg;
        float s1[kLoSeg], s2[kLoSeg], bb[kLoSeg + kLoTaps - 1];
#pragma unroll
        for (int k = 0; k < kLoSeg + kLoTaps - 1; ++k) bb[k] = b[k] * b[k];
        lo_box6(b, s1);
        lo_box6(bb, s2);
#pragma unroll
        for (int r = 0; r < kLoSeg; ++r) {
            float sg = 0.f;
#pragma unroll
            for (int k = 0; k < kLoTaps; ++k) sg = fmaf(P.g2[k], b[r + k], sg);
            dst[r] = sg; dst[kLoBl * kLoRs + r] = s1[r]; dst[2 * kLoBl * kLoRs + r] = s2[r];
        }
    }
    __syncthreads();
    // lateral pass + NCC for the tile and one pixel around it: a thread owns one depth column and a block of up to
    // kLoBlk lateral positions; the lanes are consecutive depth positions
    if (threadIdx.x < 3 * kLoRa) {
        const int blk = threadIdx.x / kLoRa, ri = threadIdx.x - blk * kLoRa;
        const int nl0 = blk == 0 ? 0 : kLoBlk + (blk - 1) * (kLoBlk - 1);         // blocks of 12, 11, 11 rows
        const int n_out = blk == 0 ? kLoBlk : kLoBlk - 1;
        float o[3][kLoBlk];
#pragma unroll
        for (int q = 0; q < 3; ++q) {
            const float *col = sR + q * kLoBl * kLoRs + nl0 * kLoRs + ri;
            float w[kLoBlk + kLoTaps - 1];
#pragma unroll
            for (int k = 0; k < kLoBlk + kLoTaps - 1; ++k) w[k] = (k < n_out + kLoTaps - 1) ? col[k * kLoRs] : 0.f;
            if (q == 0) {
#pragma unroll
                for (int r = 0; r < kLoBlk; ++r) {
                    float acc = 0.f;
#pragma unroll
                    for (int k = 0; k < kLoTaps; ++k) acc = fmaf(P.g1[k], w[r + k], acc);
                    o[0][r] = acc;
                }
            } else {
                lo_box6(w, o[q]);
                lo_box6(w + kLoSeg, o[q] + kLoSeg);
            }
        }
#pragma unroll
        for (int r = 0; r < kLoBlk; ++r) {
            if (r < n_out) {
                const float var = o[2][r] - o[1][r] * o[1][r] * (1.f / 121.f);
                const float den = var * P.g_den;
                sN[(nl0 + r) * kLoRs + ri] = den > 0.f ? (o[0][r] - P.g_mean * o[1][r]) * rsqrtf(den) : 0.f;
            }
        }
    }
    __syncthreads();
    const float thr = P.threshold_rel * __uint_as_float(P.frame_max[f]);
    for (int t = threadIdx.x; t < kLoTl * kLoTa; t += kLoThreads) {
        const int tl = t / kLoTa, ti = t - tl * kLoTa;
        const int l = l0 + tl, i = i0 + ti;
        if (l < 1 || l > n_lat - 2 || i < 1 || i > n_z - 2) continue;                       // interior pixels only
        const float *nn = sN + (tl + 1) * kLoRs + ti + 1;
        const float n0 = nn[0];
        if (!(n0 >= P.ncc_min)) continue;
        const bool peak = n0 > nn[1] && n0 > nn[kLoRs - 1] && n0 > nn[kLoRs] && n0 > nn[kLoRs + 1] &&
                          n0 >= nn[-1] && n0 >= nn[-kLoRs + 1] && n0 >= nn[-kLoRs] && n0 >= nn[-kLoRs - 1];
        if (!peak) continue;
        const float2 x = __ldg(v + (long long)l * n_z + i);
        const float b = sqrtf(x.x * x.x + x.y * x.y);
        if (!(b >= thr)) continue;
        auto parab = [](float mm, float cc, float pp) { const float d = mm - 2.f * cc + pp; return d == 0.f ? 0.f : 0.5f * (mm - pp) / d; };
        const float dl = parab(nn[-kLoRs], n0, nn[kLoRs]), di = parab(nn[-1], n0, nn[1]);
        const int slot = atomicAdd(P.count + (long long)f * n_pl + pl, 1);
        if (slot < P.capacity) P.loc[((long long)f * n_pl + pl) * P.capacity + slot] = make_float4((float)l + dl, (float)i + di, n0, b);
    }
}

}  // namespace ulm
