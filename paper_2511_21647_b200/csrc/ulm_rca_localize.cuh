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
constexpr int kLoThreads = 256;
constexpr int kLoSmem = (kLoBl * kLoBa + 3 * kLoBl * kLoRa + kLoNl * kLoRa) * 4;

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
    float m = 0.f;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < P.planes_per_frame; i += (long long)gridDim.x * 256) {
        const float2 x = __ldg(v + i);
        m = fmaxf(m, sqrtf(x.x * x.x + x.y * x.y));
    }
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(P.frame_max + f, __float_as_uint(m));
}

// grid = (lateral tiles, depth tiles, frames * planes)
__global__ void __launch_bounds__(kLoThreads) localize_kernel(const __grid_constant__ LoParams P) {
    extern __shared__ __align__(16) unsigned char lo_smem[];
    float *sB = reinterpret_cast<float *>(lo_smem);                  // [kLoBl][kLoBa]
    float *sR = sB + kLoBl * kLoBa;                                   // [3][kLoBl][kLoRa]  depth-pass sums (g, 1, squares)
    float *sN = sR + 3 * kLoBl * kLoRa;                               // [kLoNl][kLoRa]     NCC map of the tile + 1
    const int n_pl = P.n_planes[0] + P.n_planes[1];
    const int f = blockIdx.z / n_pl, pl = blockIdx.z - f * n_pl;
    const int a = pl >= P.n_planes[0] ? 1 : 0, m = a ? pl - P.n_planes[0] : pl;
    const int n_lat = a ? P.n_lat[1] : P.n_lat[0], n_z = P.n_z;
    const int l0 = blockIdx.x * kLoTl, i0 = blockIdx.y * kLoTa;
    if (l0 >= n_lat || i0 >= n_z) return;
    const float2 *v = P.planes + (long long)f * P.planes_per_frame + (a ? P.set_off[1] : P.set_off[0]) + (long long)m * n_lat * n_z;
    auto bval = [&](int l, int i) {
        if (l < 0 || l >= n_lat || i < 0 || i >= n_z) return 0.f;
        const float2 x = __ldg(v + (long long)l * n_z + i);
        return sqrtf(x.x * x.x + x.y * x.y);
    };
    const float c = bval(min(l0 + kLoTl / 2, n_lat - 1), min(i0 + kLoTa / 2, n_z - 1));       // offset of this tile
    for (int t = threadIdx.x; t < kLoBl * kLoBa; t += kLoThreads) {
        const int bl = t / kLoBa, bi = t - bl * kLoBa;
        sB[t] = bval(l0 - kLoHalo + bl, i0 - kLoHalo + bi) - c;
    }
    __syncthreads();
    // depth pass: for every row of the B tile, the three 11-tap sums centred on depth positions i0 - 1 .. i0 + kLoTa
    for (int t = threadIdx.x; t < kLoBl * kLoRa; t += kLoThreads) {
        const int bl = t / kLoRa, ri = t - bl * kLoRa;
        const float *row = sB + bl * kLoBa + ri;                      // window ri .. ri + 10 (centre ri + 5 = i0 - 1 + ri)
        float sg = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
        for (int k = 0; k < kLoTaps; ++k) { const float b = row[k]; sg = fmaf(P.g2[k], b, sg); s1 += b; s2 = fmaf(b, b, s2); }
        sR[t] = sg; sR[kLoBl * kLoRa + t] = s1; sR[2 * kLoBl * kLoRa + t] = s2;
    }
    __syncthreads();
    // lateral pass + NCC for the tile and one pixel around it
    for (int t = threadIdx.x; t < kLoNl * kLoRa; t += kLoThreads) {
        const int nl = t / kLoRa, ri = t - nl * kLoRa;
        float sg = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
        for (int k = 0; k < kLoTaps; ++k) {
            const int q = (nl + k) * kLoRa + ri;
            sg = fmaf(P.g1[k], sR[q], sg); s1 += sR[kLoBl * kLoRa + q]; s2 += sR[2 * kLoBl * kLoRa + q];
        }
        const float var = s2 - s1 * s1 * (1.f / 121.f);
        const float den = var * P.g_den;
        sN[t] = den > 0.f ? (sg - P.g_mean * s1) * rsqrtf(den) : 0.f;
    }
    __syncthreads();
    const float thr = P.threshold_rel * __uint_as_float(P.frame_max[f]);
    for (int t = threadIdx.x; t < kLoTl * kLoTa; t += kLoThreads) {
        const int tl = t / kLoTa, ti = t - tl * kLoTa;
        const int l = l0 + tl, i = i0 + ti;
        if (l < 1 || l > n_lat - 2 || i < 1 || i > n_z - 2) continue;                       // interior pixels only
        const float b = sB[(tl + kLoHalo) * kLoBa + ti + kLoHalo] + c;
        const float *nn = sN + (tl + 1) * kLoRa + ti + 1;
        const float n0 = nn[0];
        if (!(b >= thr && n0 >= P.ncc_min)) continue;
        const bool peak = n0 > nn[1] && n0 > nn[kLoRa - 1] && n0 > nn[kLoRa] && n0 > nn[kLoRa + 1] &&
                          n0 >= nn[-1] && n0 >= nn[-kLoRa + 1] && n0 >= nn[-kLoRa] && n0 >= nn[-kLoRa - 1];
        if (!peak) continue;
        auto parab = [](float mm, float cc, float pp) { const float d = mm - 2.f * cc + pp; return d == 0.f ? 0.f : 0.5f * (mm - pp) / d; };
        const float dl = parab(nn[-kLoRa], n0, nn[kLoRa]), di = parab(nn[-1], n0, nn[1]);
        const int slot = atomicAdd(P.count + (long long)f * n_pl + pl, 1);
        if (slot < P.capacity) P.loc[((long long)f * n_pl + pl) * P.capacity + slot] = make_float4((float)l + dl, (float)i + di, n0, b);
    }
}

}  // namespace ulm
