// ulm_rca_clutter.cuh -- eigen-based clutter filter on the Stage-1 slice stacks (Section II.A.2; reading
// = DESIGN.md section 12) for sm_100a.
//
//   CF-1  C_e = I_e^H I_e  for every transmit event e: I_e[p][f] = slice value of pixel p in frame f, i.e. with the
//         frame-major slices X[f][p]:  C[i][j] = sum_p conj(X[i][p]) X[j][p]   (n_t x n_t Hermitian, 32 <= n_t <= 320)
//   CF-2  the `rank` eigenvectors U_c of the largest eigenvalues of C_e (the clutter subspace)
//   CF-3  X_f[f][p] = X[f][p] - sum_m conj(U_c[f][m]) t_m[p],   t_m[p] = sum_f U_c[f][m] X[f][p]
//
// CF-1 is the one dense contraction of the pipeline (2K batched 300 x 29 520 x 300 complex GEMMs) and runs on the
// 5th-generation tensor cores: the real and imaginary parts of X are split into bf16 (hi, lo) pairs by
// clutter_split_kernel (Y = Y_hi + Y_lo carries 16 significant bits), stacked as the rows of a real matrix
// Y = [Re X; Im X] (2 NTP x K, K-major), and clutter_gram_kernel forms the upper triangle of G = Y Y^T with
// tcgen05.mma (kind::f16, bf16 x bf16 -> fp32 in TMEM) as  Y_hi Y_hi^T + Y_hi Y_lo^T + Y_lo Y_hi^T  ("bf16 x 3"; the
// dropped lo x lo term is 2^-16 relative): operand tiles arrive by TMA (cp.async.bulk.tensor, 128-byte swizzle) through
// a 3-stage mbarrier ring, one elected thread issues the MMAs, four warps drain the accumulator with tcgen05.ld.  K is
// split over several CTAs whose partial tiles are added in a fixed order by clutter_assemble_kernel, which also folds
// G back into  C = (RR + II) + j (RI - RI^T).
// CF-2: only the clutter subspace enters the filter, so the full decomposition is not needed: clutter_eig_kernel (one
// CTA per event) runs a blocked orthogonal iteration  Q <- orth(C Q)  on 32 vectors (re-orthonormalised twice per
// step), then a Rayleigh-Ritz step whose 32 x 32 Hermitian problem is solved by a cyclic Jacobi in shared memory.
// CF-3: clutter_project_kernel, one thread per pixel, two passes over the frames (coefficients, then subtraction).
#pragma once

#include <cuda.h>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

constexpr int kCfB = 32;             // vectors of the orthogonal iteration
constexpr int kCfMaxRank = 24;       // clutter rank at most (leaves 8 guard vectors)
constexpr int kCfMaxFrames = 320;    // n_t at most (64 row groups of 5 in clutter_eig_kernel; 2 NTP = 640 Gram rows)
constexpr int kCfTile = 128;         // Gram tile (UMMA M = N = 128)
constexpr int kCfBK = 64;            // k-block: 64 bf16 = one 128-byte swizzle row
constexpr int kCfStages = 3;
constexpr int kCfTileBytes = kCfTile * kCfBK * 2;           // 16 KB
constexpr int kCfStageBytes = 4 * kCfTileBytes;             // A_hi, A_lo, B_hi, B_lo
constexpr int kCfGramThreads = 192;                          // warp 0 TMA, warp 1 MMA, warps 2..5 epilogue
constexpr int kCfGramSmem = kCfStages * kCfStageBytes + 1024 /* alignment slack */ + 256 /* barriers */;

struct CfEvents {            // per-event geometry of the compound = 0 slice layout (device arrays)
    const long long *off;    // [n_events] float2 offset of the event's slice inside a frame
    const int *n_pix;        // [n_events]
};

// ------------------------------------------------------------------------------------------------------------------
// bf16 (hi, lo) split:  Y[e][row][p], rows [0, n_t) = Re X[f][p], rows [NTP, NTP + n_t) = Im X[f][p]  (other rows and the
// columns p >= n_pix stay zero from the plan's initial clear)
// ------------------------------------------------------------------------------------------------------------------
struct CfSplitParams {
    const float2 *x;
    long long frame_stride;          // float2 per frame
    CfEvents ev;
    __nv_bfloat16 *y_hi, *y_lo;
    long long ld;                    // elements per row of Y
    int n_t, ntp, n_events;
};

// a thread = 8 consecutive pixels of one (event, frame): four 16-byte loads, one 16-byte store per output plane
// (scalar tail / unaligned slices: one pixel at a time)
__global__ void __launch_bounds__(256) clutter_split_kernel(const __grid_constant__ CfSplitParams P) {
    const int e = blockIdx.z, f = blockIdx.y;
    const int n_pix = P.ev.n_pix[e];
    const int p = (blockIdx.x * 256 + threadIdx.x) * 8;
    if (p >= n_pix) return;
    const float2 *x = P.x + (long long)f * P.frame_stride + P.ev.off[e] + p;
    const long long row_re = ((long long)e * 2 * P.ntp + f) * P.ld + p;
    const long long row_im = row_re + (long long)P.ntp * P.ld;
    auto split1 = [](float v, __nv_bfloat16 &h, __nv_bfloat16 &l) {
        h = __float2bfloat16_rn(v);
        l = __float2bfloat16_rn(v - __bfloat162float(h));
    };
    const bool vec = p + 8 <= n_pix && ((reinterpret_cast<unsigned long long>(x) & 15ull) == 0) && ((P.ld & 7) == 0);
    if (vec) {
        float4 v[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) v[q] = __ldg(reinterpret_cast<const float4 *>(x) + q);
        __align__(16) __nv_bfloat16 rh[8], rl[8], ih[8], il[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            split1(v[q].x, rh[2 * q], rl[2 * q]); split1(v[q].y, ih[2 * q], il[2 * q]);
            split1(v[q].z, rh[2 * q + 1], rl[2 * q + 1]); split1(v[q].w, ih[2 * q + 1], il[2 * q + 1]);
        }
        *reinterpret_cast<uint4 *>(P.y_hi + row_re) = *reinterpret_cast<const uint4 *>(rh);
        *reinterpret_cast<uint4 *>(P.y_lo + row_re) = *reinterpret_cast<const uint4 *>(rl);
        *reinterpret_cast<uint4 *>(P.y_hi + row_im) = *reinterpret_cast<const uint4 *>(ih);
        *reinterpret_cast<uint4 *>(P.y_lo + row_im) = *reinterpret_cast<const uint4 *>(il);
    } else {
        for (int q = 0; q < 8 && p + q < n_pix; ++q) {
            const float2 v = __ldg(x + q);
            __nv_bfloat16 h, l;
            split1(v.x, h, l); P.y_hi[row_re + q] = h; P.y_lo[row_re + q] = l;
            split1(v.y, h, l); P.y_hi[row_im + q] = h; P.y_lo[row_im + q] = l;
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// PTX helpers: mbarrier, TMA tensor load, tcgen05
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cf_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cf_mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void cf_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// Bounded wait: a protocol mistake must end in a trap (an error the host sees), never in a hung GPU.
__device__ __forceinline__ void cf_mbar_wait(uint32_t bar, uint32_t parity) {
    const long long t0 = clock64();
    for (;;) {
        uint32_t ok;
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (clock64() - t0 > 4000000000ll) __trap();      // ~2 s
    }
}
__device__ __forceinline__ void cf_tma_load_2d(uint32_t dst, const CUtensorMap *map, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
// shared-memory matrix descriptor: K-major tile of 128-byte rows, 128-byte swizzle, 8-row groups 1024 bytes apart
__device__ __forceinline__ uint64_t cf_smem_desc(uint32_t addr) {
    return (uint64_t)((addr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: D fp32, A and B bf16, both K-major, N = 128, M = 128
constexpr uint32_t kCfIdesc = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(kCfTile >> 3) << 17) | ((uint32_t)(kCfTile >> 4) << 24);
__device__ __forceinline__ void cf_mma(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t accumulate) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(kCfIdesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void cf_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

struct CfGramParams {
    float *partial;                  // [event][split][2 NTP][2 NTP] fp32 (upper-triangular tiles only)
    int nr;                          // 2 NTP
    int n_kblocks, n_splits;         // k-blocks of 64 over the longest event; K splits
    int n_tiles_1d;                  // nr / 128
};

// One CTA = one (tile (bm <= bn), K split, event).
__global__ void __launch_bounds__(kCfGramThreads, 1) clutter_gram_kernel(const __grid_constant__ CUtensorMap map_hi,
                                                                         const __grid_constant__ CUtensorMap map_lo,
                                                                         const __grid_constant__ CfGramParams P) {
    extern __shared__ unsigned char cf_raw[];
    unsigned char *smem = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(cf_raw) + 1023) & ~uintptr_t(1023));
    uint64_t *bars = reinterpret_cast<uint64_t *>(smem + kCfStages * kCfStageBytes);
    uint64_t *full = bars, *empty = bars + kCfStages, *tmem_full = bars + 2 * kCfStages;
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(bars + 2 * kCfStages + 1);

    // tile index -> (bm, bn), bm <= bn
    int bm = 0, t = blockIdx.x;
    while (t >= P.n_tiles_1d - bm) { t -= P.n_tiles_1d - bm; ++bm; }
    const int bn = bm + t;
    const bool diag = bm == bn;
    const int split = blockIdx.y, e = blockIdx.z;
    const int kb0 = (int)((long long)P.n_kblocks * split / P.n_splits);
    const int kb1 = (int)((long long)P.n_kblocks * (split + 1) / P.n_splits);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kCfStages; ++s) { cf_mbar_init(cf_smem_u32(&full[s]), 1); cf_mbar_init(cf_smem_u32(&empty[s]), 1); }
        cf_mbar_init(cf_smem_u32(tmem_full), 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {                 // this warp owns the tensor-memory allocation (128 fp32 columns x 128 lanes)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(cf_smem_u32(tmem_slot)), "r"(128u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = *tmem_slot;

    if (warp == 0) {
        // ===================== TMA producer (one thread) =====================
        if (lane == 0) {
            const int row_a = e * P.nr + bm * kCfTile, row_b = e * P.nr + bn * kCfTile;
            uint32_t stage = 0, phase = 0;
            for (int kb = kb0; kb < kb1; ++kb) {
                cf_mbar_wait(cf_smem_u32(&empty[stage]), phase ^ 1);
                const uint32_t bar = cf_smem_u32(&full[stage]);
                const uint32_t dst = cf_smem_u32(smem + stage * kCfStageBytes);
                cf_mbar_expect_tx(bar, (diag ? 2 : 4) * kCfTileBytes);
                cf_tma_load_2d(dst, &map_hi, kb * kCfBK, row_a, bar);
                cf_tma_load_2d(dst + kCfTileBytes, &map_lo, kb * kCfBK, row_a, bar);
                if (!diag) {
                    cf_tma_load_2d(dst + 2 * kCfTileBytes, &map_hi, kb * kCfBK, row_b, bar);
                    cf_tma_load_2d(dst + 3 * kCfTileBytes, &map_lo, kb * kCfBK, row_b, bar);
                }
                if (++stage == kCfStages) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (one thread) =====================
        if (lane == 0) {
            uint32_t stage = 0, phase = 0;
            for (int kb = kb0; kb < kb1; ++kb) {
                cf_mbar_wait(cf_smem_u32(&full[stage]), phase);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t a_hi = cf_smem_u32(smem + stage * kCfStageBytes), a_lo = a_hi + kCfTileBytes;
                const uint32_t b_hi = diag ? a_hi : a_hi + 2 * kCfTileBytes, b_lo = diag ? a_lo : a_hi + 3 * kCfTileBytes;
#pragma unroll
                for (int k4 = 0; k4 < kCfBK / 16; ++k4) {           // UMMA K = 16 bf16 = 32 bytes along the swizzled row
                    const uint64_t dah = cf_smem_desc(a_hi + k4 * 32), dal = cf_smem_desc(a_lo + k4 * 32);
                    const uint64_t dbh = cf_smem_desc(b_hi + k4 * 32), dbl = cf_smem_desc(b_lo + k4 * 32);
                    cf_mma(tmem_base, dah, dbh, (kb > kb0 || k4 > 0) ? 1u : 0u);
                    cf_mma(tmem_base, dah, dbl, 1u);
                    cf_mma(tmem_base, dal, dbh, 1u);
                }
                cf_commit(cf_smem_u32(&empty[stage]));             // frees the stage once these MMAs have read it
                if (++stage == kCfStages) { stage = 0; phase ^= 1; }
            }
            cf_commit(cf_smem_u32(tmem_full));                      // accumulator complete
        }
    } else {
        // ===================== epilogue: TMEM -> registers -> global partial tile =====================
        const int q = warp & 3;                                     // the TMEM lane quarter this warp may access
        if (kb1 > kb0) {
            cf_mbar_wait(cf_smem_u32(tmem_full), 0);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        }
        const int row = bm * kCfTile + q * 32 + lane;
        float *dst = P.partial + (((long long)e * P.n_splits + split) * P.nr + row) * P.nr + bn * kCfTile;
#pragma unroll 1
        for (int c = 0; c < kCfTile / 32; ++c) {
            uint32_t v[32];
            if (kb1 > kb0) {
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)(c * 32);
                asm volatile(
                    "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
                    "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                    : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
                      "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
                      "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
                      "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
                    : "r"(taddr) : "memory");
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            } else {
#pragma unroll
                for (int i = 0; i < 32; ++i) v[i] = 0u;
            }
#pragma unroll
            for (int i = 0; i < 32; i += 4)
                *reinterpret_cast<uint4 *>(dst + c * 32 + i) = make_uint4(v[i], v[i + 1], v[i + 2], v[i + 3]);
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 2) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(128u) : "memory");
}

// C[e][i][j] = (RR + II)[i][j] + j (RI[i][j] - RI[j][i]) from the partial Gram tiles, splits added in order
struct CfAssembleParams {
    const float *partial;
    float2 *cov;                     // [event][n_t][n_t]
    int nr, ntp, n_t, n_splits, n_events;
};
__global__ void __launch_bounds__(256) clutter_assemble_kernel(const __grid_constant__ CfAssembleParams P) {
    const int e = blockIdx.z, i = blockIdx.y, j = blockIdx.x * 256 + threadIdx.x;
    if (j >= P.n_t) return;
    auto g = [&](int a, int b) {     // G is symmetric; only tiles with row block <= column block were computed
        if (a / kCfTile > b / kCfTile) { const int t = a; a = b; b = t; }
        float s = 0.f;
        for (int sp = 0; sp < P.n_splits; ++sp) s += __ldg(P.partial + (((long long)e * P.n_splits + sp) * P.nr + a) * P.nr + b);
        return s;
    };
    const float re = g(i, j) + g(P.ntp + i, P.ntp + j);
    const float im = g(i, P.ntp + j) - g(j, P.ntp + i);
    P.cov[((long long)e * P.n_t + i) * P.n_t + j] = make_float2(re, im);
}

// ------------------------------------------------------------------------------------------------------------------
// CF-2: clutter subspace of one event's covariance: blocked orthogonal iteration + Rayleigh-Ritz (Jacobi)
// ------------------------------------------------------------------------------------------------------------------
constexpr int kCfEigThreads = 512;
constexpr int kCfQs = kCfB + 1;      // padded row stride of Q / Z (float2)
constexpr int kCfKc = 16;            // columns of C staged per step
__host__ __device__ inline int clutter_eig_smem_bytes(int n_t) {
    return (2 * n_t * kCfQs + n_t * (kCfKc + 1) + 2 * kCfB * kCfQs) * 8 + 128 * 4;
}

struct CfEigParams {
    const float2 *cov;               // [event][n_t][n_t]
    float2 *uc;                      // [event][n_t][kCfB]  Ritz vectors, descending Ritz value
    float *lam;                      // [event][kCfB]       Ritz values, descending
    int n_t, iters;                  // iters = upper limit of the orthogonal iterations
    int n_track;                     // the leading n_track (= rank) vectors decide convergence
};

__device__ __forceinline__ float2 cf_cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ float2 cf_cmul_conj(float2 a, float2 b) {       // conj(a) b
    return make_float2(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x);
}
__device__ __forceinline__ float cf_warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// modified Gram-Schmidt of the kCfB columns of z (in place) -> q; both [n_t][kCfQs].  All threads of the CTA.
// track != nullptr: track[c] keeps the squared norm of the orthogonalised column c < n_track (the running estimate of
// lambda_c^2) and track[kCfB] is set to 1 when their PRODUCT moved by more than 2e-6 relative since the last call (the
// sum of the logarithms of the ratios).  The product of the leading diagonal of R is |det| of C restricted to
// the span of the leading n_track columns: it does not see rotations INSIDE that span (which the Rayleigh-Ritz step
// resolves exactly and the filter does not depend on), only the convergence of the span itself.
__device__ void cf_mgs(float2 *z, float2 *q, int n_t, float *track = nullptr, int n_track = 0) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = kCfEigThreads / 32;
    float nn_max = 0.f, drift = 0.f;
    for (int c = 0; c < kCfB; ++c) {
        // every warp forms the norm of column c itself (no extra barrier)
        float nn = 0.f;
        for (int i = lane; i < n_t; i += 32) { const float2 v = z[i * kCfQs + c]; nn += v.x * v.x + v.y * v.y; }
        nn = cf_warp_sum(nn);
        // a column that has (numerically) no component outside the span of the previous ones -- C of rank < 32, e.g. an
        // ensemble of repeated frames -- is deflated to zero instead of being normalised into noise
        nn_max = fmaxf(nn_max, nn);
        const bool live = nn > 1e-12f * nn_max && nn > 1e-36f;
        const float inv = live ? rsqrtf(nn) : 0.f, inv2 = live ? 1.f / nn : 0.f;
        if (track && c < n_track && threadIdx.x == 0) {
            // log of the ratio to the last call's value; a column that died or came to life counts as a move
            drift += (live && track[c] > 0.f) ? log1pf((nn - track[c]) / track[c]) : ((live || track[c] != 0.f) ? 1.f : 0.f);
            track[c] = live ? nn : 0.f;
            if (c == n_track - 1 && fabsf(drift) > 2e-6f) track[kCfB] = 1.f;
        }
        for (int c2 = c + 1 + warp; c2 < kCfB; c2 += n_warps) {
            float pr = 0.f, pi = 0.f;
            for (int i = lane; i < n_t; i += 32) {
                const float2 d = cf_cmul_conj(z[i * kCfQs + c], z[i * kCfQs + c2]);
                pr += d.x; pi += d.y;
            }
            pr = cf_warp_sum(pr) * inv2; pi = cf_warp_sum(pi) * inv2;
            for (int i = lane; i < n_t; i += 32) {
                const float2 a = z[i * kCfQs + c];
                float2 b = z[i * kCfQs + c2];
                b.x -= pr * a.x - pi * a.y; b.y -= pr * a.y + pi * a.x;
                z[i * kCfQs + c2] = b;
            }
        }
        if (warp == n_warps - 1)
            for (int i = lane; i < n_t; i += 32) { const float2 v = z[i * kCfQs + c]; q[i * kCfQs + c] = make_float2(v.x * inv, v.y * inv); }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kCfEigThreads, 1) clutter_eig_kernel(const __grid_constant__ CfEigParams P) {
    extern __shared__ __align__(16) unsigned char cf_eig_smem[];
    const int n_t = P.n_t, e = blockIdx.x;
    float2 *q = reinterpret_cast<float2 *>(cf_eig_smem);             // [n_t][kCfQs]
    float2 *z = q + n_t * kCfQs;                                      // [n_t][kCfQs]
    float2 *cs = z + n_t * kCfQs;                                     // [n_t][kCfKc + 1] staged columns of C
    float2 *h = cs + n_t * (kCfKc + 1);                               // [kCfB][kCfQs]
    float2 *w = h + kCfB * kCfQs;                                     // [kCfB][kCfQs]
    int *order = reinterpret_cast<int *>(w + kCfB * kCfQs);           // [kCfB]
    float *track = reinterpret_cast<float *>(order + kCfB);           // [kCfB + 1]
    const float2 *cov = P.cov + (long long)e * n_t * n_t;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

    // start vectors: a fixed integer hash of (row, column), so that every eigenvector has a component in the block
    for (int i = tid; i < n_t * kCfB; i += kCfEigThreads) {
        const int r = i / kCfB, c = i - r * kCfB;
        uint32_t s = (uint32_t)(r * 2654435761u) ^ (uint32_t)(c * 40503u + 0x9E3779B9u);
        s ^= s >> 15; s *= 2246822519u; s ^= s >> 13; s *= 3266489917u; s ^= s >> 16;
        z[r * kCfQs + c] = make_float2((float)(s & 0xFFFF) / 32768.f - 1.f, (float)(s >> 16) / 32768.f - 1.f);
    }
    __syncthreads();
    cf_mgs(z, q, n_t);

    // Z = C Q: thread (row group of 5, column group of 4) -- 5 x 4 outputs, C staged kCfKc columns at a time
    const int n_rg = (n_t + 4) / 5;                                   // row groups
    const int rg = tid / (kCfB / 4), cg = tid % (kCfB / 4);
    const bool mm_ok = rg < n_rg;
    auto multiply = [&]() {
        float2 acc[5][4];
#pragma unroll
        for (int a = 0; a < 5; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) acc[a][b] = make_float2(0.f, 0.f);
        // the next chunk of C (kCfKc columns of all rows) is fetched into registers while the current one is used
        constexpr int PF = (kCfMaxFrames * kCfKc + kCfEigThreads - 1) / kCfEigThreads;
        float2 pre[PF];
        auto fetch = [&](int k0) {
#pragma unroll
            for (int r_ = 0; r_ < PF; ++r_) {
                const int i = tid + r_ * kCfEigThreads, r = i / kCfKc, kk = i - r * kCfKc;
                pre[r_] = (r < n_t && k0 + kk < n_t) ? __ldg(cov + (long long)r * n_t + k0 + kk) : make_float2(0.f, 0.f);
            }
        };
        fetch(0);
        for (int k0 = 0; k0 < n_t; k0 += kCfKc) {
            __syncthreads();                                          // previous chunk consumed
#pragma unroll
            for (int r_ = 0; r_ < PF; ++r_) {
                const int i = tid + r_ * kCfEigThreads, r = i / kCfKc, kk = i - r * kCfKc;
                if (r < n_t) cs[r * (kCfKc + 1) + kk] = pre[r_];
            }
            __syncthreads();
            if (k0 + kCfKc < n_t) fetch(k0 + kCfKc);
            if (mm_ok) {
#pragma unroll 4
                for (int kk = 0; kk < kCfKc; ++kk) {
                    const int k = min(k0 + kk, n_t - 1);              // a staged zero multiplies the clamped row
                    float2 qv[4];
#pragma unroll
                    for (int b = 0; b < 4; ++b) qv[b] = q[k * kCfQs + cg * 4 + b];
#pragma unroll
                    for (int a = 0; a < 5; ++a) {
                        const float2 cv = cs[min(rg * 5 + a, n_t - 1) * (kCfKc + 1) + kk];
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            acc[a][b].x = fmaf(cv.x, qv[b].x, acc[a][b].x); acc[a][b].x = fmaf(-cv.y, qv[b].y, acc[a][b].x);
                            acc[a][b].y = fmaf(cv.x, qv[b].y, acc[a][b].y); acc[a][b].y = fmaf(cv.y, qv[b].x, acc[a][b].y);
                        }
                    }
                }
            }
        }
        if (mm_ok)
#pragma unroll
            for (int a = 0; a < 5; ++a)
                if (rg * 5 + a < n_t)
#pragma unroll
                    for (int b = 0; b < 4; ++b) z[(rg * 5 + a) * kCfQs + cg * 4 + b] = acc[a][b];
        __syncthreads();
    };

    // Orthogonal iteration Q <- orth(C Q).  One Gram-Schmidt pass per step is enough while iterating (what it leaves
    // of the dominant vectors in the later columns stays inside the span that matters); the basis is re-orthonormalised
    // twice at the end.  Stop: three steps after the squared norms of the leading n_track orthogonalised columns -- the
    // running lambda^2 estimates, which converge twice as fast as the vectors -- have settled to 1e-6, or at P.iters.
    if (tid <= kCfB) track[tid] = 0.f;
    __syncthreads();
    int settled = -1;
    for (int it = 0; it < P.iters; ++it) {
        multiply();
        if (tid == 0) track[kCfB] = 0.f;
        __syncthreads();
        cf_mgs(z, q, n_t, track, P.n_track);
        const bool moved = track[kCfB] != 0.f;                         // uniform: written before the barriers of cf_mgs
        if (!moved && settled < 0) settled = it;
        if (moved) settled = -1;
        if (settled >= 0 && it >= settled + 3) break;
    }
    for (int pass = 0; pass < 2; ++pass) {
        for (int i = tid; i < n_t * kCfB; i += kCfEigThreads) { const int r = i / kCfB, c = i - r * kCfB; z[r * kCfQs + c] = q[r * kCfQs + c]; }
        __syncthreads();
        cf_mgs(z, q, n_t);
    }

    // Rayleigh-Ritz: H = Q^H (C Q), Hermitian part
    multiply();
    for (int i = tid; i < kCfB * kCfB; i += kCfEigThreads) {
        const int a = i / kCfB, b = i - a * kCfB;
        float2 s = make_float2(0.f, 0.f);
        for (int r = 0; r < n_t; ++r) { const float2 d = cf_cmul_conj(q[r * kCfQs + a], z[r * kCfQs + b]); s.x += d.x; s.y += d.y; }
        w[a * kCfQs + b] = s;         // scratch
    }
    __syncthreads();
    for (int i = tid; i < kCfB * kCfB; i += kCfEigThreads) {
        const int a = i / kCfB, b = i - a * kCfB;
        const float2 u = w[a * kCfQs + b], v = w[b * kCfQs + a];
        h[a * kCfQs + b] = a == b ? make_float2(u.x, 0.f) : make_float2(0.5f * (u.x + v.x), 0.5f * (u.y - v.y));
    }
    __syncthreads();
    for (int i = tid; i < kCfB * kCfB; i += kCfEigThreads) { const int a = i / kCfB, b = i - a * kCfB; w[a * kCfQs + b] = make_float2(a == b ? 1.f : 0.f, 0.f); }
    __syncthreads();

    // cyclic two-sided Jacobi on the 32 x 32 Hermitian H by warp 0 (lane = row / column index); W accumulates the rotations
    if (warp == 0) {
        for (int sweep = 0; sweep < 16; ++sweep) {
            float off = 0.f;
            for (int b = 0; b < kCfB; ++b) if (b != lane) { const float2 v = h[lane * kCfQs + b]; off += v.x * v.x + v.y * v.y; }
            float dg = h[lane * kCfQs + lane].x; dg *= dg;
            off = cf_warp_sum(off); dg = cf_warp_sum(dg);
            if (off <= 1e-14f * dg) break;
            for (int p = 0; p < kCfB - 1; ++p)
                for (int qq = p + 1; qq < kCfB; ++qq) {
                    const float2 apq = h[p * kCfQs + qq];
                    const float mag = sqrtf(apq.x * apq.x + apq.y * apq.y);
                    if (mag > 0.f) {                                    // warp-uniform
                        const float2 ph = make_float2(apq.x / mag, apq.y / mag);
                        const float tau = (h[qq * kCfQs + qq].x - h[p * kCfQs + p].x) / (2.f * mag);
                        const float tt = (tau >= 0.f ? 1.f : -1.f) / (fabsf(tau) + sqrtf(1.f + tau * tau));
                        const float cs_ = rsqrtf(1.f + tt * tt), sn = tt * cs_;
                        const float2 sph = make_float2(sn * ph.x, sn * ph.y);                 // s e^{j phi}
                        // columns p, q of H and W:  new_p = c x_p - s conj(ph) x_q,  new_q = s ph x_p + c x_q   (row = lane)
                        {
                            const float2 xp = h[lane * kCfQs + p], xq = h[lane * kCfQs + qq];
                            const float2 a1 = cf_cmul_conj(sph, xq), a2 = cf_cmul(sph, xp);
                            h[lane * kCfQs + p] = make_float2(cs_ * xp.x - a1.x, cs_ * xp.y - a1.y);
                            h[lane * kCfQs + qq] = make_float2(a2.x + cs_ * xq.x, a2.y + cs_ * xq.y);
                            const float2 wp = w[lane * kCfQs + p], wq = w[lane * kCfQs + qq];
                            const float2 b1 = cf_cmul_conj(sph, wq), b2 = cf_cmul(sph, wp);
                            w[lane * kCfQs + p] = make_float2(cs_ * wp.x - b1.x, cs_ * wp.y - b1.y);
                            w[lane * kCfQs + qq] = make_float2(b2.x + cs_ * wq.x, b2.y + cs_ * wq.y);
                        }
                        __syncwarp();
                        // rows p, q of H:  new_p = c y_p - s ph y_q,  new_q = s conj(ph) y_p + c y_q   (column = lane)
                        {
                            const float2 yp = h[p * kCfQs + lane], yq = h[qq * kCfQs + lane];
                            const float2 a1 = cf_cmul(sph, yq), a2 = cf_cmul_conj(sph, yp);
                            h[p * kCfQs + lane] = make_float2(cs_ * yp.x - a1.x, cs_ * yp.y - a1.y);
                            h[qq * kCfQs + lane] = make_float2(a2.x + cs_ * yq.x, a2.y + cs_ * yq.y);
                        }
                        __syncwarp();
                    }
                }
        }
        // descending order of the Ritz values (rank by counting; ties by index)
        // (a non-finite value can only come from non-finite input; it is ranked last so that the order stays a permutation)
        auto clean = [](float v) { return (v == v && fabsf(v) < 3.0e38f) ? v : -3.0e38f; };
        const float mine = clean(h[lane * kCfQs + lane].x);
        int rank = 0;
        for (int b = 0; b < kCfB; ++b) { const float o = clean(h[b * kCfQs + b].x); rank += (o > mine) || (o == mine && b < lane); }
        order[rank] = lane;
        P.lam[e * kCfB + rank] = mine;
    }
    __syncthreads();
    // Ritz vectors U = Q W[:, order]
    for (int i = tid; i < n_t * kCfB; i += kCfEigThreads) {
        const int r = i / kCfB, m = i - r * kCfB, col = order[m];
        float2 s = make_float2(0.f, 0.f);
        for (int b = 0; b < kCfB; ++b) { const float2 d = cf_cmul(q[r * kCfQs + b], w[b * kCfQs + col]); s.x += d.x; s.y += d.y; }
        P.uc[((long long)e * n_t + r) * kCfB + m] = s;
    }
}

// ------------------------------------------------------------------------------------------------------------------
// CF-3: projection, one thread per pixel of one event
// ------------------------------------------------------------------------------------------------------------------
struct CfProjectParams {
    const float2 *x;
    float2 *out;
    long long frame_stride;
    CfEvents ev;
    const float2 *uc;                // [event][n_t][kCfB]
    int n_t, rank;
};

template <int R>
__global__ void __launch_bounds__(128) clutter_project_kernel(const __grid_constant__ CfProjectParams P) {
    extern __shared__ __align__(16) unsigned char cf_prj_smem[];
    float2 *us = reinterpret_cast<float2 *>(cf_prj_smem);            // [n_t][R]
    const int e = blockIdx.y, n_t = P.n_t;
    for (int i = threadIdx.x; i < n_t * R; i += 128) {
        const int f = i / R, m = i - f * R;
        us[i] = m < P.rank ? __ldg(P.uc + ((long long)e * n_t + f) * kCfB + m) : make_float2(0.f, 0.f);
    }
    __syncthreads();
    const int p = blockIdx.x * 128 + threadIdx.x;
    if (p >= P.ev.n_pix[e]) return;
    const float2 *x = P.x + P.ev.off[e] + p;
    float2 *o = P.out + P.ev.off[e] + p;
    float2 t[R];
#pragma unroll
    for (int m = 0; m < R; ++m) t[m] = make_float2(0.f, 0.f);
    for (int f = 0; f < n_t; ++f) {
        const float2 v = x[(long long)f * P.frame_stride];          // plain loads: out may alias x (in-place filtering)
#pragma unroll
        for (int m = 0; m < R; ++m) {
            const float2 u = us[f * R + m];
            t[m].x = fmaf(u.x, v.x, t[m].x); t[m].x = fmaf(-u.y, v.y, t[m].x);
            t[m].y = fmaf(u.x, v.y, t[m].y); t[m].y = fmaf(u.y, v.x, t[m].y);
        }
    }
    for (int f = 0; f < n_t; ++f) {
        float2 v = x[(long long)f * P.frame_stride];
#pragma unroll
        for (int m = 0; m < R; ++m) {           // v -= conj(u) t
            const float2 u = us[f * R + m];
            v.x = fmaf(-u.x, t[m].x, v.x); v.x = fmaf(-u.y, t[m].y, v.x);
            v.y = fmaf(-u.x, t[m].y, v.y); v.y = fmaf(u.y, t[m].x, v.y);
        }
        o[(long long)f * P.frame_stride] = v;
    }
}

}  // namespace ulm
