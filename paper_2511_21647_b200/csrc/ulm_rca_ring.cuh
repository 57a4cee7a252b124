// ulm_rca_ring.cuh -- the hot kernel: shared-memory ring DAS for sm_100a.
//
// One persistent CTA per SM walks work items (frame group of F frames) x (aperture) x (pixel tile).  For a
// work item the receive elements j are the outer loop and the transmit angles k the middle loop; for
// every (j, k) a "stage" = the window of W IQ entries of channel j / event k that the tile can touch,
// for all F frames, is brought from the IQ scratch into a shared-memory ring by one elected producer
// thread with cp.async.bulk (TMA, SASS UBLKCP) completing on an mbarrier; 12 consumer warps gather from
// it.  Everything that does not depend on the frame -- receive delay H(p, j), sample index, interpolation
// weight, phase rotation, apodisation -- is computed once per (pixel, j, k) and reused for the F frames,
// whose accumulators stay in registers; the angle sum is taken in the same registers (the transmit phase
// is folded into the per-(j, k) phasor), so one float2 per pixel and frame is written at the end and no
// per-angle image or volume ever reaches HBM.
//
// Lanes of a warp are consecutive lateral pixels at one depth: their sample indices form a slowly varying
// monotone run, so the 16-byte LDS.128 gathers hit distinct or identical (broadcast) bank groups.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "ulm_rca_device.cuh"

namespace ulm {

constexpr int kRingConsumerWarps = 12;
constexpr int kRingConsumers = kRingConsumerWarps * 32;     // 384 consumer threads
constexpr int kRingThreads = kRingConsumers + 32;           // + 1 producer warp
constexpr int kRingPx = 4;                                  // pixels per consumer thread
constexpr int kRingTilePixels = kRingConsumers * kRingPx;   // 1536
constexpr int kRingMaxStages = 8;
constexpr int kRingMaxRx = 256;                             // receive elements per aperture
constexpr int kRingMaxTz = 96;                              // tile rows
constexpr int kRingMaxBt = 2048;                            // n_tx * tile rows

struct RingConfig {
    int frames = 0, tile_pixels = 0, window = 0, stages = 0, smem_bytes = 0;
    int ws = 0;          // compile-time frame stride (entries) of a stage, >= window
    int n_sms = 0;
};

struct RingTables {
    int n_tiles = 0;
    int tx = 0, tz = 0, tiles_x = 0, tiles_z = 0;
    int *d_s0 = nullptr;     // [tile][j][k] window start, relative to the scratch origin
    ~RingTables() { if (d_s0) cudaFree(d_s0); }
};

struct RingApertureDesc {
    int n_tx, n_rx, n_lat, n_ax;
    double lat0, dlat, z0, dz, ref;
    const double *angles, *t0;
};

struct RingApertureArgs {
    int e0, n_tx, n_rx, n_lat, n_ax;
    const float *xs, *zs, *ejs, *xm, *zm, *ejm, *win;
    const int *n0;
    const float *f0m;
    long long out_base;
    // filled by ring_launch from RingTables:
    const int *s0;
    int n_tiles, tx, tz, tiles_x;
};

struct RingLaunch {
    const float4 *iq;
    int l_row, n_rx_max, n_events;
    float2 *out;
    long long out_frame_stride;
    int n_frames;
    double fcfs, fct;
    int n_lo;
    float two_f;
    RingApertureArgs ap[2];
    // filled by ring_launch:
    int window, n_stages, n_groups, n_work;
};

// ---- PTX helpers (mbarrier + bulk async copy) --------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LAB_DONE_%=;\n"
        "bra LAB_WAIT_%=;\n"
        "LAB_DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void consumer_bar() {
    asm volatile("bar.sync 1, %0;" ::"n"(kRingConsumers) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

template <int F, int WS, bool APOD>
__global__ void __launch_bounds__(kRingThreads, 1) das_ring_kernel(const RingLaunch P) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int kStageBytes = F * WS * 16;
    const int NS = P.n_stages;
    unsigned char *p_misc = smem + (size_t)NS * kStageBytes;
    float *s_bt = reinterpret_cast<float *>(p_misc);                       // [k][tz]
    float *s_ejs = s_bt + kRingMaxBt;                                      // [n_rx]
    float *s_win = s_ejs + kRingMaxRx;
    float *s_ejm = s_win + kRingMaxRx;
    float4 *s_hdr = reinterpret_cast<float4 *>(s_ejm + kRingMaxRx);        // [NS] {off, phi, -, -}
    uint64_t *s_full = reinterpret_cast<uint64_t *>(s_hdr + kRingMaxStages);
    uint64_t *s_empty = s_full + kRingMaxStages;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(smem_u32(&s_full[i]), 1);
            mbar_init(smem_u32(&s_empty[i]), kRingConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    const int tiles_all = P.ap[0].n_tiles + P.ap[1].n_tiles;
    uint32_t stage_ctr = 0;     // global stage counter (identical sequence in producer and consumers)

    if (warp == kRingConsumerWarps) {
        // =================================== PRODUCER WARP ===================================
        for (int w = blockIdx.x; w < P.n_work; w += gridDim.x) {
            const int g = w / tiles_all;
            int tt = w - g * tiles_all;
            const int a = tt >= P.ap[0].n_tiles ? 1 : 0;
            if (a) tt -= P.ap[0].n_tiles;
            const RingApertureArgs &A = P.ap[a];
            const int iz0 = (tt / A.tiles_x) * A.tz;
            const int n_st = A.n_rx * A.n_tx;
            const int *s0_tab = A.s0 + (size_t)tt * n_st;
            const int f_first = g * F;
            for (int sb = 0; sb < n_st; sb += 32) {
                // each lane fetches the window start and the tile's reference n0 of one stage
                const int my = sb + lane;
                int my_s0 = 0, my_nref = 0;
                if (my < n_st) {
                    my_s0 = __ldg(s0_tab + my);
                    my_nref = __ldg(A.n0 + (my % A.n_tx) * A.n_ax + iz0);
                }
                const int cnt = min(32, n_st - sb);
                for (int i = 0; i < cnt; ++i) {
                    const int s0 = __shfl_sync(0xffffffffu, my_s0, i);
                    const int nref = __shfl_sync(0xffffffffu, my_nref, i);
                    if (lane == 0) {
                        const int st = sb + i;
                        const int j = st / A.n_tx, k = st - j * A.n_tx;
                        const uint32_t slot = stage_ctr % NS, phase = (stage_ctr / NS) & 1;
                        mbar_wait(smem_u32(&s_empty[slot]), phase ^ 1);
                        double cyc = P.fcfs * ((double)(P.n_lo + s0) + 0.5) + P.fct;
                        cyc -= floor(cyc);
                        s_hdr[slot] = make_float4((float)(nref - s0), (float)cyc, 0.f, 0.f);
                        const uint32_t bar = smem_u32(&s_full[slot]);
                        const uint32_t bytes = (uint32_t)P.window * 16u;
                        mbar_expect_tx(bar, bytes * F);
                        const uint32_t dst = smem_u32(smem) + slot * kStageBytes;
#pragma unroll
                        for (int f = 0; f < F; ++f) {
                            const int fr = min(f_first + f, P.n_frames - 1);
                            const float4 *src = P.iq + ((long long)(fr * P.n_events + A.e0 + k) * P.n_rx_max + j) * P.l_row + s0;
                            bulk_g2s(dst + f * (WS * 16), src, bytes, bar);
                        }
                    }
                    ++stage_ctr;
                }
            }
        }
        return;
    }

    // ===================================== CONSUMER WARPS =====================================
    const int t = threadIdx.x;
    for (int w = blockIdx.x; w < P.n_work; w += gridDim.x) {
        const int g = w / tiles_all;
        int tt = w - g * tiles_all;
        const int a = tt >= P.ap[0].n_tiles ? 1 : 0;
        if (a) tt -= P.ap[0].n_tiles;
        const RingApertureArgs &A = P.ap[a];
        const int tile_z = tt / A.tiles_x, tile_x = tt - tile_z * A.tiles_x;
        const int ix0 = tile_x * A.tx, iz0 = tile_z * A.tz;
        const int tx = min(A.tx, A.n_lat - ix0), tz = min(A.tz, A.n_ax - iz0);
        const int npx = tx * tz;

        consumer_bar();     // everybody has left the previous work item: the tables may be rewritten
        for (int i = t; i < A.n_tx * tz; i += kRingConsumers) {
            const int k = i / tz, izl = i - k * tz;
            const int base = k * A.n_ax + iz0;
            s_bt[k * A.tz + izl] = (float)(A.n0[base + izl] - A.n0[base]) + A.f0m[base + izl];
        }
        for (int i = t; i < A.n_rx; i += kRingConsumers) {
            s_ejs[i] = A.ejs[i];
            if (APOD) { s_win[i] = A.win[i]; s_ejm[i] = A.ejm[i]; }
        }
        consumer_bar();

        // this thread's pixels
        float xs[kRingPx], zs[kRingPx], xm[kRingPx], zm[kRingPx];
        int bt_off[kRingPx], pix[kRingPx];
#pragma unroll
        for (int m = 0; m < kRingPx; ++m) {
            int q = t + m * kRingConsumers;
            const bool ok = q < npx;
            if (!ok) q = npx - 1;
            const int izl = q / tx, ixl = q - izl * tx;
            xs[m] = A.xs[ix0 + ixl];
            zs[m] = A.zs[iz0 + izl];
            if (APOD) { xm[m] = A.xm[ix0 + ixl]; zm[m] = A.zm[iz0 + izl]; }
            bt_off[m] = izl;
            pix[m] = ok ? (ix0 + ixl) * A.n_ax + iz0 + izl : -1;
        }
        float accr[kRingPx][F], acci[kRingPx][F];
#pragma unroll
        for (int m = 0; m < kRingPx; ++m)
#pragma unroll
            for (int f = 0; f < F; ++f) accr[m][f] = acci[m][f] = 0.f;

        const float fcfs = (float)P.fcfs;
        for (int j = 0; j < A.n_rx; ++j) {
            float H[kRingPx], wgt[kRingPx];
            const float ej = s_ejs[j];
#pragma unroll
            for (int m = 0; m < kRingPx; ++m) {
                const float dxs = xs[m] - ej;
                const float dx2 = dxs * dxs;
                const float den = sqrtf(fmaf(zs[m], zs[m], dx2)) + zs[m];
                H[m] = den > 0.f ? __fdividef(dx2, den) : 0.f;
                if (APOD) {
                    float wv = s_win[j];
                    if (P.two_f > 0.f) {
                        const float lhs = __fmul_rn(fabsf(__fsub_rn(xm[m], s_ejm[j])), P.two_f);
                        if (!(lhs <= zm[m])) wv = 0.f;
                    }
                    wgt[m] = wv;
                }
            }
            for (int k = 0; k < A.n_tx; ++k) {
                const uint32_t slot = stage_ctr % NS, phase = (stage_ctr / NS) & 1;
                mbar_wait(smem_u32(&s_full[slot]), phase);
                const float4 hdr = s_hdr[slot];
                // entry address = stage base + 16 * rint(upm); the magic-constant bits are folded into cbase
                const uint32_t cbase = smem_u32(smem) + slot * kStageBytes - ((uint32_t)kMagicBits << 4);
                const float *bt = s_bt + k * A.tz;
#pragma unroll
                for (int m = 0; m < kRingPx; ++m) {
                    const float upm = (bt[bt_off[m]] + hdr.x) + H[m];
                    const float tt_ = upm + kMagic;
                    const float al = upm - (tt_ - kMagic);
                    const uint32_t addr = ((uint32_t)__float_as_int(tt_) << 4) + cbase;
                    float s, c;
                    sincos_cycles(fmaf(fcfs, upm, hdr.y), s, c);
                    if (APOD) { s *= wgt[m]; c *= wgt[m]; }
                    float4 e[F];
#pragma unroll
                    for (int f = 0; f < F; ++f) e[f] = lds128(addr + f * (WS * 16));
#pragma unroll
                    for (int f = 0; f < F; ++f) {
                        const float vr = fmaf(al, e[f].z, e[f].x), vi = fmaf(al, e[f].w, e[f].y);
                        accr[m][f] = fmaf(c, vr, accr[m][f]);
                        accr[m][f] = fmaf(-s, vi, accr[m][f]);
                        acci[m][f] = fmaf(s, vr, acci[m][f]);
                        acci[m][f] = fmaf(c, vi, acci[m][f]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&s_empty[slot]));
                ++stage_ctr;
            }
        }
        // projection write: one float2 per pixel and frame
#pragma unroll
        for (int m = 0; m < kRingPx; ++m) {
            if (pix[m] < 0) continue;
#pragma unroll
            for (int f = 0; f < F; ++f) {
                const int fr = g * F + f;
                if (fr < P.n_frames)
                    P.out[(long long)fr * P.out_frame_stride + A.out_base + pix[m]] = make_float2(accr[m][f], acci[m][f]);
            }
        }
    }
}

}  // namespace ulm
