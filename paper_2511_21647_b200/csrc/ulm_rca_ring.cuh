// ulm_rca_ring.cuh -- the hot kernel: shared-memory ring DAS for sm_100a.
//
// One persistent CTA per SM walks work items (frame group of F frames) x (aperture) x (pixel tile).  For a
// work item the receive elements j are the outer loop and the transmit angles k the inner loop; for
// every (j, k) a "stage" = the window of W scratch entries of channel j / event k that the tile can touch
// (all F frames of the group are interleaved inside an entry, so a stage is ONE contiguous block) is
// brought from the IQ scratch into a shared-memory ring by one elected producer thread with one
// cp.async.bulk (TMA, SASS UBLKCP) completing on an mbarrier; 12 consumer warps gather from it.
// Everything that does not depend on the frame -- receive delay H(p, j), sample index, interpolation
// weight, phase rotation E(a) of the fractional delay (the sample's own phase is already in the entry), apodisation --
// is computed once per (pixel, j, k) and reused for the F frames, whose accumulators stay in registers; the angle
// sum is taken in the same registers, so one float2 per pixel and frame is written at the end and no per-angle
// image or volume ever reaches HBM.
// The per-item tables (transmit delay rows of the tile, element coordinates, window offsets) are double-buffered and
// written by a second warp of the producer group one work item ahead, so the consumer warps never meet at a CTA-wide
// barrier: each flows from item to item on its own (full/empty mbarriers per table buffer, as for the ring).
//
// Pixel mapping: the image is cut into horizontal strips of PX rows; a consumer thread owns the PX
// vertically adjacent pixels of one (strip, column) position and a tile is 384 consecutive positions, so the
// lanes of a warp are lateral neighbours at the same depths: their sample indices form a slowly varying
// monotone run; compact entries (10 F bytes = odd multiple of 8 B) are gathered with LDS.64, whose 16 lanes of a
// half-warp hit 16 different bank pairs or the same address (measured: 2 cycles per warp-level LDS.64 = 128 B/clk
// up to one entry per lane, profiles/r01_smem_microbench.md); full entries (odd multiple of 16 B) with LDS.128.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "ulm_rca_device.cuh"

namespace ulm {

constexpr int kRingConsumerWarps = 12;
constexpr int kRingConsumers = kRingConsumerWarps * 32;     // 384 consumer threads = positions per tile
constexpr int kRingThreads = kRingConsumers + 128;          // + 1 producer warp group (1 working warp)
constexpr int kRingConsumerRegs = 160;                      // setmaxnreg targets: 3 x 160 + 32 = 512 per SM sub-partition
constexpr int kRingProducerRegs = 32;
constexpr int kRingMaxStages = 8;
constexpr int kRingMaxRx = 256;                             // receive elements per aperture
constexpr int kRingMaxTab = 512;                            // n_tx * tile rows (per table buffer)

struct RingApertureArgs {
    int e0, n_tx, n_rx, n_lat, n_ax;
    const float *xs, *zs, *ejs, *xm, *zm, *ejm, *win;
    const int *n0;           // [k][iz] floor(U0) - n_lo
    const float *f0m;        // [k][iz] U0 - floor(U0) - 0.5
    long long out_base;
    // filled by ring_launch from RingTables:
    const int *dj;           // [tile][j] floor(min H over the tile) - 2
    const int *wj;           // [tile][j] entries of the stages of element j (multiple of 8, <= window)
    int n_tiles;
};

struct RingLaunch {
    const unsigned char *iq;
    int l_row, n_rx_max, n_events;
    float2 *out;
    long long out_frame_stride;
    int n_frames;
    int per_angle;           // 1: compound = 0 -- a work item is one transmit angle of a tile, the output is one slice
                             // per event [event][lat][ax] (out_base = first slice of the aperture)
    float fcfs;
    float two_f;
    RingApertureArgs ap[2];
    // filled by ring_launch:
    int window, stage_stride, n_stages, n_groups, n_work;
    // Tail splitting: the first n_whole work items (a multiple of the grid size) are processed whole; each of the
    // remaining n_items - n_whole items -- the last, partially filled round of the persistent grid -- is cut into
    // split_s slices of the receive elements, work item n_whole + v = (item n_whole + v / split_s, slice v % split_s),
    // whose partial sums go to `partial` [v][thread][PX][F] and are added in slice order by ring_combine_kernel.
    int n_items, n_whole, split_s;
    float2 *partial;
    // DUAL kernels: a work item covers TWO consecutive frame groups (2 F frames) of a tile of PX = 2 rows: the stage
    // brings the windows of both groups (identical delays) and the index / weight / phasor arithmetic of a (pixel,
    // element, angle) term is shared by 2 F frames.  n_groups then counts PAIRS; n_fgroups = the real frame groups.
    int n_fgroups, stage_half;     // stage_half = byte offset of the second group's window inside a ring slot
    int g_first;                   // first frame group (pair) this launch works on: item w belongs to group g_first + w / (items per group)
};

// (item, slice) of work item w; slice = -1: whole item
__device__ __forceinline__ void ring_work(const RingLaunch &P, int w, int &item, int &slice) {
    if (w < P.n_whole) { item = w; slice = -1; }
    else { const int v = w - P.n_whole; item = P.n_whole + v / P.split_s; slice = v - (item - P.n_whole) * P.split_s; }
}
// receive elements of a slice: j = jb, jb + js, ... < n_rx (nj of them).  The slices interleave the elements, so each
// holds the same mix of near and far elements (whose stages differ in bank conflicts and window length)
__device__ __forceinline__ void ring_slice(const RingLaunch &P, int slice, int n_rx, int &jb, int &js, int &nj) {
    if (slice < 0) { jb = 0; js = 1; nj = n_rx; }
    else { jb = slice; js = P.split_s; nj = (n_rx - slice + P.split_s - 1) / P.split_s; }
}

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
// non-blocking phase test (acquire): true when the phase with the given parity has completed
__device__ __forceinline__ bool mbar_test(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ unsigned long long lds64(uint32_t addr) {
    unsigned long long v;
    asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}

// the fields of ap[a] for a run-time a, selected field by field (indexing the kernel parameter with a
// run-time index would copy the whole struct to local memory)
#define ULM_AP(field) (a ? P.ap[1].field : P.ap[0].field)

template <int F, int PX, bool D32, bool APOD, bool W2 = false, bool DUAL = false>
__global__ void __launch_bounds__(kRingThreads, 1) das_ring_kernel(const __grid_constant__ RingLaunch P) {
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int EB = entry_bytes(F, D32);
    constexpr int NAB = DUAL ? 2 : 1, FE = NAB * F;      // frame groups / frames of a work item
    static_assert(!(DUAL && D32), "the two-group items exist for compact entries only");
    const int NS = P.n_stages;
    unsigned char *p_misc = smem + (size_t)NS * P.stage_stride;
    // [k][row] {frac(U0_k(z_row)) - 0.5, floor(U0_k(z_row)) - floor(U0_k(z_iz0))}: the integer row offset is added
    // to the entry index in integer arithmetic, so the fp32 delay sum carries only the fraction and H
    // two buffers of: s_tab [kRingMaxTab] float2, then s_ejs, s_win, s_ejm, s_dj [kRingMaxRx] floats each
    constexpr int kTabBufBytes = kRingMaxTab * 8 + 4 * kRingMaxRx * 4;
    int *s_hdr = reinterpret_cast<int *>(p_misc + 2 * kTabBufBytes);       // [NS] entry shift of the stage
    uint64_t *s_full = reinterpret_cast<uint64_t *>(s_hdr + kRingMaxStages);
    uint64_t *s_empty = s_full + kRingMaxStages;
    uint64_t *t_full = s_empty + kRingMaxStages;                           // [2] table buffer written / released
    uint64_t *t_empty = t_full + 2;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < NS; ++i) {
            mbar_init(smem_u32(&s_full[i]), 1);
            mbar_init(smem_u32(&s_empty[i]), kRingConsumerWarps);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(smem_u32(&t_full[i]), 1);
            mbar_init(smem_u32(&t_empty[i]), kRingConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // work items of a frame group: (aperture, tile) -- with per_angle (aperture, angle, tile)
    const int items0 = P.ap[0].n_tiles * (P.per_angle ? P.ap[0].n_tx : 1);
    const int tiles_all = items0 + P.ap[1].n_tiles * (P.per_angle ? P.ap[1].n_tx : 1);
    // ring position of the next stage (identical sequence in producer and consumers): slot and phase parity are
    // carried along instead of dividing a stage counter by the run-time ring depth
    uint32_t slot = 0, phase = 0;

    if (warp >= kRingConsumerWarps) {
        // ============ PRODUCER WARP GROUP: gives its registers to the consumers; one warp works ============
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRingProducerRegs));
        if (warp == kRingConsumerWarps + 1) {
            // ---- table warp: writes the tables of work item i into buffer i & 1, one item ahead of the consumers
            uint32_t tbuf = 0, tphase = 0;
            for (int ww = blockIdx.x; ww < P.n_work; ww += gridDim.x) {
                int w, slice;
                ring_work(P, ww, w, slice);
                const int gl = w / tiles_all, g = gl + P.g_first;
                int tt = w - gl * tiles_all;
                const int a = tt >= items0 ? 1 : 0;
                if (a) tt -= items0;
                const int n_tx = ULM_AP(n_tx), n_rx = ULM_AP(n_rx), n_lat = ULM_AP(n_lat), n_ax = ULM_AP(n_ax);
                const int n_tiles_a = ULM_AP(n_tiles);
                const int k0 = P.per_angle ? tt / n_tiles_a : 0;
                const int k1 = P.per_angle ? k0 + 1 : n_tx;
                tt -= (P.per_angle ? k0 : 0) * n_tiles_a;
                const int pos0 = tt * kRingConsumers;
                const int iz0 = (pos0 / n_lat) * PX;
                const int n_pos = n_lat * ((n_ax + PX - 1) / PX);
                const int last_pos = min(pos0 + kRingConsumers, n_pos) - 1;
                const int rows = min(n_ax, (last_pos / n_lat + 1) * PX) - iz0;
                const int rows_cap = kRingMaxTab / n_tx;
                unsigned char *buf = p_misc + tbuf * kTabBufBytes;
                float2 *s_tab = reinterpret_cast<float2 *>(buf);
                float *s_ejs = reinterpret_cast<float *>(buf + kRingMaxTab * 8);
                float *s_win = s_ejs + kRingMaxRx, *s_ejm = s_win + kRingMaxRx, *s_dj = s_ejm + kRingMaxRx;
                mbar_wait(smem_u32(&t_empty[tbuf]), tphase ^ 1);      // every consumer warp has left the item that used it
                const int *n0 = ULM_AP(n0);
                const float *f0m = ULM_AP(f0m);
                for (int i = lane; i < (k1 - k0) * rows; i += 32) {
                    const int k = k0 + i / rows, r = i - (k - k0) * rows;
                    const int base = k * n_ax + iz0;
                    s_tab[k * rows_cap + r] = make_float2(__ldg(f0m + base + r), __int_as_float(__ldg(n0 + base + r) - __ldg(n0 + base)));
                }
                const float *ejs = ULM_AP(ejs), *win = ULM_AP(win), *ejm = ULM_AP(ejm);
                const int *dj = ULM_AP(dj) + (size_t)tt * n_rx;
                for (int i = lane; i < n_rx; i += 32) {
                    s_ejs[i] = __ldg(ejs + i);
                    s_dj[i] = (float)__ldg(dj + i);
                    if (APOD) { s_win[i] = __ldg(win + i); s_ejm[i] = __ldg(ejm + i); }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&t_full[tbuf]));
                if (++tbuf == 2) { tbuf = 0; tphase ^= 1; }
            }
            return;
        }
        if (warp != kRingConsumerWarps) return;
        for (int ww = blockIdx.x; ww < P.n_work; ww += gridDim.x) {
            int w, slice;
            ring_work(P, ww, w, slice);
            const int gl = w / tiles_all, g = gl + P.g_first;
            int tt = w - gl * tiles_all;
            const int a = tt >= items0 ? 1 : 0;
            if (a) tt -= items0;
            const int n_rx = ULM_AP(n_rx), n_lat = ULM_AP(n_lat), n_ax = ULM_AP(n_ax);
            int jb, js, nj;
            ring_slice(P, slice, n_rx, jb, js, nj);
            const int n_tiles_a = ULM_AP(n_tiles);
            const int k0 = P.per_angle ? tt / n_tiles_a : 0;              // first angle of the item
            const int n_tx = P.per_angle ? 1 : ULM_AP(n_tx);              // angles of the item
            tt -= (P.per_angle ? k0 : 0) * n_tiles_a;
            const int e0 = ULM_AP(e0) + k0;
            const int *n0 = ULM_AP(n0), *dj = ULM_AP(dj) + (size_t)tt * n_rx, *wj = ULM_AP(wj) + (size_t)tt * n_rx;
            const int iz0 = ((tt * kRingConsumers) / n_lat) * PX;          // first row of the tile
            const int n_st = nj * n_tx;
            const size_t grp_bytes = (size_t)P.n_events * P.n_rx_max * P.l_row * EB;
            const unsigned char *grp = P.iq + (size_t)(NAB * g) * grp_bytes;
            const bool has_b = DUAL && NAB * g + 1 < P.n_fgroups;      // the last pair may hold one group only
            for (int sb = 0; sb < n_st; sb += 32) {
                // each lane fetches the (unclamped) window start of one stage
                const int my = sb + lane;
                int my_s0 = 0, my_w = 0;
                if (my < n_st) {
                    my_s0 = __ldg(n0 + (k0 + my % n_tx) * n_ax + iz0) + __ldg(dj + jb + (my / n_tx) * js);
                    my_w = __ldg(wj + jb + (my / n_tx) * js);
                }
                const int cnt = min(32, n_st - sb);
                for (int i = 0; i < cnt; ++i) {
                    const int s0_raw = __shfl_sync(0xffffffffu, my_s0, i);
                    const int wlen = __shfl_sync(0xffffffffu, my_w, i);
                    if (lane == 0) {
                        const int st = sb + i;
                        const int j = jb + (st / n_tx) * js, k = st % n_tx;
                        // compact entries are 8-byte multiples: an even first entry keeps the copy 16-byte aligned
                        // (the window has two spare entries at either end, ring_plan_aperture)
                        const int s0 = max(0, min(s0_raw, P.l_row - wlen)) & (D32 ? ~0 : ~1);
                        mbar_wait(smem_u32(&s_empty[slot]), phase ^ 1);
                        s_hdr[slot] = s0_raw - s0 - kMagicBits;     // entry shift, with the magic-constant bits folded in
                        const uint32_t bar = smem_u32(&s_full[slot]);
                        const uint32_t bytes = (uint32_t)wlen * EB;
                        mbar_expect_tx(bar, has_b ? 2u * bytes : bytes);
                        const unsigned char *src = grp + (((size_t)(e0 + k) * P.n_rx_max + j) * P.l_row + s0) * EB;
                        bulk_g2s(smem_u32(smem) + slot * P.stage_stride, src, bytes, bar);
                        if (has_b) bulk_g2s(smem_u32(smem) + slot * P.stage_stride + P.stage_half, src + grp_bytes, bytes, bar);
                    }
                    if (++slot == (uint32_t)NS) { slot = 0; phase ^= 1; }
                }
            }
        }
        return;
    }

    // ===================================== CONSUMER WARPS =====================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRingConsumerRegs));
    const int t = threadIdx.x;
    const float th = kTwoPi * P.fcfs;       // 2 pi fc / fs
    uint32_t cbuf = 0, cphase = 0;           // table buffer / phase parity of the next work item
    for (int ww = blockIdx.x; ww < P.n_work; ww += gridDim.x) {
        int w, slice;
        ring_work(P, ww, w, slice);
        const int gl = w / tiles_all, g = gl + P.g_first;
        int tt = w - gl * tiles_all;
        const int a = tt >= items0 ? 1 : 0;
        if (a) tt -= items0;
        const int n_tx = ULM_AP(n_tx), n_rx = ULM_AP(n_rx), n_lat = ULM_AP(n_lat), n_ax = ULM_AP(n_ax);
        int jb, js, nj;
        ring_slice(P, slice, n_rx, jb, js, nj);
        const int n_tiles_a = ULM_AP(n_tiles);
        const int k0 = P.per_angle ? tt / n_tiles_a : 0;                     // angles [k0, k1) of the item
        const int k1 = P.per_angle ? k0 + 1 : n_tx;
        tt -= (P.per_angle ? k0 : 0) * n_tiles_a;
        const int pos0 = tt * kRingConsumers;
        const int iz0 = (pos0 / n_lat) * PX;                                // first row of the tile
        const int n_pos = n_lat * ((n_ax + PX - 1) / PX);
        const int last_pos = min(pos0 + kRingConsumers, n_pos) - 1;
        const int rows = min(n_ax, (last_pos / n_lat + 1) * PX) - iz0;      // rows the tile touches
        const int rows_cap = kRingMaxTab / n_tx;                             // table row stride (>= rows, host-checked)

        // the tables of this item (written by the table warp, possibly long ago)
        unsigned char *tb_ = p_misc + cbuf * kTabBufBytes;
        float2 *s_tab = reinterpret_cast<float2 *>(tb_);
        float *s_ejs = reinterpret_cast<float *>(tb_ + kRingMaxTab * 8);
        float *s_win = s_ejs + kRingMaxRx, *s_ejm = s_win + kRingMaxRx, *s_dj = s_ejm + kRingMaxRx;
        const uint32_t my_tab_empty = smem_u32(&t_empty[cbuf]);
        mbar_wait(smem_u32(&t_full[cbuf]), cphase);
        if (++cbuf == 2) { cbuf = 0; cphase ^= 1; }

        // this thread's PX vertically adjacent pixels
        int pos = pos0 + t;
        const bool active = pos <= last_pos;
        if (!active) pos = last_pos;
        const int strip = pos / n_lat, ix = pos - strip * n_lat;
        const int r0 = strip * PX - iz0;                                     // tile-relative first row
        const float xs = ULM_AP(xs)[ix];
        float zs[PX], xm = 0.f, zm[PX];
        if (APOD) xm = ULM_AP(xm)[ix];
#pragma unroll
        for (int m = 0; m < PX; ++m) {
            const int iz = min(strip * PX + m, n_ax - 1);
            zs[m] = ULM_AP(zs)[iz];
            if (APOD) zm[m] = ULM_AP(zm)[iz];
        }
        const uint32_t tab_addr = smem_u32(s_tab + min(r0, rows - 1));
        // rows past the image bottom re-read the last table row (their results are never stored)
        uint32_t tab_off[PX];
#pragma unroll
        for (int m = 0; m < PX; ++m) tab_off[m] = (uint32_t)(min(r0 + m, rows - 1) - min(r0, rows - 1)) * 8u;

        // accumulators: (frame 2p, frame 2p+1) pairs of real / imaginary parts for FFMA2
        unsigned long long accR2[PX][FE / 2], accI2[PX][FE / 2];
#pragma unroll
        for (int m = 0; m < PX; ++m)
#pragma unroll
            for (int f = 0; f < FE / 2; ++f) accR2[m][f] = accI2[m][f] = 0ull;

        bool ready = false;      // the full barrier of the next stage was already seen complete
        for (int j = jb; j < n_rx; j += js) {
            float Hs[PX], wv[PX];
            {
                const float dxs = xs - s_ejs[j];
                const float dx2 = dxs * dxs;
                const float djf = s_dj[j];
#pragma unroll
                for (int m = 0; m < PX; ++m) {
                    const float den = sqrtf(fmaf(zs[m], zs[m], dx2)) + zs[m];
                    const float H = den > 0.f ? __fdividef(dx2, den) : 0.f;
                    Hs[m] = H - djf;
                    if (APOD) {
                        wv[m] = s_win[j];
                        if (P.two_f > 0.f) {
                            const float lhs = __fmul_rn(fabsf(__fsub_rn(xm, s_ejm[j])), P.two_f);
                            if (!(lhs <= zm[m])) wv[m] = 0.f;
                        }
                    }
                }
            }
            for (int k = k0; k < k1; ++k) {
                // the table row of the first pixel does not depend on the ring: fetched before the barrier wait
                const uint32_t tk = tab_addr + (uint32_t)(k * rows_cap) * 8u;
                unsigned long long tbn = lds64(tk + tab_off[0]);
                if (!ready) mbar_wait(smem_u32(&s_full[slot]), phase);
                // entry address = stage base + EB * (rint(upm) + shift); hdr = shift - magic-constant bits
                const uint32_t cbase = smem_u32(smem) + slot * P.stage_stride;
                const int hdr = s_hdr[slot];
                const uint32_t my_empty = smem_u32(&s_empty[slot]);
                // ring position of the next stage; its barrier is tested now (non-blocking) and the answer is used
                // at the top of the next iteration, so the latency of the test is hidden behind this stage's work
                if (++slot == (uint32_t)NS) { slot = 0; phase ^= 1; }
                ready = mbar_test(smem_u32(&s_full[slot]), phase);
                // per-pixel setup of this stage: entry address, interpolation weight, phasor T_k(z) R(p, j)
                struct PixCtx { uint32_t addr; Alpha A; float c, s; };
                auto prep_tb = [&](int m, unsigned long long tb) {
                    uint32_t fbits, ioff;
                    split_u2(tb, fbits, ioff);
                    const float upm = __uint_as_float(fbits) + Hs[m];
                    const float tt_ = upm + kMagic;
                    const float al = upm - (tt_ - kMagic);
                    PixCtx x;
                    x.addr = (uint32_t)(__float_as_int(tt_) + (int)ioff + hdr) * EB + cbase;
                    x.A = make_alpha<W2>(al);
                    // E(a) = exp(j 2 pi (fc/fs) a), a = al + 0.5 in [0, 1]: the whole phase rotation of this gather
                    __sincosf(fmaf(th, al, 0.5f * th), &x.s, &x.c);
                    if (APOD) { x.c *= wv[m]; x.s *= wv[m]; }
                    return x;
                };
                auto prep = [&](int m) { return prep_tb(m, lds64(tk + tab_off[m])); };
                if constexpr (D32) {
#pragma unroll
                    for (int m = 0; m < PX; ++m) {
                        const PixCtx x = prep(m);
                        const unsigned long long AA = pack_f2(x.A.al, x.A.al), CC = pack_f2(x.c, x.c), SS = pack_f2(x.s, x.s),
                                                 NS = pack_f2(-x.s, -x.s);
#pragma unroll
                        for (int q = 0; q < F / 2; ++q)
                            pair_mac2_full(lds128(x.addr + 16u * q), lds128(x.addr + 8u * F + 16u * q), AA, CC, SS, NS,
                                           accR2[m][q], accI2[m][q]);
                    }
                } else {
                    // software pipeline over (pixel, 4-frame chunk): the five LDS.64 of step i + 1 (three mid word
                    // pairs, two d word pairs) are issued before the 32 FMAs of step i
                    constexpr int NQ = F / 4, NS2 = NAB * NQ, NSTEP = PX * NS2;
                    const uint32_t half = DUAL ? (uint32_t)P.stage_half : 0u;      // window of the second frame group
                    unsigned long long buf[2][5];
                    PixCtx cur = prep_tb(0, tbn), nxt = cur;
                    if (PX > 1) tbn = lds64(tk + tab_off[1]);
                    buf[0][0] = lds64(cur.addr); buf[0][1] = lds64(cur.addr + 8u); buf[0][2] = lds64(cur.addr + 16u);
                    buf[0][3] = lds64(cur.addr + 6u * F); buf[0][4] = lds64(cur.addr + 6u * F + 8u);
#pragma unroll
                    for (int st = 0; st < NSTEP; ++st) {
                        const int m = st / NS2, r = st % NS2, ab = r / NQ, q = r % NQ;
                        if (st + 1 < NSTEP) {
                            const int m1 = (st + 1) / NS2, r1 = (st + 1) % NS2, ab1 = r1 / NQ, q1 = r1 % NQ;
                            if (r1 == 0) {
                                // the table row of pixel m1 was requested a whole pixel earlier
                                nxt = prep_tb(m1, tbn);
                                if (m1 + 1 < PX) tbn = lds64(tk + tab_off[m1 + 1]);
                            }
                            const uint32_t a1 = (r1 == 0 ? nxt.addr : cur.addr) + (ab1 ? half : 0u);
                            unsigned long long *b = buf[(st + 1) & 1];
                            b[0] = lds64(a1 + 24u * q1); b[1] = lds64(a1 + 24u * q1 + 8u); b[2] = lds64(a1 + 24u * q1 + 16u);
                            b[3] = lds64(a1 + 6u * F + 16u * q1); b[4] = lds64(a1 + 6u * F + 16u * q1 + 8u);
                        }
                        const unsigned long long *b = buf[st & 1];
                        chunk_mac2<W2>(b[0], b[1], b[2], b[3], b[4], cur.A.ah, cur.A.ah2, pack_f2(cur.c, cur.c),
                                   pack_f2(cur.s, cur.s), pack_f2(-cur.s, -cur.s), accR2[m] + ab * (F / 2) + 2 * q,
                                   accI2[m] + ab * (F / 2) + 2 * q);
                        if (r == NS2 - 1) cur = nxt;
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(my_empty);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(my_tab_empty);      // this warp is done with the item's tables
        if (slice >= 0) {
            // partial sums of a slice: [work item - n_whole][thread][PX][FE], added in slice order by ring_combine_kernel
            float2 *dst = P.partial + ((size_t)(ww - P.n_whole) * kRingConsumers + t) * (PX * FE);
#pragma unroll
            for (int m = 0; m < PX; ++m)
#pragma unroll
                for (int f = 0; f < FE; f += 2) {
                    float r0, r1, i0, i1;
                    unpack_f2(accR2[m][f / 2], r0, r1);
                    unpack_f2(accI2[m][f / 2], i0, i1);
                    *reinterpret_cast<float4 *>(dst + m * FE + f) = make_float4(r0, i0, r1, i1);
                }
        } else if (active) {
            // projection write: one float2 per pixel and frame; the PX pixels of a thread are contiguous in memory
            // (axial index fastest), so a whole strip is written as 16-byte stores (pixel pairs) when it is aligned
            const long long out_base = ULM_AP(out_base) + (P.per_angle ? (long long)k0 * n_lat * n_ax : 0);
            const int izs = strip * PX;
            const bool vec = (PX % 2 == 0) && izs + PX <= n_ax &&
                             (((P.out_frame_stride | out_base | (long long)n_ax) & 1) == 0) &&
                             ((reinterpret_cast<unsigned long long>(P.out) & 15ull) == 0);
#pragma unroll
            for (int f = 0; f < FE; ++f) {
                const int fr = g * FE + f;       // (the frames of the NAB groups of an item are consecutive)
                if (fr >= P.n_frames) break;
                float2 *dst = P.out + (long long)fr * P.out_frame_stride + out_base + (long long)ix * n_ax + izs;
                float re[PX], im[PX];
#pragma unroll
                for (int m = 0; m < PX; ++m) {
                    float r0, r1, i0, i1;
                    unpack_f2(accR2[m][f / 2], r0, r1);
                    unpack_f2(accI2[m][f / 2], i0, i1);
                    re[m] = (f & 1) ? r1 : r0;
                    im[m] = (f & 1) ? i1 : i0;
                }
                if (vec) {
#pragma unroll
                    for (int m = 0; m < PX; m += 2)
                        *reinterpret_cast<float4 *>(dst + m) = make_float4(re[m], im[m], re[m + 1], im[m + 1]);
                } else {
#pragma unroll
                    for (int m = 0; m < PX; ++m)
                        if (izs + m < n_ax) dst[m] = make_float2(re[m], im[m]);
                }
            }
        }
    }
}

// Adds the split_s partial sums of every split work item in slice order (deterministic) and writes the pixels.
// grid = (split items, PX), block = kRingConsumers.  F = frames of a work item (2 x 12 for the two-group items).
template <int F, int PX>
__global__ void __launch_bounds__(kRingConsumers) ring_combine_kernel(const __grid_constant__ RingLaunch P) {
    const int w = P.n_whole + blockIdx.x, m = blockIdx.y, t = threadIdx.x;
    const int items0 = P.ap[0].n_tiles * (P.per_angle ? P.ap[0].n_tx : 1);
    const int tiles_all = items0 + P.ap[1].n_tiles * (P.per_angle ? P.ap[1].n_tx : 1);
    const int gl = w / tiles_all, g = gl + P.g_first;
    int tt = w - gl * tiles_all;
    const int a = tt >= items0 ? 1 : 0;
    if (a) tt -= items0;
    const int n_lat = ULM_AP(n_lat), n_ax = ULM_AP(n_ax), n_tiles_a = ULM_AP(n_tiles);
    const int k0 = P.per_angle ? tt / n_tiles_a : 0;
    tt -= (P.per_angle ? k0 : 0) * n_tiles_a;
    const int n_pos = n_lat * ((n_ax + PX - 1) / PX);
    const int pos = tt * kRingConsumers + t;
    if (pos >= n_pos) return;
    const int strip = pos / n_lat, ix = pos - strip * n_lat, iz = strip * PX + m;
    if (iz >= n_ax) return;
    const long long out_base = ULM_AP(out_base) + (P.per_angle ? (long long)k0 * n_lat * n_ax : 0);
    const float2 *src = P.partial + ((size_t)blockIdx.x * P.split_s * kRingConsumers + t) * (PX * F) + m * F;
    const size_t slice_stride = (size_t)kRingConsumers * PX * F;
    for (int f = 0; f < F; ++f) {
        const int fr = g * F + f;
        if (fr >= P.n_frames) break;
        float2 acc = src[f];
        for (int s_ = 1; s_ < P.split_s; ++s_) {
            const float2 v = src[s_ * slice_stride + f];
            acc.x += v.x; acc.y += v.y;
        }
        P.out[(long long)fr * P.out_frame_stride + out_base + (long long)ix * n_ax + iz] = acc;
    }
}

#undef ULM_AP

}  // namespace ulm
