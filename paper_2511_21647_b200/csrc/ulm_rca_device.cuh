// ulm_rca_device.cuh -- device-side data layout, the demodulation/staging pre-pass and the generic
// gather kernel of the RCA projection beamformer (sm_100a).
//
// Numerics shared by every DAS kernel:
//   u = (tau - t_start) fs is split as  u = U0[k][iz] + H(p, j)  with
//     U0 = (t0_k + (z cos th_k + ref sin th_k)/c + z/c - t_start) fs   -- host, fp64, stored as
//          integer n0 (relative to the scratch origin) + fraction f0m = frac - 0.5 (fp32)
//     H  = (sqrt(dx^2 + z^2) - z) fs/c = dx_s^2 / (sqrt(dx_s^2 + z_s^2) + z_s)   -- device, fp32, <= ~400
//   so no fp32 quantity ever carries the full ~1300-sample delay.  floor(u) is taken with the
//   add-magic-constant trick on (u - 0.5).
//   Phase rotation: exp(j 2 pi fc tau) with tau = t_n + a / fs (n = floor(u), a = u - n) factors into
//   rho_n = exp(j 2 pi fc t_n), which depends on the sample only and is applied ONCE by the pre-pass to the
//   scratch entry of sample n, and E(a) = exp(j 2 pi (fc/fs) a), a in [0, 1], the only phasor the DAS kernels
//   evaluate (per pixel, element and angle; shared by all frames).  With th = 2 pi fc / fs:
//     term = E(a) [ (1 - a) A_n + a B_n ],   A_n = iq[n] rho_n = s[n],   B_n = iq[n+1] rho_n = s[n+1] exp(-j th),
//   s = the analytic RF signal.  Entries hold mid = (A_n + B_n)/2 and d = B_n - A_n.
//
// IQ scratch ("entries"): frames are processed in groups of F (4 or 12) and paired (2p, 2p+1).  For frame group g,
// event e, receive element j and sample n the scratch holds ONE compact entry of 10 F bytes:
//     mid section, 24 B per chunk of 4 frames (frame pairs a, b) of  mid = (iq[n] + iq[n+1]) / 2  as "fp24" = the top
//       three bytes of the fp32 value (16 mantissa bits): words W0..W5 carry re_a0, re_a1, im_a0, im_a1, re_b0, re_b1 in
//       their top three bytes; the low bytes of W0, W2, W4 are bytes 3, 2, 1 of im_b0 and those of W1, W3, W5 the same
//       of im_b1 (two PRMT each to reassemble; the six direct values are used as loaded, their low mantissa byte
//       being a byte of another value, i.e. a zero-mean error below 2^-16 relative)
//     d section,    4 B per frame:  half2 (dr, di)  of  d/16 = (iq[n+1] - iq[n]) / 16
// so that the interpolated sample is mid + a' d with a' = a - 0.5 in [-0.5, 0.5]: the value carries 17 significant
// bits, only the small difference term is fp16, and every LDS.64 of the mid section delivers an aligned
// (frame 2p, frame 2p+1) register pair for the packed fp32x2 FMA (FFMA2).  "Full" entries keep mid and d in fp32 (16 F + 16 bytes, LDS.128).
// Compact entry sizes 40 / 120 B are odd multiples of 8 B: the LDS.64 gathers of the 16 lanes of a half-warp fall into
// 16 different bank pairs whenever their entries differ; full entry sizes 80 / 208 B are odd multiples of 16 B.
#pragma once

#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

constexpr float kMagic = 12582912.0f;        // 1.5 * 2^23: (x + kMagic) - kMagic = rint(x) for |x| < 2^22
constexpr int kMagicBits = 0x4B400000;
constexpr int kMaxTaps = 129;
constexpr float kTwoPi = 6.283185307179586f;
constexpr float kDScale = 0.0625f;           // d is stored / 16 (|d| can exceed the fp16 range) ...
constexpr float kAlScale = 16.0f;            // ... and a' is multiplied by 16 before it is rounded to fp16
constexpr int kDemodSlots = 128;             // entry slots of the shared-memory image of a chunk (16 thread groups x 8)
constexpr int kDemodChunk = 126;             // entries per demodulation CTA (even: every chunk of 10 F-byte entries starts 16-byte aligned)

// D32 = false: compact entries (fp24 mid + fp16 difference term, 10 F bytes); true: full entries (fp32 mid and
// difference term, 16 F bytes + 16 bytes of padding that keep the entry an odd multiple of 16 B)
__host__ __device__ constexpr int entry_bytes(int F, bool D32) { return D32 ? 16 * F + 16 : 10 * F; }

// Demodulation constants (per plan); they travel inside the kernel parameters (constant bank 0: unrolled taps are
// FFMA constant operands), so plans with different filters can be alive and in flight at the same time.
struct DemodConst {
    int half_len;            // L
    float gd[kMaxTaps];      // dense taps: gd[t] = 2 h[t - L], t = 0..2L   ({1} for IQ input)
    float qd[17];            // quadrature path (fs = 4 fc, L = 8): qd[8] = h[0], qd[t] = h[m] j^(m-1) for odd m = t - 8
    // analytic path (RF input, fs = 8 fc, 33 taps): two REAL filters ga[t] = gd[t] cos(theta m), gb[t] = gd[t] sin(theta m),
    // m = t - L, theta = 2 pi fc / fs, give s[n] = iq[n] rho_n = A + jB directly; rot1 = (cos theta, sin theta)
    float ga[33], gb[33];
    float rot1[2];
};

struct DemodParams {
    const int16_t *rf;       // [frame][event][channel][sample] (x2 for IQ input)
    unsigned char *iq;       // entries: [group][event][rx elem (n_rx_max)][l_row][entry_bytes(F, D32)]
    const float2 *mixer;     // exp(-j 2 pi fc t_n) for n = mix_n0 ..  (mixing of RF input; its conjugate is rho_n)
    int mix_n0;
    int n_frames, n_events, channels_per_event, n_samples;   // n_events = event rows of the scratch (folded or real)
    int n_events_real;       // events per frame of the channel data
    const short2 *ev_map;    // [n_events] the real events (first, second or -1) whose channel data are added into a row
    int n_row_tx, n_rows, n_cols, n_rx_max;
    int full_channels;       // 1: channels_per_event = n_rows + n_cols
    int n_lo, l_row;         // scratch origin (absolute sample of entry 0) and entries per row
    int chunks_per_row;
    DemodConst dc;
};


// d(f32) = a(f16) * b(f16) + c(f32), one FHFMA on sm_100a
__device__ __forceinline__ float fhfma(unsigned short a, unsigned short b, float c) {
    float r;
    asm("fma.rn.f32.f16 %0, %1, %2, %3;" : "=f"(r) : "h"(a), "h"(b), "f"(c));
    return r;
}
__device__ __forceinline__ void split_h2(uint32_t v, unsigned short &lo, unsigned short &hi) {
    asm("mov.b32 {%0, %1}, %2;" : "=h"(lo), "=h"(hi) : "r"(v));
}
__device__ __forceinline__ unsigned short f2h_bits(float v) {
    unsigned short r;
    asm("cvt.rn.f16.f32 %0, %1;" : "=h"(r) : "f"(v));
    return r;
}
__device__ __forceinline__ uint32_t pack_h2(float lo, float hi) {
    uint32_t r;
    asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
    return r;
}

// Compact-entry store of one frame's (mid, d/16) in the layout described at the top of this file (fp24 mid words
// per 4-frame chunk, then one half2 word (dr, di) per frame), so that the DAS kernels read aligned
// (frame 2p, frame 2p+1) register pairs for FFMA2.
// Full-entry store of one frame: the same frame-pair layout with fp32 differences,
// mid: [re_2p, re_2p+1, im_2p, im_2p+1], then d: [dr_2p, dr_2p+1, di_2p, di_2p+1], then 16 bytes of padding.
template <int F>
__device__ __forceinline__ void store_full_entry(unsigned char *ep, int f, float mr, float mi, float dr, float di) {
    const int p = f >> 1, h = f & 1;
    float *mid = reinterpret_cast<float *>(ep) + 4 * p + h;
    mid[0] = mr;
    mid[2] = mi;
    float *d = reinterpret_cast<float *>(ep + 8 * F) + 4 * p + h;
    d[0] = dr;
    d[2] = di;
    if (f == 0) *reinterpret_cast<uint4 *>(ep + 16 * F) = make_uint4(0u, 0u, 0u, 0u);
}

// Warp-cooperative: EVERY thread with f < F of the warp must call it for the same entry slot (the threads of a
// 4-frame chunk are adjacent lanes).  Lane i of a chunk (frame 4c + i) holds
// (re_i, im_i): lanes 0 / 1 write the words W_i = re_i | byte 3 and W_{2+i} = im_i | byte 2 of im_{i+2} (fetched with
// one shuffle), lanes 2 / 3 write W_{2+i} = re_i | byte 1 of their own im_i -- whole 32-bit stores, no byte stores.
template <int F>
__device__ __forceinline__ void store_compact_entry(unsigned char *ep, int f, float mr, float mi, float dr16, float di16) {
    constexpr unsigned kMask = F == 12 ? 0x0FFF0FFFu : 0xFFFFFFFFu;      // lanes with f < F (demod_threads_per_group)
    const int i = f & 3;
    const uint32_t br = __float_as_uint(mr), bi = __float_as_uint(mi);
    const int lane = threadIdx.x & 31;
    const uint32_t v = __shfl_sync(kMask, bi, i < 2 ? lane + 2 : lane);   // im of frame 4c + i + 2 (lanes 0, 1) or own
    uint32_t *mid = reinterpret_cast<uint32_t *>(ep + 24 * (f >> 2));
    const uint32_t wa = __byte_perm(br, v, i < 2 ? 0x3217 : 0x3215);      // re | v.b3   or   re | own im.b1
    const uint32_t wb = __byte_perm(bi, v, 0x3216);                       // im | v.b2 (lanes 0, 1)
    mid[i < 2 ? i : i + 2] = wa;
    if (i < 2) mid[2 + i] = wb;
    reinterpret_cast<uint32_t *>(ep + 6 * F)[f] = pack_h2(dr16, di16);
}

// Edge rule of the interpolation (a term is 0 unless 0 <= n and n + 1 <= Ns - 1), applied to the
// shared-memory image of a chunk after it is written: entries whose two taps are not both inside the record are
// zeroed (all-zero words are zeros in every entry format).  Only the chunks that touch an end of the record do any
// work here.  Must be called by all threads of the CTA.
__device__ __forceinline__ void zero_edge_entries(unsigned char *s_out, int eb, int n_ent, int base, int n_samples) {
    if (base >= 0 && base + n_ent <= n_samples - 1) return;     // block-uniform
    __syncthreads();
    const int words = eb / 4;
    for (int idx = threadIdx.x; idx < n_ent * words; idx += blockDim.x) {
        const int n = base + idx / words;
        if (!(n >= 0 && n + 1 <= n_samples - 1)) reinterpret_cast<uint32_t *>(s_out)[idx] = 0u;
    }
}

// ---------------------------------------------------------------------------------------------------
// Demodulation / staging pre-pass: int16 RF (or IQ) -> scratch entries over the touched
// sample range only.  One CTA = one chunk of 126 entries of one (frame group, event, rx element) row, all F
// frames of the group:
//   (1) the mixed samples x = rf * exp(-j 2 pi fc t) of the F frames go to shared memory;
//   (2) thread (frame f, group of 8 entries) runs the FIR for 9 consecutive outputs with the inputs sliding
//       through registers (dense taps straight from constant memory; ZS = 2: half-band filter, fs = 4 fc: the
//       even taps other than the centre are exactly zero and are skipped at compile time; ZS = 4: every fourth tap,
//       fs = 8 fc), forms
//       mid = (a + b)/2 and d = b - a and writes them into an image of the output block in shared memory;
//   (3) one elected thread stores the block (126 x 10 F contiguous bytes) with one cp.async.bulk (TMA).
// NT = dense tap count 2L+1 (0: run-time L).  Lanes of a half-warp are the frames of one group, so every
// shared-memory access of step (2) is conflict free (row stride of x = 1 mod 16 float2).
// ---------------------------------------------------------------------------------------------------

__host__ __device__ constexpr int demod_threads_per_group(int F) { return F == 12 ? 16 : F; }
__host__ __device__ inline int demod_xs(int L) { return ((kDemodChunk + 2 + 2 * L) + 14) / 16 * 16 + 1; }
__host__ __device__ inline int demod_smem_bytes(int F, bool D32, int L) {
    return kDemodSlots * entry_bytes(F, D32) + F * demod_xs(L) * 8;
}

// AN = analytic variant (RF input, NT = 33, ZS = 4, i.e. fs = 8 fc): no mixer; the staging buffer holds the REAL samples
// and the two real filters ga / gb (17 + 24 non-zero taps: ga[m] = 0 for m = 2 mod 4, both 0 for m = 0 mod 4, m != 0,
// gb[0] = 0 -- checked on the host) give the analytic signal s[n] = A + jB, so an entry needs one constant rotation
// B_n = s[n+1] exp(-j theta) instead of two table rotations: 41 real FMAs per output instead of 50 + mixing.
template <int NT, int ZS, bool IQ_INPUT, int F, bool D32, bool AN = false>
__global__ void __launch_bounds__(256) demod_kernel(const __grid_constant__ DemodParams P) {
    static_assert(!AN || (!IQ_INPUT && NT == 33 && ZS == 4), "analytic variant: RF input, 33 taps at fs = 8 fc");
    extern __shared__ __align__(128) unsigned char s_raw[];
    constexpr int EB = entry_bytes(F, D32);
    constexpr int OUT_BYTES = kDemodSlots * EB;      // every entry slot a thread can address (a multiple of 128 B)
    constexpr int R = 8;                       // entries per thread
    constexpr int TPG = demod_threads_per_group(F);
    const int L = NT > 0 ? (NT - 1) / 2 : P.dc.half_len;
    const int XW = kDemodChunk + 2 + 2 * L;    // mixed samples per frame: iq[0..128] needs x[0 .. 128 + 2L]
    const int XS = demod_xs(L);                // row stride of s_x (float2)
    unsigned char *s_out = s_raw;              // [126][EB] image of the output block
    float2 *s_x = reinterpret_cast<float2 *>(s_raw + OUT_BYTES);   // [F][XS]

    // grid = (chunk lanes, n_rx_max, groups * n_events): a CTA walks the chunks blockIdx.x, blockIdx.x + gridDim.x, ...
    // of its row; the global loads of the next chunk are in flight while the current one is filtered and stored
    const int j = blockIdx.y;
    const int g = blockIdx.z / P.n_events, e = blockIdx.z - g * P.n_events;
    const long long row = (long long)blockIdx.z * P.n_rx_max + j;     // (group * n_events + e) * n_rx_max + j
    const int row_tx = e < P.n_row_tx;
    const int n_rx = row_tx ? P.n_cols : P.n_rows;
    if (j >= n_rx) return;                      // rows of the shorter aperture stay unused
    const int ch = row_tx ? (P.full_channels ? P.n_rows + j : j) : j;

    // (1) mixed samples: half h of the CTA takes frames [h F/2, (h+1) F/2), a thread takes the sample columns i0 and
    // i0 + 128 (XW <= 256); the record address is formed once, the frames are reached by stepping
    constexpr int FH = F / 2;
    const int h = threadIdx.x >> 7, i0 = threadIdx.x & 127;
    const long long frame_stride = (long long)P.n_events_real * P.channels_per_event * P.n_samples;
    const int fr0 = g * F + h * FH;
    const int f_last = min(FH - 1, P.n_frames - 1 - fr0);       // < 0: this half of the group has no frame at all
    const short2 ev = __ldg(P.ev_map + e);                      // real event(s) folded into this scratch row
    const bool two = ev.y >= 0;                                  // folded pair: everything downstream is linear
    const long long rec0 = (long long)min(fr0, P.n_frames - 1) * frame_stride +
                           ((long long)ev.x * P.channels_per_event + ch) * (long long)P.n_samples;
    const long long off_b = two ? (long long)(ev.y - ev.x) * P.channels_per_event * (long long)P.n_samples : 0;
    const bool second = i0 + 128 < XW;
    // prefetched samples of the next chunk: [sample column][frame], first / second event (IQ input: packed re | im)
    int ra[2][FH], rb[2][FH];
    auto issue_loads = [&](int chunk) {
        const int base = P.n_lo + chunk * kDemodChunk;
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
            if (rep == 1 && !second) break;
            const int n = base - L + i0 + rep * 128;
            long long src = rec0 + min(max(n, 0), P.n_samples - 1);     // clamped: the loads are unconditional
#pragma unroll
            for (int f = 0; f < FH; ++f) {
                if (IQ_INPUT) {
                    ra[rep][f] = __ldg(reinterpret_cast<const int *>(P.rf) + src);
                    rb[rep][f] = two ? __ldg(reinterpret_cast<const int *>(P.rf) + src + off_b) : 0;
                } else {
                    ra[rep][f] = __ldg(P.rf + src);
                    rb[rep][f] = two ? (int)__ldg(P.rf + src + off_b) : 0;
                }
                if (f < f_last) src += frame_stride;
            }
        }
    };
    auto store_x = [&](int chunk) {
        const int base = P.n_lo + chunk * kDemodChunk;
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
            if (rep == 1 && !second) break;
            const int i = i0 + rep * 128;
            const int n = base - L + i;
            const bool inb = n >= 0 && n < P.n_samples;
            float2 *dst = s_x + (h * FH) * XS + i;
            if (AN) {
                float *dr_ = reinterpret_cast<float *>(s_x) + (h * FH) * XS + i;
#pragma unroll
                for (int f = 0; f < FH; ++f) dr_[f * XS] = (inb && f <= f_last) ? (float)(ra[rep][f] + rb[rep][f]) : 0.f;
                continue;
            }
            float2 m = make_float2(1.f, 0.f);
            if (!IQ_INPUT && inb) m = __ldg(P.mixer + (n - P.mix_n0));
#pragma unroll
            for (int f = 0; f < FH; ++f) {
                const bool ok = inb && f <= f_last;
                if (IQ_INPUT) {
                    const int a = ra[rep][f], b = rb[rep][f];
                    const float re = (float)((short)(a & 0xffff) + (short)(b & 0xffff));
                    const float im = (float)((a >> 16) + (b >> 16));
                    dst[f * XS] = ok ? make_float2(re, im) : make_float2(0.f, 0.f);
                } else {
                    const float re = ok ? (float)(ra[rep][f] + rb[rep][f]) : 0.f;
                    dst[f * XS] = make_float2(re * m.x, re * m.y);
                }
            }
        }
    };

    const int f = threadIdx.x % TPG, grp = threadIdx.x / TPG;
    int chunk = blockIdx.x;
    if (chunk < P.chunks_per_row) issue_loads(chunk);
    for (; chunk < P.chunks_per_row; chunk += gridDim.x) {
    const int base = P.n_lo + chunk * kDemodChunk;   // absolute sample of this chunk's first iq value
    store_x(chunk);                                  // consumes the prefetched registers
    if (chunk + (int)gridDim.x < P.chunks_per_row) issue_loads(chunk + gridDim.x);
    // the image of the previous chunk must have been read by its bulk store before it is overwritten
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncthreads();

    // (2) FIR: iq[base + r] = sum_{i = r .. r + 2L} gd[r + 2L - i] x[i]   (x index relative to base - L)
    const int n_ent = min(kDemodChunk, P.l_row - chunk * kDemodChunk);
    // every lane with f < F of a warp that holds at least one valid entry runs the whole loop (the compact store is
    // warp-cooperative); entries past n_ent are computed from whatever the staging buffer holds and never stored
    if (f < F && ((threadIdx.x & ~31) / TPG) * R < n_ent) {
        const int r0 = grp * R;
        const float2 *x = s_x + f * XS + r0;
        float ar[R + 1], ai[R + 1];
#pragma unroll
        for (int q = 0; q <= R; ++q) ar[q] = ai[q] = 0.f;
        if (AN) {
            const float *xr = reinterpret_cast<const float *>(s_x) + f * XS + r0;
#pragma unroll
            for (int u = 0; u < R + NT; ++u) {
                const float xv = xr[u];
#pragma unroll
                for (int q = 0; q <= R; ++q) {
                    const int t = q - u + (NT - 1);
                    const int m4 = ((t - NT / 2) % 4 + 4) % 4;
                    if (t >= 0 && t < NT && (m4 != 0 || t == NT / 2)) {
                        if (m4 != 2) ar[q] = fmaf(P.dc.ga[t], xv, ar[q]);
                        if (t != NT / 2) ai[q] = fmaf(P.dc.gb[t], xv, ai[q]);
                    }
                }
            }
        } else if (NT > 0) {
#pragma unroll
            for (int u = 0; u < R + NT; ++u) {
                const float2 xv = x[u];
#pragma unroll
                for (int q = 0; q <= R; ++q) {
                    const int t = q - u + (NT - 1);
                    if (t >= 0 && t < NT && !(ZS > 0 && t != NT / 2 && ((t - NT / 2) % ZS) == 0)) {
                        ar[q] = fmaf(P.dc.gd[t], xv.x, ar[q]);
                        ai[q] = fmaf(P.dc.gd[t], xv.y, ai[q]);
                    }
                }
            }
        } else {
            for (int u = 0; u <= R + 2 * L; ++u) {
                const float2 xv = x[u];
#pragma unroll
                for (int q = 0; q <= R; ++q) {
                    const int t = q - u + 2 * L;
                    if (t >= 0 && t <= 2 * L) {
                        ar[q] = fmaf(P.dc.gd[t], xv.x, ar[q]);
                        ai[q] = fmaf(P.dc.gd[t], xv.y, ai[q]);
                    }
                }
            }
        }
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const int ent = r0 + q;               // < kDemodSlots: slots past n_ent are written but never copied out
            const float m0r = 0.5f * (ar[q] + ar[q + 1]), m0i = 0.5f * (ai[q] + ai[q + 1]);
            const float d0r = ar[q + 1] - ar[q], d0i = ai[q + 1] - ai[q];
            float mr, mi, dr, di;
            if (AN) {
                // A_n = s[n] = (ar, ai)[q];  B_n = s[n+1] exp(-j theta)
                const float c1 = P.dc.rot1[0], s1 = P.dc.rot1[1];
                const float br = fmaf(ar[q + 1], c1, ai[q + 1] * s1), bi = fmaf(ai[q + 1], c1, -ar[q + 1] * s1);
                mr = 0.5f * (ar[q] + br); mi = 0.5f * (ai[q] + bi);
                dr = br - ar[q]; di = bi - ai[q];
            } else {
                // rotate by rho_n = conj(mixer[n]) (one broadcast load per entry: all frames share n)
                const float2 mx = __ldg(P.mixer + (base + ent - P.mix_n0));
                mr = fmaf(m0r, mx.x, m0i * mx.y); mi = fmaf(m0i, mx.x, -m0r * mx.y);
                dr = fmaf(d0r, mx.x, d0i * mx.y); di = fmaf(d0i, mx.x, -d0r * mx.y);
            }
            unsigned char *ep = s_out + ent * EB;
            if (D32) {
                store_full_entry<F>(ep, f, mr, mi, dr, di);
            } else {
                store_compact_entry<F>(ep, f, mr, mi, kDScale * dr, kDScale * di);
            }
        }
    }
    // (3) one bulk store of the block: generic-proxy writes -> async proxy, then TMA shared -> global
    zero_edge_entries(s_out, EB, n_ent, base, P.n_samples);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();                                 // image complete; everybody is done reading s_x
    if (threadIdx.x == 0) {
        unsigned char *dst = P.iq + ((size_t)row * P.l_row + (size_t)chunk * kDemodChunk) * EB;
        const uint32_t src = (uint32_t)__cvta_generic_to_shared(s_out);
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"((uint32_t)(n_ent * EB))
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    }   // chunk loop
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// ---------------------------------------------------------------------------------------------------
// Quadrature-sampled variant of the pre-pass (RF input, fs = 4 fc exactly, default 17-tap filter): the analytic
// signal is  s[n] = iq[n] rho_n = A + j B  with the REAL filters  A = g[0] rf[n],
// B = sum_{m odd} g[m] j^(m-1) rf[n-m]  (the even taps of the half-band filter are exactly zero): 9 real FMAs
// per output instead of 34 complex ones, no mixer and no rotation at all (A_n = s[n], B_n = s[n+1] (-j) = B' - jA').
// The taps are stored halved (qd = g/2) so that mid = a' + b' and d/16 = (b' - a')/8 need no further scaling.
// Same CTA decomposition, shared-memory image and TMA store as demod_kernel.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ constexpr int demod_quad_xs() { return 225; }    // >= 1.5 * 145 + 4, = 1 mod 32 (words)
__host__ __device__ inline int demod_quad_smem_bytes(int F, bool D32) {
    return kDemodSlots * entry_bytes(F, D32) + F * demod_quad_xs() * 4;
}

template <int F, bool D32>
__device__ __forceinline__ void demod_quad_emit(const float (&A)[9], const float (&B)[9], int r0, int f,
                                                unsigned char *s_out) {
    constexpr int EB = entry_bytes(F, D32);
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const int ent = r0 + q;                   // < kDemodSlots: slots past n_ent are written but never copied out
        // halved A_n = s[n] = A + jB and B_n = s[n+1] exp(-j pi/2) = B' - jA'
        const float mr = A[q] + B[q + 1], mi = B[q] - A[q + 1];
        const float dr = B[q + 1] - A[q], di = -A[q + 1] - B[q];                                       // = (d)/2
        unsigned char *ep = s_out + ent * EB;
        if (D32) {
            store_full_entry<F>(ep, f, mr, mi, 2.f * dr, 2.f * di);
        } else {
            store_compact_entry<F>(ep, f, mr, mi, 2.f * kDScale * dr, 2.f * kDScale * di);
        }
    }
}

// PAIR: the raw samples are read as aligned int16 pairs (one 4-byte load for two samples; needs an even record length):
// column c of a staging row then holds sample base - L - (n_lo & 1) + c and the filter reads one column further right.
template <int F, bool D32, bool PAIR = false>
__global__ void __launch_bounds__(256, 4) demod_quad_kernel(const __grid_constant__ DemodParams P) {
    extern __shared__ __align__(128) unsigned char s_raw[];
    constexpr int EB = entry_bytes(F, D32);
    constexpr int OUT_BYTES = kDemodSlots * EB;      // every entry slot a thread can address (a multiple of 128 B)
    constexpr int L = 8, XW = kDemodChunk + 2 + 2 * L, XS = demod_quad_xs();
    constexpr int TPG = demod_threads_per_group(F), FH = F / 2;
    unsigned char *s_out = s_raw;
    float *s_x = reinterpret_cast<float *>(s_raw + OUT_BYTES);      // [F][XS], sample i at i + 4 (i >> 3)

    // grid = (chunk lanes, n_rx_max, groups * n_events): a CTA walks the chunks blockIdx.x, blockIdx.x + gridDim.x, ...
    // of its row; the global loads of the next chunk are in flight while the current one is filtered and stored
    const int j = blockIdx.y;
    const int g = blockIdx.z / P.n_events, e = blockIdx.z - g * P.n_events;
    const long long row = (long long)blockIdx.z * P.n_rx_max + j;     // (group * n_events + e) * n_rx_max + j
    const int row_tx = e < P.n_row_tx;
    const int n_rx = row_tx ? P.n_cols : P.n_rows;
    if (j >= n_rx) return;
    const int ch = row_tx ? (P.full_channels ? P.n_rows + j : j) : j;

    // (1) raw samples: half h of the CTA takes frames [h FH, (h+1) FH), a thread takes samples i0 and (i0 < 16) i0 + 128.
    // The record address is formed once; the frames are reached by stepping a pointer (no per-frame 64-bit products).
    const int h = threadIdx.x >> 7, i0 = threadIdx.x & 127;
    const long long frame_stride = (long long)P.n_events_real * P.channels_per_event * P.n_samples;
    const int fr0 = g * F + h * FH;
    const int f_last = min(FH - 1, P.n_frames - 1 - fr0);       // < 0: this half of the group has no frame at all
    const short2 ev = __ldg(P.ev_map + e);                      // real event(s) folded into this scratch row
    const bool two = ev.y >= 0;                                  // folded pair: the FIR is linear, the records are added
    const int16_t *rec = P.rf + (long long)min(fr0, P.n_frames - 1) * frame_stride +
                         ((long long)ev.x * P.channels_per_event + ch) * (long long)P.n_samples;
    const long long off_b = two ? (long long)(ev.y - ev.x) * P.channels_per_event * (long long)P.n_samples : 0;
    const bool second = !PAIR && i0 + 128 < XW;
    const int odd = PAIR ? (P.n_lo & 1) : 0;                    // L and kDemodChunk are even: the same for every chunk
    constexpr int NPAIRS = (XW + 2) / 2;
    int ra[2][FH], rb[2][FH];        // prefetched samples of the next chunk: [sample column][frame], first / second event
    // unconditional loads from clamped addresses (out-of-range samples and frames are zeroed when they are consumed)
    auto issue_loads = [&](int chunk) {
        const int base = P.n_lo + chunk * kDemodChunk;
        if (PAIR) {
            if (i0 < NPAIRS) {
                const int n = base - L - odd + 2 * i0;           // even: the pair (n, n + 1) is 4-byte aligned, both in or both out
                const int *src = reinterpret_cast<const int *>(rec + min(max(n, 0), P.n_samples - 2));
#pragma unroll
                for (int f = 0; f < FH; ++f) {
                    ra[0][f] = __ldg(src);
                    rb[0][f] = two ? __ldg(src + off_b / 2) : 0;
                    if (f < f_last) src += frame_stride / 2;
                }
            }
            return;
        }
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
            if (rep == 1 && !second) break;
            const int n = base - L + i0 + rep * 128;
            const int16_t *src = rec + min(max(n, 0), P.n_samples - 1);
#pragma unroll
            for (int f = 0; f < FH; ++f) {
                ra[rep][f] = __ldg(src);
                rb[rep][f] = two ? (int)__ldg(src + off_b) : 0;
                if (f < f_last) src += frame_stride;
            }
        }
    };
    auto store_x = [&](int chunk) {
        const int base = P.n_lo + chunk * kDemodChunk;
        if (PAIR) {
            if (i0 < NPAIRS) {
                const int n = base - L - odd + 2 * i0, c = 2 * i0;
                const bool inb = n >= 0 && n < P.n_samples;
                float *dst = s_x + (h * FH) * XS + c + 4 * (c >> 3);
#pragma unroll
                for (int f = 0; f < FH; ++f) {
                    const int va = ra[0][f], vb = rb[0][f];
                    const bool ok = inb && f <= f_last;
                    dst[f * XS] = ok ? (float)((int)(short)(va & 0xffff) + (int)(short)(vb & 0xffff)) : 0.f;
                    dst[f * XS + 1] = ok ? (float)((va >> 16) + (vb >> 16)) : 0.f;
                }
            }
            return;
        }
#pragma unroll
        for (int rep = 0; rep < 2; ++rep) {
            if (rep == 1 && !second) break;
            const int i = i0 + rep * 128;
            const int n = base - L + i;
            const bool inb = n >= 0 && n < P.n_samples;
            float *dst = s_x + (h * FH) * XS + i + 4 * (i >> 3);
#pragma unroll
            for (int f = 0; f < FH; ++f) dst[f * XS] = (inb && f <= f_last) ? (float)(ra[rep][f] + rb[rep][f]) : 0.f;
        }
    };

    const int f = threadIdx.x % TPG, grp = threadIdx.x / TPG;
    int chunk = blockIdx.x;
    if (chunk < P.chunks_per_row) issue_loads(chunk);
    for (; chunk < P.chunks_per_row; chunk += gridDim.x) {
        const int base = P.n_lo + chunk * kDemodChunk;
        store_x(chunk);                                      // consumes the prefetched registers
        if (chunk + (int)gridDim.x < P.chunks_per_row) issue_loads(chunk + gridDim.x);
        // the image of the previous chunk must have been read by its bulk store before it is overwritten
        if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        __syncthreads();

        // (2) real FIRs A, B for 9 consecutive outputs, mid / d into the output image
        const int n_ent = min(kDemodChunk, P.l_row - chunk * kDemodChunk);
        // every lane with f < F of a warp that holds at least one valid entry runs the whole loop (the compact store is
        // warp-cooperative); entries past n_ent are computed from whatever the staging buffer holds and never stored
        if (f < F && ((threadIdx.x & ~31) / TPG) * 8 < n_ent) {
            const int r0 = grp * 8;
            const float *x = s_x + f * XS + r0 + (r0 >> 1);         // r0 + 4 (r0 >> 3)
            // PAIR: column u + odd; one step to the right crosses a padded group boundary after u = 7 mod 8
            const float *x1 = x + odd, *x5 = x + 5 * odd;
            float A[9], B[9];
#pragma unroll
            for (int q = 0; q < 9; ++q) B[q] = 0.f;
#pragma unroll
            for (int u = 0; u < 9 + 2 * L; ++u) {
                const float xv = PAIR ? ((u & 7) == 7 ? x5 : x1)[u + 4 * (u >> 3)] : x[u + 4 * (u >> 3)];
#pragma unroll
                for (int q = 0; q < 9; ++q) {
                    const int t = q - u + 2 * L;                    // tap m = t - L
                    if (t == L) A[q] = P.dc.qd[L] * xv;
                    else if (t >= 0 && t <= 2 * L && ((t - L) & 1)) B[q] = fmaf(P.dc.qd[t], xv, B[q]);
                }
            }
            demod_quad_emit<F, D32>(A, B, r0, f, s_out);
        }
        zero_edge_entries(s_out, EB, n_ent, base, P.n_samples);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        __syncthreads();                                     // image complete; everybody is done reading s_x
        if (threadIdx.x == 0) {
            unsigned char *dst = P.iq + ((size_t)row * P.l_row + (size_t)chunk * kDemodChunk) * EB;
            const uint32_t src = (uint32_t)__cvta_generic_to_shared(s_out);
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"((uint32_t)(n_ent * EB))
                         : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// One aperture (image) of the generic DAS kernel.
constexpr int kVolMirrorMaxAngles = 32;

struct DasParams {
    const unsigned char *iq;
    int l_row, n_rx_max, n_events;
    int e0, n_tx, n_rx, n_lat, n_ax;
    const float *xs, *zs, *ejs;      // lateral pixel / depth / element coordinates in samples (coord * fs / c)
    const float *xm, *zm, *ejm;      // the same in metres, fp32-rounded (f-number decision only)
    const float *win;                // [n_rx]
    float two_f;                     // 2 * f_number (0 = no mask)
    const int *n0;                   // [plane][k][iz]  floor(U0) - n_lo
    const float *f0m;                // [plane][k][iz]  U0 - floor(U0) - 0.5
    float fcfs;
    float2 *out;                     // frame 0 of this batch
    long long out_frame_stride;      // float2 per frame
    long long out_base;              // offset of this aperture inside a frame
    long long s_lat, s_plane, s_k;   // strides (float2) of lateral index, plane index, angle index
    int n_planes, per_angle, accumulate;
    int n_frames;                    // frames in this batch
    // single-frame volume path (unpack_frame_kernel + das_volume_kernel)
    const float4 *rows;              // [event][rx elem (n_rx_max)][l_row] {mid.re, mid.im, d.re, d.im} of ONE frame, fp32
    const int2 *tab;                 // [plane][iz][k (tab_kpad, even)] {bits of f0m, n0}
    int tab_kpad;
    // mirror form of the same table (das_volume_mirror_kernel; nullptr when the geometry is not mirror-symmetric):
    // [plane < n_planes / 2][iz][slot (mtab_kpad, even)]; slots 2 i, 2 i + 1 = angles mk[2 i], mk[2 i + 1] = a pair
    // (th, -th), i < n_mpairs; then one slot per self-mirrored angle (th = 0), mk[2 n_mpairs + i], i < n_msingle
    const int2 *mtab;
    int mtab_kpad, n_mpairs, n_msingle;
    short mk[kVolMirrorMaxAngles];
};

// the interpolation weight a' = a - 0.5 of one gather: al (fp32) for full entries; ah = 16 a' rounded to fp16 for
// compact entries, whose difference term is stored / 16 in fp16 -- there the whole interpolation
// v = mid + (16 a') (d / 16) is ONE mixed-precision FMA per component (FHFMA: fp16 x fp16 product exact, fp32 addend,
// one rounding), so the only errors are the fp16 roundings of the two factors
// W2 ("exact-weight" compact entries, precision = 3): 16 a' = ah + al2 with al2 = fp16(16 a' - ah), so the weight is
// carried with 22 significant bits and the interpolation is two FHFMAs per component, v = ah d + (al2 d + mid): the
// only format error left is the fp16 rounding of the stored difference term.
struct Alpha {
    float al;
    unsigned short ah, ah2;
};
__device__ __forceinline__ float h2f_bits(unsigned short h) {
    float r;
    asm("cvt.f32.f16 %0, %1;" : "=f"(r) : "h"(h));
    return r;
}
template <bool W2 = false>
__device__ __forceinline__ Alpha make_alpha(float al) {
    Alpha a;
    a.al = al;
    a.ah = f2h_bits(kAlScale * al);
    a.ah2 = W2 ? f2h_bits(fmaf(kAlScale, al, -h2f_bits(a.ah))) : (unsigned short)0;
    return a;
}

// packed fp32x2 helpers (sm_100 FFMA2: two fp32 FMAs in one issue slot)
__device__ __forceinline__ unsigned long long pack_f2(float lo, float hi) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack_f2(unsigned long long v, float &lo, float &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long ffma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

// im_b0 / im_b1 of a compact chunk from the low bytes of its six mid words (two PRMT each)
__device__ __forceinline__ uint32_t fp24_gather(uint32_t w0, uint32_t w1, uint32_t w2) {
    return __byte_perm(__byte_perm(w0, w1, 0x0400), w2, 0x3245);
}

// Four frames (two frame pairs a, b) of a compact entry: w[0..5] = the mid words, dd[0..3] = the half2 words (dr, di)
// of the four frames (difference term / 16).
// Scalar version (generic kernel): v = mid + ah * d (one FHFMA per component), acc += (c + j s) v.
// nv = number of valid frames among the four.
template <bool W2 = false>
__device__ __forceinline__ void chunk_mac(const uint32_t (&w)[6], const uint32_t (&dd)[4], const Alpha &A, float c,
                                          float s, float *accr, float *acci, int nv = 4) {
    const uint32_t re[4] = {w[0], w[1], w[4], w[5]};
    const uint32_t im[4] = {w[2], w[3], fp24_gather(w[0], w[2], w[4]), fp24_gather(w[1], w[3], w[5])};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (i >= nv) break;
        unsigned short dr, di;
        split_h2(dd[i], dr, di);
        float mr = __uint_as_float(re[i]), mi = __uint_as_float(im[i]);
        if (W2) { mr = fhfma(A.ah2, dr, mr); mi = fhfma(A.ah2, di, mi); }
        const float vr = fhfma(A.ah, dr, mr);
        const float vi = fhfma(A.ah, di, mi);
        accr[i] = fmaf(c, vr, accr[i]); accr[i] = fmaf(-s, vi, accr[i]);
        acci[i] = fmaf(s, vr, acci[i]); acci[i] = fmaf(c, vi, acci[i]);
    }
}

__device__ __forceinline__ void split_u2(unsigned long long v, uint32_t &lo, uint32_t &hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=r"(lo), "=r"(hi) : "l"(v));
}

// Packed version (ring kernel): m01 / m23 / m45 = the mid words as loaded by three LDS.64 (already the register
// pairs (re_a0, re_a1), (im_a0, im_a1), (re_b0, re_b1)), da / db = the d words of pairs a / b.  The interpolation is
// one FHFMA per component and frame, the complex multiply-accumulate of a frame pair runs as FFMA2 on
// (frame 2p, frame 2p+1) register pairs; aR / aI are pairs of real / imaginary accumulators; CC = (c, c), SS = (s, s),
// NS = (-s, -s).  Each half is an ordinary round-to-nearest fp32 FMA, so the results are bit-identical to chunk_mac.
template <bool W2 = false>
__device__ __forceinline__ void chunk_mac2(unsigned long long m01, unsigned long long m23, unsigned long long m45,
                                           unsigned long long da, unsigned long long db, unsigned short ah,
                                           unsigned short ah2, unsigned long long CC, unsigned long long SS,
                                           unsigned long long NS, unsigned long long *aR, unsigned long long *aI) {
    // interpolation of one component: mid + (ah + ah2) d, the small residual term first
    auto lerp = [&](unsigned short d, uint32_t mid) {
        float m = __uint_as_float(mid);
        if (W2) m = fhfma(ah2, d, m);
        return fhfma(ah, d, m);
    };
    uint32_t w0, w1, w2, w3, w4, w5, d0, d1, d2, d3;
    split_u2(m01, w0, w1); split_u2(m23, w2, w3); split_u2(m45, w4, w5);
    split_u2(da, d0, d1); split_u2(db, d2, d3);
    unsigned short r0, r1, i0, i1;
    {
        split_h2(d0, r0, i0);
        split_h2(d1, r1, i1);
        const unsigned long long VR = pack_f2(lerp(r0, w0), lerp(r1, w1));
        const unsigned long long VI = pack_f2(lerp(i0, w2), lerp(i1, w3));
        aR[0] = ffma2(CC, VR, aR[0]); aR[0] = ffma2(NS, VI, aR[0]);
        aI[0] = ffma2(SS, VR, aI[0]); aI[0] = ffma2(CC, VI, aI[0]);
    }
    {
        split_h2(d2, r0, i0);
        split_h2(d3, r1, i1);
        const unsigned long long VR = pack_f2(lerp(r0, w4), lerp(r1, w5));
        const unsigned long long VI = pack_f2(lerp(i0, fp24_gather(w0, w2, w4)), lerp(i1, fp24_gather(w1, w3, w5)));
        aR[1] = ffma2(CC, VR, aR[1]); aR[1] = ffma2(NS, VI, aR[1]);
        aI[1] = ffma2(SS, VR, aI[1]); aI[1] = ffma2(CC, VI, aI[1]);
    }
}

// One frame pair of a full entry in FFMA2 (ring kernel): m = [re, re, im, im], d = [dr, dr, di, di], AA = (a', a').
__device__ __forceinline__ void pair_mac2_full(const uint4 &m, const uint4 &d, unsigned long long AA, unsigned long long CC,
                                               unsigned long long SS, unsigned long long NS, unsigned long long &aR,
                                               unsigned long long &aI) {
    const unsigned long long VR = ffma2(AA, pack_f2(__uint_as_float(d.x), __uint_as_float(d.y)),
                                        pack_f2(__uint_as_float(m.x), __uint_as_float(m.y)));
    const unsigned long long VI = ffma2(AA, pack_f2(__uint_as_float(d.z), __uint_as_float(d.w)),
                                        pack_f2(__uint_as_float(m.z), __uint_as_float(m.w)));
    aR = ffma2(CC, VR, aR); aR = ffma2(NS, VI, aR);
    aI = ffma2(SS, VR, aI); aI = ffma2(CC, VI, aI);
}

// interpolate-and-accumulate of F frames from one entry in global memory (generic kernel):
// v = mid + a' d  (a' in fp32; compact: d converted from fp16),  acc += (c + j s) v.
// Full entries are read as 16-byte units, compact entries (8-byte aligned) as 8-byte units.
template <int F, bool D32, bool W2 = false>
__device__ __forceinline__ void entry_mac(const unsigned char *ent, const Alpha &A, float c, float s, float *accr,
                                          float *acci, int nv = F) {
    if (D32) {
        const uint4 *e4 = reinterpret_cast<const uint4 *>(ent);
#pragma unroll
        for (int q = 0; q < F / 2; ++q) {        // frame pair q: m = [re, re, im, im], d = [dr, dr, di, di]
            if (2 * q >= nv) break;
            const uint4 m = __ldg(e4 + q), d = __ldg(e4 + F / 2 + q);
            const float mv[4] = {__uint_as_float(m.x), __uint_as_float(m.y), __uint_as_float(m.z), __uint_as_float(m.w)};
            const float dv[4] = {__uint_as_float(d.x), __uint_as_float(d.y), __uint_as_float(d.z), __uint_as_float(d.w)};
#pragma unroll
            for (int i = 0; i < 2; ++i) {
                const float vr = fmaf(A.al, dv[i], mv[i]), vi = fmaf(A.al, dv[2 + i], mv[2 + i]);
                const int f = 2 * q + i;
                accr[f] = fmaf(c, vr, accr[f]); accr[f] = fmaf(-s, vi, accr[f]);
                acci[f] = fmaf(s, vr, acci[f]); acci[f] = fmaf(c, vi, acci[f]);
            }
        }
    } else {
        const uint2 *e2 = reinterpret_cast<const uint2 *>(ent);
#pragma unroll
        for (int q = 0; q < F / 4; ++q) {
            if (4 * q >= nv) break;
            const uint2 a = __ldg(e2 + 3 * q), b = __ldg(e2 + 3 * q + 1), cc = __ldg(e2 + 3 * q + 2);
            const uint2 da = __ldg(e2 + (6 * F) / 8 + 2 * q), db = __ldg(e2 + (6 * F) / 8 + 2 * q + 1);
            const uint32_t w[6] = {a.x, a.y, b.x, b.y, cc.x, cc.y};
            const uint32_t dd[4] = {da.x, da.y, db.x, db.y};
            chunk_mac<W2>(w, dd, A, c, s, accr + 4 * q, acci + 4 * q, nv - 4 * q);
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Generic gather kernel: one thread = one pixel x the F frames of one group, gathers straight from the
// IQ scratch through L1/L2.  Serves per-angle slices (compound = 0), the 3-D comparator (config 4) and any
// shape the shared-memory ring kernel does not cover.  grid = (pixel blocks, frame groups, plane * angle groups).
// ---------------------------------------------------------------------------------------------------
template <int F, bool D32, bool APOD, bool W2 = false>
__global__ void __launch_bounds__(128) das_generic_kernel(DasParams P) {
    const int npix = P.n_lat * P.n_ax;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= npix) return;
    const int il = p % P.n_lat, iz = p / P.n_lat;     // lanes = lateral neighbours: their entries are adjacent in the scratch
    const int g = blockIdx.y;
    const int n_kgroups = P.per_angle ? P.n_tx : 1;
    const int plane = blockIdx.z / n_kgroups;
    const int k_begin = P.per_angle ? (int)(blockIdx.z % n_kgroups) : 0;
    const int k_end = P.per_angle ? k_begin + 1 : P.n_tx;

    const float xs = P.xs[il], zs = P.zs[iz];
    const float zs2 = zs * zs;
    float accr[F], acci[F];
#pragma unroll
    for (int f = 0; f < F; ++f) accr[f] = acci[f] = 0.f;
    const int tab0 = (plane * P.n_tx) * P.n_ax + iz;
    const int nv = min(F, P.n_frames - g * F);          // valid frames of this group (block-uniform)
    const size_t grow = (size_t)g * P.n_events * P.n_rx_max;

    for (int j = 0; j < P.n_rx; ++j) {
        const float dxs = xs - P.ejs[j];
        const float dx2 = dxs * dxs;
        const float r = sqrtf(dx2 + zs2);
        const float den = r + zs;
        const float H = den > 0.f ? __fdividef(dx2, den) : 0.f;
        float w = P.win[j];
        if (APOD) {
            if (P.two_f > 0.f) {
                const float lhs = __fmul_rn(fabsf(__fsub_rn(P.xm[il], P.ejm[j])), P.two_f);
                if (!(lhs <= P.zm[iz])) w = 0.f;
            }
            if (w == 0.f) continue;
        }
        for (int k = k_begin; k < k_end; ++k) {
            const int t = tab0 + k * P.n_ax;
            const float upm = P.f0m[t] + H;
            const float tt = upm + kMagic;
            const float al = upm - (tt - kMagic);
            const int idx = P.n0[t] + (__float_as_int(tt) - kMagicBits);
            float s, c;
            __sincosf(fmaf(kTwoPi * P.fcfs, al, 0.5f * kTwoPi * P.fcfs), &s, &c);     // E(a), a = al + 0.5 in [0, 1]
            if (APOD) { s *= w; c *= w; }
            const unsigned char *ent = P.iq + ((grow + (size_t)(P.e0 + k) * P.n_rx_max + j) * P.l_row + idx) * entry_bytes(F, D32);
            entry_mac<F, D32, W2>(ent, make_alpha<W2>(al), c, s, accr, acci, nv);
        }
    }
    const long long o = P.out_base + (long long)il * P.s_lat + (long long)plane * P.s_plane +
                        (long long)k_begin * P.s_k + iz;
#pragma unroll
    for (int f = 0; f < F; ++f) {
        const int fr = g * F + f;
        if (fr < P.n_frames) {
            float2 *dst = P.out + (long long)fr * P.out_frame_stride + o;
            float2 v = make_float2(accr[f], acci[f]);
            if (P.accumulate) { const float2 old = *dst; v.x += old.x; v.y += old.y; }
            *dst = v;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Single-frame volume path (config 4, the conventional comparator, is ONE frame: the frame groups of the scratch,
// which let the projection kernels share all index arithmetic between 4 / 12 frames, have nothing to share there).
// unpack_frame_kernel copies frame f of a group out of the scratch entries into plain fp32 rows
// {mid.re, mid.im, d.re, d.im} (16 B per sample: one LDG.128 per gather-sample); das_volume_kernel gathers from them.
// ---------------------------------------------------------------------------------------------------
template <int F, bool D32>
__global__ void __launch_bounds__(256) unpack_frame_kernel(const unsigned char *iq, float4 *rows, long long n_entries, int f) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n_entries) return;
    const unsigned char *ep = iq + i * entry_bytes(F, D32);
    float4 o;
    if (D32) {
        const float *mid = reinterpret_cast<const float *>(ep) + 4 * (f >> 1) + (f & 1);
        const float *d = reinterpret_cast<const float *>(ep + 8 * F) + 4 * (f >> 1) + (f & 1);
        o = make_float4(mid[0], mid[2], d[0], d[2]);
    } else {
        const uint32_t *w = reinterpret_cast<const uint32_t *>(ep + 24 * (f >> 2));
        const int i4 = f & 3;
        uint32_t re, im;
        if (i4 < 2) { re = w[i4]; im = w[2 + i4]; }
        else { re = w[2 + i4]; im = fp24_gather(w[i4 - 2], w[i4], w[i4 + 2]); }
        const uint32_t dw = reinterpret_cast<const uint32_t *>(ep + 6 * F)[f];
        const float2 dd = __half22float2(*reinterpret_cast<const __half2 *>(&dw));
        // fp24 = the top three bytes of the fp32 value (truncated): the low byte is set to the middle of the cell.
        // An all-zero value (edge rule) stays exactly zero.
        const uint32_t rb = re & 0xFFFFFF00u, ib = im & 0xFFFFFF00u;
        o = make_float4(__uint_as_float(rb ? (rb | 0x80u) : 0u), __uint_as_float(ib ? (ib | 0x80u) : 0u),
                        dd.x * kAlScale, dd.y * kAlScale);
    }
    rows[i] = o;
}

// One thread = one (lateral, depth) pixel x NP consecutive planes (the y pixels of the volume for the row-transmit
// events, the x pixels for the column-transmit ones).  The receive excess H(pixel, element) is shared by the planes
// and the angles; neighbouring planes differ by a fraction of a sample in transmit delay, so their gathers hit the
// same L1 lines.  Per gather-sample: half a broadcast LDG.128 of {f0m, n0} x 2 angles, floor / fraction by the magic constant,
// E(a) by two MUFU, one LDG.128 of the fp32 entry, 2 FMA for the interpolation, 4 FMA for the complex
// multiply-accumulate.  grid = (pixel blocks, plane groups).
template <int NP, bool APOD>
__global__ void __launch_bounds__(128) das_volume_kernel(DasParams P) {
    const int npix = P.n_lat * P.n_ax;
    const int p = blockIdx.x * 128 + threadIdx.x;
    if (p >= npix) return;
    const int il = p % P.n_lat, iz = p / P.n_lat;
    const int plane0 = blockIdx.y * NP;
    const float xs = P.xs[il], zs = P.zs[iz];
    const float zs2 = zs * zs;
    const float th = kTwoPi * P.fcfs, th0 = 0.5f * th;
    float ar[NP], ai[NP];
    const int2 *tq[NP];
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        ar[q] = ai[q] = 0.f;
        tq[q] = P.tab + ((size_t)min(plane0 + q, P.n_planes - 1) * P.n_ax + iz) * P.tab_kpad;
        asm("" : "+l"(tq[q]));      // keep it a pointer register pair (address = one IMAD.WIDE per load)
    }
    const size_t ev_stride = (size_t)P.n_rx_max * P.l_row;
    // one gather-sample of plane q: t = {bits of f0m, n0} of (plane, angle, depth row), row = the (angle, element) row
    auto term = [&](int tf, int tn, const float4 *row, float H, float w, float &accr, float &acci) {
        const float upm = __int_as_float(tf) + H;
        const float tt = upm + kMagic;
        const float al = upm - (tt - kMagic);
        const int idx = tn + (__float_as_int(tt) - kMagicBits);
        float s, c;
        __sincosf(fmaf(th, al, th0), &s, &c);       // E(a), a = al + 0.5 in [0, 1]
        if (APOD) { s *= w; c *= w; }
        const float4 e = __ldg(row + idx);
        const float vr = fmaf(al, e.z, e.x), vi = fmaf(al, e.w, e.y);
        accr = fmaf(c, vr, accr); accr = fmaf(-s, vi, accr);
        acci = fmaf(s, vr, acci); acci = fmaf(c, vi, acci);
    };
    for (int j = 0; j < P.n_rx; ++j) {
        const float dxs = xs - P.ejs[j];
        const float dx2 = dxs * dxs;
        const float den = sqrtf(dx2 + zs2) + zs;
        const float H = den > 0.f ? __fdividef(dx2, den) : 0.f;
        float w = 1.f;
        if (APOD) {
            w = P.win[j];
            if (P.two_f > 0.f) {
                const float lhs = __fmul_rn(fabsf(__fsub_rn(P.xm[il], P.ejm[j])), P.two_f);
                if (!(lhs <= P.zm[iz])) w = 0.f;
            }
            if (w == 0.f) continue;
        }
        const float4 *row = P.rows + ((size_t)P.e0 * P.n_rx_max + j) * P.l_row;
        // the table rows are [plane][iz][angle], padded to an even angle count: one LDG.128 serves two angles
        int k = 0;
        for (; k + 1 < P.n_tx; k += 2, row += 2 * ev_stride) {
            const float4 *row1 = row + ev_stride;
            asm("" : "+l"(row), "+l"(row1));
#pragma unroll
            for (int q = 0; q < NP; ++q) {
                const int4 t = __ldg(reinterpret_cast<const int4 *>(tq[q] + k));
                term(t.x, t.y, row, H, w, ar[q], ai[q]);
                term(t.z, t.w, row1, H, w, ar[q], ai[q]);
            }
        }
        if (k < P.n_tx) {
#pragma unroll
            for (int q = 0; q < NP; ++q) {
                const int2 t = __ldg(tq[q] + k);
                term(t.x, t.y, row, H, w, ar[q], ai[q]);
            }
        }
    }
#pragma unroll
    for (int q = 0; q < NP; ++q) {
        if (plane0 + q >= P.n_planes) break;
        float2 *dst = P.out + P.out_base + (long long)il * P.s_lat + (long long)(plane0 + q) * P.s_plane + iz;
        float2 v = make_float2(ar[q], ai[q]);
        if (P.accumulate) { const float2 old = *dst; v.x += old.x; v.y += old.y; }
        *dst = v;
    }
}

// The volume DAS on MIRROR PAIRS.  On a centred grid with a symmetric angle set the transmit delay of (plane y, angle th)
// equals that of (plane -y, angle -th): the split delay, the entry index, the interpolation weight and the phasor E(a)
// of a term -- all that a single frame cannot share with other frames -- are computed once and serve two gathers (row
// of event th into plane y, row of event -th into plane -y); the table entry is read once as well.  An angle th = 0 has
// the same delay on every plane pair: one gather serves both planes.  Thread = one (lateral, depth) pixel x NPH planes
// of the lower half and their mirrors; lanes = lateral neighbours as in das_volume_kernel.
template <int NPH, bool APOD>
__global__ void __launch_bounds__(128) das_volume_mirror_kernel(DasParams P) {
    const int npix = P.n_lat * P.n_ax;
    const int p = blockIdx.x * 128 + threadIdx.x;
    if (p >= npix) return;
    const int il = p % P.n_lat, iz = p / P.n_lat;
    const int half = P.n_planes / 2, plane0 = blockIdx.y * NPH;
    const float xs = P.xs[il], zs = P.zs[iz];
    const float zs2 = zs * zs;
    const float th = kTwoPi * P.fcfs, th0 = 0.5f * th;
    float ar[2][NPH], ai[2][NPH];
    const int2 *tq[NPH];
#pragma unroll
    for (int q = 0; q < NPH; ++q) {
        ar[0][q] = ai[0][q] = ar[1][q] = ai[1][q] = 0.f;
        tq[q] = P.mtab + ((size_t)min(plane0 + q, half - 1) * P.n_ax + iz) * P.mtab_kpad;
        asm("" : "+l"(tq[q]));
    }
    const size_t ev_stride = (size_t)P.n_rx_max * P.l_row;
    struct Idx { int idx; float al, c, s; };
    auto index_of = [&](int tf, int tn, float H, float w) {
        Idx r;
        const float upm = __int_as_float(tf) + H;
        const float tt = upm + kMagic;
        r.al = upm - (tt - kMagic);
        r.idx = tn + (__float_as_int(tt) - kMagicBits);
        __sincosf(fmaf(th, r.al, th0), &r.s, &r.c);          // E(a), a = al + 0.5 in [0, 1]
        if (APOD) { r.s *= w; r.c *= w; }
        return r;
    };
    auto mac = [&](const float4 e, const Idx &x, float &accr, float &acci) {
        const float vr = fmaf(x.al, e.z, e.x), vi = fmaf(x.al, e.w, e.y);
        accr = fmaf(x.c, vr, accr); accr = fmaf(-x.s, vi, accr);
        acci = fmaf(x.s, vr, acci); acci = fmaf(x.c, vi, acci);
    };
    const float4 *rows0 = P.rows + (size_t)P.e0 * ev_stride;
    for (int j = 0; j < P.n_rx; ++j) {
        const float dxs = xs - P.ejs[j];
        const float dx2 = dxs * dxs;
        const float den = sqrtf(dx2 + zs2) + zs;
        const float H = den > 0.f ? __fdividef(dx2, den) : 0.f;
        float w = 1.f;
        if (APOD) {
            w = P.win[j];
            if (P.two_f > 0.f) {
                const float lhs = __fmul_rn(fabsf(__fsub_rn(P.xm[il], P.ejm[j])), P.two_f);
                if (!(lhs <= P.zm[iz])) w = 0.f;
            }
            if (w == 0.f) continue;
        }
        const float4 *rowj = rows0 + (size_t)j * P.l_row;
        for (int i = 0; i < P.n_mpairs; ++i) {
            const float4 *ra = rowj + (size_t)P.mk[2 * i] * ev_stride, *rb = rowj + (size_t)P.mk[2 * i + 1] * ev_stride;
            asm("" : "+l"(ra), "+l"(rb));
#pragma unroll
            for (int q = 0; q < NPH; ++q) {
                const int4 t = __ldg(reinterpret_cast<const int4 *>(tq[q] + 2 * i));
                const Idx x1 = index_of(t.x, t.y, H, w);      // (plane, th) and (mirror plane, -th)
                mac(__ldg(ra + x1.idx), x1, ar[0][q], ai[0][q]);
                mac(__ldg(rb + x1.idx), x1, ar[1][q], ai[1][q]);
                const Idx x2 = index_of(t.z, t.w, H, w);      // (plane, -th) and (mirror plane, th)
                mac(__ldg(rb + x2.idx), x2, ar[0][q], ai[0][q]);
                mac(__ldg(ra + x2.idx), x2, ar[1][q], ai[1][q]);
            }
        }
        for (int i = 0; i < P.n_msingle; ++i) {
            const float4 *ra = rowj + (size_t)P.mk[2 * P.n_mpairs + i] * ev_stride;
#pragma unroll
            for (int q = 0; q < NPH; ++q) {
                const int2 t = __ldg(tq[q] + 2 * P.n_mpairs + i);
                const Idx x = index_of(t.x, t.y, H, w);
                const float4 e = __ldg(ra + x.idx);
                mac(e, x, ar[0][q], ai[0][q]);
                mac(e, x, ar[1][q], ai[1][q]);
            }
        }
    }
#pragma unroll
    for (int q = 0; q < NPH; ++q) {
        if (plane0 + q >= half) break;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int pl = h == 0 ? plane0 + q : P.n_planes - 1 - (plane0 + q);
            float2 *dst = P.out + P.out_base + (long long)il * P.s_lat + (long long)pl * P.s_plane + iz;
            float2 v = make_float2(ar[h][q], ai[h][q]);
            if (P.accumulate) { const float2 old = *dst; v.x += old.x; v.y += old.y; }
            *dst = v;
        }
    }
}

// Register-only FFMA loop for the FP32 roofline denominator.
__global__ void __launch_bounds__(256) fp32_peak_kernel(float *sink, int iters, float a, float b) {
    float x[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456f) sink[0] = s;
}

}  // namespace ulm
