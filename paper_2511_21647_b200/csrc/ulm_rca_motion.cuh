// ulm_rca_motion.cuh -- Fourier-domain NCC rigid motion estimation on the Stage-1 slices (Section
// II.A.3; reading = DESIGN.md section 13) for sm_100a.
//
//   ME-1  a(l, i) = |S(l, i)| (B-mode), mean removed, zero-padded to N1 x N2 = next powers of two >= n_lat, n_ax
//   ME-2  c(d) = IFFT2( FFT2(a_f) conj(FFT2(a_ref)) ) / (|a_f| |a_ref|)          ("two forward and one inverse" transform)
//   ME-3  integer argmax of c (first in row-major order), signed shift, 3-point parabola per axis
//   ME-4  per frame: mean over the row-tx events -> (dx, dz_RC), over the column-tx events -> (dy, dz_CR),
//         motion = (dx, dy, (dz_RC + dz_CR) / 2) in metres
//
// The paper uses cuFFT (cufftPlanMany) plus a correlation kernel; here the transforms are hand-written: one warp per
// line, the whole transform in registers (R-point butterflies per lane, 32-point butterflies across the lanes by
// shuffles; forward = decimation in frequency, inverse = the same network backwards, so no bit-reversal pass exists),
// every pass over global memory coalesced, and the product with the reference spectrum and the inverse lateral
// transform fused into the forward lateral pass:
//   motion_stats_kernel     mean and mean-removed energy of every B-mode image (one pass)
//   motion_fwd_z_kernel     FFT along depth of 32 lateral lines per CTA, written transposed  T1[img][kz][l]; an image =
//                           TWO frames, (a_2p, a_2p+1) as real / imaginary part: correlating with the fixed reference is
//                           linear in the frame, so Re / Im of the final map are the two frames' correlation maps
//   motion_lat_kernel<REF>  FFT along the lateral axis of 32 kz rows per CTA; REF: store the reference spectrum;
//                           else multiply by its conjugate, inverse lateral FFT, write transposed  T2[img][dl][kz]
//   motion_peak_kernel      inverse FFT along depth line by line, running argmax, neighbours, parabola -> (d_lat, d_ax, ncc)
//   motion_combine_kernel   ME-4
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace ulm {

struct MoEvents {                 // per-event geometry (device arrays)
    const long long *off;         // float2 offset of the event's slice inside a frame
    const int *n_lat, *n_ax;      // slice size
    const int *log1, *log2;       // log2 of the padded FFT sizes N1 (lateral), N2 (axial)
    const long long *t1_off, *t2_off, *ref_off;   // float2 offsets of the event's block inside one frame's T1 / T2 and inside F_ref
};

struct MoParams {
    const float2 *x;              // slices [frame][event][lat][ax]
    long long frame_stride;
    MoEvents ev;
    int n_events, n_frames, ref_frame;
    int n_pairs;                  // packed images: frames (2 p, 2 p + 1) in the real / imaginary part; image n_pairs = the reference frame alone
    float2 *stats;                // [frame][event] {mean, sum of squares of the mean-removed image}
    float2 *t1, *t2, *fref;       // scratch
    long long t1_frame, t2_frame; // float2 per packed image of T1 / T2
    const float2 *tw;             // twiddles exp(-2 pi i k / 1024), k < 1024
    float4 *per_event;            // [frame][event] {d_lat px, d_ax px, ncc, 0}
    float4 *motion;               // [frame] {dx, dy, dz (m), mean ncc}
    int n_row_tx;
    float dlat[2], dz[2];         // grid steps of the x-z / y-z slices
};

constexpr int kMoMaxN = 512;      // padded FFT length at most
constexpr int kMoLines = 32;      // lines per CTA of the transposing kernels
constexpr int kMoThreads = 256;

// ------------------------------------------------------------------------------------------------------------------
// Warp FFT in registers.  N = 32 R points (R = 2^LOGR <= 16): lane m holds x[32 r + m] in v[r] (the layout of a
// coalesced load).  N = R x 32 Cooley-Tukey:
//     X[k1 + R k2] = sum_m W_32^{m k2} W_N^{m k1} sum_r x[32 r + m] W_R^{r k1}
// mo_fft_dif: R-point DIF butterflies in registers, twiddle W_N^{m k1}, 32-point DIF butterflies across the lanes with
// xor shuffles.  Result in PERMUTED order: register slot q of lane l holds X[brev_R(q) + R brev_5(l)]
// (mo_perm).  mo_fft_dit runs the same network backwards (DIT butterflies with the conjugate twiddles): it takes the
// permuted order and returns natural order, x[32 r + m] in v[r] of lane m.  A forward transform, a pointwise product
// and the inverse therefore never need a bit-reversal pass, and no stage goes through shared memory.
// SIGN = -1: exponent -2 pi i nk/N (forward); +1: the (unnormalised) inverse.  tw[k] = exp(-2 pi i k / 1024).
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float2 mo_cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
template <int SIGN> __device__ __forceinline__ float2 mo_tw(const float2 *tw, int idx) {
    float2 w = __ldg(tw + idx);
    if (SIGN > 0) w.y = -w.y;
    return w;
}
// exp(SIGN 2 pi i j / len) for the register butterflies, len <= 16: compile-time constants after unrolling
template <int SIGN> __device__ __forceinline__ float2 mo_w16(int j16) {
    constexpr float c[8] = {1.f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f, 0.f, -0.38268343236508977f,
                            -0.70710678118654752f, -0.92387953251128674f};
    constexpr float s[8] = {0.f, 0.38268343236508977f, 0.70710678118654752f, 0.92387953251128674f, 1.f, 0.92387953251128674f,
                            0.70710678118654752f, 0.38268343236508977f};
    return make_float2(c[j16], SIGN > 0 ? s[j16] : -s[j16]);
}
__host__ __device__ constexpr int mo_brev_c(int q, int bits) {
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((q >> b) & 1) << (bits - 1 - b);
    return r;
}
// frequency index held by (register slot q, lane l) after mo_fft_dif
template <int LOGR> __device__ __forceinline__ int mo_perm(int q, int l) {
    return mo_brev_c(q, LOGR) + ((int)(__brev((unsigned)l) >> 27) << LOGR);
}

template <int LOGR, int SIGN>
__device__ __forceinline__ void mo_fft_dif(float2 (&v)[1 << LOGR], const float2 *tw, int lane) {
    constexpr int R = 1 << LOGR;
    // R-point DIF over the register index (natural r -> bit-reversed slot)
#pragma unroll
    for (int len = R; len >= 2; len >>= 1) {
        const int half = len / 2;
#pragma unroll
        for (int base = 0; base < R; base += len)
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const float2 u = v[base + j], w = v[base + j + half];
                v[base + j] = make_float2(u.x + w.x, u.y + w.y);
                const float2 d = make_float2(u.x - w.x, u.y - w.y);
                v[base + j + half] = j == 0 ? d : mo_cmul(d, mo_w16<SIGN>(j * (16 / len)));
            }
    }
    // twiddle W_N^{m k1}, k1 = brev_R(slot)
#pragma unroll
    for (int q = 1; q < R; ++q) v[q] = mo_cmul(v[q], mo_tw<SIGN>(tw, (lane * mo_brev_c(q, LOGR) * (32 >> LOGR)) & 1023));
    // 32-point DIF across the lanes
#pragma unroll
    for (int h = 16; h >= 1; h >>= 1) {
        const bool upper = (lane & h) != 0;
        const float2 w = mo_tw<SIGN>(tw, (lane & (h - 1)) * (512 / h));
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const float bx = __shfl_xor_sync(0xffffffffu, v[q].x, h), by = __shfl_xor_sync(0xffffffffu, v[q].y, h);
            if (upper) v[q] = mo_cmul(make_float2(bx - v[q].x, by - v[q].y), w);
            else v[q] = make_float2(v[q].x + bx, v[q].y + by);
        }
    }
}

template <int LOGR, int SIGN>
__device__ __forceinline__ void mo_fft_dit(float2 (&v)[1 << LOGR], const float2 *tw, int lane) {
    constexpr int R = 1 << LOGR;
#pragma unroll
    for (int h = 1; h <= 16; h <<= 1) {
        const bool upper = (lane & h) != 0;
        const float2 w = mo_tw<SIGN>(tw, (lane & (h - 1)) * (512 / h));
#pragma unroll
        for (int q = 0; q < R; ++q) {
            const float2 t = upper ? mo_cmul(v[q], w) : v[q];
            const float bx = __shfl_xor_sync(0xffffffffu, t.x, h), by = __shfl_xor_sync(0xffffffffu, t.y, h);
            v[q] = upper ? make_float2(bx - t.x, by - t.y) : make_float2(t.x + bx, t.y + by);
        }
    }
#pragma unroll
    for (int q = 1; q < R; ++q) v[q] = mo_cmul(v[q], mo_tw<SIGN>(tw, (lane * mo_brev_c(q, LOGR) * (32 >> LOGR)) & 1023));
#pragma unroll
    for (int len = 2; len <= R; len <<= 1) {
        const int half = len / 2;
#pragma unroll
        for (int base = 0; base < R; base += len)
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const float2 u = v[base + j];
                const float2 t = j == 0 ? v[base + j + half] : mo_cmul(v[base + j + half], mo_w16<SIGN>(j * (16 / len)));
                v[base + j] = make_float2(u.x + t.x, u.y + t.y);
                v[base + j + half] = make_float2(u.x - t.x, u.y - t.y);
            }
    }
}

// call(LOGR) for the run-time transform length 2^logn (32 .. 512), LOGR = logn - 5 as a compile-time constant
#define ULM_MO_DISPATCH(logn, call)                    \
    switch (logn) {                                    \
        case 5: call(0); break;                        \
        case 6: call(1); break;                        \
        case 7: call(2); break;                        \
        case 8: call(3); break;                        \
        default: call(4); break;                       \
    }

// One pass over the image: sums of (a - c) and (a - c)^2 with the pilot value c = a[0] (a large common offset of the
// image then cancels before the squares are taken); mean = c + S1 / n, mean-removed energy = S2 - S1^2 / n.
__global__ void __launch_bounds__(kMoThreads) motion_stats_kernel(const __grid_constant__ MoParams P) {
    const int e = blockIdx.x, f = blockIdx.y;
    const int n = P.ev.n_lat[e] * P.ev.n_ax[e];
    const float2 *x = P.x + (long long)f * P.frame_stride + P.ev.off[e];
    __shared__ float red[2][kMoThreads / 32];
    const float2 x0 = __ldg(x);
    const float c = sqrtf(x0.x * x0.x + x0.y * x0.y);
    float s1 = 0.f, s2 = 0.f;
    auto add = [&](float re, float im) { const float d = sqrtf(re * re + im * im) - c; s1 += d; s2 = fmaf(d, d, s2); };
    if ((reinterpret_cast<unsigned long long>(x) & 15ull) == 0) {
        const float4 *x4 = reinterpret_cast<const float4 *>(x);
        const int n4 = n >> 1;
        int i = threadIdx.x;
        for (; i + 3 * kMoThreads < n4; i += 4 * kMoThreads) {
            float4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) v[u] = __ldg(x4 + i + u * kMoThreads);
#pragma unroll
            for (int u = 0; u < 4; ++u) { add(v[u].x, v[u].y); add(v[u].z, v[u].w); }
        }
        for (; i < n4; i += kMoThreads) { const float4 v = __ldg(x4 + i); add(v.x, v.y); add(v.z, v.w); }
        if ((n & 1) && threadIdx.x == 0) { const float2 v = __ldg(x + n - 1); add(v.x, v.y); }
    } else {
        for (int i = threadIdx.x; i < n; i += kMoThreads) { const float2 v = __ldg(x + i); add(v.x, v.y); }
    }
    for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(0xffffffffu, s1, o); s2 += __shfl_xor_sync(0xffffffffu, s2, o); }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = s1; red[1][threadIdx.x >> 5] = s2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        float t1 = 0.f, t2 = 0.f;
        for (int i = 0; i < kMoThreads / 32; ++i) { t1 += red[0][i]; t2 += red[1][i]; }
        P.stats[(long long)f * P.n_events + e] = make_float2(c + t1 / (float)n, fmaxf(t2 - t1 * t1 / (float)n, 0.f));
    }
}

// depth FFT of the CTA's 32 lateral lines (one warp per line, 4 lines per warp) into the shared-memory tile s[line][position]
template <int LOGR>
__device__ __forceinline__ void mo_fwd_z_lines(const MoParams &P, float2 *s, int rs, const float2 *xa, const float2 *xb, int n_lat,
                                               int n_ax, int l0, float mean_a, float mean_b, int warp, int lane) {
    constexpr int R = 1 << LOGR;
    // the raw samples of the warp's next line are requested before the transform of the current one
    float2 ca[R], cb[R];
    auto fetch = [&](int li) {
        const int l = l0 + li;
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = 32 * r + lane;
            ca[r] = cb[r] = make_float2(0.f, 0.f);
            if (l < n_lat && i < n_ax) {
                ca[r] = __ldg(xa + (long long)l * n_ax + i);
                if (xb) cb[r] = __ldg(xb + (long long)l * n_ax + i);
            }
        }
    };
    fetch(warp);
    for (int li = warp; li < kMoLines; li += kMoThreads / 32) {
        const int l = l0 + li;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int i = 32 * r + lane;
            float a = 0.f, b = 0.f;
            if (i < n_ax) {
                a = sqrtf(ca[r].x * ca[r].x + ca[r].y * ca[r].y) - mean_a;
                if (xb) b = sqrtf(cb[r].x * cb[r].x + cb[r].y * cb[r].y) - mean_b;
            }
            v[r] = make_float2(a, b);
        }
        if (li + kMoThreads / 32 < kMoLines) fetch(li + kMoThreads / 32);
        if (l >= n_lat) continue;                                      // warp-uniform; such lines are written as zeros below
        mo_fft_dif<LOGR, -1>(v, P.tw, lane);
#pragma unroll
        for (int q = 0; q < R; ++q) s[li * rs + 32 * q + lane] = v[q];
    }
}

// grid = (lateral tiles of 32 lines, events, packed images + 1): image p < n_pairs = frames (2 p, 2 p + 1) as real and
// imaginary part (the correlation with the fixed reference is linear in the frame, so the whole transform chain runs once
// for two frames and the real / imaginary part of the result is the correlation map of the first / second one); image
// n_pairs = the reference frame alone (its spectrum is the other factor and must stay unmixed)
#ifndef ULM_MO_FZ
#define ULM_MO_FZ 2
#endif
__global__ void __launch_bounds__(kMoThreads, ULM_MO_FZ) motion_fwd_z_kernel(const __grid_constant__ MoParams P) {
    extern __shared__ __align__(16) unsigned char mo_smem[];
    const int e = blockIdx.y, img = blockIdx.z;
    const int fa = img < P.n_pairs ? 2 * img : P.ref_frame, fb = (img < P.n_pairs && 2 * img + 1 < P.n_frames) ? 2 * img + 1 : -1;
    const int n_lat = P.ev.n_lat[e], n_ax = P.ev.n_ax[e], log2_ = P.ev.log2[e], n2 = 1 << log2_;
    const int l0 = blockIdx.x * kMoLines;
    if (l0 >= n_lat) return;
    float2 *s = reinterpret_cast<float2 *>(mo_smem);                  // [32][n2 + 1]
    const int rs = n2 + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float mean_a = P.stats[(long long)fa * P.n_events + e].x, mean_b = fb >= 0 ? P.stats[(long long)fb * P.n_events + e].x : 0.f;
    const float2 *xa = P.x + (long long)fa * P.frame_stride + P.ev.off[e];
    const float2 *xb = fb >= 0 ? P.x + (long long)fb * P.frame_stride + P.ev.off[e] : nullptr;
#define ULM_MO_CALL(LR) mo_fwd_z_lines<LR>(P, s, rs, xa, xb, n_lat, n_ax, l0, mean_a, mean_b, warp, lane)
    ULM_MO_DISPATCH(log2_, ULM_MO_CALL)
#undef ULM_MO_CALL
    __syncthreads();
    // transposed, coalesced write: T1[image][event block][kz position][l]  (kz in the permuted order of mo_fft_dif: every
    // later pass treats the kz rows independently and the final inverse depth transform takes exactly that order)
    float2 *t1 = P.t1 + (long long)img * P.t1_frame + P.ev.t1_off[e];
    const int n_lat_p = (n_lat + 31) / 32 * 32;
    for (int kz = warp; kz < n2; kz += kMoThreads / 32)
        t1[(long long)kz * n_lat_p + l0 + lane] = (l0 + lane < n_lat) ? s[lane * rs + kz] : make_float2(0.f, 0.f);
}

// lateral FFT of the CTA's 32 kz rows; REF: store the spectrum (permuted order); else product with the conjugate
// reference spectrum (same permuted order on both sides), inverse lateral FFT (natural order out) into the tile s[row][dl]
template <int LOGR, bool REF>
__device__ __forceinline__ void mo_lat_rows(const MoParams &P, float2 *s, int rs, const float2 *t1, float2 *fref, int n_lat,
                                            int n_lat_p, int n1, int kz0, int warp, int lane) {
    constexpr int R = 1 << LOGR;
    float2 nx[R];                                                      // the next row, requested a row ahead
    auto fetch = [&](int ri) {
        const int kz = kz0 + ri;                                       // n2 is a multiple of 32: always a valid row
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int l = 32 * r + lane;
            nx[r] = l < n_lat ? __ldg(t1 + (long long)kz * n_lat_p + l) : make_float2(0.f, 0.f);
        }
    };
    fetch(warp);
    for (int ri = warp; ri < kMoLines; ri += kMoThreads / 32) {
        const int kz = kz0 + ri;
        float2 v[R];
#pragma unroll
        for (int r = 0; r < R; ++r) v[r] = nx[r];
        if (ri + kMoThreads / 32 < kMoLines) fetch(ri + kMoThreads / 32);
        mo_fft_dif<LOGR, -1>(v, P.tw, lane);
        if (REF) {
#pragma unroll
            for (int q = 0; q < R; ++q) fref[(long long)kz * n1 + 32 * q + lane] = v[q];
        } else {
#pragma unroll
            for (int q = 0; q < R; ++q) {
                const float2 a = v[q], r = __ldg(fref + (long long)kz * n1 + 32 * q + lane);
                v[q] = make_float2(a.x * r.x + a.y * r.y, a.y * r.x - a.x * r.y);     // a conj(r)
            }
            mo_fft_dit<LOGR, +1>(v, P.tw, lane);
#pragma unroll
            for (int r = 0; r < R; ++r) s[ri * rs + 32 * r + lane] = v[r];
        }
    }
}

// grid = (kz tiles of 32 rows, events, packed images [REF: 1, the reference image])
#ifndef ULM_MO_LAT
#define ULM_MO_LAT 2
#endif
template <bool REF>
__global__ void __launch_bounds__(kMoThreads, ULM_MO_LAT) motion_lat_kernel(const __grid_constant__ MoParams P) {
    extern __shared__ __align__(16) unsigned char mo_smem[];
    const int e = blockIdx.y, img = REF ? P.n_pairs : blockIdx.z;
    const int n_lat = P.ev.n_lat[e], log1 = P.ev.log1[e], n1 = 1 << log1, n2 = 1 << P.ev.log2[e];
    const int kz0 = blockIdx.x * kMoLines;
    if (kz0 >= n2) return;
    const int rs = n1 + 1;
    float2 *s = reinterpret_cast<float2 *>(mo_smem);                  // [32][n1 + 1]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_lat_p = (n_lat + 31) / 32 * 32;
    const float2 *t1 = P.t1 + (long long)img * P.t1_frame + P.ev.t1_off[e];
    float2 *fref = P.fref + P.ev.ref_off[e];
#define ULM_MO_CALL(LR) mo_lat_rows<LR, REF>(P, s, rs, t1, fref, n_lat, n_lat_p, n1, kz0, warp, lane)
    ULM_MO_DISPATCH(log1, ULM_MO_CALL)
#undef ULM_MO_CALL
    if (REF) return;
    __syncthreads();
    // transposed, coalesced write: T2[image][event block][dl][kz position]
    float2 *t2 = P.t2 + (long long)img * P.t2_frame + P.ev.t2_off[e];
    for (int dl = warp; dl < n1; dl += kMoThreads / 32) t2[(long long)dl * n2 + kz0 + lane] = s[lane * rs + dl];
}

// running maxima of the two correlation maps (real part: first frame of the image, imaginary part: second frame) over the
// lateral-shift lines of one warp: inverse depth FFT of each line in registers, the values to the warp's rows in shared
// memory (the depth neighbours of a new maximum are read from them)
struct MoBest { float val, m, p; int idx; };
__device__ __forceinline__ void mo_best_update(MoBest &B, const float *row, float best, int bi, int dl, int n2) {
    for (int o = 16; o > 0; o >>= 1) {
        const float ov = __shfl_xor_sync(0xffffffffu, best, o);
        const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
        if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
    }
    const int idx = dl * n2 + bi;
    if (best > B.val || (best == B.val && idx < B.idx)) {
        B.val = best; B.idx = idx;
        B.m = row[(bi + n2 - 1) & (n2 - 1)];
        B.p = row[(bi + 1) & (n2 - 1)];
    }
}
template <int LOGR>
__device__ __forceinline__ void mo_peak_lines(const MoParams &P, float *row_a, float *row_b, const float2 *t2, int n1, int n2,
                                              int warp, int lane, MoBest &Ba, MoBest &Bb) {
    constexpr int R = 1 << LOGR;
    float2 nx[R];                                                      // the next line, requested a line ahead
    auto fetch = [&](int dl) {
#pragma unroll
        for (int q = 0; q < R; ++q) nx[q] = __ldg(t2 + (long long)dl * n2 + 32 * q + lane);
    };
    if (warp < n1) fetch(warp);
    for (int dl = warp; dl < n1; dl += kMoThreads / 32) {
        float2 v[R];
#pragma unroll
        for (int q = 0; q < R; ++q) v[q] = nx[q];
        if (dl + kMoThreads / 32 < n1) fetch(dl + kMoThreads / 32);
        mo_fft_dit<LOGR, +1>(v, P.tw, lane);
        float best_a = -3.0e38f, best_b = -3.0e38f;
        int bi_a = 0, bi_b = 0;
#pragma unroll
        for (int r = 0; r < R; ++r) {                                  // depth shift 32 r + lane, ascending: first maximum
            row_a[32 * r + lane] = v[r].x;
            row_b[32 * r + lane] = v[r].y;
            if (v[r].x > best_a) { best_a = v[r].x; bi_a = 32 * r + lane; }
            if (v[r].y > best_b) { best_b = v[r].y; bi_b = 32 * r + lane; }
        }
        __syncwarp();
        mo_best_update(Ba, row_a, best_a, bi_a, dl, n2);
        mo_best_update(Bb, row_b, best_b, bi_b, dl, n2);
        __syncwarp();
    }
}

// c(dl, dz) by one direct inverse DFT sum over the (permuted) kz positions of line dl:
// sum_kz T2[dl][pos] exp(+2 pi i kz dz / n2)  (real part: first frame, imaginary part: second frame)
template <int LOGR>
__device__ __forceinline__ float2 mo_direct(const MoParams &P, const float2 *t2, int dl, int dz, int n2, int lane) {
    float ar = 0.f, ai = 0.f;
    for (int pos = lane; pos < n2; pos += 32) {
        const int kz = mo_perm<LOGR>(pos >> 5, pos & 31);
        const float2 v = __ldg(t2 + (long long)dl * n2 + pos);
        const float2 w = __ldg(P.tw + ((kz * dz) & (n2 - 1)) * (32 >> LOGR));      // exp(-2 pi i kz dz / n2); the inverse uses its conjugate
        ar += v.x * w.x + v.y * w.y;                                                   // v conj(w)
        ai += v.y * w.x - v.x * w.y;
    }
    for (int o = 16; o > 0; o >>= 1) { ar += __shfl_xor_sync(0xffffffffu, ar, o); ai += __shfl_xor_sync(0xffffffffu, ai, o); }
    return make_float2(ar, ai);
}

// grid = (events, packed images): inverse FFT along depth of every lateral-shift line, running maxima, sub-pixel peaks of
// the image's two frames
#ifndef ULM_MO_PK
#define ULM_MO_PK 2
#endif
__global__ void __launch_bounds__(kMoThreads, ULM_MO_PK) motion_peak_kernel(const __grid_constant__ MoParams P) {
    __shared__ float rows[kMoThreads / 32][2][kMoMaxN];
    __shared__ float b_val[2][kMoThreads / 32], b_m[2][kMoThreads / 32], b_p[2][kMoThreads / 32];
    __shared__ int b_idx[2][kMoThreads / 32];
    __shared__ float nb[2][2];
    const int e = blockIdx.x, img = blockIdx.y;
    const int log1 = P.ev.log1[e], log2_ = P.ev.log2[e], n1 = 1 << log1, n2 = 1 << log2_;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float2 *t2 = P.t2 + (long long)img * P.t2_frame + P.ev.t2_off[e];
    MoBest B[2] = {{-3.0e38f, 0.f, 0.f, 0x7fffffff}, {-3.0e38f, 0.f, 0.f, 0x7fffffff}};
#define ULM_MO_CALL(LR) mo_peak_lines<LR>(P, rows[warp][0], rows[warp][1], t2, n1, n2, warp, lane, B[0], B[1])
    ULM_MO_DISPATCH(log2_, ULM_MO_CALL)
#undef ULM_MO_CALL
    if (lane == 0)
        for (int h = 0; h < 2; ++h) { b_val[h][warp] = B[h].val; b_idx[h][warp] = B[h].idx; b_m[h][warp] = B[h].m; b_p[h][warp] = B[h].p; }
    __syncthreads();
    int w_best[2] = {0, 0};
    for (int h = 0; h < 2; ++h)
        for (int w = 1; w < kMoThreads / 32; ++w)
            if (b_val[h][w] > b_val[h][w_best[h]] || (b_val[h][w] == b_val[h][w_best[h]] && b_idx[h][w] < b_idx[h][w_best[h]])) w_best[h] = w;
    // the lateral neighbours c(dl +- 1, dz) of either frame's peak (warps 0, 1: first frame; warps 2, 3: second frame)
    if (warp < 4) {
        const int h = warp >> 1, pk = b_idx[h][w_best[h]], dl_pk = pk / n2, dz_pk = pk - dl_pk * n2;
        const int dl = (dl_pk + ((warp & 1) == 0 ? n1 - 1 : 1)) & (n1 - 1);
        float2 acc = make_float2(0.f, 0.f);
#define ULM_MO_CALL(LR) acc = mo_direct<LR>(P, t2, dl, dz_pk, n2, lane)
        ULM_MO_DISPATCH(log2_, ULM_MO_CALL)
#undef ULM_MO_CALL
        if (lane == 0) nb[h][warp & 1] = h ? acc.y : acc.x;
    }
    __syncthreads();
    if (threadIdx.x < 2) {
        const int h = threadIdx.x, f = 2 * img + h;
        if (f < P.n_frames) {
            const float c0 = b_val[h][w_best[h]], cm2 = b_m[h][w_best[h]], cp2 = b_p[h][w_best[h]];
            const int pk = b_idx[h][w_best[h]], dl_pk = pk / n2, dz_pk = pk - dl_pk * n2;
            const float2 sf = P.stats[(long long)f * P.n_events + e], sr = P.stats[(long long)P.ref_frame * P.n_events + e];
            const float den = sqrtf(sf.y) * sqrtf(sr.y) * (float)n1 * (float)n2;
            const float inv = den > 0.f ? 1.f / den : 0.f;
            auto parab = [](float m, float c, float p) { const float d = m - 2.f * c + p; return d == 0.f ? 0.f : 0.5f * (m - p) / d; };
            const float d1 = parab(nb[h][0], c0, nb[h][1]), d2 = parab(cm2, c0, cp2);
            const int s1 = dl_pk < n1 / 2 ? dl_pk : dl_pk - n1, s2 = dz_pk < n2 / 2 ? dz_pk : dz_pk - n2;
            P.per_event[(long long)f * P.n_events + e] = make_float4((float)s1 + d1, (float)s2 + d2, c0 * inv, 0.f);
        }
    }
}

__global__ void __launch_bounds__(128) motion_combine_kernel(const __grid_constant__ MoParams P) {
    const int f = blockIdx.x * 128 + threadIdx.x;
    if (f >= P.n_frames) return;
    const int kr = P.n_row_tx, kc = P.n_events - kr;
    float dx = 0.f, dzr = 0.f, dy = 0.f, dzc = 0.f, ncc = 0.f;
    for (int e = 0; e < P.n_events; ++e) {
        const float4 v = P.per_event[(long long)f * P.n_events + e];
        if (e < kr) { dx += v.x; dzr += v.y; } else { dy += v.x; dzc += v.y; }
        ncc += v.z;
    }
    if (kr) { dx = dx / kr * P.dlat[0]; dzr = dzr / kr * P.dz[0]; }
    if (kc) { dy = dy / kc * P.dlat[1]; dzc = dzc / kc * P.dz[1]; }
    const float dzv = (kr && kc) ? 0.5f * (dzr + dzc) : (kr ? dzr : dzc);
    P.motion[f] = make_float4(dx, dy, dzv, ncc / P.n_events);
}

}  // namespace ulm
