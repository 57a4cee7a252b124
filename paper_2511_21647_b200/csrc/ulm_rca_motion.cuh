// ulm_rca_motion.cuh -- Fourier-domain NCC rigid motion estimation on the Stage-1 slices (Section
// II.A.3; reading = DESIGN.md section 13) for sm_100a.
//
//   ME-1  a(l, i) = |S(l, i)| (B-mode), mean removed, zero-padded to N1 x N2 = next powers of two >= n_lat, n_ax
//   ME-2  c(d) = IFFT2( FFT2(a_f) conj(FFT2(a_ref)) ) / (|a_f| |a_ref|)          ("two forward and one inverse" transform)
//   ME-3  integer argmax of c (first in row-major order), signed shift, 3-point parabola per axis
//   ME-4  per frame: mean over the row-tx events -> (dx, dz_RC), over the column-tx events -> (dy, dz_CR),
//         motion = (dx, dy, (dz_RC + dz_CR) / 2) in metres
//
// The paper uses cuFFT (cufftPlanMany) plus a correlation kernel; here the transforms are hand-written radix-2 FFTs, one
// warp per line in shared memory, organised so that every pass over global memory is coalesced and the product with
// the reference spectrum and the inverse lateral transform are fused into the forward lateral pass:
//   motion_stats_kernel     mean and mean-removed energy of every B-mode image
//   motion_fwd_z_kernel     FFT along depth of 32 lateral lines per CTA, written transposed  T1[img][kz][l]
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
    float2 *stats;                // [frame][event] {mean, sum of squares of the mean-removed image}
    float2 *t1, *t2, *fref;       // scratch
    long long t1_frame, t2_frame; // float2 per frame of T1 / T2
    const float2 *tw;             // twiddles exp(-2 pi i k / 1024), k < 1024
    float4 *per_event;            // [frame][event] {d_lat px, d_ax px, ncc, 0}
    float4 *motion;               // [frame] {dx, dy, dz (m), mean ncc}
    int n_row_tx;
    float dlat[2], dz[2];         // grid steps of the x-z / y-z slices
};

constexpr int kMoMaxN = 512;      // padded FFT length at most
constexpr int kMoLines = 32;      // lines per CTA of the transposing kernels
constexpr int kMoThreads = 256;

// In-place radix-2 FFT of n = 2^logn points held BIT-REVERSED in s[] (shared memory) by one warp.
// tw[k] = exp(-2 pi i k / 1024); INV conjugates the twiddles (no 1/n scaling).
template <bool INV>
__device__ __forceinline__ void mo_warp_fft(float2 *s, int logn, const float2 *tw, int lane) {
    const int n = 1 << logn;
    for (int lg = 1; lg <= logn; ++lg) {
        const int half = 1 << (lg - 1), tstep = 1024 >> lg;
        for (int b = lane; b < n / 2; b += 32) {
            const int pos = b & (half - 1), i0 = ((b >> (lg - 1)) << lg) + pos, i1 = i0 + half;
            float2 w = tw[pos * tstep];
            if (INV) w.y = -w.y;
            const float2 u = s[i0], v = s[i1];
            const float2 t = make_float2(w.x * v.x - w.y * v.y, w.x * v.y + w.y * v.x);
            s[i0] = make_float2(u.x + t.x, u.y + t.y);
            s[i1] = make_float2(u.x - t.x, u.y - t.y);
        }
        __syncwarp();
    }
}
__device__ __forceinline__ int mo_brev(int i, int logn) { return (int)(__brev((unsigned)i) >> (32 - logn)); }

__global__ void __launch_bounds__(kMoThreads) motion_stats_kernel(const __grid_constant__ MoParams P) {
    const int e = blockIdx.x, f = blockIdx.y;
    const int n = P.ev.n_lat[e] * P.ev.n_ax[e];
    const float2 *x = P.x + (long long)f * P.frame_stride + P.ev.off[e];
    __shared__ float red[kMoThreads / 32];
    __shared__ float s_mean;
    auto block_sum = [&](float v) {
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        __syncthreads();
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
        __syncthreads();
        float t = 0.f;
        for (int i = 0; i < kMoThreads / 32; ++i) t += red[i];
        return t;
    };
    float s = 0.f;
    for (int i = threadIdx.x; i < n; i += kMoThreads) { const float2 v = __ldg(x + i); s += sqrtf(v.x * v.x + v.y * v.y); }
    const float mean = block_sum(s) / (float)n;
    float q = 0.f;
    for (int i = threadIdx.x; i < n; i += kMoThreads) { const float2 v = __ldg(x + i); const float d = sqrtf(v.x * v.x + v.y * v.y) - mean; q += d * d; }
    const float ss = block_sum(q);
    if (threadIdx.x == 0) P.stats[(long long)f * P.n_events + e] = make_float2(mean, ss);
    (void)s_mean;
}

// grid = (lateral tiles of 32 lines, events, frames)
__global__ void __launch_bounds__(kMoThreads) motion_fwd_z_kernel(const __grid_constant__ MoParams P) {
    extern __shared__ __align__(16) unsigned char mo_smem[];
    const int e = blockIdx.y, f = blockIdx.z;
    const int n_lat = P.ev.n_lat[e], n_ax = P.ev.n_ax[e], log2_ = P.ev.log2[e], n2 = 1 << log2_;
    const int l0 = blockIdx.x * kMoLines;
    if (l0 >= n_lat) return;
    float2 *s = reinterpret_cast<float2 *>(mo_smem);                  // [32][n2 + 1]
    const int rs = n2 + 1;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float mean = P.stats[(long long)f * P.n_events + e].x;
    const float2 *x = P.x + (long long)f * P.frame_stride + P.ev.off[e];
    for (int li = warp; li < kMoLines; li += kMoThreads / 32) {
        const int l = l0 + li;
        float2 *row = s + li * rs;
        for (int i = lane; i < n2; i += 32) {
            float a = 0.f;
            if (l < n_lat && i < n_ax) { const float2 v = __ldg(x + (long long)l * n_ax + i); a = sqrtf(v.x * v.x + v.y * v.y) - mean; }
            row[mo_brev(i, log2_)] = make_float2(a, 0.f);
        }
        __syncwarp();
        mo_warp_fft<false>(row, log2_, P.tw, lane);
    }
    __syncthreads();
    // transposed, coalesced write: T1[frame][event block][kz][l]
    float2 *t1 = P.t1 + (long long)f * P.t1_frame + P.ev.t1_off[e];
    const int n_lat_p = (n_lat + 31) / 32 * 32;
    for (int kz = warp; kz < n2; kz += kMoThreads / 32)
        t1[(long long)kz * n_lat_p + l0 + lane] = (l0 + lane < n_lat) ? s[lane * rs + kz] : make_float2(0.f, 0.f);
}

// grid = (kz tiles of 32 rows, events, frames [REF: 1])
template <bool REF>
__global__ void __launch_bounds__(kMoThreads) motion_lat_kernel(const __grid_constant__ MoParams P) {
    extern __shared__ __align__(16) unsigned char mo_smem[];
    const int e = blockIdx.y, f = REF ? P.ref_frame : blockIdx.z;
    const int n_lat = P.ev.n_lat[e], log1 = P.ev.log1[e], n1 = 1 << log1, n2 = 1 << P.ev.log2[e];
    const int kz0 = blockIdx.x * kMoLines;
    if (kz0 >= n2) return;
    const int rs = n1 + 1;
    float2 *s = reinterpret_cast<float2 *>(mo_smem);                  // [32][n1 + 1]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_lat_p = (n_lat + 31) / 32 * 32;
    const float2 *t1 = P.t1 + (long long)f * P.t1_frame + P.ev.t1_off[e];
    float2 *fref = P.fref + P.ev.ref_off[e];
    for (int ri = warp; ri < kMoLines; ri += kMoThreads / 32) {
        const int kz = kz0 + ri;                                       // n2 is a multiple of 32: always a valid row
        float2 *row = s + ri * rs;
        for (int l = lane; l < n1; l += 32)
            row[mo_brev(l, log1)] = l < n_lat ? __ldg(t1 + (long long)kz * n_lat_p + l) : make_float2(0.f, 0.f);
        __syncwarp();
        mo_warp_fft<false>(row, log1, P.tw, lane);
        if (REF) {
            for (int k = lane; k < n1; k += 32) fref[(long long)kz * n1 + k] = row[k];
        } else {
            // product with the conjugate reference spectrum, permuted in place into bit-reversed order for the inverse
            for (int k = lane; k < n1; k += 32) {
                const int j = mo_brev(k, log1);
                if (k <= j) {
                    const float2 a = row[k], r = __ldg(fref + (long long)kz * n1 + k);
                    const float2 b = row[j], q = __ldg(fref + (long long)kz * n1 + j);
                    row[j] = make_float2(a.x * r.x + a.y * r.y, a.y * r.x - a.x * r.y);     // a conj(r)
                    row[k] = make_float2(b.x * q.x + b.y * q.y, b.y * q.x - b.x * q.y);
                }
            }
            __syncwarp();
            mo_warp_fft<true>(row, log1, P.tw, lane);
        }
    }
    if (REF) return;
    __syncthreads();
    // transposed, coalesced write: T2[frame][event block][dl][kz]
    float2 *t2 = P.t2 + (long long)f * P.t2_frame + P.ev.t2_off[e];
    for (int dl = warp; dl < n1; dl += kMoThreads / 32) t2[(long long)dl * n2 + kz0 + lane] = s[lane * rs + dl];
}

// grid = (events, frames): inverse FFT along depth of every lateral-shift line, running maximum, sub-pixel peak
__global__ void __launch_bounds__(kMoThreads) motion_peak_kernel(const __grid_constant__ MoParams P) {
    __shared__ __align__(16) float2 s[kMoThreads / 32][kMoMaxN];
    __shared__ float b_val[kMoThreads / 32], b_m[kMoThreads / 32], b_p[kMoThreads / 32];
    __shared__ int b_idx[kMoThreads / 32];
    __shared__ float nb[2];
    const int e = blockIdx.x, f = blockIdx.y;
    const int log1 = P.ev.log1[e], log2_ = P.ev.log2[e], n1 = 1 << log1, n2 = 1 << log2_;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float2 *t2 = P.t2 + (long long)f * P.t2_frame + P.ev.t2_off[e];
    float best = -3.0e38f, best_m = 0.f, best_p = 0.f;
    int best_idx = 0x7fffffff;
    for (int dl = warp; dl < n1; dl += kMoThreads / 32) {
        float2 *row = s[warp];
        for (int k = lane; k < n2; k += 32) row[mo_brev(k, log2_)] = __ldg(t2 + (long long)dl * n2 + k);
        __syncwarp();
        mo_warp_fft<true>(row, log2_, P.tw, lane);
        float v = -3.0e38f;
        int vi = 0;
        for (int k = lane; k < n2; k += 32) if (row[k].x > v) { v = row[k].x; vi = k; }      // first maximum of this lane
        for (int o = 16; o > 0; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, v, o);
            const int oi = __shfl_xor_sync(0xffffffffu, vi, o);
            if (ov > v || (ov == v && oi < vi)) { v = ov; vi = oi; }
        }
        const int idx = dl * n2 + vi;
        if (v > best || (v == best && idx < best_idx)) {
            best = v; best_idx = idx;
            best_m = row[(vi + n2 - 1) & (n2 - 1)].x;
            best_p = row[(vi + 1) & (n2 - 1)].x;
        }
        __syncwarp();
    }
    if (lane == 0) { b_val[warp] = best; b_idx[warp] = best_idx; b_m[warp] = best_m; b_p[warp] = best_p; }
    __syncthreads();
    int w_best = 0;
    for (int w = 1; w < kMoThreads / 32; ++w)
        if (b_val[w] > b_val[w_best] || (b_val[w] == b_val[w_best] && b_idx[w] < b_idx[w_best])) w_best = w;
    const float c0 = b_val[w_best], cm2 = b_m[w_best], cp2 = b_p[w_best];
    const int pk = b_idx[w_best], dl_pk = pk / n2, dz_pk = pk - dl_pk * n2;
    // the lateral neighbours c(dl +- 1, dz): one direct inverse DFT sum over kz each (warps 0 and 1)
    if (warp < 2) {
        const int dl = (dl_pk + (warp == 0 ? n1 - 1 : 1)) & (n1 - 1);
        float acc = 0.f;
        for (int k = lane; k < n2; k += 32) {
            const float2 v = __ldg(t2 + (long long)dl * n2 + k);
            const float2 w = P.tw[((k * dz_pk) & (n2 - 1)) * (1024 >> log2_)];       // exp(-2 pi i k dz / n2); the inverse needs its conjugate
            acc += v.x * w.x + v.y * w.y;                                                    // Re(v conj(w))
        }
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) nb[warp] = acc;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const float2 sf = P.stats[(long long)f * P.n_events + e], sr = P.stats[(long long)P.ref_frame * P.n_events + e];
        const float den = sqrtf(sf.y) * sqrtf(sr.y) * (float)n1 * (float)n2;
        const float inv = den > 0.f ? 1.f / den : 0.f;
        auto parab = [](float m, float c, float p) { const float d = m - 2.f * c + p; return d == 0.f ? 0.f : 0.5f * (m - p) / d; };
        const float d1 = parab(nb[0], c0, nb[1]), d2 = parab(cm2, c0, cp2);
        const int s1 = dl_pk < n1 / 2 ? dl_pk : dl_pk - n1, s2 = dz_pk < n2 / 2 ? dz_pk : dz_pk - n2;
        P.per_event[(long long)f * P.n_events + e] = make_float4((float)s1 + d1, (float)s2 + d2, c0 * inv, 0.f);
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
