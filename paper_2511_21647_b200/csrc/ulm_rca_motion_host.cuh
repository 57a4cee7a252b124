// ulm_rca_motion_host.cuh -- host side of the motion estimation: scratch and the launch sequence.
#pragma once

#include <algorithm>
#include <cmath>
#include <vector>

#include "ulm_rca_motion.cuh"

namespace ulm {

struct MotionPlan {
    bool ready = false;
    int n_events = 0, n_row_tx = 0, max_frames = 0;
    long long frame_stride = 0, t1_frame = 0, t2_frame = 0, ref_total = 0;
    int max_n1 = 0, max_n2 = 0, max_lat_tiles = 0, max_kz_tiles = 0;
    float dlat[2] = {0, 0}, dz[2] = {0, 0};
    void *d_off = nullptr, *d_nlat = nullptr, *d_nax = nullptr, *d_log1 = nullptr, *d_log2 = nullptr;
    void *d_t1off = nullptr, *d_t2off = nullptr, *d_refoff = nullptr;
    void *stats = nullptr, *t1 = nullptr, *t2 = nullptr, *fref = nullptr, *tw = nullptr, *per_event = nullptr;
    cudaEvent_t ev[2] = {nullptr, nullptr};
    ~MotionPlan() {
        for (void *p : {d_off, d_nlat, d_nax, d_log1, d_log2, d_t1off, d_t2off, d_refoff, stats, t1, t2, fref, tw, per_event}) if (p) cudaFree(p);
        for (auto &e : ev) if (e) cudaEventDestroy(e);
    }
};

namespace mohost {
inline int ilog2_ceil(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }
template <class T> inline bool up(void **dst, const std::vector<T> &v) {
    return cudaMalloc(dst, std::max<size_t>(1, v.size()) * sizeof(T)) == cudaSuccess &&
           (v.empty() || cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice) == cudaSuccess);
}
}  // namespace mohost

// n_lat / n_ax per event (row-tx events first), offsets of the slices inside a frame
inline const char *motion_build(MotionPlan &M, const std::vector<long long> &off, const std::vector<int> &n_lat,
                                const std::vector<int> &n_ax, int n_row_tx, long long frame_stride, int max_frames,
                                const float dlat[2], const float dz[2], bool timing) {
    using namespace mohost;
    M.n_events = (int)off.size(); M.n_row_tx = n_row_tx; M.max_frames = max_frames; M.frame_stride = frame_stride;
    for (int a = 0; a < 2; ++a) { M.dlat[a] = dlat[a]; M.dz[a] = dz[a]; }
    std::vector<int> log1, log2;
    std::vector<long long> t1off, t2off, refoff;
    for (int e = 0; e < M.n_events; ++e) {
        const int l1 = std::max(5, ilog2_ceil(n_lat[e])), l2 = std::max(5, ilog2_ceil(n_ax[e]));
        if ((1 << l1) > kMoMaxN || (1 << l2) > kMoMaxN) return "slices larger than 512 pixels along an axis";
        log1.push_back(l1); log2.push_back(l2);
        t1off.push_back(M.t1_frame); t2off.push_back(M.t2_frame); refoff.push_back(M.ref_total);
        M.t1_frame += (long long)(1 << l2) * ((n_lat[e] + 31) / 32 * 32);
        M.t2_frame += (long long)(1 << l1) * (1 << l2);
        M.ref_total += (long long)(1 << l1) * (1 << l2);
        M.max_n1 = std::max(M.max_n1, 1 << l1); M.max_n2 = std::max(M.max_n2, 1 << l2);
        M.max_lat_tiles = std::max(M.max_lat_tiles, (n_lat[e] + kMoLines - 1) / kMoLines);
        M.max_kz_tiles = std::max(M.max_kz_tiles, (1 << l2) / kMoLines);
    }
    std::vector<float2> tw(1024);
    for (int k = 0; k < 1024; ++k) tw[k] = make_float2((float)std::cos(-2.0 * M_PI * k / 1024.0), (float)std::sin(-2.0 * M_PI * k / 1024.0));
    if (!up(&M.d_off, off) || !up(&M.d_nlat, n_lat) || !up(&M.d_nax, n_ax) || !up(&M.d_log1, log1) || !up(&M.d_log2, log2) ||
        !up(&M.d_t1off, t1off) || !up(&M.d_t2off, t2off) || !up(&M.d_refoff, refoff) || !up(&M.tw, tw))
        return "table upload failed";
    if (cudaMalloc(&M.stats, (size_t)max_frames * M.n_events * sizeof(float2)) != cudaSuccess ||
        // packed images: two frames each, + the reference frame alone (T1 only)
        cudaMalloc(&M.t1, (size_t)((max_frames + 1) / 2 + 1) * M.t1_frame * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&M.t2, (size_t)((max_frames + 1) / 2) * M.t2_frame * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&M.fref, (size_t)M.ref_total * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&M.per_event, (size_t)max_frames * M.n_events * sizeof(float4)) != cudaSuccess)
        return "scratch allocation failed";
    const int smem1 = kMoLines * (M.max_n2 + 1) * 8, smem2 = kMoLines * (M.max_n1 + 1) * 8;
    if (cudaFuncSetAttribute(motion_fwd_z_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem1) != cudaSuccess ||
        cudaFuncSetAttribute(motion_lat_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2) != cudaSuccess ||
        cudaFuncSetAttribute(motion_lat_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2) != cudaSuccess)
        return "kernel attribute failed";
    if (timing) for (auto &e : M.ev) if (cudaEventCreate(&e) != cudaSuccess) return "event creation failed";
    M.ready = true;
    return nullptr;
}

// n_frames <= max_frames frames against frame ref_frame of the same call
inline cudaError_t motion_launch(const MotionPlan &M, const float2 *x, int n_frames, int ref_frame, float4 *motion,
                                 float4 *per_event_out, cudaStream_t st, int *launches) {
    cudaError_t e;
    MoParams P{};
    P.x = x; P.frame_stride = M.frame_stride;
    P.ev = MoEvents{static_cast<const long long *>(M.d_off), static_cast<const int *>(M.d_nlat), static_cast<const int *>(M.d_nax),
                    static_cast<const int *>(M.d_log1), static_cast<const int *>(M.d_log2), static_cast<const long long *>(M.d_t1off),
                    static_cast<const long long *>(M.d_t2off), static_cast<const long long *>(M.d_refoff)};
    P.n_events = M.n_events; P.n_frames = n_frames; P.ref_frame = ref_frame; P.n_pairs = (n_frames + 1) / 2;
    P.stats = static_cast<float2 *>(M.stats); P.t1 = static_cast<float2 *>(M.t1); P.t2 = static_cast<float2 *>(M.t2);
    P.fref = static_cast<float2 *>(M.fref); P.t1_frame = M.t1_frame; P.t2_frame = M.t2_frame; P.tw = static_cast<const float2 *>(M.tw);
    P.per_event = static_cast<float4 *>(M.per_event); P.motion = motion; P.n_row_tx = M.n_row_tx;
    for (int a = 0; a < 2; ++a) { P.dlat[a] = M.dlat[a]; P.dz[a] = M.dz[a]; }
    const int smem1 = kMoLines * (M.max_n2 + 1) * 8, smem2 = kMoLines * (M.max_n1 + 1) * 8;
    if (M.ev[0] && (e = cudaEventRecord(M.ev[0], st)) != cudaSuccess) return e;
    motion_stats_kernel<<<dim3(M.n_events, n_frames), kMoThreads, 0, st>>>(P);
    motion_fwd_z_kernel<<<dim3(M.max_lat_tiles, M.n_events, P.n_pairs + 1), kMoThreads, smem1, st>>>(P);
    motion_lat_kernel<true><<<dim3(M.max_kz_tiles, M.n_events, 1), kMoThreads, smem2, st>>>(P);
    motion_lat_kernel<false><<<dim3(M.max_kz_tiles, M.n_events, P.n_pairs), kMoThreads, smem2, st>>>(P);
    motion_peak_kernel<<<dim3(M.n_events, P.n_pairs), kMoThreads, 0, st>>>(P);
    motion_combine_kernel<<<(n_frames + 127) / 128, 128, 0, st>>>(P);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (M.ev[1] && (e = cudaEventRecord(M.ev[1], st)) != cudaSuccess) return e;
    *launches += 6;
    if (per_event_out)
        return cudaMemcpyAsync(per_event_out, M.per_event, (size_t)n_frames * M.n_events * sizeof(float4), cudaMemcpyDeviceToDevice, st);
    return cudaSuccess;
}

}  // namespace ulm
