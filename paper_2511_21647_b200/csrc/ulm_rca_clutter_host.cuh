// ulm_rca_clutter_host.cuh -- host side of the clutter filter: scratch, TMA tensor maps of the
// bf16 operand planes, and the launch sequence split -> Gram (tcgen05) -> assemble -> eigen-subspace -> projection.
#pragma once

#include <algorithm>
#include <vector>

#include "ulm_rca_clutter.cuh"

namespace ulm {

struct ClutterPlan {
    bool ready = false;
    int n_events = 0, max_t = 0, iters = 24, n_splits = 1;
    long long frame_stride = 0, k_max = 0, ld = 0;
    std::vector<long long> off;
    std::vector<int> n_pix;
    void *d_off = nullptr, *d_npix = nullptr;
    void *y_hi = nullptr, *y_lo = nullptr, *partial = nullptr, *cov = nullptr, *uc = nullptr, *lam = nullptr;
    size_t y_bytes = 0, partial_bytes = 0;
    int ntp_cached = 0;               // padded frame count the operand planes are currently laid out / cleared for
    CUtensorMap map_hi{}, map_lo{};
    cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    ~ClutterPlan() {
        for (void *p : {d_off, d_npix, y_hi, y_lo, partial, cov, uc, lam}) if (p) cudaFree(p);
        for (auto &e : ev) if (e) cudaEventDestroy(e);
    }
};

inline int clutter_ntp(int n_t) { return (n_t + 63) / 64 * 64; }

using cf_encode_fn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tensor maps of Y_hi / Y_lo for a given padded frame count: 2-D bf16 [n_events * 2 NTP rows][k_max], row pitch ld
inline const char *clutter_make_maps(ClutterPlan &C, int ntp) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
        qres != cudaDriverEntryPointSuccess)
        return "cuTensorMapEncodeTiled is not available";
    const cf_encode_fn encode = reinterpret_cast<cf_encode_fn>(fn);
    const cuuint64_t dims[2] = {(cuuint64_t)C.k_max, (cuuint64_t)C.n_events * 2 * ntp};
    const cuuint64_t strides[1] = {(cuuint64_t)C.ld * 2};
    const cuuint32_t box[2] = {(cuuint32_t)kCfBK, (cuuint32_t)kCfTile};
    const cuuint32_t estr[2] = {1, 1};
    for (int i = 0; i < 2; ++i) {
        const CUresult r = encode(i == 0 ? &C.map_hi : &C.map_lo, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, i == 0 ? C.y_hi : C.y_lo, dims,
                                  strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                  CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return "cuTensorMapEncodeTiled failed";
    }
    return nullptr;
}

// off / n_pix: float2 offset and pixel count of every event's slice inside a frame of the compound = 0 layout
inline const char *clutter_build(ClutterPlan &C, const std::vector<long long> &off, const std::vector<int> &n_pix,
                                 long long frame_stride, int max_t, bool timing) {
    C.n_events = (int)off.size();
    C.max_t = max_t;
    C.off = off; C.n_pix = n_pix;
    C.frame_stride = frame_stride;
    C.k_max = *std::max_element(n_pix.begin(), n_pix.end());
    C.ld = (C.k_max + 7) / 8 * 8;                                   // 16-byte row pitch
    const int ntp = clutter_ntp(max_t), nr = 2 * ntp;
    const int n_kblocks = (int)((C.k_max + kCfBK - 1) / kCfBK);
    const int tiles = (nr / kCfTile) * (nr / kCfTile + 1) / 2;
    int sms = 148, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    // K splits: about six CTAs per SM in total, at least 32 k-blocks each
    C.n_splits = std::max(1, std::min({8, n_kblocks / 32, (6 * sms + tiles * C.n_events - 1) / (tiles * C.n_events)}));
    C.y_bytes = (size_t)C.n_events * nr * C.ld * 2;
    C.partial_bytes = (size_t)C.n_events * C.n_splits * nr * nr * sizeof(float);
    if (cudaMalloc(&C.d_off, off.size() * sizeof(long long)) != cudaSuccess || cudaMalloc(&C.d_npix, n_pix.size() * sizeof(int)) != cudaSuccess ||
        cudaMalloc(&C.y_hi, C.y_bytes) != cudaSuccess || cudaMalloc(&C.y_lo, C.y_bytes) != cudaSuccess ||
        cudaMalloc(&C.partial, C.partial_bytes) != cudaSuccess ||
        cudaMalloc(&C.cov, (size_t)C.n_events * max_t * max_t * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&C.uc, (size_t)C.n_events * max_t * kCfB * sizeof(float2)) != cudaSuccess ||
        cudaMalloc(&C.lam, (size_t)C.n_events * kCfB * sizeof(float)) != cudaSuccess)
        return "scratch allocation failed";
    if (cudaMemcpy(C.d_off, off.data(), off.size() * sizeof(long long), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(C.d_npix, n_pix.data(), n_pix.size() * sizeof(int), cudaMemcpyHostToDevice) != cudaSuccess)
        return "table upload failed";
    if (cudaFuncSetAttribute(clutter_gram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kCfGramSmem) != cudaSuccess ||
        cudaFuncSetAttribute(clutter_eig_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, clutter_eig_smem_bytes(kCfMaxFrames)) != cudaSuccess ||
        cudaFuncSetAttribute(clutter_project_kernel<24>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCfMaxFrames * 24 * 8) != cudaSuccess ||
        cudaFuncSetAttribute(clutter_project_kernel<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCfMaxFrames * 16 * 8) != cudaSuccess)
        return "kernel attribute failed";
    if (timing) for (auto &e : C.ev) if (cudaEventCreate(&e) != cudaSuccess) return "event creation failed";
    C.ready = true;
    return nullptr;
}

// The whole filter for n_t frames (32 <= n_t <= max_t).  Returns a CUDA status; *why gets a reason for non-CUDA failures.
inline cudaError_t clutter_launch(ClutterPlan &C, const float2 *x, int n_t, int rank, float2 *out, float *lam_out, float2 *cov_out,
                                  cudaStream_t st, int *launches, const char **why) {
    cudaError_t e;
    const int ntp = clutter_ntp(n_t), nr = 2 * ntp;
    const CfEvents ev{static_cast<const long long *>(C.d_off), static_cast<const int *>(C.d_npix)};
    if (C.ntp_cached != ntp) {
        // rows that hold no frame (padding) and columns past an event's last pixel must read as zero
        if ((e = cudaMemsetAsync(C.y_hi, 0, C.y_bytes, st)) != cudaSuccess) return e;
        if ((e = cudaMemsetAsync(C.y_lo, 0, C.y_bytes, st)) != cudaSuccess) return e;
        if (const char *w = clutter_make_maps(C, ntp)) { *why = w; return cudaErrorUnknown; }
        C.ntp_cached = ntp;
    }
    if (C.ev[0] && (e = cudaEventRecord(C.ev[0], st)) != cudaSuccess) return e;
    CfSplitParams S{};
    S.x = x; S.frame_stride = C.frame_stride; S.ev = ev; S.y_hi = static_cast<__nv_bfloat16 *>(C.y_hi);
    S.y_lo = static_cast<__nv_bfloat16 *>(C.y_lo); S.ld = C.ld; S.n_t = n_t; S.ntp = ntp; S.n_events = C.n_events;
    clutter_split_kernel<<<dim3((unsigned)((C.k_max + 2047) / 2048), n_t, C.n_events), 256, 0, st>>>(S);      // 8 pixels per thread
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (C.ev[1] && (e = cudaEventRecord(C.ev[1], st)) != cudaSuccess) return e;

    CfGramParams G{};
    G.partial = static_cast<float *>(C.partial); G.nr = nr; G.n_kblocks = (int)((C.k_max + kCfBK - 1) / kCfBK);
    G.n_splits = C.n_splits; G.n_tiles_1d = nr / kCfTile;
    const int tiles = G.n_tiles_1d * (G.n_tiles_1d + 1) / 2;
    clutter_gram_kernel<<<dim3(tiles, C.n_splits, C.n_events), kCfGramThreads, kCfGramSmem, st>>>(C.map_hi, C.map_lo, G);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (C.ev[2] && (e = cudaEventRecord(C.ev[2], st)) != cudaSuccess) return e;
    CfAssembleParams A{};
    A.partial = static_cast<const float *>(C.partial); A.cov = static_cast<float2 *>(C.cov); A.nr = nr; A.ntp = ntp; A.n_t = n_t;
    A.n_splits = C.n_splits; A.n_events = C.n_events;
    clutter_assemble_kernel<<<dim3((n_t + 255) / 256, n_t, C.n_events), 256, 0, st>>>(A);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (C.ev[3] && (e = cudaEventRecord(C.ev[3], st)) != cudaSuccess) return e;

    CfEigParams E{};
    E.cov = static_cast<const float2 *>(C.cov); E.uc = static_cast<float2 *>(C.uc); E.lam = static_cast<float *>(C.lam);
    E.n_t = n_t; E.iters = rank > 0 ? C.iters : 0; E.n_track = rank;
    clutter_eig_kernel<<<C.n_events, kCfEigThreads, clutter_eig_smem_bytes(n_t), st>>>(E);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (C.ev[4] && (e = cudaEventRecord(C.ev[4], st)) != cudaSuccess) return e;

    CfProjectParams J{};
    J.x = x; J.out = out; J.frame_stride = C.frame_stride; J.ev = ev; J.uc = static_cast<const float2 *>(C.uc); J.n_t = n_t; J.rank = rank;
    const dim3 pg((unsigned)((C.k_max + 127) / 128), C.n_events);
    if (rank <= 8) clutter_project_kernel<8><<<pg, 128, n_t * 8 * 8, st>>>(J);
    else if (rank <= 16) clutter_project_kernel<16><<<pg, 128, n_t * 16 * 8, st>>>(J);
    else clutter_project_kernel<24><<<pg, 128, n_t * 24 * 8, st>>>(J);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    if (C.ev[5] && (e = cudaEventRecord(C.ev[5], st)) != cudaSuccess) return e;
    *launches += 5;
    if (lam_out && (e = cudaMemcpyAsync(lam_out, C.lam, (size_t)C.n_events * kCfB * sizeof(float), cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return e;
    if (cov_out && (e = cudaMemcpyAsync(cov_out, C.cov, (size_t)C.n_events * n_t * n_t * sizeof(float2), cudaMemcpyDeviceToDevice, st)) != cudaSuccess) return e;
    return cudaSuccess;
}

}  // namespace ulm
