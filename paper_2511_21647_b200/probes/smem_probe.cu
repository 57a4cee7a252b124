// smem_probe.cu -- stand-alone micro-benchmark (not part of libulm_rca.so): FP32 / mixed-precision pipe rates and the
// shared-memory wavefront cost of LDS.32/.64/.128 when the lanes of a warp read overlapping, slowly advancing
// entries (the access pattern of the DAS gather).  Build: python -m paper_2511_21647_b200.build --probe
#include <cstdio>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <vector>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)

template<int MODE> __global__ void __launch_bounds__(512) pipe_kernel(float* sink, int iters, float a, float b, unsigned hbits) {
    float x[16];
    unsigned h = hbits + threadIdx.x;
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 1e-3f + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < 16; ++i) {
                if (MODE == 0) x[i] = fmaf(x[i], a, b);                       // FFMA 3-reg
                else if (MODE == 1) { asm volatile("fma.rn.f32.f16 %0, %1, %2, %0;" : "+f"(x[i]) : "h"((unsigned short)(h & 0xffff)), "h"((unsigned short)(h >> 16))); }
                else if (MODE == 2) { x[i] = fmaf(x[i], a, x[(i + 1) & 15]); }   // FFMA with 3 distinct regs
                else if (MODE == 3) { float s, c; __sincosf(x[i], &s, &c); x[i] = s + c; }
                else if (MODE == 4) { x[i] = __half2float(__float2half_rn(x[i])) + a; }
                else if (MODE == 5) { asm volatile("fma.rn.f32.f16 %0, %1, %2, %3;" : "=f"(x[i]) : "h"((unsigned short)(h & 0xffff)), "h"((unsigned short)(h >> 16)), "f"(x[(i+1)&15])); }
            }
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += x[i];
    if (s == 123.456f) sink[0] = s;
}

// smem: each lane loads WIDTH bytes at entry index idx[lane] (entry stride STRIDE bytes), repeated; measures cycles/load per SM
template<int WIDTH> __global__ void __launch_bounds__(512) lds_kernel(float* sink, const int* lane_entry, int stride_bytes, int iters, long long* cycles) {
    extern __shared__ __align__(16) unsigned char sm[];
    for (int i = threadIdx.x; i < 48 * 1024 / 4; i += blockDim.x) ((float*)sm)[i] = i;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    unsigned addr = (unsigned)__cvta_generic_to_shared(sm) + lane_entry[lane] * stride_bytes + (threadIdx.x >> 5) * 0;
    float acc = 0.f;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 16; ++r) {
            const unsigned a = addr + r * 2304 + ((it & 7) << 4);
            if (WIDTH == 4) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a) : "memory"); acc += v; }
            if (WIDTH == 8) { float v, w; asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v), "=f"(w) : "r"(a) : "memory"); acc += v + w; }
            if (WIDTH == 16) { float v, w, y, z; asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v), "=f"(w), "=f"(y), "=f"(z) : "r"(a) : "memory"); acc += v + w + y + z; }
        }
    }
    long long t1 = clock64();
    if (acc == 123.456f) sink[0] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template<int MODE> double run_pipe(int sms, float* sink) {
    cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
    const int blocks = sms * 4, iters = 2000;
    pipe_kernel<MODE><<<blocks, 512>>>(sink, 100, 0.999f, 0.001f, 0x3c003800u);
    cudaEventRecord(a);
    pipe_kernel<MODE><<<blocks, 512>>>(sink, iters, 0.999f, 0.001f, 0x3c003800u);
    cudaEventRecord(b); cudaEventSynchronize(b);
    float ms; cudaEventElapsedTime(&ms, a, b);
    double ops = 64.0 * iters * 512.0 * blocks;   // thread-level ops
    return ops / (ms * 1e-3) / sms / 1.965e9;     // ops per clk per SM (at 1965 MHz)
}

template<int WIDTH> double run_lds(const std::vector<int>& pat, int stride, float* sink, int* d_pat, long long* d_cyc) {
    cudaMemcpy(d_pat, pat.data(), 32 * sizeof(int), cudaMemcpyHostToDevice);
    const int iters = 2000, warps = 16;
    lds_kernel<WIDTH><<<1, warps * 32, 48 * 1024>>>(sink, d_pat, stride, iters, d_cyc);
    lds_kernel<WIDTH><<<1, warps * 32, 48 * 1024>>>(sink, d_pat, stride, iters, d_cyc);
    cudaDeviceSynchronize();
    long long c; cudaMemcpy(&c, d_cyc, sizeof(c), cudaMemcpyDeviceToHost);
    return (double)c / (iters * 16.0 * warps);    // cycles per warp-level load instruction on the SM
}

int main() {
    int sms; CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0));
    float* sink; CK(cudaMalloc(&sink, 4));
    int* d_pat; CK(cudaMalloc(&d_pat, 128)); long long* d_cyc; CK(cudaMalloc(&d_cyc, 8 * 1024));
    printf("SMs %d\n", sms);
    printf("pipe ops/clk/SM (@1965MHz): FFMA(acc,a,b imm-like) %.1f | FHFMA acc %.1f | FFMA 3reg %.1f | sincos(2 MUFU+..)/thread-op %.1f | F2F roundtrip %.1f | FHFMA 3-operand %.1f\n",
           run_pipe<0>(sms, sink), run_pipe<1>(sms, sink), run_pipe<2>(sms, sink), run_pipe<3>(sms, sink), run_pipe<4>(sms, sink), run_pipe<5>(sms, sink));
    CK(cudaGetLastError());
    const double steps[] = {0.0, 0.25, 0.3, 0.4, 0.45, 0.5, 0.6, 0.75, 1.0, 1.5, 2.0};
    const double offs[] = {0.0, 0.35, 0.7};
    const int strides[] = {8, 16, 144, 120, 40, 112, 64, 128};
    for (int stride : strides) {
        for (double s : steps) for (double off : offs) {
            if (off != 0.0 && (s == 0.0 || s >= 1.0)) continue;
            std::vector<int> pat(32);
            for (int l = 0; l < 32; ++l) pat[l] = (int)(l * s + off);
            double c4 = (stride % 4 == 0) ? run_lds<4>(pat, stride, sink, d_pat, d_cyc) : 0;
            double c8 = (stride % 8 == 0) ? run_lds<8>(pat, stride, sink, d_pat, d_cyc) : 0;
            double c16 = (stride % 16 == 0) ? run_lds<16>(pat, stride, sink, d_pat, d_cyc) : 0;
            printf("stride %3d B step %.2f offset %.2f entries/lane: cycles per warp-LDS  .32: %.2f  .64: %.2f  .128: %.2f\n", stride, s, off, c4, c8, c16);
        }
    }
    CK(cudaGetLastError());
    return 0;
}
