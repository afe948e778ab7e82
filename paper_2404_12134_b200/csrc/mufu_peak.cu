// mufu_peak.cu -- live measurement of the special-function (MUFU: ex2 / lg2 / rcp .approx.f32) issue rate of the
// device, the denominator of the "alu" roofline bench.py reports.  Not part of the numerical
// path: it runs independent dependent-chains of one MUFU instruction per thread on every SM and divides the count
// by the CUDA-event time.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sdtw.h"

namespace {

constexpr int CHAINS = 8;      // independent chains per thread (covers the MUFU latency at 32 warps/SM)
constexpr int INNER = 64;      // unrolled MUFU per chain per outer iteration

template <int KIND>
__device__ __forceinline__ float mufu_step(float x) {
    float y;
    if constexpr (KIND == 0) asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(-x));          // stays in (0.5, 1]
    else if constexpr (KIND == 1) asm volatile("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x + 3.f)); // -> ~2.2
    else asm volatile("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x + 0.5f));                          // -> ~0.78 (a bare
                                                                 // rcp(rcp(x)) chain is folded away by ptxas)
    return y;
}

template <int KIND>
__global__ void __launch_bounds__(1024) mufu_chain_kernel(int outer, float seed, float* sink) {
    float x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = seed + 0.01f * (float)(c + (threadIdx.x & 7));
    for (int o = 0; o < outer; ++o) {
#pragma unroll
        for (int i = 0; i < INNER; ++i) {
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) x[c] = mufu_step<KIND>(x[c]);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
    if (s == 123456.789f) *sink = s;    // never true; keeps the chains alive
}

thread_local int g_peak_cuda_error = 0;

}  // namespace

extern "C" int sdtw_measure_mufu_peak(int32_t kind, double* ops_per_s, int32_t* sm_count) {
    if (kind < 0 || kind > 2 || !ops_per_s) return SDTW_ERR_INVALID_ARG;
    int dev = 0;
    cudaDeviceProp prop;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { g_peak_cuda_error = (int)e; return SDTW_ERR_CUDA; }
    if (prop.major != 10) return SDTW_ERR_UNSUPPORTED;
    const int grid = prop.multiProcessorCount * 2, block = 1024, outer = 256;
    float* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaStream_t st = nullptr;
    e = cudaMalloc(&sink, 4);
    if (e == cudaSuccess) e = cudaStreamCreate(&st);
    if (e == cudaSuccess) e = cudaEventCreate(&e0);
    if (e == cudaSuccess) e = cudaEventCreate(&e1);
    double best = 0.0;
    for (int rep = 0; rep < 4 && e == cudaSuccess; ++rep) {   // rep 0 warms up
        cudaEventRecord(e0, st);
        if (kind == 0) mufu_chain_kernel<0><<<grid, block, 0, st>>>(outer, 0.3f, sink);
        else if (kind == 1) mufu_chain_kernel<1><<<grid, block, 0, st>>>(outer, 0.3f, sink);
        else mufu_chain_kernel<2><<<grid, block, 0, st>>>(outer, 0.3f, sink);
        cudaEventRecord(e1, st);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e == cudaSuccess && rep > 0 && ms > 0.f) {
            const double ops = (double)grid * block * CHAINS * INNER * (double)outer;
            const double r = ops / (ms * 1e-3);
            if (r > best) best = r;
        }
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (st) cudaStreamDestroy(st);
    if (sink) cudaFree(sink);
    if (e != cudaSuccess) { g_peak_cuda_error = (int)e; return SDTW_ERR_CUDA; }
    *ops_per_s = best;
    if (sm_count) *sm_count = prop.multiProcessorCount;
    return SDTW_OK;
}
