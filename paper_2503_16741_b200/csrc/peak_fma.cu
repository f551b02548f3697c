// peak_fma.cu -- ct_measure_fp32_peak: the measured fp32 FMA throughput of the device, the denominator of the
// roofline that binds this path ("the builder measures it first with an FMA-only microbenchmark").
//
// FMA-only kernel: every thread carries 8 independent FMA chains in registers (16 with the packed form), no memory
// traffic, one CTA of 1024 threads per SM and several waves; timed with CUDA events on the caller's stream.
// kind 0: scalar FFMA (one fused multiply-add per lane and instruction); kind 1: FFMA2 (sm_100 packed pair, two
// per lane and instruction).  Two mixes, for the design record: kind 2 interleaves FFMA2 with scalar
// FFMA 1:1 on independent chains (3 FMAs per lane and pair of instructions), kind 3 interleaves FFMA2 with an ALU-pipe
// FMNMX (its flops count the FFMA2 only).
#include <cuda_runtime.h>

#include "ctsf_internal.h"

namespace {

constexpr int PK_CHAINS = 8, PK_UNROLL = 8, PK_THREADS = 1024;

template <int KIND>
__global__ void __launch_bounds__(PK_THREADS, 1) peak_fma_kernel(float *sink, float seed, int iters)
{
    float2 acc[PK_CHAINS];
    float side[PK_CHAINS];
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) {
        acc[i] = make_float2(seed + (float)(threadIdx.x + i), seed - (float)i);
        side[i] = seed * 0.5f + (float)i;
    }
    const float b = 1.0f - seed * 1e-7f, c = seed * 1e-7f;
    const float2 b2 = make_float2(b, b), c2 = make_float2(c, c);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < PK_UNROLL; ++r)
#pragma unroll
            for (int i = 0; i < PK_CHAINS; ++i) {
                if (KIND == 0) acc[i].x = fmaf(acc[i].x, b, c);
                if (KIND == 1) acc[i] = __ffma2_rn(acc[i], b2, c2);
                if (KIND == 2) { acc[i] = __ffma2_rn(acc[i], b2, c2); side[i] = fmaf(side[i], b, c); }
                if (KIND == 3) { acc[i] = __ffma2_rn(acc[i], b2, c2); side[i] = fmaxf(side[i], acc[i].y); }
            }
    }
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) s += acc[i].x + acc[i].y + side[i];
    if (s == 12345.678f) sink[0] = s;                // never true: keeps the chains alive
}

}  // namespace

extern "C" ct_status_t ct_measure_fp32_peak(int32_t kind, double *flops_per_s, double *seconds, ct_stream_t stream)
{
    if (!flops_per_s || kind < 0 || kind > 3) return CT_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        n_sm < 1) { cudaGetLastError(); return CT_ERR_CUDA; }
    float *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ct_status_t rc = CT_OK;
    if (cudaMalloc((void **)&sink, sizeof(float)) != cudaSuccess) { cudaGetLastError(); return CT_ERR_ALLOC; }
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = CT_ERR_CUDA;
    const int waves = 4, iters = 8192;
    auto launch = [&](int it) {
        if (kind == 0) peak_fma_kernel<0><<<n_sm * waves, PK_THREADS, 0, st>>>(sink, 1.0f, it);
        if (kind == 1) peak_fma_kernel<1><<<n_sm * waves, PK_THREADS, 0, st>>>(sink, 1.0f, it);
        if (kind == 2) peak_fma_kernel<2><<<n_sm * waves, PK_THREADS, 0, st>>>(sink, 1.0f, it);
        if (kind == 3) peak_fma_kernel<3><<<n_sm * waves, PK_THREADS, 0, st>>>(sink, 1.0f, it);
    };
    float best_ms = 0.0f;
    if (rc == CT_OK) {
        launch(64);                                   // warm-up (clocks, instruction cache)
        for (int rep = 0; rep < 3 && rc == CT_OK; ++rep) {
            cudaEventRecord(e0, st);
            launch(iters);
            cudaEventRecord(e1, st);
            float ms = 0.0f;
            if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) rc = CT_ERR_CUDA;
            else if (rep == 0 || ms < best_ms) best_ms = ms;
        }
    }
    if (rc == CT_OK && cudaGetLastError() != cudaSuccess) rc = CT_ERR_CUDA;
    if (rc == CT_OK && best_ms > 0.0f) {
        const double fma = (double)n_sm * waves * PK_THREADS * (double)iters * PK_UNROLL * PK_CHAINS * (kind == 0 ? 1.0 : (kind == 2 ? 3.0 : 2.0));
        *flops_per_s = 2.0 * fma / (best_ms * 1e-3);
        if (seconds) *seconds = best_ms * 1e-3;
    } else if (rc == CT_OK) rc = CT_ERR_CUDA;
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    if (rc != CT_OK) cudaGetLastError();
    return rc;
}
