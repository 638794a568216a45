// qmmm_probe.cu -- same-run roofline denominators (north_star: "FMA peak, measured by a
// microbenchmark in the same run").  Register-only kernels: every thread runs CHAINS
// independent dependent chains of one instruction kind, full occupancy, every SM.
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "../../include/qmmm_field.h"

namespace {

constexpr int CHAINS = 8;
constexpr int UNROLL = 32;     // instructions per chain per loop trip

__global__ void __launch_bounds__(256) probe_ffma(int iters, float a, float b, float *sink) {
    float x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = a + threadIdx.x * 1e-6f + c;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) x[c] = fmaf(x[c], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
    if (s == 12345.678f) sink[0] = s;      // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) probe_dfma(int iters, double a, double b, double *sink) {
    double x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = a + threadIdx.x * 1e-6 + c;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < CHAINS; ++c) x[c] = fma(x[c], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
    if (s == 12345.678) sink[0] = s;
}

__global__ void __launch_bounds__(256) probe_mufu(int iters, float a, float *sink) {
    float x[CHAINS];
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) x[c] = a + threadIdx.x * 1e-3f + c;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < UNROLL; ++u)
#pragma unroll
            for (int c = 0; c < CHAINS; ++c)
                asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x[c]));
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < CHAINS; ++c) s += x[c];
    if (s == 12345.678f) sink[0] = s;
}

__global__ void probe_empty() {}

thread_local std::string g_probe_error;

}  // namespace

extern "C" qmmm_status qmmm_probe_peak(int kind, int iters, double *rate, double *seconds,
                                       void *stream) {
    if (!rate || kind < 0 || kind > 3) return QMMM_ERR_INVALID_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return QMMM_ERR_CUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess)
        return QMMM_ERR_CUDA;
    void *sink = nullptr;
    if (cudaMalloc(&sink, 64) != cudaSuccess) return QMMM_ERR_ALLOC;
    const int threads = 256, ctas = sms * 8;     // 2048 threads/SM resident
    if (iters <= 0) iters = kind == 1 ? 512 : (kind == 2 ? 256 : 2048);
    float ms = 0.f;
    cudaError_t err = cudaSuccess;
    if (kind == 3) {
        const int reps = 200;
        for (int i = 0; i < 20; ++i) { probe_empty<<<1, 32, 0, st>>>(); cudaStreamSynchronize(st); }
        cudaEventRecord(e0, st);
        cudaStreamSynchronize(st);
        // host-timed: launch + sync round trip
        struct timespec t0, t1;
        clock_gettime(CLOCK_MONOTONIC, &t0);
        for (int i = 0; i < reps; ++i) { probe_empty<<<1, 32, 0, st>>>(); cudaStreamSynchronize(st); }
        clock_gettime(CLOCK_MONOTONIC, &t1);
        const double s = (t1.tv_sec - t0.tv_sec) + 1e-9 * (t1.tv_nsec - t0.tv_nsec);
        *rate = s / reps;
        if (seconds) *seconds = s;
        err = cudaGetLastError();
    } else {
        for (int rep = 0; rep < 2; ++rep) {      // rep 0 = warm-up
            cudaEventRecord(e0, st);
            if (kind == 0) probe_ffma<<<ctas, threads, 0, st>>>(iters, 0.999f, 1e-3f, (float *)sink);
            if (kind == 1) probe_dfma<<<ctas, threads, 0, st>>>(iters, 0.999, 1e-3, (double *)sink);
            if (kind == 2) probe_mufu<<<ctas, threads, 0, st>>>(iters, 1.5f, (float *)sink);
            cudaEventRecord(e1, st);
            err = cudaStreamSynchronize(st);
            if (err != cudaSuccess) break;
            cudaEventElapsedTime(&ms, e0, e1);
        }
        const double ops = static_cast<double>(ctas) * threads * CHAINS * UNROLL * iters;
        *rate = ops / (ms * 1e-3);
        if (seconds) *seconds = ms * 1e-3;
        if (err == cudaSuccess) err = cudaGetLastError();
    }
    cudaFree(sink);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return err == cudaSuccess ? QMMM_OK : QMMM_ERR_CUDA;
}
