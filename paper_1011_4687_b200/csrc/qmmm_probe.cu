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

// Read bandwidth: every thread streams 128-bit loads over the buffer (grid-stride), `passes`
// times; the xor keeps the loads alive.  A 33 MB buffer stays in the 126 MB L2 after the
// warm-up launch (the config-2 charge arrays are 8.4 / 16.8 MB, its source lists 33 / 67 MB);
// a 537 MB buffer (config 4's FP64 source list) streams from HBM.
__global__ void __launch_bounds__(256) probe_read(const uint4 *buf, size_t n16, int passes, uint4 *sink) {
    uint4 acc = make_uint4(0u, 0u, 0u, 0u);
    const size_t stride = static_cast<size_t>(gridDim.x) * blockDim.x;
    for (int p = 0; p < passes; ++p) {
        size_t i = static_cast<size_t>(blockIdx.x) * blockDim.x + threadIdx.x;
        for (; i + 3 * stride < n16; i += 4 * stride) {
            const uint4 a = __ldcg(buf + i), b = __ldcg(buf + i + stride), c = __ldcg(buf + i + 2 * stride),
                        d = __ldcg(buf + i + 3 * stride);
            acc.x ^= a.x ^ b.x ^ c.x ^ d.x; acc.y ^= a.y ^ b.y ^ c.y ^ d.y;
            acc.z ^= a.z ^ b.z ^ c.z ^ d.z; acc.w ^= a.w ^ b.w ^ c.w ^ d.w;
        }
        for (; i < n16; i += stride) {
            const uint4 a = __ldcg(buf + i);
            acc.x ^= a.x; acc.y ^= a.y; acc.z ^= a.z; acc.w ^= a.w;
        }
    }
    if ((acc.x ^ acc.y ^ acc.z ^ acc.w) == 0x12345678u) sink[0] = acc;     // never true (buffer is zero)
}

}  // namespace

namespace qmmm { void set_last_error(const char *msg); }      // qmmm_field.cu (thread-local message)

namespace {
qmmm_status probe_fail(qmmm_status st, const char *msg) {
    qmmm::set_last_error(msg);
    return st;
}
}  // namespace

extern "C" qmmm_status qmmm_probe_peak(int kind, int iters, double *rate, double *seconds,
                                       void *stream) {
    if (!rate || kind < 0 || kind > 5) return probe_fail(QMMM_ERR_INVALID_ARG, "probe_peak: NULL rate or unknown kind");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return probe_fail(QMMM_ERR_CUDA, "probe_peak: cudaGetDevice failed");
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    void *sink = nullptr, *buf = nullptr;
    auto cleanup = [&]() {
        if (sink) cudaFree(sink);
        if (buf) cudaFree(buf);
        if (e0) cudaEventDestroy(e0);
        if (e1) cudaEventDestroy(e1);
    };
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) {
        cleanup();
        return probe_fail(QMMM_ERR_CUDA, "probe_peak: cudaEventCreate failed");
    }
    if (cudaMalloc(&sink, 64) != cudaSuccess) {
        cudaGetLastError();
        cleanup();
        return probe_fail(QMMM_ERR_ALLOC, "probe_peak: out of device memory");
    }
    const int threads = 256, ctas = sms * 8;     // 2048 threads/SM resident
    float ms = 0.f;
    cudaError_t err = cudaSuccess;
    if (kind >= 4) {
        // kind 4: 33 MB (L2-resident after the warm-up), kind 5: 537 MB (HBM)
        const size_t bytes = kind == 4 ? (size_t(33) << 20) : (size_t(537) << 20);
        const int passes = iters > 0 ? iters : (kind == 4 ? 16 : 2);
        if (cudaMalloc(&buf, bytes) != cudaSuccess) {
            cudaGetLastError();
            cleanup();
            return probe_fail(QMMM_ERR_ALLOC, "probe_peak: out of device memory for the bandwidth buffer");
        }
        err = cudaMemsetAsync(buf, 0, bytes, st);
        for (int rep = 0; rep < 2 && err == cudaSuccess; ++rep) {      // rep 0 = warm-up
            cudaEventRecord(e0, st);
            probe_read<<<ctas, threads, 0, st>>>(static_cast<const uint4 *>(buf), bytes / 16, passes,
                                                  static_cast<uint4 *>(sink));
            cudaEventRecord(e1, st);
            err = cudaStreamSynchronize(st);
            if (err == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
        }
        *rate = static_cast<double>(bytes) * passes / (ms * 1e-3);      // bytes per second
        if (seconds) *seconds = ms * 1e-3;
        if (err == cudaSuccess) err = cudaGetLastError();
        cleanup();
        return err == cudaSuccess ? QMMM_OK : probe_fail(QMMM_ERR_CUDA, cudaGetErrorString(err));
    }
    if (iters <= 0) iters = kind == 1 ? 512 : (kind == 2 ? 256 : 2048);
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
    cleanup();
    return err == cudaSuccess ? QMMM_OK : probe_fail(QMMM_ERR_CUDA, cudaGetErrorString(err));
}
