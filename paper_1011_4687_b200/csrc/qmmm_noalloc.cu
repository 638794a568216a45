// qmmm_noalloc.cu -- qmmm_field_eval_noalloc: ONE evaluation entry point that allocates nothing.
//
// Why: qmmm_field_create allocates (packed source copies, the partials workspace, tickets,
// mailboxes), so the handle-based calls are closed to callers that cannot call cudaMalloc at
// all: code under CUDA-graph capture, tight serving loops, harnesses that forbid allocation.
// This entry point evaluates Eq. 4 and its field straight from the caller's
// device arrays, in FP64, with the one kind of scratch memory the evaluation kernels need --
// the per-slice partials of Eq. 5-6 (U = B[1] + ... + B[N_B]) and the arrival
// tickets of the point blocks -- in a file-scope __device__ array of fixed size.
//
// The array (NA_SCRATCH_BYTES = 2 MiB + 4 KiB) lives in every GPU that loads the library, until
// the process exits.  Every call shares it:
//   * calls that OVERLAP on the GPU (two streams, two host threads, two processes' worth of
//     ranks are fine -- one array per process and device -- but two calls of ONE process in
//     flight at once on ONE device) race on it and give wrong results.  Serialise them.
//   * it keeps the last call's contents.  The partials need no clearing (every slot that is read
//     has been written by this call first); the tickets must start at zero and are cleared on
//     the caller's stream at the start of every call (cudaMemsetAsync: no allocation), so a call
//     that died half way cannot poison the next one.
//
// In host code the array's name is a host-side stand-in, not a device address: its device
// address is taken once per device, with that device current, by cudaGetSymbolAddress in this
// translation unit, and only that pointer is handed to the kernel.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <string>

#include "../../include/qmmm_field.h"

namespace qmmm { void set_last_error(const char *msg); }      // qmmm_field.cu (thread-local message)

namespace {

constexpr int NA_THREADS = 256;                     // threads per CTA (8 warps)
constexpr int NA_WARPS = NA_THREADS / 32;
constexpr int NA_PPB = 8;                           // evaluation points per CTA (and per thread: registers)
constexpr int64_t NA_MAX_POINTS = QMMM_NOALLOC_MAX_POINTS;
constexpr int NA_MAX_POINT_BLOCKS = static_cast<int>((NA_MAX_POINTS + NA_PPB - 1) / NA_PPB);
constexpr size_t NA_TICKET_BYTES = 4096;            // >= NA_MAX_POINT_BLOCKS ints, keeps the partials 256-aligned
constexpr size_t NA_PARTIAL_DOUBLES = size_t(1) << 18;              // slices x points x 4 <= this (2 MiB)
constexpr size_t NA_SCRATCH_BYTES = NA_TICKET_BYTES + NA_PARTIAL_DOUBLES * sizeof(double);
static_assert(NA_MAX_POINT_BLOCKS * sizeof(int) <= NA_TICKET_BYTES, "tickets do not fit their region");
static_assert(NA_MAX_POINTS * 4 <= static_cast<int64_t>(NA_PARTIAL_DOUBLES), "one slice of the largest batch must fit");
constexpr int MAX_DEVICES = 64;

// [tickets: NA_MAX_POINT_BLOCKS ints, padded to 4 KiB][partials: [slices][P][4] doubles]
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_SCRATCH_BYTES];

struct NaParams {
    const double *src_xyz, *src_q, *nuc_xyz, *nuc_Z, *elec;
    double *V, *E;
    int64_t M, K;
    int P, slices;
    int *tickets;            // device address inside g_noalloc_scratch (from cudaGetSymbolAddress)
    double *partial;         // likewise
};

// grid = (point blocks, slices).  A CTA owns NA_PPB points (in registers of every thread) and one
// slice of the M cells + K nuclei (thread-strided: Eq. 8, the coalesced order);
// fixed-order butterfly + shared-memory sum per CTA; partial[slice][point][4]; the CTA that takes
// the last ticket of its point block adds the slices in index order (no floating-point atomics:
// bitwise reproducible) and writes V, E.
__global__ void __launch_bounds__(NA_THREADS) noalloc_eval_kernel(const NaParams p) {
    __shared__ double pts_s[NA_PPB * 3];
    __shared__ double red_s[NA_WARPS][NA_PPB * 4];
    __shared__ int last_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid < NA_PPB * 3) {
        int pi = blockIdx.x * NA_PPB + tid / 3;
        pi = pi < p.P ? pi : p.P - 1;                        // clamp: duplicates are not written
        pts_s[tid] = p.elec[static_cast<int64_t>(pi) * 3 + tid % 3];
    }
    __syncthreads();
    double px[NA_PPB], py[NA_PPB], pz[NA_PPB], V[NA_PPB], Ex[NA_PPB], Ey[NA_PPB], Ez[NA_PPB];
#pragma unroll
    for (int e = 0; e < NA_PPB; ++e) {
        px[e] = pts_s[3 * e]; py[e] = pts_s[3 * e + 1]; pz[e] = pts_s[3 * e + 2];
        V[e] = Ex[e] = Ey[e] = Ez[e] = 0.0;
    }
    const int64_t total = p.M + p.K;
    const int64_t lo = total / p.slices * blockIdx.y + (total % p.slices) * blockIdx.y / p.slices;
    const int64_t hi = total / p.slices * (blockIdx.y + 1) + (total % p.slices) * (blockIdx.y + 1) / p.slices;
    for (int64_t j = lo + tid; j < hi; j += NA_THREADS) {
        const bool cell = j < p.M;
        const double *pos = cell ? p.src_xyz + 3 * j : p.nuc_xyz + 3 * (j - p.M);
        const double q = cell ? p.src_q[j] : p.nuc_Z[j - p.M];            // nuclei enter with +Z
        const double sx = pos[0], sy = pos[1], sz = pos[2];
#pragma unroll
        for (int e = 0; e < NA_PPB; ++e) {
            const double dx = px[e] - sx, dy = py[e] - sy, dz = pz[e] - sz;
            const double y = rsqrt(fma(dz, dz, fma(dy, dy, dx * dx)));
            const double t = q * y;                                        // q / r
            const double g = t * (y * y);                                  // q / r^3
            V[e] += t;
            Ex[e] = fma(g, dx, Ex[e]);
            Ey[e] = fma(g, dy, Ey[e]);
            Ez[e] = fma(g, dz, Ez[e]);
        }
    }
#pragma unroll
    for (int e = 0; e < NA_PPB; ++e)
#pragma unroll
        for (int m = 16; m >= 1; m >>= 1) {
            V[e] += __shfl_xor_sync(0xffffffffu, V[e], m);
            Ex[e] += __shfl_xor_sync(0xffffffffu, Ex[e], m);
            Ey[e] += __shfl_xor_sync(0xffffffffu, Ey[e], m);
            Ez[e] += __shfl_xor_sync(0xffffffffu, Ez[e], m);
        }
    if (lane == 0) {
#pragma unroll
        for (int e = 0; e < NA_PPB; ++e) {
            red_s[warp][4 * e] = V[e]; red_s[warp][4 * e + 1] = Ex[e];
            red_s[warp][4 * e + 2] = Ey[e]; red_s[warp][4 * e + 3] = Ez[e];
        }
    }
    __syncthreads();
    if (tid < NA_PPB * 4) {                                  // value tid = 4 e + component
        double a = 0.0;
        for (int w = 0; w < NA_WARPS; ++w) a += red_s[w][tid];
        const int pi = blockIdx.x * NA_PPB + tid / 4;
        if (pi < p.P) p.partial[(static_cast<int64_t>(blockIdx.y) * p.P + pi) * 4 + (tid & 3)] = a;
    }
    __threadfence();                                         // this CTA's partials are visible
    __syncthreads();
    if (tid == 0) {
        last_s = atomicAdd(p.tickets + blockIdx.x, 1) == p.slices - 1;     // integer ticket only
        __threadfence();                                     // the other CTAs' partials, seen through the ticket
    }
    __syncthreads();
    if (!last_s) return;
    // last CTA of the point block: group g = warp adds slices g, g + 8, ... in index order, then the
    // eight groups are added in index order
    {
        const int pi = blockIdx.x * NA_PPB + lane / 4;
        double a = 0.0;
        if (pi < p.P)
            for (int s = warp; s < p.slices; s += NA_WARPS)
                a += __ldcg(p.partial + (static_cast<int64_t>(s) * p.P + pi) * 4 + (lane & 3));
        __syncthreads();                                     // red_s is reused
        red_s[warp][lane] = a;
        __syncthreads();
        if (warp == 0 && pi < p.P) {
            double r = 0.0;
            for (int w = 0; w < NA_WARPS; ++w) r += red_s[w][lane];
            if ((lane & 3) == 0) p.V[pi] = r;
            else if (p.E) p.E[3 * static_cast<int64_t>(pi) + (lane & 3) - 1] = r;
        }
    }
    if (tid == 0) p.tickets[blockIdx.x] = 0;                 // at rest again (the next call clears them anyway)
}

// Per device: the scratch array's device address and the SM count, resolved once.
struct NaDevice {
    bool ready = false;
    unsigned char *scratch = nullptr;
    int sm_count = 0;
};
NaDevice g_na_dev[MAX_DEVICES];
std::mutex g_na_mu;

qmmm_status na_fail(qmmm_status st, const std::string &msg) {
    qmmm::set_last_error(msg.c_str());
    return st;
}

// Set-up of the current device `dev`: cudaGetSymbolAddress with that device current.
qmmm_status na_setup(int dev, NaDevice **out) {
    if (dev < 0 || dev >= MAX_DEVICES) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: device ordinal out of range");
    std::lock_guard<std::mutex> lk(g_na_mu);
    NaDevice &d = g_na_dev[dev];
    if (!d.ready) {
        int major = 0, sms = 0;
        cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return na_fail(QMMM_ERR_CUDA, std::string("eval_noalloc: cudaDeviceGetAttribute: ") + cudaGetErrorString(e));
        if (major != 10)
            return na_fail(QMMM_ERR_UNSUPPORTED_DEVICE, "eval_noalloc: this library is built for sm_100a (B200) only");
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);   // the DEVICE address of the array on this device
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return na_fail(QMMM_ERR_CUDA, std::string("eval_noalloc: cudaGetSymbolAddress(g_noalloc_scratch): ") +
                                              cudaGetErrorString(e));
        }
        d.scratch = static_cast<unsigned char *>(ptr);
        d.sm_count = sms > 0 ? sms : 1;
        d.ready = true;
    }
    *out = &d;
    return QMMM_OK;
}

}  // namespace

extern "C" qmmm_status qmmm_field_eval_noalloc(const double *src_xyz, const double *src_q, int64_t M,
                                               const double *nuc_xyz, const double *nuc_Z, int64_t K,
                                               const double *elec_xyz, int64_t P, double *V, double *E,
                                               void *stream) {
    if (M < 0 || K < 0) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: negative M or K");
    if (M > 0 && (!src_xyz || !src_q)) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: NULL source array with M > 0");
    if (K > 0 && (!nuc_xyz || !nuc_Z)) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: NULL nuclear array with K > 0");
    if (!elec_xyz || !V) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: NULL elec_xyz or V");
    if (P < 1) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: P < 1");
    if (P > NA_MAX_POINTS)
        return na_fail(QMMM_ERR_INVALID_ARG,
                       "eval_noalloc: P = " + std::to_string(P) + " exceeds QMMM_NOALLOC_MAX_POINTS = " +
                           std::to_string(NA_MAX_POINTS) + " (the fixed scratch array holds no more; split the batch, "
                           "or use qmmm_field_create / qmmm_field_eval)");
    if (M > (int64_t(1) << 40) || K > (int64_t(1) << 40)) return na_fail(QMMM_ERR_INVALID_ARG, "eval_noalloc: M or K too large");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return na_fail(QMMM_ERR_CUDA, std::string("eval_noalloc: cudaGetDevice: ") + cudaGetErrorString(e));
    NaDevice *d = nullptr;
    qmmm_status st = na_setup(dev, &d);
    if (st != QMMM_OK) return st;

    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const int pb = static_cast<int>((P + NA_PPB - 1) / NA_PPB);
    // slices: about two CTAs per SM in all, at least 256 sources each, and slices x P x 4 doubles
    // must fit the partials region of the scratch array
    const int64_t total = M + K;
    int64_t slices = (2 * static_cast<int64_t>(d->sm_count) + pb - 1) / pb;
    slices = slices < (total + NA_THREADS - 1) / NA_THREADS ? slices : (total + NA_THREADS - 1) / NA_THREADS;
    const int64_t cap = static_cast<int64_t>(NA_PARTIAL_DOUBLES) / (4 * P);
    if (slices > cap) slices = cap;
    if (slices > 65535) slices = 65535;
    if (slices < 1) slices = 1;

    NaParams prm;
    prm.src_xyz = src_xyz; prm.src_q = src_q; prm.nuc_xyz = nuc_xyz; prm.nuc_Z = nuc_Z; prm.elec = elec_xyz;
    prm.V = V; prm.E = E;
    prm.M = M; prm.K = K;
    prm.P = static_cast<int>(P);
    prm.slices = static_cast<int>(slices);
    prm.tickets = reinterpret_cast<int *>(d->scratch);
    prm.partial = reinterpret_cast<double *>(d->scratch + NA_TICKET_BYTES);
    // the tickets must start at zero whatever an earlier (possibly failed) call left behind
    e = cudaMemsetAsync(prm.tickets, 0, static_cast<size_t>(pb) * sizeof(int), s);
    if (e != cudaSuccess) return na_fail(QMMM_ERR_CUDA, std::string("eval_noalloc: cudaMemsetAsync: ") + cudaGetErrorString(e));
    noalloc_eval_kernel<<<dim3(pb, static_cast<unsigned>(slices)), NA_THREADS, 0, s>>>(prm);
    e = cudaGetLastError();
    if (e != cudaSuccess) return na_fail(QMMM_ERR_CUDA, std::string("eval_noalloc: kernel launch: ") + cudaGetErrorString(e));
    return QMMM_OK;
}
