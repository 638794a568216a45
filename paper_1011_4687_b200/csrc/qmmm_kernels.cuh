// qmmm_kernels.cuh -- sm_100a device code of the pairwise hot loop.
//
// Mapping (PAPER.md:119-132, :177-184 restated for Blackwell):
//   * the source sum is split over CTAs ("blocks", Eq. 5-6); inside a CTA the 32 lanes
//     of a warp own different sources in thread-strided order (Eq. 8, the coalesced
//     order) and every thread keeps EPT evaluation points in registers (the paper's
//     "r_new in constant memory": uniform data kept next to the ALUs);
//   * sources live in HBM as 128-source SoA chunks x[128] y[128] z[128] q[128]; a
//     producer warp stages up to 8 chunks per pipeline stage into shared memory with
//     TMA bulk copies (cp.async.bulk + mbarrier complete_tx), consumers read them with
//     conflict-free 128-bit LDS (lane l owns sources 4l..4l+3 of a chunk);
//   * per-thread FP64 running sums, fixed-order warp-shuffle + shared-memory reduction,
//     one partial {V,Ex,Ey,Ez} per (slice, point) in a workspace, and a second kernel
//     that adds the slices in index order and the nuclear term (always FP64).
// No floating-point atomics anywhere: results are bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmmm {

constexpr int CHUNK = 128;          // sources per SoA chunk (4 per lane)
constexpr int BLOCK_CHUNKS = 8;     // chunks per origin block (FP32 tile-local coordinates)
constexpr int COMPUTE_WARPS = 8;    // consumer warps per CTA; +1 producer warp
constexpr int CTA_THREADS = 32 * (COMPUTE_WARPS + 1);
constexpr int STAGE_HDR = 128;      // bytes reserved per stage for the block origin

struct PairParams {
    const char *chunks;      // FP64: [n_chunks][4][128] double ; FP32: [n_chunks][4][128] float
    const double *origins;   // FP32 only: [n_blocks][4] (cx, cy, cz, pad)
    const double *elec;      // [P][3]
    double *partial;         // [slices][P][4]
    int P;
    int n_chunks;
    int slices;
    int point_warps;         // WP; source-split warps WS = COMPUTE_WARPS / WP
    int stages;
};

// ----------------------------------------------------------------------------- PTX helpers
__device__ __forceinline__ uint32_t smem_u32(const void *p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier.
__device__ __forceinline__ void tma_bulk_g2s(void *dst, const void *src, uint32_t bytes,
                                             uint64_t *bar) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
            "r"(smem_u32(dst)),
        "l"(src), "r"(bytes), "r"(smem_u32(bar))
        : "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void compute_warps_sync() {   // named barrier 1: consumers only
    asm volatile("bar.sync 1, %0;" ::"n"(32 * COMPUTE_WARPS) : "memory");
}
__device__ __forceinline__ float rsqrt_mufu_f32(float x) {          // MUFU.RSQ
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ double rsqrt_mufu_f64(double x) {        // MUFU.RSQ64H seed
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

// ----------------------------------------------------------------------------- pair math
// FP64 reciprocal square root: hardware seed (about 20+ bits) + ONE cubically convergent
// refinement  y <- y (1 + e/2 + 3 e^2/8),  e = 1 - x y^2  (relative error 2.5 eps0^3).
__device__ __forceinline__ double rsqrt_refined_f64(double x) {
    double y0 = rsqrt_mufu_f64(x);
    double t = x * y0;
    double e = fma(-t, y0, 1.0);
    double c = fma(0.375, e, 0.5);
    double u = y0 * e;
    return fma(u, c, y0);
}

// One FP64 pair: 18 DP-pipe instructions + 1 MUFU.
__device__ __forceinline__ void pair_f64(double rx, double ry, double rz, double sx, double sy,
                                         double sz, double q, double &V, double &Ex, double &Ey,
                                         double &Ez) {
    double dx = rx - sx, dy = ry - sy, dz = rz - sz;
    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    double y = rsqrt_refined_f64(r2);
    double p = q * y;
    V += p;
    double s = p * (y * y);
    Ex = fma(s, dx, Ex);
    Ey = fma(s, dy, Ey);
    Ez = fma(s, dz, Ez);
}

// One FP32 pair: 17 FP32-pipe instructions + 1 MUFU.RSQ (MUFU seed + one Newton step).
__device__ __forceinline__ void pair_f32(float ax, float ay, float az, float ox, float oy,
                                         float oz, float q, float &V, float &Ex, float &Ey,
                                         float &Ez) {
    float dx = ax - ox, dy = ay - oy, dz = az - oz;
    float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    float y0 = rsqrt_mufu_f32(r2);
    float t = r2 * y0;
    float e = fmaf(-t, y0, 1.0f);
    float h = 0.5f * y0;
    float y = fmaf(h, e, y0);
    float p = q * y;
    V += p;
    float s = p * (y * y);
    Ex = fmaf(s, dx, Ex);
    Ey = fmaf(s, dy, Ey);
    Ez = fmaf(s, dz, Ez);
}

// Slice s of S covers chunks [lo, hi): an even split at chunk granularity.
__device__ __host__ __forceinline__ void slice_range(int n_chunks, int S, int s, int &lo, int &hi) {
    lo = static_cast<int>((static_cast<int64_t>(n_chunks) * s) / S);
    hi = static_cast<int>((static_cast<int64_t>(n_chunks) * (s + 1)) / S);
}
// A pipeline stage never straddles an origin block: [c, min(hi, next block boundary)).
__device__ __forceinline__ int stage_end(int c, int hi) {
    int e = (c / BLOCK_CHUNKS + 1) * BLOCK_CHUNKS;
    return e < hi ? e : hi;
}

// Butterfly all-reduce over the 32 lanes in a fixed order (deterministic).
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    return v;
}

// ----------------------------------------------------------------------------- pair kernel
// grid = (slices, point_blocks).  REAL = double (FP64 path) or float (FP32-acc64 path).
template <typename REAL, int EPT>
__global__ void __launch_bounds__(CTA_THREADS, 1) pair_kernel(const PairParams prm) {
    constexpr bool F32 = sizeof(REAL) == 4;
    constexpr int CHUNK_BYTES = 4 * CHUNK * sizeof(REAL);
    constexpr int STAGE_BYTES = STAGE_HDR + BLOCK_CHUNKS * CHUNK_BYTES;

    extern __shared__ __align__(128) unsigned char smem[];
    // layout: [stages x STAGE_BYTES] [full barriers] [empty barriers] [reduction scratch]
    const int stages = prm.stages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + static_cast<size_t>(stages) * STAGE_BYTES);
    uint64_t *empty = full + 8;
    double *red = reinterpret_cast<double *>(empty + 8);   // [COMPUTE_WARPS][EPT*4]
    double *elec_s = red + COMPUTE_WARPS * EPT * 4;          // [WP*EPT][3]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WP = prm.point_warps, WS = COMPUTE_WARPS / WP;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.x, lo, hi);

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], COMPUTE_WARPS);
        }
        fence_barrier_init();
    }
    // stage the CTA's evaluation points (FP64) in shared memory
    const int ppb = WP * EPT;
    for (int i = threadIdx.x; i < ppb * 3; i += CTA_THREADS) {
        int p = blockIdx.y * ppb + i / 3;
        p = p < prm.P ? p : prm.P - 1;                       // clamp: duplicates are not written
        elec_s[i] = prm.elec[static_cast<int64_t>(p) * 3 + (i % 3)];
    }
    __syncthreads();

    if (warp == COMPUTE_WARPS) {
        // ===================== producer warp: one lane drives the TMA pipeline ==========
        if (lane == 0) {
            int c = lo, k = 0;
            while (c < hi) {
                const int ce = stage_end(c, hi);
                const int slot = k % stages;
                if (k >= stages) mbar_wait(&empty[slot], ((k / stages) - 1) & 1);
                unsigned char *dst = smem + static_cast<size_t>(slot) * STAGE_BYTES;
                const uint32_t bytes = static_cast<uint32_t>(ce - c) * CHUNK_BYTES;
                if constexpr (F32) {
                    mbar_expect_tx(&full[slot], bytes + 32);
                    tma_bulk_g2s(dst, prm.origins + 4 * (c / BLOCK_CHUNKS), 32, &full[slot]);
                } else {
                    mbar_expect_tx(&full[slot], bytes);
                }
                tma_bulk_g2s(dst + STAGE_HDR, prm.chunks + static_cast<size_t>(c) * CHUNK_BYTES,
                             bytes, &full[slot]);
                c = ce;
                ++k;
            }
        }
        return;
    }

    // ========================= consumer warps ============================================
    const int wp = warp % WP, ws = warp / WP;
    double V[EPT], Ex[EPT], Ey[EPT], Ez[EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) V[e] = Ex[e] = Ey[e] = Ez[e] = 0.0;

    REAL rx[EPT], ry[EPT], rz[EPT];
    if constexpr (!F32) {
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            rx[e] = static_cast<REAL>(elec_s[(wp * EPT + e) * 3 + 0]);
            ry[e] = static_cast<REAL>(elec_s[(wp * EPT + e) * 3 + 1]);
            rz[e] = static_cast<REAL>(elec_s[(wp * EPT + e) * 3 + 2]);
        }
    }

    int c = lo, k = 0;
    while (c < hi) {
        const int ce = stage_end(c, hi);
        const int slot = k % stages;
        mbar_wait(&full[slot], (k / stages) & 1);
        const unsigned char *st = smem + static_cast<size_t>(slot) * STAGE_BYTES;
        const REAL *data = reinterpret_cast<const REAL *>(st + STAGE_HDR);
        const int nch = ce - c;

        if constexpr (F32) {
            // tile-local coordinates: a = r_i - c_block formed in FP64, rounded once to FP32;
            // the rounding residual delta is applied as a first-order correction at the flush:
            // V(a_hat + delta) = V(a_hat) - E(a_hat) . delta.
            const double *org = reinterpret_cast<const double *>(st);
            const double cx = org[0], cy = org[1], cz = org[2];
            float v32[EPT], ex32[EPT], ey32[EPT], ez32[EPT];
            float ddx[EPT], ddy[EPT], ddz[EPT];   // rounding residuals (|delta| <= ulp/2 of a)
#pragma unroll
            for (int e = 0; e < EPT; ++e) {
                const double a0 = elec_s[(wp * EPT + e) * 3 + 0] - cx;
                const double a1 = elec_s[(wp * EPT + e) * 3 + 1] - cy;
                const double a2 = elec_s[(wp * EPT + e) * 3 + 2] - cz;
                rx[e] = static_cast<REAL>(a0);
                ry[e] = static_cast<REAL>(a1);
                rz[e] = static_cast<REAL>(a2);
                ddx[e] = static_cast<float>(a0 - static_cast<double>(rx[e]));
                ddy[e] = static_cast<float>(a1 - static_cast<double>(ry[e]));
                ddz[e] = static_cast<float>(a2 - static_cast<double>(rz[e]));
                v32[e] = ex32[e] = ey32[e] = ez32[e] = 0.0f;
            }
            for (int ch = ws; ch < nch; ch += WS) {
                const float *b = reinterpret_cast<const float *>(data) + ch * 4 * CHUNK + 4 * lane;
                const float4 X = *reinterpret_cast<const float4 *>(b);
                const float4 Y = *reinterpret_cast<const float4 *>(b + CHUNK);
                const float4 Z = *reinterpret_cast<const float4 *>(b + 2 * CHUNK);
                const float4 Q = *reinterpret_cast<const float4 *>(b + 3 * CHUNK);
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                    pair_f32(rx[e], ry[e], rz[e], X.x, Y.x, Z.x, Q.x, v32[e], ex32[e], ey32[e], ez32[e]);
                    pair_f32(rx[e], ry[e], rz[e], X.y, Y.y, Z.y, Q.y, v32[e], ex32[e], ey32[e], ez32[e]);
                    pair_f32(rx[e], ry[e], rz[e], X.z, Y.z, Z.z, Q.z, v32[e], ex32[e], ey32[e], ez32[e]);
                    pair_f32(rx[e], ry[e], rz[e], X.w, Y.w, Z.w, Q.w, v32[e], ex32[e], ey32[e], ez32[e]);
                }
            }
#pragma unroll
            for (int e = 0; e < EPT; ++e) {      // flush FP32 run -> FP64 running sums
                float corr = ex32[e] * ddx[e];
                corr = fmaf(ey32[e], ddy[e], corr);
                corr = fmaf(ez32[e], ddz[e], corr);
                V[e] += static_cast<double>(v32[e]) - static_cast<double>(corr);
                Ex[e] += static_cast<double>(ex32[e]);
                Ey[e] += static_cast<double>(ey32[e]);
                Ez[e] += static_cast<double>(ez32[e]);
            }
        } else {
            for (int ch = ws; ch < nch; ch += WS) {
                const double *b = reinterpret_cast<const double *>(data) + ch * 4 * CHUNK + 2 * lane;
                // lane owns sources 2l, 2l+1 and 64+2l, 64+2l+1 of the chunk (two conflict-free
                // 128-bit loads per array)
#pragma unroll
                for (int half = 0; half < 2; ++half) {
                    const double2 X = *reinterpret_cast<const double2 *>(b + half * 64);
                    const double2 Y = *reinterpret_cast<const double2 *>(b + CHUNK + half * 64);
                    const double2 Z = *reinterpret_cast<const double2 *>(b + 2 * CHUNK + half * 64);
                    const double2 Q = *reinterpret_cast<const double2 *>(b + 3 * CHUNK + half * 64);
#pragma unroll
                    for (int e = 0; e < EPT; ++e) {
                        pair_f64(rx[e], ry[e], rz[e], X.x, Y.x, Z.x, Q.x, V[e], Ex[e], Ey[e], Ez[e]);
                        pair_f64(rx[e], ry[e], rz[e], X.y, Y.y, Z.y, Q.y, V[e], Ex[e], Ey[e], Ez[e]);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);
        c = ce;
        ++k;
    }

    // ---- in-CTA reduction (paper: shared memory; here shuffle + smem) ----
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
        V[e] = warp_sum(V[e]);
        Ex[e] = warp_sum(Ex[e]);
        Ey[e] = warp_sum(Ey[e]);
        Ez[e] = warp_sum(Ez[e]);
    }
    if (lane == 0) {
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            double *r = red + (warp * EPT + e) * 4;
            r[0] = V[e]; r[1] = Ex[e]; r[2] = Ey[e]; r[3] = Ez[e];
        }
    }
    compute_warps_sync();
    // warps with ws == 0 add the WS source-split partners in index order and store
    if (ws == 0 && lane < EPT * 4) {
        double acc = 0.0;
        for (int s = 0; s < WS; ++s) acc += red[((s * WP + wp) * EPT) * 4 + lane];
        const int p = (blockIdx.y * WP + wp) * EPT + lane / 4;
        if (p < prm.P)
            prm.partial[(static_cast<int64_t>(blockIdx.x) * prm.P + p) * 4 + (lane & 3)] = acc;
    }
}

// ----------------------------------------------------------------------------- FP32 packed
// FP32-acc64 pair kernel for EPT >= 2: two evaluation points share one f32x2 register pair
// (sm_100 FADD2 / FMUL2 / FFMA2; the source scalar is a broadcast operand), so the 17
// FP32-pipe operations of a pair cost 8.5 issue slots and the issue port is no longer the
// limiter.  The per-thread FP64 running sums live in shared memory (one conflict-free
// column per thread) instead of 8*EPT registers, which leaves the register file to the
// interleaved FP32 chains: ptxas serialises the pairs when the doubles stay in registers.
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 bc(float a) { return make_float2(a, a); }   // broadcast operand

// One 128-source chunk: the lane's 4 sources x EP2 point pairs, written stage by stage so
// that EP2 independent chains are in flight around every MUFU.
template <int EP2>
__device__ __forceinline__ void chunk_f32x2(const float *b, const float2 (&rx)[EP2],
                                            const float2 (&ry)[EP2], const float2 (&rz)[EP2],
                                            float2 (&V)[EP2], float2 (&Ex)[EP2],
                                            float2 (&Ey)[EP2], float2 (&Ez)[EP2]) {
    const float4 X = *reinterpret_cast<const float4 *>(b);
    const float4 Y = *reinterpret_cast<const float4 *>(b + CHUNK);
    const float4 Z = *reinterpret_cast<const float4 *>(b + 2 * CHUNK);
    const float4 Q = *reinterpret_cast<const float4 *>(b + 3 * CHUNK);
    const float xs[4] = {X.x, X.y, X.z, X.w}, ys[4] = {Y.x, Y.y, Y.z, Y.w};
    const float zs[4] = {Z.x, Z.y, Z.z, Z.w}, qs[4] = {Q.x, Q.y, Q.z, Q.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        float2 dx[EP2], dy[EP2], dz[EP2], r2[EP2], y0[EP2];
        const float2 nx = bc(-xs[k]), ny = bc(-ys[k]), nz = bc(-zs[k]), qq = bc(qs[k]);
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            dx[e] = __fadd2_rn(rx[e], nx);
            dy[e] = __fadd2_rn(ry[e], ny);
            dz[e] = __fadd2_rn(rz[e], nz);
            r2[e] = __ffma2_rn(dz[e], dz[e], __ffma2_rn(dy[e], dy[e], __fmul2_rn(dx[e], dx[e])));
        }
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            y0[e].x = rsqrt_mufu_f32(r2[e].x);
            y0[e].y = rsqrt_mufu_f32(r2[e].y);
        }
#pragma unroll
        for (int e = 0; e < EP2; ++e) {       // one Newton step, then V and E (17 FP32 ops/pair)
            const float2 t = __fmul2_rn(r2[e], y0[e]);
            const float2 err = __ffma2_rn(f2(-t.x, -t.y), y0[e], bc(1.0f));
            const float2 h = __fmul2_rn(y0[e], bc(0.5f));
            const float2 y = __ffma2_rn(h, err, y0[e]);
            const float2 p = __fmul2_rn(y, qq);
            V[e] = __fadd2_rn(V[e], p);
            const float2 s = __fmul2_rn(p, __fmul2_rn(y, y));
            Ex[e] = __ffma2_rn(s, dx[e], Ex[e]);
            Ey[e] = __ffma2_rn(s, dy[e], Ey[e]);
            Ez[e] = __ffma2_rn(s, dz[e], Ez[e]);
        }
    }
}

// grid = (slices, point_blocks); EPT = 2 * EP2 points per thread; 8 warps, no producer warp:
// a 9th warp would put 3 warps on one SM sub-partition and cap every thread at 168
// registers.  Warp 0 drives the TMA pipeline inline, one stage ahead of its own consumption.
constexpr int F32X2_THREADS = 32 * COMPUTE_WARPS;

template <int EP2>
__global__ void __launch_bounds__(F32X2_THREADS, 1) pair_kernel_f32x2(const PairParams prm) {
    constexpr int EPT = 2 * EP2;
    constexpr int CHUNK_BYTES = 4 * CHUNK * sizeof(float);
    constexpr int STAGE_BYTES = STAGE_HDR + BLOCK_CHUNKS * CHUNK_BYTES;
    constexpr int NT = F32X2_THREADS;

    extern __shared__ __align__(128) unsigned char smem[];
    // layout: [stages x STAGE_BYTES] [full barriers] [empty barriers] [elec] [acc columns]
    const int stages = prm.stages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + static_cast<size_t>(stages) * STAGE_BYTES);
    uint64_t *empty = full + 8;
    double *elec_s = reinterpret_cast<double *>(empty + 8);   // [WP*EPT][3], WP <= 8
    double *acc = elec_s + COMPUTE_WARPS * EPT * 3;            // [EPT*4][NT]

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WP = prm.point_warps, WS = COMPUTE_WARPS / WP;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.x, lo, hi);

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], COMPUTE_WARPS);
        }
        fence_barrier_init();
    }
    const int ppb = WP * EPT;
    for (int i = threadIdx.x; i < ppb * 3; i += NT) {
        int p = blockIdx.y * ppb + i / 3;
        p = p < prm.P ? p : prm.P - 1;
        elec_s[i] = prm.elec[static_cast<int64_t>(p) * 3 + (i % 3)];
    }
    __syncthreads();

    // producer cursor (used by warp 0 only): next pipeline step to load
    int pc = lo, pk = 0;
    auto produce = [&]() {
        if (pc >= hi) return;
        const int ce = stage_end(pc, hi);
        const int slot = pk % stages;
        if (pk >= stages) mbar_wait(&empty[slot], ((pk / stages) - 1) & 1);
        if (lane == 0) {
            unsigned char *dst = smem + static_cast<size_t>(slot) * STAGE_BYTES;
            const uint32_t bytes = static_cast<uint32_t>(ce - pc) * CHUNK_BYTES;
            mbar_expect_tx(&full[slot], bytes + 32);
            tma_bulk_g2s(dst, prm.origins + 4 * (pc / BLOCK_CHUNKS), 32, &full[slot]);
            tma_bulk_g2s(dst + STAGE_HDR, prm.chunks + static_cast<size_t>(pc) * CHUNK_BYTES, bytes,
                         &full[slot]);
        }
        pc = ce;
        ++pk;
    };
    if (warp == 0)
        for (int i = 0; i < stages - 1; ++i) produce();

    const int wp = warp % WP, ws = warp / WP;
    double *my = acc + threadIdx.x;                 // column of this thread: my[i * NT]
#pragma unroll
    for (int i = 0; i < EPT * 4; ++i) my[i * NT] = 0.0;
    const double *pe = elec_s + wp * EPT * 3;

    int c = lo, k = 0;
    while (c < hi) {
        const int ce = stage_end(c, hi);
        const int slot = k % stages;
        if (warp == 0) produce();          // step k + stages - 1 into the slot freed by step k - 1
        mbar_wait(&full[slot], (k / stages) & 1);
        const unsigned char *st = smem + static_cast<size_t>(slot) * STAGE_BYTES;
        const float *data = reinterpret_cast<const float *>(st + STAGE_HDR);
        const int nch = ce - c;
        // tile-local coordinates a = r_i - c_block, formed in FP64 and rounded once
        const double *org = reinterpret_cast<const double *>(st);
        const double cx = org[0], cy = org[1], cz = org[2];
        float2 rx[EP2], ry[EP2], rz[EP2], v[EP2], ex[EP2], ey[EP2], ez[EP2];
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            rx[e] = f2(static_cast<float>(pe[6 * e + 0] - cx), static_cast<float>(pe[6 * e + 3] - cx));
            ry[e] = f2(static_cast<float>(pe[6 * e + 1] - cy), static_cast<float>(pe[6 * e + 4] - cy));
            rz[e] = f2(static_cast<float>(pe[6 * e + 2] - cz), static_cast<float>(pe[6 * e + 5] - cz));
            v[e] = ex[e] = ey[e] = ez[e] = f2(0.0f, 0.0f);
        }
        for (int ch = ws; ch < nch; ch += WS)
            chunk_f32x2<EP2>(data + ch * 4 * CHUNK + 4 * lane, rx, ry, rz, v, ex, ey, ez);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);   // the stage's source data is consumed
        // flush the FP32 run into the FP64 column; the rounding residual delta of a enters as
        // the first-order correction V(a_hat + delta) = V(a_hat) - E(a_hat) . delta
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
#pragma unroll
            for (int hlf = 0; hlf < 2; ++hlf) {
                const int pi = 2 * e + hlf;
                const float ax = hlf ? rx[e].y : rx[e].x, ay = hlf ? ry[e].y : ry[e].x;
                const float az = hlf ? rz[e].y : rz[e].x;
                const float fx = hlf ? ex[e].y : ex[e].x, fy = hlf ? ey[e].y : ey[e].x;
                const float fz = hlf ? ez[e].y : ez[e].x, fv = hlf ? v[e].y : v[e].x;
                const float ddx = static_cast<float>((pe[3 * pi + 0] - cx) - static_cast<double>(ax));
                const float ddy = static_cast<float>((pe[3 * pi + 1] - cy) - static_cast<double>(ay));
                const float ddz = static_cast<float>((pe[3 * pi + 2] - cz) - static_cast<double>(az));
                const float corr = fmaf(fz, ddz, fmaf(fy, ddy, fx * ddx));
                my[(4 * pi + 0) * NT] += static_cast<double>(fv) - static_cast<double>(corr);
                my[(4 * pi + 1) * NT] += static_cast<double>(fx);
                my[(4 * pi + 2) * NT] += static_cast<double>(fy);
                my[(4 * pi + 3) * NT] += static_cast<double>(fz);
            }
        }
        c = ce;
        ++k;
    }

    // ---- in-CTA reduction: fixed-order butterfly per value, then the WS partners in order ----
    double *red = acc;      // reuse: after the barrier, [COMPUTE_WARPS][EPT*4] at the front
    double mine = 0.0;
#pragma unroll
    for (int i = 0; i < EPT * 4; ++i) {
        const double t = warp_sum(my[i * NT]);
        if (lane == i) mine = t;
    }
    __syncthreads();                                 // every column has been read
    if (lane < EPT * 4) red[warp * EPT * 4 + lane] = mine;
    __syncthreads();
    if (ws == 0 && lane < EPT * 4) {
        double a = 0.0;
        for (int s = 0; s < WS; ++s) a += red[(s * WP + wp) * EPT * 4 + lane];
        const int p = (blockIdx.y * WP + wp) * EPT + lane / 4;
        if (p < prm.P)
            prm.partial[(static_cast<int64_t>(blockIdx.x) * prm.P + p) * 4 + (lane & 3)] = a;
    }
}

// ----------------------------------------------------------------------------- finalize
// Adds the slice partials in index order, then the nuclear term (always FP64, PAPER.md:117
// keeps U_nuc in double), and writes V, E.  TPP threads cooperate on one point.
struct FinalizeParams {
    const double *partial;   // [slices][P][4]
    const double *nuc;       // [K][4] packed x, y, z, Z
    const double *elec;      // [P][3]
    double *V;               // [P]
    double *E;               // [P][3] or NULL
    int P, slices, K, tpp;   // tpp: 32 or 256 threads per point
};

__global__ void __launch_bounds__(256) finalize_kernel(const FinalizeParams prm) {
    __shared__ double red[8][4];
    const int tpp = prm.tpp;
    const int per_cta = 256 / tpp;
    const int sub = threadIdx.x / tpp, t = threadIdx.x % tpp;
    const int p = blockIdx.x * per_cta + sub;
    const bool live = p < prm.P;
    const int pc = live ? p : prm.P - 1;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    for (int s = t; s < prm.slices; s += tpp) {
        const double4 v = *reinterpret_cast<const double4 *>(
            prm.partial + (static_cast<int64_t>(s) * prm.P + pc) * 4);
        a0 += v.x; a1 += v.y; a2 += v.z; a3 += v.w;
    }
    const double rx = prm.elec[3 * static_cast<int64_t>(pc) + 0];
    const double ry = prm.elec[3 * static_cast<int64_t>(pc) + 1];
    const double rz = prm.elec[3 * static_cast<int64_t>(pc) + 2];
    for (int j = t; j < prm.K; j += tpp) {
        const double4 n = *reinterpret_cast<const double4 *>(prm.nuc + 4 * static_cast<int64_t>(j));
        pair_f64(rx, ry, rz, n.x, n.y, n.z, n.w, a0, a1, a2, a3);
    }
    a0 = warp_sum(a0); a1 = warp_sum(a1); a2 = warp_sum(a2); a3 = warp_sum(a3);
    if (tpp == 256) {
        const int w = threadIdx.x >> 5;
        if ((threadIdx.x & 31) == 0) { red[w][0] = a0; red[w][1] = a1; red[w][2] = a2; red[w][3] = a3; }
        __syncthreads();
        if (threadIdx.x < 4) {
            double acc = 0.0;
            for (int i = 0; i < 8; ++i) acc += red[i][threadIdx.x];
            if (threadIdx.x == 0) prm.V[p] = acc;
            else if (prm.E) prm.E[3 * static_cast<int64_t>(p) + threadIdx.x - 1] = acc;
        }
    } else if (live && t == 0) {
        prm.V[p] = a0;
        if (prm.E) {
            prm.E[3 * static_cast<int64_t>(p) + 0] = a1;
            prm.E[3 * static_cast<int64_t>(p) + 1] = a2;
            prm.E[3 * static_cast<int64_t>(p) + 2] = a3;
        }
    }
}

// ----------------------------------------------------------------------------- packing
// a0: pack {R_j, q_j} once per environment.
// Pads (j >= M) replicate the last real source with charge 0: they contribute exactly 0.
__global__ void pack_f64_kernel(const double *xyz, const double *q, int64_t M, int64_t Mpad,
                                double *chunks) {
    const int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (j >= Mpad) return;
    const int64_t src = j < M ? j : M - 1;
    const int64_t ch = j / CHUNK;
    const int i = static_cast<int>(j % CHUNK);
    // within a chunk the FP64 consumer reads element pairs (2l, 2l+1) and (64+2l, 64+2l+1):
    // storage order is the natural one.
    double *c = chunks + ch * 4 * CHUNK;
    c[i] = xyz[3 * src + 0];
    c[CHUNK + i] = xyz[3 * src + 1];
    c[2 * CHUNK + i] = xyz[3 * src + 2];
    c[3 * CHUNK + i] = j < M ? q[src] : 0.0;
}

// One warp per origin block: centre of the bounding box of the block's real sources.
__global__ void origins_kernel(const double *xyz, int64_t M, int64_t n_blocks, double *origins) {
    const int64_t b = (blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (b >= n_blocks) return;
    const int64_t j0 = b * BLOCK_CHUNKS * CHUNK;
    int64_t j1 = j0 + BLOCK_CHUNKS * CHUNK;
    if (j1 > M) j1 = M;
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t j = j0 + lane; j < j1; j += 32)
        for (int k = 0; k < 3; ++k) {
            const double v = xyz[3 * j + k];
            lo[k] = fmin(lo[k], v);
            hi[k] = fmax(hi[k], v);
        }
    for (int k = 0; k < 3; ++k)
        for (int m = 16; m >= 1; m >>= 1) {
            lo[k] = fmin(lo[k], __shfl_xor_sync(0xffffffffu, lo[k], m));
            hi[k] = fmax(hi[k], __shfl_xor_sync(0xffffffffu, hi[k], m));
        }
    if (lane == 0) {
        for (int k = 0; k < 3; ++k) origins[4 * b + k] = 0.5 * (lo[k] + hi[k]);
        origins[4 * b + 3] = 0.0;
    }
}

__global__ void pack_f32_kernel(const double *xyz, const double *q, int64_t M, int64_t Mpad,
                                const double *origins, float *chunks) {
    const int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (j >= Mpad) return;
    const int64_t src = j < M ? j : M - 1;
    const int64_t ch = j / CHUNK;
    const int i = static_cast<int>(j % CHUNK);
    const double *o = origins + 4 * (ch / BLOCK_CHUNKS);
    float *c = chunks + ch * 4 * CHUNK;
    c[i] = static_cast<float>(xyz[3 * src + 0] - o[0]);
    c[CHUNK + i] = static_cast<float>(xyz[3 * src + 1] - o[1]);
    c[2 * CHUNK + i] = static_cast<float>(xyz[3 * src + 2] - o[2]);
    c[3 * CHUNK + i] = j < M ? static_cast<float>(q[src]) : 0.0f;
}

__global__ void pack_nuclei_kernel(const double *xyz, const double *Z, int64_t K, double *out) {
    const int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (j >= K) return;
    out[4 * j + 0] = xyz[3 * j + 0];
    out[4 * j + 1] = xyz[3 * j + 1];
    out[4 * j + 2] = xyz[3 * j + 2];
    out[4 * j + 3] = Z[j];
}

}  // namespace qmmm
