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
//   * per-thread FP64 running sums (cells in FP64 or FP32-acc64, nuclei always FP64),
//     fixed-order warp-shuffle + shared-memory reduction, one partial {V,Ex,Ey,Ez} per
//     (slice, point) in a workspace; the last CTA of a point block to arrive (integer
//     ticket) adds the slices in a fixed order and writes V, E: one launch per evaluation.
// No floating-point atomics anywhere: results are bitwise reproducible.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qmmm {

constexpr int CHUNK = 128;          // sources per SoA chunk (4 per lane)
#ifndef QMMM_BLOCK_CHUNKS
#define QMMM_BLOCK_CHUNKS 16
#endif
constexpr int BLOCK_CHUNKS = QMMM_BLOCK_CHUNKS;    // chunks per origin block (FP32 tile-local coordinates) = FP32 stage
constexpr int STAGE_CHUNKS_F64 = 8; // chunks per FP64 pipeline stage
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
    double lattice;          // FP32 only: coordinate quantum (power of two), and its inverse
    double inv_lattice;
    const double *nuc;       // [K][4] packed x, y, z, Z (always FP64)
    int K;
    double *V;               // [P]       final outputs, written by the last CTA of a point block
    double *E;               // [P][3] or NULL
    int *counters;           // [point_blocks] arrival tickets, zero between evaluations
    // per-move mailbox (qmmm_field_eval_host with few points): when host_flag is set, the CTA
    // that completes the LAST point block publishes seq to pinned host memory
    unsigned long long *host_flag;
    unsigned long long seq;
    int *done;               // point blocks finished (zero between evaluations)
    // grid layout (qmmm_grid.cuh): chunks = gchunks of charges only, n_chunks = their number,
    // nuc = nuclei in grid units; sums are formed in grid units and scaled at the partial store
    double g_org[3];         // position of node (0,0,0), bohr
    double g_inv_h[3];       // 1 / spacing per axis: u = (r - org) * inv_h puts the nodes at integers
    double g_sx, g_sy;       // hx / hz, hy / hz: distances are measured in units of hz
    int g_ortho;             // cells are not cubic (g_sx or g_sy differs from 1)
    double g_scaleV, g_scaleE;   // 1/hz, 1/hz^2
    int g_n[3], g_segs;      // nodes per axis (row = ix * ny + iy); z segments (gchunks) per row tile
    int g_dzt;               // grid kernels: dz table in shared memory (qmmm_grid.cuh, DZT)
    int g_accv;              // FP32 batched dz-table kernel: accurate V (z2 table, FP64 rxy2, compensated row sums)
    int g_fine;              // FP32 grid kernel: coordinate lattice per gchunk instead of per grid (long axes)
    // FP32 copies (list and grid) store q_j * 2^k with 2^k * max|q| in [0.5, 1): tiny charges keep
    // their full FP32 precision (no denormals, no flush), and the result does not depend on the
    // unit of charge.  q_unscale = 2^-k multiplies the cells' FP64 sums before the nuclei are added.
    double q_unscale;
    int g_light;             // host side only: FP64 grid kernel with 4 consumer warps (overlapped few-point evaluations)
    // push-model collection (overlapped few-point evaluations): tagged 64-byte records instead
    // of partials + fence + ticket; NULL = the ticket path
    unsigned long long *push_slots;   // [slices][P][8] words
    unsigned long long push_seq;      // tag of this evaluation (never 0, never reused)
    // per-move mailbox with the push collection: the collecting CTA writes one tagged record
    // {tag, V, Ex, Ey, Ez, tag} per point straight into pinned host memory (no system-scope
    // fence, no flag); NULL = V / E as usual
    unsigned long long *host_records; // [P][8] words, device-mapped host memory
    // per-move mailbox, up to INLINE_POINTS points: the coordinates travel as kernel parameters
    // (constant bank) instead of being read from pinned host memory over PCIe by every CTA
    int inline_pts;
    double pts[3 * 32];
    int pdl;                 // host side only: launch with programmatic stream serialization
    int *dev_err;            // device-mapped host word: set when a bounded wait gave up (never expected)
    int kernel_id;           // host side only: which instantiation was launched (qmmm_field_info.last_kernel)
#ifdef QMMM_PHASE_TIMING
    long long *dbg;          // [CTAs][10] clock64 at phase boundaries + globaltimer (diagnostic build)
#endif
};

constexpr int INLINE_POINTS = 32;
// coordinate idx (= 3 p + component) of the evaluation points
__device__ __forceinline__ double point_coord(const PairParams &prm, int64_t idx) {
    return prm.inline_pts ? prm.pts[idx] : prm.elec[idx];
}

// ----------------------------------------------------------------------------- PTX helpers
#ifdef QMMM_PHASE_TIMING
#define QMMM_MARK(i)                                                                          \
    do {                                                                                      \
        if (threadIdx.x == 0)                                                                 \
            prm.dbg[(blockIdx.y * gridDim.x + blockIdx.x) * 10 + (i)] = clock64();            \
    } while (0)
#define QMMM_MARK_GT(i)                                                                       \
    do {                                                                                      \
        if (threadIdx.x == 0) {                                                               \
            long long t;                                                                      \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));                             \
            prm.dbg[(blockIdx.y * gridDim.x + blockIdx.x) * 10 + (i)] = t;                    \
        }                                                                                     \
    } while (0)
#else
#define QMMM_MARK(i) do {} while (0)
#define QMMM_MARK_GT(i) do {} while (0)
#endif
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
// Programmatic dependent launch (qmmm_field_set_overlap).  Every evaluation kernel lets its
// successor in the stream start at once (launch_dependents, first instruction) and touches
// what a predecessor may still be using -- the partials workspace, the tickets, V and E --
// only after pdl_wait(): prologue, source walk, nuclear term and in-CTA reduction of evaluation
// n + 1 overlap the tail (fence, ticket, last-CTA sum) of evaluation n.  Both instructions are
// no-ops for launches without the attribute.
__device__ __forceinline__ void pdl_launch_dependents() {
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

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

// Tile-local coordinate of an evaluation point on the handle's coordinate lattice: the FP32
// offsets of the sources are multiples of the same power-of-two quantum, so the FP32
// subtraction d = a - o is EXACT (no rounding) whenever |d| < 2^24 quanta, i.e. for every
// point inside the environment's bounding box.  Plain FP32 rounding of d is coherent over
// a regular grid and biases V by ~2e-8 hartree per point.
__device__ __forceinline__ float lattice_round(double a64, double lattice, double inv_lattice) {
    return static_cast<float>(rint(a64 * inv_lattice) * lattice);
}
// The same with a quantum chosen per (point, origin block): the block's sources lie within
// `radius` of its origin on every axis, so every |a - o| < |a| + radius =: reach < 2^ex, and a
// lattice of 2^(ex - 24) -- never coarser than the handle's, of which the source offsets are
// multiples -- still makes d = a - o exact.  For the blocks NEAR a point this is far finer than
// the handle's quantum (2^-24 of the whole environment's extent), and those are the blocks
// that matter for the residual dd = (r - c) - a: V is corrected for it to first order
// (V(a + dd) = V(a) - E(a) . dd) but E itself is evaluated at a, with a relative error of about
// 3 |dd| / (distance to the cell) per term.  Returns a, sets dd.
__device__ __forceinline__ float lattice_round_local(double a64, double radius, double lattice,
                                                     double inv_lattice, float &dd) {
    const double reach = fabs(a64) + radius;                                  // radius >= 2 lattice > 0
    const int ex = ((__double2hiint(reach) >> 20) & 0x7ff) - 1022;            // reach < 2^ex
    double lam = __hiloint2double((ex - 24 + 1023) << 20, 0);
    double inv = __hiloint2double((24 - ex + 1023) << 20, 0);
    if (lam > lattice) { lam = lattice; inv = inv_lattice; }
    const double al = rint(a64 * inv) * lam;
    dd = static_cast<float>(a64 - al);
    return static_cast<float>(al);                                            // exact: |al| < 2^24 quanta
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

// Potential only (the paper's own computation, Eq. 4): 13 DP-pipe instructions + 1 MUFU.
__device__ __forceinline__ void pair_f64_v(double rx, double ry, double rz, double sx, double sy,
                                           double sz, double q, double &V) {
    double dx = rx - sx, dy = ry - sy, dz = rz - sz;
    double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    V = fma(q, rsqrt_refined_f64(r2), V);
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
template <int BC = BLOCK_CHUNKS>
__device__ __forceinline__ int stage_end(int c, int hi) {
    int e = (c / BC + 1) * BC;
    return e < hi ? e : hi;
}

// Butterfly all-reduce over the 32 lanes in a fixed order (deterministic).
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    return v;
}

// ----------------------------------------------------------------------------- epilogue
// a5: the nuclear term, always FP64 (the paper keeps U_nuc in double on the
// CPU).  The K nuclei are split over the source slices like the cells; inside
// a CTA over the source-split warps and the lanes.  Every thread adds its share for its EPT
// points to its FP64 sums before the in-CTA reduction.
template <int EPT>
__device__ __forceinline__ void nuclei_share(const PairParams &prm, const double *pe, int ws,
                                             int WS, int lane, double (&V)[EPT], double (&Ex)[EPT],
                                             double (&Ey)[EPT], double (&Ez)[EPT]) {
    int klo, khi;
    slice_range(prm.K, prm.slices, blockIdx.y, klo, khi);
    for (int j = klo + ws * 32 + lane; j < khi; j += 32 * WS) {
        const double2 a = *reinterpret_cast<const double2 *>(prm.nuc + 4 * static_cast<int64_t>(j));
        const double2 b = *reinterpret_cast<const double2 *>(prm.nuc + 4 * static_cast<int64_t>(j) + 2);
#pragma unroll
        for (int e = 0; e < EPT; ++e)
            pair_f64(pe[3 * e], pe[3 * e + 1], pe[3 * e + 2], a.x, a.y, b.x, b.y, V[e], Ex[e], Ey[e],
                     Ez[e]);
    }
}

// a4, cross-CTA part: the paper adds the block sums B[1..N_B] "by reduction" (PAPER.md:132,
// Eq. 5).  Each CTA has stored its partial; the CTA that takes the LAST ticket of its point
// block (an integer atomic; no floating-point atomics anywhere) adds the slices in a fixed
// order -- lane-strided, then the butterfly -- so the result does not depend on which CTA
// that is.  NT threads (whole warps) call this; sync() is their barrier.
template <int NT, typename SYNC>
__device__ __forceinline__ void finish_point_block(const PairParams &prm, int ppb, int tid,
                                                   int *flag, double *scratch /*[NT]*/, SYNC sync,
                                                   unsigned long long seq) {
    __threadfence();                                   // this CTA's partials are visible
    sync();
    if (tid == 0) {
        *flag = atomicAdd(prm.counters + blockIdx.x, 1) == prm.slices - 1;
        __threadfence();                               // the other CTAs' partials, seen through the ticket
    }
    sync();
    if (!*flag) return;
    QMMM_MARK(7);
    // thread = (group g, value v): nval = 4*ppb values {V,Ex,Ey,Ez} x points (a power of two
    // <= NT); group g adds slices g, g+G, g+2G, ... on eight interleaved accumulators (all
    // loads independent and coalesced over v), then the G groups are added in index order.
    const int nval = 4 * ppb, G = NT / nval;
    const int v = tid % nval, g = tid / nval;
    const int p = blockIdx.x * ppb + v / 4;
    double a[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};   // 8 loads in flight per thread
    if (p < prm.P) {
        const double *src = prm.partial + static_cast<int64_t>(p) * 4 + (v & 3);
        const int64_t stride = static_cast<int64_t>(prm.P) * 4;
        int sidx = g;
        for (; sidx + 7 * G < prm.slices; sidx += 8 * G) {
            double t[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) t[k] = __ldcg(src + (sidx + k * G) * stride);
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] += t[k];
        }
        // tail (< 8 G slices left): same accumulator order, compile-time indices (a[] stays in
        // registers) and all loads in flight together
        double t[8];
#pragma unroll
        for (int k = 0; k < 8; ++k)
            t[k] = sidx + k * G < prm.slices ? __ldcg(src + (sidx + k * G) * stride) : 0.0;
#pragma unroll
        for (int k = 0; k < 8; ++k) a[k] += t[k];
    }
    scratch[tid] = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
    sync();
    if (g == 0 && p < prm.P) {
        double a = 0.0;
        for (int k = 0; k < G; ++k) a += scratch[k * nval + v];
        if ((v & 3) == 0) prm.V[p] = a;
        else if (prm.E) prm.E[3 * static_cast<int64_t>(p) + (v & 3) - 1] = a;
    }
    if (tid == 0) prm.counters[blockIdx.x] = 0;        // ready for the next evaluation
    if (prm.host_flag) {
        __threadfence_system();                        // V, E (mapped host memory) before the flag
        sync();
        if (tid == 0 && atomicAdd(prm.done, 1) == static_cast<int>(gridDim.x) - 1) {
            *prm.done = 0;
            __threadfence_system();
            *reinterpret_cast<volatile unsigned long long *>(prm.host_flag) = seq;
        }
    }
}

// ---------------------------------------------------------------- push-model cross-CTA sum
// For overlapped few-point evaluations (qmmm_field_set_overlap) the serial tail of an
// evaluation -- partial store, fence, ticket atomic, fence, last-CTA loads -- is what bounds
// the period of a sequence (measured in isolation: 2.6 us at 37 CTAs, 3.4 us at 148).  Here
// every CTA instead stores each of its points' partials as ONE tagged 64-byte record of four
// self-validating 16-byte units {tag, V} {tag, Ex} {tag, Ey} {tag, Ez} (no fence, no atomic)
// and the CTA of slice 0 collects: its threads poll the records with volatile 16-byte loads
// until all four units carry this evaluation's tag (1.4 us at 37 CTAs, 2.5 us at 148), then add
// the slices in exactly the order of finish_point_block.
//
// What the protocol rests on: a naturally aligned 16-byte vector store / load of one thread
// (st.v2.u64 / ld.v2.u64) is performed as one access, so a unit is seen whole or not at all;
// nothing is assumed about the order in which the four units of a record, or different
// records, become visible.  (An earlier layout -- six 8-byte stores, tags at both ends of a
// 48-byte record -- assumed that a 32-byte sector is written atomically.)
//
// Tags.  A record is taken when its tags equal prm.push_seq, which is unique per evaluation
// ISSUED by the host -- but a kernel parameter, so a CUDA graph replays an evaluation with the
// same tag.  The collector therefore CLEARS the tags of every record it has consumed: when the
// same graph node runs again, its slots are untagged until this replay's CTAs push.  The
// clearing stores cannot race with the next evaluation's pushes: those are issued after its
// griddepcontrol.wait (overlapped launches) or after the kernel boundary (serial launches),
// i.e. after this grid has completed and its memory operations are visible.  A record that
// never arrives (cannot happen: every CTA of the grid pushes unconditionally) ends the poll
// after PUSH_HARD_NS with NaN results and sets the handle's device error word
// (qmmm_field_info.device_errors; the host-buffer calls return QMMM_ERR_CUDA).
constexpr int PUSH_SLOT_WORDS = 8;
constexpr long long PUSH_HARD_NS = 2000000000ll;
__device__ __forceinline__ long long push_global_ns() {
    long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
struct push_u64x2 { unsigned long long x, y; };
__device__ __forceinline__ push_u64x2 push_ld_v2(const unsigned long long *p) {
    push_u64x2 r;
    asm volatile("ld.volatile.global.v2.u64 {%0, %1}, [%2];" : "=l"(r.x), "=l"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ void push_st_v2(unsigned long long *p, unsigned long long a, unsigned long long b) {
    asm volatile("st.volatile.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
// Warps with ws == 0 call this with all 32 lanes: lane 4 e + c holds value c of the warp's
// point e (first point pbase); EPT <= 4.  One 16-byte store {tag, value} per lane.
template <int EPT>
__device__ __forceinline__ void push_records(const PairParams &prm, double a, int pbase, int lane) {
    static_assert(EPT <= 4, "four units per point, at most sixteen lanes");
    const int e = lane >> 2, c = lane & 3;
    const int p = pbase + e;
    if (lane < 4 * EPT && p < prm.P)
        push_st_v2(prm.push_slots + (static_cast<int64_t>(blockIdx.y) * prm.P + p) * PUSH_SLOT_WORDS + 2 * c,
                   prm.push_seq, static_cast<unsigned long long>(__double_as_longlong(a)));
}
// All NT threads of every CTA call this after the records are pushed.  rec_s: shared memory
// for slices * ppb * 4 doubles (the idle stage buffers), scratch: NT doubles, flag: one int.
template <int NT, typename SYNC>
__device__ __forceinline__ void finish_point_block_push(const PairParams &prm, int ppb, int tid, int *flag,
                                                        double *rec_s, double *scratch, SYNC sync) {
    if (blockIdx.y != 0) return;                       // slice 0 of each point block collects
    if (tid == 0) *flag = 1;
    sync();
    const long long t0 = push_global_ns();
    const int nrec = prm.slices * ppb;
    for (int r = tid; r < nrec; r += NT) {
        const int sl = r / ppb, pp = r - sl * ppb;
        const int p = blockIdx.x * ppb + pp;
        double *dst = rec_s + 4 * r;
        if (p >= prm.P) { dst[0] = dst[1] = dst[2] = dst[3] = 0.0; continue; }
        unsigned long long *q = prm.push_slots + (static_cast<int64_t>(sl) * prm.P + p) * PUSH_SLOT_WORDS;
        for (;;) {
            const push_u64x2 a = push_ld_v2(q), b = push_ld_v2(q + 2), c = push_ld_v2(q + 4), d = push_ld_v2(q + 6);
            if (a.x == prm.push_seq && b.x == prm.push_seq && c.x == prm.push_seq && d.x == prm.push_seq) {
                dst[0] = __longlong_as_double(static_cast<long long>(a.y));
                dst[1] = __longlong_as_double(static_cast<long long>(b.y));
                dst[2] = __longlong_as_double(static_cast<long long>(c.y));
                dst[3] = __longlong_as_double(static_cast<long long>(d.y));
                // consumed: untag, so that a replay of this launch (CUDA graph: same tag) waits
                // for its own records
#pragma unroll
                for (int u = 0; u < 4; ++u) push_st_v2(q + 2 * u, 0ull, 0ull);
                break;
            }
            if (push_global_ns() - t0 > PUSH_HARD_NS) {
                *flag = 0;
                if (prm.dev_err) *reinterpret_cast<volatile int *>(prm.dev_err) = 1;
                break;
            }
        }
    }
    sync();
    const bool ok = *flag != 0;
    // same association as finish_point_block: thread = (group g, value v)
    const int nval = 4 * ppb, G = NT / nval;
    const int v = tid % nval, g = tid / nval;
    const int p = blockIdx.x * ppb + v / 4;
    double a[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (p < prm.P && g < G) {
        const double *src = rec_s + v;                 // record (sl, pp): rec_s[(sl * ppb + pp) * 4 + c]
        int sidx = g;
        for (; sidx + 7 * G < prm.slices; sidx += 8 * G)
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] += src[(sidx + k * G) * nval];
#pragma unroll
        for (int k = 0; k < 8; ++k)
            if (sidx + k * G < prm.slices) a[k] += src[(sidx + k * G) * nval];
    }
    scratch[tid] = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
    sync();
    const bool mine = g == 0 && p < prm.P;
    double r = 0.0;
    if (mine) {
        for (int k = 0; k < G; ++k) r += scratch[k * nval + v];
        if (!ok) r = __longlong_as_double(0x7ff8000000000000ll);
    }
    if (prm.host_records) {
        // thread (g == 0, v) holds value v & 3 of the CTA's point v >> 2: one 16-byte store
        // {tag, value} into the point's record in pinned host memory
        if (mine)
            push_st_v2(prm.host_records + static_cast<int64_t>(p) * PUSH_SLOT_WORDS + 2 * (v & 3), prm.push_seq,
                       static_cast<unsigned long long>(__double_as_longlong(r)));
    } else if (mine) {
        if ((v & 3) == 0) prm.V[p] = r;
        else if (prm.E) prm.E[3 * static_cast<int64_t>(p) + (v & 3) - 1] = r;
    }
}

// ----------------------------------------------------------------------------- pair kernel
// grid = (point_blocks, slices).  REAL = double (FP64 path) or float (FP32-acc64 path).
template <typename REAL, int EPT, bool WITH_E = true>
__global__ void __launch_bounds__(CTA_THREADS, 1) pair_kernel(const PairParams prm) {
    constexpr bool F32 = sizeof(REAL) == 4;
    constexpr int CHUNK_BYTES = 4 * CHUNK * sizeof(REAL);
    constexpr int SC = F32 ? BLOCK_CHUNKS : STAGE_CHUNKS_F64;     // chunks per stage
    constexpr int STAGE_BYTES = STAGE_HDR + SC * CHUNK_BYTES;

    extern __shared__ __align__(128) unsigned char smem[];
    pdl_launch_dependents();
    QMMM_MARK_GT(8);
    QMMM_MARK(0);
    // layout: [stages x STAGE_BYTES] [full barriers] [empty barriers] [reduction scratch]
    const int stages = prm.stages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + static_cast<size_t>(stages) * STAGE_BYTES);
    uint64_t *empty = full + 8;
    int *flag = reinterpret_cast<int *>(empty + 8);        // last-CTA flag (16 bytes reserved)
    double *red = reinterpret_cast<double *>(empty + 10);  // [COMPUTE_WARPS][EPT*4]
    double *elec_s = red + 32 * COMPUTE_WARPS;               // [WP*EPT][3]; red has one double per thread

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WP = prm.point_warps, WS = COMPUTE_WARPS / WP;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.y, lo, hi);

    // The producer lane initialises the barriers itself and sends the first `stages` loads at
    // once; everybody else meanwhile stages the CTA's evaluation points (FP64) in shared memory.
    const bool producer = warp == COMPUTE_WARPS && lane == 0;
    int pc = lo, pk = 0;                                     // producer cursor
    auto load_step = [&]() {                                 // one pipeline step: [pc, stage end)
        const int ce = stage_end<SC>(pc, hi);
        const int slot = pk % stages;
        if (pk >= stages) mbar_wait(&empty[slot], ((pk / stages) - 1) & 1);
        unsigned char *dst = smem + static_cast<size_t>(slot) * STAGE_BYTES;
        const uint32_t bytes = static_cast<uint32_t>(ce - pc) * CHUNK_BYTES;
        if constexpr (F32) {
            mbar_expect_tx(&full[slot], bytes + 32);
            tma_bulk_g2s(dst, prm.origins + 4 * (pc / SC), 32, &full[slot]);
        } else {
            mbar_expect_tx(&full[slot], bytes);
        }
        tma_bulk_g2s(dst + STAGE_HDR, prm.chunks + static_cast<size_t>(pc) * CHUNK_BYTES, bytes,
                     &full[slot]);
        pc = ce;
        ++pk;
    };
    if (producer) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], COMPUTE_WARPS);
        }
        fence_barrier_init();
        while (pc < hi && pk < stages) load_step();
    }
    const int ppb = WP * EPT;
    for (int i = threadIdx.x; i < ppb * 3; i += CTA_THREADS) {
        int p = blockIdx.x * ppb + i / 3;
        p = p < prm.P ? p : prm.P - 1;                       // clamp: duplicates are not written
        elec_s[i] = point_coord(prm, static_cast<int64_t>(p) * 3 + (i % 3));
    }
    __syncthreads();
    QMMM_MARK(1);

    if (warp == COMPUTE_WARPS) {
        // ===================== producer warp: one lane drives the TMA pipeline ==========
        if (lane == 0)
            while (pc < hi) load_step();
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

    QMMM_MARK(2);
    int c = lo, k = 0;
    while (c < hi) {
        const int ce = stage_end<SC>(c, hi);
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
            const double cx = org[0], cy = org[1], cz = org[2], rad = org[3];
            float v32[EPT], ex32[EPT], ey32[EPT], ez32[EPT];
            float ddx[EPT], ddy[EPT], ddz[EPT];   // lattice residuals (|delta| <= half a local quantum)
#pragma unroll
            for (int e = 0; e < EPT; ++e) {
                const double a0 = elec_s[(wp * EPT + e) * 3 + 0] - cx;
                const double a1 = elec_s[(wp * EPT + e) * 3 + 1] - cy;
                const double a2 = elec_s[(wp * EPT + e) * 3 + 2] - cz;
                rx[e] = lattice_round_local(a0, rad, prm.lattice, prm.inv_lattice, ddx[e]);
                ry[e] = lattice_round_local(a1, rad, prm.lattice, prm.inv_lattice, ddy[e]);
                rz[e] = lattice_round_local(a2, rad, prm.lattice, prm.inv_lattice, ddz[e]);
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
                        if constexpr (WITH_E) {
                            pair_f64(rx[e], ry[e], rz[e], X.x, Y.x, Z.x, Q.x, V[e], Ex[e], Ey[e], Ez[e]);
                            pair_f64(rx[e], ry[e], rz[e], X.y, Y.y, Z.y, Q.y, V[e], Ex[e], Ey[e], Ez[e]);
                        } else {
                            pair_f64_v(rx[e], ry[e], rz[e], X.x, Y.x, Z.x, Q.x, V[e]);
                            pair_f64_v(rx[e], ry[e], rz[e], X.y, Y.y, Z.y, Q.y, V[e]);
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);
        c = ce;
        ++k;
    }

    QMMM_MARK(3);
    // FP64 path: the nuclei are ordinary sources at the end of the FP64 chunk array
    if constexpr (F32) {
        // the FP32 copy stores the cell charges times a power of two (PairParams::q_unscale)
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            V[e] *= prm.q_unscale; Ex[e] *= prm.q_unscale; Ey[e] *= prm.q_unscale; Ez[e] *= prm.q_unscale;
        }
        nuclei_share<EPT>(prm, elec_s + wp * EPT * 3, ws, WS, lane, V, Ex, Ey, Ez);
    }

    QMMM_MARK(4);
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
    pdl_wait();                                  // the previous evaluation is done with the workspace
    // warps with ws == 0 add the WS source-split partners in index order and store
    if (ws == 0) {
        double acc = 0.0;
        if (lane < EPT * 4)
            for (int s = 0; s < WS; ++s) acc += red[((s * WP + wp) * EPT) * 4 + lane];
        const int p = (blockIdx.x * WP + wp) * EPT + lane / 4;
        if (prm.push_slots)                      // few points, single wave: tagged records
            push_records<EPT>(prm, acc, (blockIdx.x * WP + wp) * EPT, lane);
        else if (lane < EPT * 4 && p < prm.P)
            prm.partial[(static_cast<int64_t>(blockIdx.y) * prm.P + p) * 4 + (lane & 3)] = acc;
    }
    QMMM_MARK(5);
    if (prm.push_slots) {                        // (uniform over the grid)
        finish_point_block_push<32 * COMPUTE_WARPS>(prm, WP * EPT, threadIdx.x, flag,
                                                    reinterpret_cast<double *>(smem), red,
                                                    [] { compute_warps_sync(); });
        QMMM_MARK(6);
        QMMM_MARK_GT(9);
        return;
    }
    finish_point_block<32 * COMPUTE_WARPS>(prm, WP * EPT, threadIdx.x, flag, red,
                                           [] { compute_warps_sync(); }, prm.seq);
    QMMM_MARK(6);
    QMMM_MARK_GT(9);
}

// ----------------------------------------------------------------------------- FP32 packed
// FP32-acc64 pair kernel for EPT >= 2: two evaluation points share one f32x2 register pair
// (sm_100 FADD2 / FMUL2 / FFMA2; the source scalar is a broadcast operand), so the 14
// FP32-pipe operations of a pair cost 7 issue slots and the issue port is no longer the
// limiter.  The per-thread FP64 running sums live in shared memory (one conflict-free
// column per thread) instead of 8*EPT registers, which leaves the register file to the
// interleaved FP32 chains: ptxas serialises the pairs when the doubles stay in registers.
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 bc(float a) { return make_float2(a, a); }   // broadcast operand

// One 128-source chunk: the lane's 4 sources x EP2 point pairs, written stage by stage so
// that EP2 independent chains are in flight around every MUFU.
//
// The Newton step is applied to the SUM, not to every pair.  With y0 = MUFU.RSQ(r^2),
// a = q y0 and c = q y0^3 (needed for the field anyway) the refined term is
//     q y1 = q y0 (3 - r^2 y0^2) / 2 = (3 a - c r^2) / 2,
// so V = (3 sum a - sum c r^2) / 2: one extra fma per pair (T += c r^2) instead of the four
// operations of a per-pair step, algebraically the same value.  The field uses y0 itself
// (tolerance 1e-5 relative per point; the raw MUFU values give 4e-7).  14 FP32-pipe
// operations per pair: 3 sub, mul + 2 fma (r^2), a, V0 += a, y0^2, c, T, 3 fma (E).
template <int EP2>
__device__ __forceinline__ void chunk_f32x2(const float *b, const float2 (&rx)[EP2],
                                            const float2 (&ry)[EP2], const float2 (&rz)[EP2],
                                            float2 (&V)[EP2], float2 (&T)[EP2], float2 (&Ex)[EP2],
                                            float2 (&Ey)[EP2], float2 (&Ez)[EP2]) {
    const float4 X = *reinterpret_cast<const float4 *>(b);
    const float4 Y = *reinterpret_cast<const float4 *>(b + CHUNK);
    const float4 Z = *reinterpret_cast<const float4 *>(b + 2 * CHUNK);
    const float4 Q = *reinterpret_cast<const float4 *>(b + 3 * CHUNK);
    const float xs[4] = {X.x, X.y, X.z, X.w}, ys[4] = {Y.x, Y.y, Y.z, Y.w};
    const float zs[4] = {Z.x, Z.y, Z.z, Z.w}, qs[4] = {Q.x, Q.y, Q.z, Q.w};
    // V0 and T are summed as trees of short FP32 runs (4 sources -> 4 chunks -> stage): a long
    // FP32 running sum of slowly varying same-sign terms drifts systematically (DESIGN.md
    // "FP32 path": +8e-8 hartree per point at 64 terms), a 4-term run does not.
    float2 Vc[EP2], Tc[EP2];
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
        for (int e = 0; e < EP2; ++e) {
            const float2 a = __fmul2_rn(y0[e], qq);
            Vc[e] = k == 0 ? a : __fadd2_rn(Vc[e], a);
            const float2 c = __fmul2_rn(a, __fmul2_rn(y0[e], y0[e]));
            Tc[e] = k == 0 ? __fmul2_rn(c, r2[e]) : __ffma2_rn(c, r2[e], Tc[e]);
            Ex[e] = __ffma2_rn(c, dx[e], Ex[e]);
            Ey[e] = __ffma2_rn(c, dy[e], Ey[e]);
            Ez[e] = __ffma2_rn(c, dz[e], Ez[e]);
        }
    }
#pragma unroll
    for (int e = 0; e < EP2; ++e) {
        V[e] = __fadd2_rn(V[e], Vc[e]);
        T[e] = __fadd2_rn(T[e], Tc[e]);
    }
}

// grid = (point_blocks, slices); EPT = 2 * EP2 points per thread; NW consumer warps and no
// producer warp: a 9th warp would put 3 warps on one SM sub-partition and cap every thread
// at 168 registers.  Warp 0 drives the TMA pipeline inline, stages-1 steps ahead.
//   NW = 8,  EP2 = 4 : 2 warps per sub-partition, 8 points per thread (<= 255 registers)
//   NW = 16, EP2 = 2 : 4 warps per sub-partition, 4 points per thread (<= 128 registers)
// Shared memory: [stages x STAGE] [full/empty barriers] [elec FP64] [a/dd scratch per warp]
//                [FP64 columns: EPT*4 doubles per thread, stored as double2 rows].
template <int EP2, int NW>
struct F32x2Layout {
    static constexpr int EPT = 2 * EP2;
    static constexpr int NT = 32 * NW;
    static constexpr int CHUNK_BYTES = 4 * CHUNK * sizeof(float);
    static constexpr int STAGE_BYTES = STAGE_HDR + BLOCK_CHUNKS * CHUNK_BYTES;
    static constexpr int BAR_BYTES = 18 * sizeof(uint64_t);     // 8 full, 8 empty, last-CTA flag
    static constexpr int ELEC_BYTES = NW * EPT * 3 * sizeof(double);
    static constexpr int SCRATCH_BYTES = NW * 2 * 3 * EPT * sizeof(float);
    static constexpr int ACC_BYTES = EPT * 4 * NT * sizeof(double);
    __host__ __device__ static constexpr size_t total(int stages) {
        return static_cast<size_t>(stages) * STAGE_BYTES + BAR_BYTES + ELEC_BYTES + SCRATCH_BYTES +
               ACC_BYTES;
    }
};

template <int EP2, int NW>
__global__ void __launch_bounds__(32 * NW, 1) pair_kernel_f32x2(const PairParams prm) {
    using L = F32x2Layout<EP2, NW>;
    constexpr int EPT = L::EPT, NT = L::NT;
    constexpr int CHUNK_BYTES = L::CHUNK_BYTES, STAGE_BYTES = L::STAGE_BYTES;

    extern __shared__ __align__(128) unsigned char smem[];
    pdl_launch_dependents();
    QMMM_MARK_GT(8);
    QMMM_MARK(0);
    const int stages = prm.stages;
    unsigned char *ptr = smem + static_cast<size_t>(stages) * STAGE_BYTES;
    uint64_t *full = reinterpret_cast<uint64_t *>(ptr);
    uint64_t *empty = full + 8;
    int *flag = reinterpret_cast<int *>(empty + 8);
    ptr += L::BAR_BYTES;
    double *elec_s = reinterpret_cast<double *>(ptr);          // [WP*EPT][3]
    ptr += L::ELEC_BYTES;
    float *scratch = reinterpret_cast<float *>(ptr);           // per warp: a[3][EPT], dd[3][EPT]
    ptr += L::SCRATCH_BYTES;
    double2 *acc = reinterpret_cast<double2 *>(ptr);           // [EPT*2][NT] double2

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WP = prm.point_warps, WS = NW / WP;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.y, lo, hi);

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], NW);
        }
        fence_barrier_init();
    }
    // ---- producer cursor (warp 0 only): next pipeline step to load -------------------------
    int pc = lo, pslot = 0;
    uint32_t pphase = 0;
    bool pwrapped = false;
    auto produce = [&]() {
        if (pc >= hi) return;
        const int ce = stage_end(pc, hi);
        if (pwrapped) mbar_wait(&empty[pslot], pphase);
        if (lane == 0) {
            unsigned char *dst = smem + static_cast<size_t>(pslot) * STAGE_BYTES;
            const uint32_t bytes = static_cast<uint32_t>(ce - pc) * CHUNK_BYTES;
            mbar_expect_tx(&full[pslot], bytes + 32);
            tma_bulk_g2s(dst, prm.origins + 4 * (pc / BLOCK_CHUNKS), 32, &full[pslot]);
            tma_bulk_g2s(dst + STAGE_HDR, prm.chunks + static_cast<size_t>(pc) * CHUNK_BYTES, bytes,
                         &full[pslot]);
        }
        pc = ce;
        if (++pslot == stages) {
            pslot = 0;
            if (pwrapped) pphase ^= 1u;
            pwrapped = true;
        }
    };
    // The first loads go out before anything else: they need only the barriers, which the
    // issuing thread has just initialised itself.
    if (warp == 0) {
        __syncwarp();
        for (int i = 0; i < stages - 1; ++i) produce();
    }
    const int ppb = WP * EPT;
    for (int i = threadIdx.x; i < ppb * 3; i += NT) {
        int p = blockIdx.x * ppb + i / 3;
        p = p < prm.P ? p : prm.P - 1;                          // clamp: duplicates are not written
        elec_s[i] = point_coord(prm, static_cast<int64_t>(p) * 3 + (i % 3));
    }
    __syncthreads();
    QMMM_MARK(1);

    const int wp = warp % WP, ws = warp / WP;
    double2 *my = acc + threadIdx.x;                 // this thread's column: my[i * NT]
#pragma unroll
    for (int i = 0; i < EPT * 2; ++i) my[i * NT] = make_double2(0.0, 0.0);
    const double *pe = elec_s + wp * EPT * 3;
    float *a_s = scratch + warp * 6 * EPT;           // a[3][EPT]
    float *dd_s = a_s + 3 * EPT;                     // dd[3][EPT]

    int slot = 0;
    uint32_t phase = 0;
    QMMM_MARK(2);
    for (int c = lo; c < hi;) {
        const int ce = stage_end(c, hi);
        if (warp == 0) produce();          // step k + stages - 1 into the slot freed by step k - 1
        mbar_wait(&full[slot], phase);
        const unsigned char *st = smem + static_cast<size_t>(slot) * STAGE_BYTES;
        const float *data = reinterpret_cast<const float *>(st + STAGE_HDR);
        const int nch = ce - c;
        // Tile-local coordinates a = r_i - c_block: formed in FP64 and rounded once, by the
        // first 3*EPT lanes for the whole warp; dd = (r_i - c_block) - a is the rounding residual.
        __syncwarp();
        if (lane < 3 * EPT) {
            const int comp = lane / EPT, pt = lane % EPT;
            const double a64 = pe[3 * pt + comp] - reinterpret_cast<const double *>(st)[comp];
            float dd32;
            a_s[lane] = lattice_round_local(a64, reinterpret_cast<const double *>(st)[3], prm.lattice,
                                            prm.inv_lattice, dd32);
            dd_s[lane] = dd32;
        }
        __syncwarp();
        float2 rx[EP2], ry[EP2], rz[EP2], v[EP2], tq[EP2], ex[EP2], ey[EP2], ez[EP2];
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            rx[e] = *reinterpret_cast<const float2 *>(a_s + 2 * e);
            ry[e] = *reinterpret_cast<const float2 *>(a_s + EPT + 2 * e);
            rz[e] = *reinterpret_cast<const float2 *>(a_s + 2 * EPT + 2 * e);
            v[e] = tq[e] = ex[e] = ey[e] = ez[e] = f2(0.0f, 0.0f);
        }
        for (int ch = ws; ch < nch;) {
            float2 v4[EP2], t4[EP2];                  // middle level of the trees: 4 chunks
#pragma unroll
            for (int e = 0; e < EP2; ++e) v4[e] = t4[e] = f2(0.0f, 0.0f);
#pragma unroll 1
            for (int g = 0; g < 4 && ch < nch; ++g, ch += WS)
                chunk_f32x2<EP2>(data + ch * 4 * CHUNK + 4 * lane, rx, ry, rz, v4, t4, ex, ey, ez);
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                v[e] = __fadd2_rn(v[e], v4[e]);
                tq[e] = __fadd2_rn(tq[e], t4[e]);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);   // the stage's source data is consumed
        // Flush the FP32 run into the FP64 columns.  The residual dd enters as the first-order
        // correction V(a + dd) = V(a) - E(a) . dd.
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            const float2 ddx = *reinterpret_cast<const float2 *>(dd_s + 2 * e);
            const float2 ddy = *reinterpret_cast<const float2 *>(dd_s + EPT + 2 * e);
            const float2 ddz = *reinterpret_cast<const float2 *>(dd_s + 2 * EPT + 2 * e);
            const float2 corr = __ffma2_rn(ez[e], ddz, __ffma2_rn(ey[e], ddy, __fmul2_rn(ex[e], ddx)));
            double2 t;                                // rows of the pair: V, Ex, Ey, Ez
            t = my[(4 * e + 0) * NT];                // V = (3 sum a - sum c r^2) / 2: the Newton step
            t.x += 1.5 * static_cast<double>(v[e].x) - 0.5 * static_cast<double>(tq[e].x) -
                   static_cast<double>(corr.x);
            t.y += 1.5 * static_cast<double>(v[e].y) - 0.5 * static_cast<double>(tq[e].y) -
                   static_cast<double>(corr.y);
            my[(4 * e + 0) * NT] = t;
            t = my[(4 * e + 1) * NT];
            t.x += static_cast<double>(ex[e].x);
            t.y += static_cast<double>(ex[e].y);
            my[(4 * e + 1) * NT] = t;
            t = my[(4 * e + 2) * NT];
            t.x += static_cast<double>(ey[e].x);
            t.y += static_cast<double>(ey[e].y);
            my[(4 * e + 2) * NT] = t;
            t = my[(4 * e + 3) * NT];
            t.x += static_cast<double>(ez[e].x);
            t.y += static_cast<double>(ez[e].y);
            my[(4 * e + 3) * NT] = t;
        }
        c = ce;
        if (++slot == stages) {
            slot = 0;
            phase ^= 1u;
        }
    }

    QMMM_MARK(3);
    // nuclear term of this CTA's share, FP64, into the same columns
    {
        double nV[EPT], nEx[EPT], nEy[EPT], nEz[EPT];
#pragma unroll
        for (int e = 0; e < EPT; ++e) nV[e] = nEx[e] = nEy[e] = nEz[e] = 0.0;
        nuclei_share<EPT>(prm, pe, ws, WS, lane, nV, nEx, nEy, nEz);
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            double2 t;
            // (the cells' sums carry the power-of-two scale of the FP32 charges: q_unscale)
            const double qu = prm.q_unscale;
            t = my[(4 * e + 0) * NT]; t.x = fma(t.x, qu, nV[2 * e]); t.y = fma(t.y, qu, nV[2 * e + 1]); my[(4 * e + 0) * NT] = t;
            t = my[(4 * e + 1) * NT]; t.x = fma(t.x, qu, nEx[2 * e]); t.y = fma(t.y, qu, nEx[2 * e + 1]); my[(4 * e + 1) * NT] = t;
            t = my[(4 * e + 2) * NT]; t.x = fma(t.x, qu, nEy[2 * e]); t.y = fma(t.y, qu, nEy[2 * e + 1]); my[(4 * e + 2) * NT] = t;
            t = my[(4 * e + 3) * NT]; t.x = fma(t.x, qu, nEz[2 * e]); t.y = fma(t.y, qu, nEz[2 * e + 1]); my[(4 * e + 3) * NT] = t;
        }
    }

    QMMM_MARK(4);
    // ---- in-CTA reduction through shared memory (paper: PAPER.md:132) ------------------------
    // Column row i = 4e+comp holds {V,Ex,Ey,Ez}[comp] of points (2e, 2e+1) for every thread.
    // Lane r < 2*EPT of each warp adds row r over the warp's 32 columns, starting at column r
    // (a rotation: the 32 lanes touch 32 different 16-byte slots, so the loads are conflict-
    // free and the order is fixed).  10x fewer instructions than 64 butterflies of shuffles.
    double *red = reinterpret_cast<double *>(acc);   // reused after the barrier: [NW][EPT*4]
    double2 tot = make_double2(0.0, 0.0);
    __syncwarp();
    if (lane < 2 * EPT) {
        const double2 *row = acc + lane * NT + warp * 32;
#pragma unroll 8
        for (int j = 0; j < 32; ++j) {
            const double2 t = row[(j + lane) & 31];
            tot.x += t.x;
            tot.y += t.y;
        }
    }
    __syncthreads();                                 // every column has been read
    if (lane < 2 * EPT) {                            // row 4e+comp -> values 8e+comp, 8e+4+comp
        red[warp * EPT * 4 + 8 * (lane >> 2) + (lane & 3)] = tot.x;
        red[warp * EPT * 4 + 8 * (lane >> 2) + 4 + (lane & 3)] = tot.y;
    }
    __syncthreads();
    pdl_wait();                                  // the previous evaluation is done with the workspace
    if (ws == 0) {
        double a = 0.0;
        if (lane < EPT * 4)
            for (int s = 0; s < WS; ++s) a += red[(s * WP + wp) * EPT * 4 + lane];
        const int p = (blockIdx.x * WP + wp) * EPT + lane / 4;
        if constexpr (EPT <= 4) {
            if (prm.push_slots) push_records<EPT>(prm, a, (blockIdx.x * WP + wp) * EPT, lane);
        }
        if (!(EPT <= 4 && prm.push_slots) && lane < EPT * 4 && p < prm.P)
            prm.partial[(static_cast<int64_t>(blockIdx.y) * prm.P + p) * 4 + (lane & 3)] = a;
    }
    QMMM_MARK(5);
    if constexpr (EPT <= 4) {
        if (prm.push_slots) {                    // (uniform over the grid)
            finish_point_block_push<NT>(prm, WP * EPT, threadIdx.x, flag, reinterpret_cast<double *>(smem), red,
                                        [] { __syncthreads(); });
            QMMM_MARK(6);
            QMMM_MARK_GT(9);
            return;
        }
    }
    finish_point_block<NT>(prm, WP * EPT, threadIdx.x, flag, red, [] { __syncthreads(); }, prm.seq);
    QMMM_MARK(6);
    QMMM_MARK_GT(9);
}

// ----------------------------------------------------------------------------- walker energy
// U_ES of one configuration (Eq. 4: the energy of the electrons in the
// environment's field, U = -sum_i V(r_i) with the library's sign convention): one warp per
// walker, lane-strided fixed-order sums, then the butterfly.  Deterministic.
__global__ void __launch_bounds__(256) walker_energy_kernel(const double *V, int64_t W, int64_t N,
                                                            double *U) {
    const int64_t w = blockIdx.x * 8ll + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (w >= W) return;
    const double *v = V + w * N;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    int64_t i = lane;
    for (; i + 96 < N; i += 128) {
        a0 += v[i]; a1 += v[i + 32]; a2 += v[i + 64]; a3 += v[i + 96];
    }
    for (; i < N; i += 32) a0 += v[i];
    const double s = warp_sum((a0 + a1) + (a2 + a3));
    if (lane == 0) U[w] = -s;
}

// ----------------------------------------------------------------------------- rank partials
// Eq. 5 across devices (U = B[1] + ... + B[N_B], one block per GPU): the
// per-rank partials parts[r][n] are added in RANK ORDER 0, 1, 2, ... (a plain left-to-right
// sum), so every rank that holds the same gathered partials gets bitwise the same result.
__global__ void __launch_bounds__(256) sum_rank_partials_kernel(const double *parts, int R, int64_t n,
                                                                double *out) {
    const int64_t i = blockIdx.x * 256ll + threadIdx.x;
    if (i >= n) return;
    double a = parts[i];
    for (int r = 1; r < R; ++r) a += parts[static_cast<int64_t>(r) * n + i];
    out[i] = a;
}

// ----------------------------------------------------------------------------- packing
// a0: pack {R_j, q_j} once per environment.
// Pads (j >= M) replicate the last real source with charge 0: they contribute exactly 0.
__global__ void pack_f64_kernel(const double *xyz, const double *q, int64_t M,
                                const double *nuc_xyz, const double *nuc_Z, int64_t K, int64_t Mpad,
                                double *chunks) {
    const int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (j >= Mpad) return;
    // FP64 copy: the M cells, then the K nuclei (charge +Z) as ordinary sources; pads replicate
    // the last real entry with charge 0.
    const int64_t jj = j < M + K ? j : M + K - 1;
    const bool cell = jj < M;
    const double *pos = cell ? xyz + 3 * jj : nuc_xyz + 3 * (jj - M);
    const double charge = j < M + K ? (cell ? q[jj] : nuc_Z[jj - M]) : 0.0;
    double *c = chunks + (j / CHUNK) * 4 * CHUNK;
    const int i = static_cast<int>(j % CHUNK);
    c[i] = pos[0];
    c[CHUNK + i] = pos[1];
    c[2 * CHUNK + i] = pos[2];
    c[3 * CHUNK + i] = charge;
}

// Bounding box of all sources: CTA b writes {lo[3], hi[3]} to part[6b..]; the host finishes.
__global__ void __launch_bounds__(256) bbox_kernel(const double *xyz, int64_t M, double *part) {
    __shared__ double sh[8][6];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t j = blockIdx.x * 256ll + threadIdx.x; j < M; j += 256ll * gridDim.x)
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
    if ((threadIdx.x & 31) == 0)
        for (int k = 0; k < 3; ++k) {
            sh[threadIdx.x >> 5][k] = lo[k];
            sh[threadIdx.x >> 5][3 + k] = hi[k];
        }
    __syncthreads();
    if (threadIdx.x < 6) {
        double v = sh[0][threadIdx.x];
        for (int w = 1; w < 8; ++w)
            v = threadIdx.x < 3 ? fmin(v, sh[w][threadIdx.x]) : fmax(v, sh[w][threadIdx.x]);
        part[6 * blockIdx.x + threadIdx.x] = v;
    }
}

// max |q| over n values (as the bits of the non-negative double: an integer maximum)
__global__ void __launch_bounds__(256) absmax_kernel(const double *q, int64_t n, unsigned long long *out) {
    double m = 0.0;
    for (int64_t j = blockIdx.x * 256ll + threadIdx.x; j < n; j += 256ll * gridDim.x) {
        const double v = fabs(q[j]);
        if (v > m && v < 1e300) m = v;
    }
    for (int k = 16; k >= 1; k >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, k));
    if ((threadIdx.x & 31) == 0 && m > 0.0)
        atomicMax(out, static_cast<unsigned long long>(__double_as_longlong(m)));
}

// One warp per origin block: centre of the bounding box of the block's real sources.
__global__ void origins_kernel(const double *xyz, int64_t M, int64_t n_blocks, double lattice,
                               double *origins) {
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
        // centre of the bounding box, plus a deterministic sub-quantum jitter so that the
        // lattice residuals of an evaluation point differ from block to block
        for (int k = 0; k < 3; ++k) {
            uint64_t hsh = (static_cast<uint64_t>(b) * 3 + k + 1) * 0x9E3779B97F4A7C15ull;
            hsh ^= hsh >> 29; hsh *= 0xBF58476D1CE4E5B9ull; hsh ^= hsh >> 32;
            const double u = static_cast<double>(hsh >> 11) * (1.0 / 9007199254740992.0) - 0.5;
            origins[4 * b + k] = 0.5 * (lo[k] + hi[k]) + u * lattice;
        }
        // reach of the block: its sources (after rounding to the lattice) lie within this
        // distance of the origin on every axis (lattice_round_local)
        double rad = 0.0;
        for (int k = 0; k < 3; ++k) rad = fmax(rad, 0.5 * (hi[k] - lo[k]));
        origins[4 * b + 3] = rad + 2.0 * lattice;
    }
}

// FP32 copy: offsets from the block origin and charges, rounded with ERROR FEEDBACK along
// memory order inside each 128-source chunk (one thread per chunk).  Plain round-to-nearest
// of a regular grid's coordinates is a coherent pattern (the same residual at every node
// with the same offset), which shifts V in the whole QM region by the same ~1e-8 hartree;
// rounding errors of the charges do the same on a smaller scale.  Here every coordinate is
// rounded to whichever of its two LATTICE neighbours keeps the running dipole residual
// sum_j q_j (x_j - c - o_j) smallest, and every charge absorbs the residual of the previous
// one, so the net monopole and dipole of the rounding errors of any run of neighbouring
// sources stay below one rounding unit.
__device__ __forceinline__ float round_feedback(double exact, double q, double &carry,
                                                double lattice, double inv_lattice) {
    const double n0 = rint(exact * inv_lattice);
    const double v0 = n0 * lattice;
    const float f0 = static_cast<float>(v0);          // exact: |offset| << 2^24 quanta
    const double r0 = exact - v0;
    if (r0 == 0.0 || q == 0.0) return f0;
    const double v1 = (r0 > 0.0 ? n0 + 1.0 : n0 - 1.0) * lattice;
    const float f1 = static_cast<float>(v1);
    const double r1 = exact - v1;
    const double c0 = carry + q * r0, c1 = carry + q * r1;
    if (fabs(c0) <= fabs(c1)) { carry = c0; return f0; }
    carry = c1;
    return f1;
}

__global__ void pack_f32_kernel(const double *xyz, const double *q, int64_t M, int64_t n_chunks,
                                const double *origins, double lattice, double q_scale, float *chunks) {
    const double inv_lattice = 1.0 / lattice;
    const int64_t ch = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (ch >= n_chunks) return;
    const double *o = origins + 4 * (ch / BLOCK_CHUNKS);
    float *c = chunks + ch * 4 * CHUNK;
    double cx = 0.0, cy = 0.0, cz = 0.0, cq = 0.0;       // running residuals
    for (int i = 0; i < CHUNK; ++i) {
        const int64_t j = ch * CHUNK + i;
        const int64_t src = j < M ? j : M - 1;           // pads: last real source, charge 0
        const double qj = j < M ? q[src] * q_scale : 0.0;   // power-of-two scale: exact
        c[i] = round_feedback(xyz[3 * src + 0] - o[0], qj, cx, lattice, inv_lattice);
        c[CHUNK + i] = round_feedback(xyz[3 * src + 1] - o[1], qj, cy, lattice, inv_lattice);
        c[2 * CHUNK + i] = round_feedback(xyz[3 * src + 2] - o[2], qj, cz, lattice, inv_lattice);
        const double want = qj + cq;
        const float q32 = static_cast<float>(want);
        cq = j < M ? want - static_cast<double>(q32) : 0.0;
        c[3 * CHUNK + i] = q32;
    }
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
