// qmmm_grid.cuh -- grid-aware compact source format.
//
// The paper's sources ARE "spatially discretized cells": nodes of a regular
// grid.  When the cells of an environment are nodes origin + (ix, iy, iz) h of a cubic grid,
// only the charges are stored (4 B FP32 / 8 B FP64 per cell instead of 16 / 32 B) and the
// coordinates are regenerated from the indices.  Everything is computed in GRID UNITS
// (u = (r - origin) / h per axis, nodes at integer coordinates; lengths in units of hz, so
// for cells that are not cubic dx, dy carry the factors hx/hz, hy/hz from the row setup on;
// V = sum / hz, E = sum / hz^2 at the end).
//
// Mapping: a "row" is the nz nodes of one (ix, iy); the 32 lanes of a warp own 32 DIFFERENT
// rows of a row tile and walk along z together.  For a point i and a row, dx, dy and
// dx^2 + dy^2 are constants of the row walk, and so is the x, y part of the field:
//     r^2  = (dx^2 + dy^2) + dz^2                       1 add (dz) + 1 fma per pair
//     Ex  += dx * sum_k s_k,  Ey += dy * sum_k s_k      1 add per pair (sum s), not 2 fma
//     Ez  += sum_k s_k dz_k                             1 fma per pair
// which, with the Newton step applied to the sum (GridRowF32 below), leaves 9 FP32 lane
// operations per pair instead of 14 for a source list, and 13 FP64 instead of 18
// (DESIGN.md section 5b).
//
// Work unit ("gchunk"): 32 rows x ZS = 64 consecutive z nodes, stored [ZS/4][32][4] (FP32) or
// [ZS/2][32][2] (FP64) so that a lane's 128-bit shared-memory loads are conflict-free.  One
// TMA bulk copy per gchunk and pipeline stage.  Slices (Eq. 5-6) are
// ranges of gchunks; the source-split warps of a CTA take different z runs of every gchunk.
// Masked-out cells are zero charges (they contribute exactly 0: r^2 carries a tiny positive
// offset so that a coincident zero-charge node cannot produce 0 * inf).
#pragma once
#include "qmmm_kernels.cuh"

namespace qmmm {

constexpr int GRID_ZS = 64;                         // z nodes per gchunk
constexpr int GRID_NODES = 32 * GRID_ZS;            // cells per gchunk

// ----------------------------------------------------------------------------- FP32 packed
template <int EP2, int NW>
struct GridF32Layout {
    static constexpr int EPT = 2 * EP2;
    static constexpr int NT = 32 * NW;
    static constexpr int STAGE_BYTES = GRID_NODES * sizeof(float);          // 8 KB
    static constexpr int BAR_BYTES = 18 * sizeof(uint64_t);                 // 8 full, 8 empty, flag
    static constexpr int ELEC_BYTES = 2 * NW * EPT * 3 * sizeof(double);    // points in units of hz, and in node units
    // whole-grid lattice a, dd per CTA point; per-warp lattice a[3][EPT], dd[3][EPT]; per-warp reference node [4]
    static constexpr int SCRATCH_BYTES = NW * 2 * 3 * EPT * sizeof(float) + NW * 6 * EPT * sizeof(float) +
                                         NW * 4 * sizeof(int);
    static constexpr int ACC_BYTES = EPT * 4 * NT * sizeof(double);
    __host__ __device__ static constexpr size_t total(int stages) {
        return static_cast<size_t>(stages) * STAGE_BYTES + BAR_BYTES + ELEC_BYTES + SCRATCH_BYTES +
               ACC_BYTES;
    }
    // dz table (DZT kernels), after everything else: [z nodes padded to whole gchunks + 1][NW][EPT]
    __host__ __device__ static constexpr size_t dzt_bytes(int segs) {
        return static_cast<size_t>(segs * 64 + 1) * NW * EPT * sizeof(float);
    }
};

// Coordinate of an evaluation point along one axis (node units) on a power-of-two lattice fine
// enough that every difference a - k to the node indices k = i_lo..i_hi is EXACT in FP32: the
// quantum is 2^-24 of the power of two above the farthest of those nodes.  a is returned
// relative to i_lo (a_rel = a - i_lo, itself exact in FP32); dd = u - a is the residual, which
// enters V as the first-order correction V(a + dd) = V(a) - E(a) . dd.
// Plain FP32 rounding of the differences would be coherent over a regular grid and bias V.
//   whole grid (i_lo = 0, i_hi = n - 1): one quantum per axis and point, 2^-24 of the axis;
//   one gchunk (the 32 rows / 64 z nodes a warp is about to walk): the quantum follows the
//     distance to THOSE nodes, so next to a point it is 2^-24 of a few dozen nodes however long
//     the axis is.  E has no first-order correction (it is evaluated at a, relative error about
//     3 |dd| / distance per term), so long axes with points close to cells need this one.
__device__ __forceinline__ void on_lattice(double u, int i_lo, int i_hi, float &a_rel, float &dd) {
    const double far = fmax(fmax(fabs(u - i_lo), fabs(u - i_hi)), 1.0);
    const int ex = ((__double2hiint(far) >> 20) & 0x7ff) - 1022;          // far < 2^ex
    const double lam = __hiloint2double((ex - 24 + 1023) << 20, 0);
    const double inv = __hiloint2double((24 - ex + 1023) << 20, 0);
    const double al = rint(u * inv) * lam;
    a_rel = static_cast<float>(al - i_lo);                     // exact: a multiple of lam, at most 2^24 quanta
    dd = static_cast<float>(u - al);
}

// v += x with the rounding error of the sum kept (fast two-sum: exact when v's exponent is not
// below x's, which always holds from the third 16-node sum of a row on; where the second sum is
// the larger one the error term may itself round -- half an ulp of that sum, in a minority of rows:
// tests/test_row_sum_identity.py), and d += dx - 2 error: V = v - d / 2 then holds the exact
// sum.  4 operations more than two plain adds, once per 16 nodes: a quarter operation per pair.
__device__ __forceinline__ void add_run(float2 &v, float2 &d, float2 x, float2 dx) {
    const float2 s = __fadd2_rn(v, x);
    const float2 bb = __ffma2_rn(v, bc(-1.0f), s);              // s - v
    const float2 er = __ffma2_rn(x, bc(-1.0f), bb);             // (s - v) - x = -(rounding error of s)
    v = s;
    d = __fadd2_rn(d, __ffma2_rn(er, bc(2.0f), dx));
}

// A run of z nodes of the lane's row for EP2 packed point pairs, software-pipelined: while
// the FMA pipe works on node n the MUFU.RSQ of node n + 1 is already in flight (two register
// sets A / B in turn).
//
// The Newton step is applied to the SUM, not to every pair.  With y0 = MUFU.RSQ(r^2),
// a = q y0 and c = q y0^3 (needed for the field anyway), the refined term is
//     q y1 = q y0 (3 - r^2 y0^2) / 2 = (3 a - c r^2) / 2,
// so V = (3 sum a - sum c r^2) / 2: ONE extra fma per pair (T += c r^2) instead of the three
// FMA-pipe operations + one integer operation of a per-pair step, and algebraically the same
// value.  (Evaluating y0 (3 - r^2 y0^2) / 2 per pair would round the correction away: the
// bracket is ~2, its ulp 2.4e-7 is the size of the MUFU error.  Raw MUFU.RSQ values have a
// mean relative error of +5.5e-9 on these inputs -- measured: 1.2e-5 hartree per 64-electron
// walker, over the tolerance -- hence the refinement.)  The FIELD uses y0 itself: its
// tolerance is 1e-5 relative per point, the raw values give 4e-7.
// Per pair: dz (the running dz steps by -1, exact on the lattice), r^2, a = q y0, V0 += a,
// y0^2, c = a y0^2, sum c, sum c dz, T += c r^2 = 9 FMA-pipe lane operations + 1 MUFU.RSQ
// (+ 10/16 for the two summation trees).
//
// TS > 0 (dz table): dz = u_z - k depends on the point and the z node only, not on the row, so
// the CTA tabulates it once in shared memory ([z node][warp][EPT] floats, TS = float2 per z
// node; formed in FP64 from the point's true coordinate, rounded once) and a node's dz is ONE
// broadcast 128-bit load for both point pairs instead of a packed add per pair: 8 FMA-pipe
// lane operations per pair instead of 9.
//
// VONLY (potential only, Eq. 4 proper; needs the table): the table holds z2 = (u_z - k)^2, formed
// in FP64 from the point's true coordinate and rounded once, rxy2 is formed in FP64 per (point,
// row) and rounded once, and r^2 = rxy2 + z2 is ONE add.  No lattice and no residual: nothing
// needs the field to be corrected with.  Per pair: r^2, a, V0 += a, y0^2, c, T += c r^2 = 6
// FMA-pipe lane operations + 1 MUFU.RSQ -- the XU pipe (16 per SM and clock) is the limit.
//
// ACCV (V + E, batched table kernel; the default, qmmm_field_set_accurate_v): the same r^2 as
// VONLY -- a z2 entry beside every dz entry of the table, rxy2 formed in FP64 per (point, row) --
// and the same compensated row sums, with dz still read for sum c dz.  Still 8 operations per
// pair (r^2 is one add instead of one fma), one more broadcast load per node, a quarter
// operation for the two-sum: +6 % time on config 3 for V rms 6.7e-8 -> 2.6e-8 hartree and the
// total over the 16,384 points of the batch 3.1e-5 -> 2.6e-6.
template <int EP2, int TS = 0, bool VONLY = false, bool ACCV = false>
struct GridRowF32 {
    static_assert(!VONLY || TS > 0, "the potential-only walk is table-driven");
    static_assert(!ACCV || (TS > 0 && !VONLY), "ACCV: V + E walk with the dz and the z2 table");
    static constexpr bool COMP = VONLY || ACCV;      // last tree level added with a two-sum
    // r^2 of the node whose table entry is t: dz^2 + rxy2, or (VONLY: the table holds z2;
    // ACCV: a z2 entry follows the node's dz entries) z2 + rxy2
    __device__ __forceinline__ void r2_of(const float2 *t, const float2 (&dz)[EP2], float2 (&r2)[EP2]) {
        if constexpr (ACCV) {
            float2 z2[EP2];
            load_dz(t + TS / 2, z2);
#pragma unroll
            for (int e = 0; e < EP2; ++e) r2[e] = __fadd2_rn(z2[e], rxy2[e]);
        } else {
#pragma unroll
            for (int e = 0; e < EP2; ++e)
                r2[e] = VONLY ? __fadd2_rn(dz[e], rxy2[e]) : __ffma2_rn(dz[e], dz[e], rxy2[e]);
        }
    }
    float2 dzA[EP2], r2A[EP2], y0A[EP2], dzB[EP2], r2B[EP2], y0B[EP2];
    float2 rxy2[EP2], S[EP2], SZ[EP2];
    const float2 *tp;                  // TS > 0: table entry of the node held in the current set

    __device__ __forceinline__ void load_dz(const float2 *t, float2 (&dz)[EP2]) {
        if constexpr (EP2 == 2) {
            const float4 d = *reinterpret_cast<const float4 *>(t);
            dz[0] = f2(d.x, d.y);
            dz[1] = f2(d.z, d.w);
        } else {
#pragma unroll
            for (int e = 0; e < EP2; ++e) dz[e] = t[e];
        }
    }
    // table variant: the run starts at the node whose entry is t
    __device__ __forceinline__ void start(const float2 *t, const float2 (&rxy2_)[EP2]) {
        tp = t;
        load_dz(t, dzA);
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            rxy2[e] = rxy2_[e];
            S[e] = SZ[e] = f2(0.0f, 0.0f);
        }
        r2_of(t, dzA, r2A);
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            y0A[e].x = rsqrt_mufu_f32(r2A[e].x);
            y0A[e].y = rsqrt_mufu_f32(r2A[e].y);
        }
    }
    __device__ __forceinline__ void start(const float2 (&azb)[EP2], const float2 (&rxy2_)[EP2]) {
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            rxy2[e] = rxy2_[e];
            S[e] = SZ[e] = f2(0.0f, 0.0f);
            dzA[e] = azb[e];
            r2A[e] = __ffma2_rn(dzA[e], dzA[e], rxy2[e]);
        }
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            y0A[e].x = rsqrt_mufu_f32(r2A[e].x);
            y0A[e].y = rsqrt_mufu_f32(r2A[e].y);
        }
    }
    // next node from the current one: dz - 1, r^2, MUFU
    __device__ __forceinline__ void step(const float2 (&dzc)[EP2], float2 (&dzn)[EP2],
                                         float2 (&r2n)[EP2], float2 (&y0n)[EP2], int j = 0) {
        if constexpr (TS > 0) {
            load_dz(tp + j * TS, dzn);                        // j-th node after the one at tp
            r2_of(tp + j * TS, dzn, r2n);
        } else {
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                dzn[e] = __fadd2_rn(dzc[e], bc(-1.0f));
                r2n[e] = __ffma2_rn(dzn[e], dzn[e], rxy2[e]);
            }
        }
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            y0n[e].x = rsqrt_mufu_f32(r2n[e].x);
            y0n[e].y = rsqrt_mufu_f32(r2n[e].y);
        }
    }
    // the sums of one node: V0 += a, T += c r^2, S += c, SZ += c dz
    __device__ __forceinline__ void acc(const float2 (&dz)[EP2], const float2 (&r2)[EP2],
                                        const float2 (&y0)[EP2], float q, float2 (&Vc)[EP2],
                                        float2 (&Tc)[EP2], bool first) {
        const float2 qq = bc(q);
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            const float2 a = __fmul2_rn(y0[e], qq);
            Vc[e] = first ? a : __fadd2_rn(Vc[e], a);
            const float2 c = __fmul2_rn(a, __fmul2_rn(y0[e], y0[e]));
            Tc[e] = first ? __fmul2_rn(c, r2[e]) : __ffma2_rn(c, r2[e], Tc[e]);
            if constexpr (!VONLY) {
                S[e] = __fadd2_rn(S[e], c);
                SZ[e] = __ffma2_rn(c, dz[e], SZ[e]);
            }
        }
    }
    // 4 nodes (one 128-bit load of charges); their V0 and T sums go to Vc, Tc
    __device__ __forceinline__ void four(const float *q4, float2 (&Vc)[EP2], float2 (&Tc)[EP2]) {
        const float4 Q = *reinterpret_cast<const float4 *>(q4);
        step(dzA, dzB, r2B, y0B, 1);
        acc(dzA, r2A, y0A, Q.x, Vc, Tc, true);
        step(dzB, dzA, r2A, y0A, 2);
        acc(dzB, r2B, y0B, Q.y, Vc, Tc, false);
        step(dzA, dzB, r2B, y0B, 3);
        acc(dzA, r2A, y0A, Q.z, Vc, Tc, false);
        step(dzB, dzA, r2A, y0A, 4);        // the last one looks one node past the run: unused
        acc(dzB, r2B, y0B, Q.w, Vc, Tc, false);
        if constexpr (TS > 0) tp += 4 * TS;
    }
    // n4 * 4 nodes starting at b ([k4][32][4] floats).  v receives the row's sum of a (V0), d the
    // sum of c r^2 - a (T - V0: the Newton term, V = V0 - d / 2).  V0 and T are summed as trees
    // of short FP32 runs (4 nodes -> 16 -> run): a long FP32 running sum of slowly varying
    // same-sign terms drifts; T - V0 is formed once per run (16 nodes
    // when compensated) and is exact, the two agree to 1e-6.
    // VONLY: the last level (16 -> run) is where the row sum reaches its full size.  It carries
    // 60 % of the tree's rounding variance and, on config 3, a systematic +6e-10 hartree per
    // point (partial sums 1 : 2 : 3 : 4 of nearly equal terms; reproduced by a CPU emulation
    // of the tree in IEEE float32), so there it is added with a fast
    // two-sum whose error term goes to d: a quarter operation per pair, +2.3 % time, rms of V
    // on config 3 4.5e-8 -> 2.7e-8 and the batch total inside 1e-5 hartree; the level below it
    // (4 -> 16) is added pairwise there, which takes its share of the drift away for nothing.
    // ACCV: the same.
    // The other V + E walks keep plain adds: their error is dominated by the FP32 dz table and
    // rxy2 (6.7e-8 -> 6.4e-8 with the two-sum alone, at +3 % time).
    __device__ __forceinline__ void run(const float *b, int n4, float2 (&v)[EP2], float2 (&d)[EP2]) {
        if ((n4 & 3) == 0) {
            float2 t[EP2];
#pragma unroll
            for (int e = 0; e < EP2; ++e) t[e] = f2(0.0f, 0.0f);
#pragma unroll 1
            for (int g = 0; g < n4; g += 4) {
                float2 v16[EP2], t16[EP2], Vc[EP2], Tc[EP2];
                four(b + g * 128, v16, t16);
                if constexpr (COMP) {
                    // the four 4-node sums pairwise, (f0 + f1) + (f2 + f3): the same three adds as
                    // one after the other, without the 1 : 2 : 3 : 4 partial sums that drift
                    // (+1.5e-10 hartree per point on config 3 at this level; 8 more live registers)
                    float2 w[EP2], tw[EP2];
                    four(b + (g + 1) * 128, Vc, Tc);
#pragma unroll
                    for (int e = 0; e < EP2; ++e) {
                        v16[e] = __fadd2_rn(v16[e], Vc[e]);
                        t16[e] = __fadd2_rn(t16[e], Tc[e]);
                    }
                    four(b + (g + 2) * 128, w, tw);
                    four(b + (g + 3) * 128, Vc, Tc);
#pragma unroll
                    for (int e = 0; e < EP2; ++e) {
                        v16[e] = __fadd2_rn(v16[e], __fadd2_rn(w[e], Vc[e]));
                        t16[e] = __fadd2_rn(t16[e], __fadd2_rn(tw[e], Tc[e]));
                    }
                } else {
#pragma unroll
                    for (int k4 = 1; k4 < 4; ++k4) {
                        four(b + (g + k4) * 128, Vc, Tc);
#pragma unroll
                        for (int e = 0; e < EP2; ++e) {
                            v16[e] = __fadd2_rn(v16[e], Vc[e]);
                            t16[e] = __fadd2_rn(t16[e], Tc[e]);
                        }
                    }
                }
#pragma unroll
                for (int e = 0; e < EP2; ++e) {
                    if constexpr (COMP) {
                        add_run(v[e], d[e], v16[e], __ffma2_rn(v16[e], bc(-1.0f), t16[e]));
                    } else {
                        v[e] = __fadd2_rn(v[e], v16[e]);
                        t[e] = __fadd2_rn(t[e], t16[e]);
                    }
                }
            }
            if constexpr (!COMP) {
#pragma unroll
                for (int e = 0; e < EP2; ++e) d[e] = __fadd2_rn(d[e], __ffma2_rn(v[e], bc(-1.0f), t[e]));
            }
        } else {
#pragma unroll 1
            for (int k4 = 0; k4 < n4; ++k4) {            // short z runs of the z-split plans
                float2 Vc[EP2], Tc[EP2];
                four(b + k4 * 128, Vc, Tc);
#pragma unroll
                for (int e = 0; e < EP2; ++e) {
                    v[e] = __fadd2_rn(v[e], Vc[e]);
                    d[e] = __fadd2_rn(d[e], __ffma2_rn(Vc[e], bc(-1.0f), Tc[e]));
                }
            }
        }
    }
};

// The same walk for ONE evaluation point (single-electron moves): the two
// halves of a register pair hold two consecutive z NODES instead of two points, so the
// packed instructions stay full with a single point.  Two chains (4 nodes = one 128-bit
// charge load) x two register sets; same 9 operations per pair.  The halves are added at
// the end of the run.
struct GridRowF32N {
    float2 dzA[2], r2A[2], y0A[2], dzB[2], r2B[2], y0B[2];
    float2 rxy2, S, SZ;

    __device__ __forceinline__ void start(float azb, float rxy2s) {
        rxy2 = bc(rxy2s);
        S = SZ = f2(0.0f, 0.0f);
        dzA[0] = f2(azb, azb - 1.0f);                  // exact (lattice)
        dzA[1] = f2(azb - 2.0f, azb - 3.0f);
#pragma unroll
        for (int e = 0; e < 2; ++e) r2A[e] = __ffma2_rn(dzA[e], dzA[e], rxy2);
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            y0A[e].x = rsqrt_mufu_f32(r2A[e].x);
            y0A[e].y = rsqrt_mufu_f32(r2A[e].y);
        }
    }
    __device__ __forceinline__ void step(const float2 (&dzc)[2], float2 (&dzn)[2], float2 (&r2n)[2],
                                         float2 (&y0n)[2]) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            dzn[e] = __fadd2_rn(dzc[e], bc(-4.0f));
            r2n[e] = __ffma2_rn(dzn[e], dzn[e], rxy2);
        }
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            y0n[e].x = rsqrt_mufu_f32(r2n[e].x);
            y0n[e].y = rsqrt_mufu_f32(r2n[e].y);
        }
    }
    __device__ __forceinline__ void acc(const float2 (&dz)[2], const float2 (&r2)[2],
                                        const float2 (&y0)[2], const float *q4, float2 &Vc,
                                        float2 &Tc, bool first) {
        const float4 Q = *reinterpret_cast<const float4 *>(q4);
        const float2 q[2] = {f2(Q.x, Q.y), f2(Q.z, Q.w)};
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const float2 a = __fmul2_rn(y0[e], q[e]);
            const float2 c = __fmul2_rn(a, __fmul2_rn(y0[e], y0[e]));
            if (first && e == 0) {
                Vc = a;
                Tc = __fmul2_rn(c, r2[e]);
            } else {
                Vc = __fadd2_rn(Vc, a);
                Tc = __ffma2_rn(c, r2[e], Tc);
            }
            S = __fadd2_rn(S, c);
            SZ = __ffma2_rn(c, dz[e], SZ);
        }
    }
    // n4 * 4 nodes starting at b; v, t receive the sums of V0 and T (both halves added)
    __device__ __forceinline__ void run(const float *b, int n4, float &v, float &t) {
        float2 vs = f2(0.0f, 0.0f), ts = f2(0.0f, 0.0f);
        int k4 = 0;
#pragma unroll 1
        for (; k4 + 1 < n4; k4 += 2) {               // 8 nodes: sets A then B
            float2 Vc, Tc;
            step(dzA, dzB, r2B, y0B);
            acc(dzA, r2A, y0A, b + k4 * 128, Vc, Tc, true);
            step(dzB, dzA, r2A, y0A);                 // the last one looks past the run: unused
            acc(dzB, r2B, y0B, b + (k4 + 1) * 128, Vc, Tc, false);
            vs = __fadd2_rn(vs, Vc);
            ts = __fadd2_rn(ts, Tc);
        }
        if (k4 < n4) {                                // odd tail: 4 nodes
            float2 Vc, Tc;
            acc(dzA, r2A, y0A, b + k4 * 128, Vc, Tc, true);
            vs = __fadd2_rn(vs, Vc);
            ts = __fadd2_rn(ts, Tc);
        }
        v = vs.x + vs.y;
        t = ts.x + ts.y;
    }
};

// grid = (point_blocks, slices); EPT = 2 * EP2 points per thread; NW warps (8 x 8 points or
// 16 x 4 points), warp 0 drives the TMA ring inline (a producer warp would cost registers).
// A pipeline stage is one gchunk, consumed by all warps: the WP point warps own different
// point groups, the WS source-split warps different z runs (ZS / WS nodes) of the same 32
// rows.  Per gchunk a thread only forms dx, dy (exact FP32 differences on the point's
// lattice) and adds the row's sums into FP32 accumulators, flushed to the FP64 columns in
// shared memory after every gchunk (GRID_FLUSH).  prm.chunks = gchunks [n_chunks][ZS/4][32][4] float;
// prm.nuc = nuclei in grid units; prm.elec in bohr (converted to grid units when staged).
#ifndef QMMM_GRID_FLUSH
#define QMMM_GRID_FLUSH 1
#endif
constexpr int GRID_FLUSH = QMMM_GRID_FLUSH;                       // gchunks per FP32 -> FP64 flush (round 2: 1; 4 measured the
                                                                  // same time on config 3 and 10 - 40 % more rounding noise in V)

// NODEPACK (EP2 = 1 only): each of the thread's two points is walked on its own with two NODES
// per register pair (GridRowF32N); a second point beyond P is skipped.  For one or two points
// per evaluation.
// FULL: every warp owns its own point group (WP = NW, no z split): the z run is the whole
// gchunk, a compile-time constant (1.3 % on config 3; the same switch made the FP64 kernel
// slower and is not used there).
// DZT (FULL only): dz from a per-CTA table in shared memory (GridRowF32<EP2, TS>), chosen by
// the launcher when the table fits beside two CTAs per SM.
// FINE: coordinate lattice per gchunk (on_lattice) -- 1 on, 0 off (the batched FULL kernels are
// compiled both ways: the switch costs registers in their loop), -1 decided by prm.g_fine.
// VONLY (E = NULL; FULL + DZT only): the potential alone, no lattice (GridRowF32<.., VONLY>).
// ACCV (FULL + DZT, V + E): accurate V (GridRowF32<.., false, ACCV>); the table is twice as large.
template <int EP2, int NW, bool NODEPACK = false, bool FULL = false, bool DZT = false, int FINE = -1,
          bool VONLY = false, bool ACCV = false>
__global__ void __launch_bounds__(32 * NW, (!NODEPACK && NW <= 8 && EP2 <= 2) ? 16 / NW : 1) grid_kernel_f32x2(const PairParams prm) {
    static_assert(!ACCV || (FULL && DZT && !VONLY), "ACCV: the batched table-driven V + E walk");
    static_assert(FINE == -1 || FULL, "the compile-time switch is for the batched FULL kernels");
    static_assert(!VONLY || (FULL && DZT && FINE == 0), "potential only: batched table-driven walk, no lattice");
    static_assert(!DZT || !NODEPACK, "dz table: the point-packed walks (every warp its own points, or z-split warps)");
    static_assert(!NODEPACK || EP2 == 1, "node packing walks single points");
    static_assert(!(NODEPACK && FULL), "FULL is a mode of the point-packed walk");
    using L = GridF32Layout<EP2, NW>;
    constexpr int EPT = L::EPT, NT = L::NT, STAGE_BYTES = L::STAGE_BYTES;

    extern __shared__ __align__(128) unsigned char smem[];
    pdl_launch_dependents();
    QMMM_MARK_GT(8);
    QMMM_MARK(0);
    // NODEPACK: warp-private pipelines, two slots per warp (prm.stages is not used)
    const int stages = NODEPACK ? 2 * NW : prm.stages;
    unsigned char *ptr = smem + static_cast<size_t>(stages) * STAGE_BYTES;
    uint64_t *full = reinterpret_cast<uint64_t *>(ptr);        // NODEPACK: 16 full barriers
    uint64_t *empty = full + 8;
    int *flag = reinterpret_cast<int *>(empty + 8);
    ptr += L::BAR_BYTES;
    double *elec_s = reinterpret_cast<double *>(ptr);          // [WP*EPT][3], units of hz (for the nuclei)
    double *u_s = elec_s + NW * EPT * 3;                       // [WP*EPT][3], node units of each axis
    ptr += L::ELEC_BYTES;
    float *lat_s = reinterpret_cast<float *>(ptr);             // whole-grid lattice: a[WP*EPT][3], then dd[WP*EPT][3]
    float *warp_s = lat_s + NW * EPT * 6;                      // per warp: a[3][EPT], dd[3][EPT] of the gchunk at hand
    int *iref_s = reinterpret_cast<int *>(warp_s + NW * EPT * 6);   // per warp: reference node of a, per axis
    ptr += L::SCRATCH_BYTES;
    double2 *acc = reinterpret_cast<double2 *>(ptr);           // [EPT*2][NT] double2

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WP = NODEPACK ? 1 : (FULL ? NW : prm.point_warps), WS = NW / WP;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.y, lo, hi);

    // ---- producer cursor (warp 0 only): next gchunk to load ---------------------------------
    int pc = lo, pslot = 0;
    uint32_t pphase = 0;
    bool pwrapped = false;
    auto produce = [&]() {
        if (pc >= hi) return;
        if (pwrapped) mbar_wait(&empty[pslot], pphase);
        if (lane == 0) {
            mbar_expect_tx(&full[pslot], STAGE_BYTES);
            tma_bulk_g2s(smem + static_cast<size_t>(pslot) * STAGE_BYTES,
                         prm.chunks + static_cast<size_t>(pc) * STAGE_BYTES, STAGE_BYTES, &full[pslot]);
        }
        ++pc;
        if (++pslot == stages) {
            pslot = 0;
            if (pwrapped) pphase ^= 1u;
            pwrapped = true;
        }
    };
    // NODEPACK: warp w walks gchunks lo + w, lo + w + NW, ... whole (all 64 z nodes) and loads
    // them itself into its own two slots: no waiting on other warps anywhere in the loop
    auto load_own = [&](int g, int sl) {           // lane 0 of the owning warp
        mbar_expect_tx(&full[sl], STAGE_BYTES);
        tma_bulk_g2s(smem + static_cast<size_t>(sl) * STAGE_BYTES,
                     prm.chunks + static_cast<size_t>(g) * STAGE_BYTES, STAGE_BYTES, &full[sl]);
    };
    if constexpr (NODEPACK) {
        if (lane == 0) {
            mbar_init(&full[2 * warp], 1);
            mbar_init(&full[2 * warp + 1], 1);
            fence_barrier_init();
            for (int i = 0; i < 2; ++i)
                if (lo + warp + i * NW < hi) load_own(lo + warp + i * NW, 2 * warp + i);
        }
        __syncwarp();
    } else {
        if (threadIdx.x == 0) {
            for (int s = 0; s < stages; ++s) {
                mbar_init(&full[s], 1);
                mbar_init(&empty[s], NW);
            }
            fence_barrier_init();
        }
        if (warp == 0) {
            __syncwarp();
            for (int i = 0; i < stages - 1; ++i) produce();
        }
    }
    const int ppb = WP * EPT;
    float *dd_all = lat_s + NW * EPT * 3;
    const bool fine = FINE >= 0 ? FINE == 1 : prm.g_fine != 0;  // local lattice per gchunk (uniform)
    // TRUEPT (the batched dz-table kernels): r^2 and the differences are those of the point's TRUE
    // position, not of its lattice position -- see the walk below; no residual, no correction, no
    // dependence of E on the length of the axes (FINE is moot: instantiated with FINE = 0 only)
    constexpr bool TRUEPT = DZT && !VONLY;
    static_assert(!(DZT && FINE == 1), "the dz-table kernels have no lattice residual to refine");
    for (int i = threadIdx.x; i < ppb * 3; i += NT) {
        int p = blockIdx.x * ppb + i / 3;
        p = p < prm.P ? p : prm.P - 1;                          // clamp: duplicates are not written
        const int comp = i % 3;
        const double u = (point_coord(prm, static_cast<int64_t>(p) * 3 + comp) - prm.g_org[comp]) * prm.g_inv_h[comp];
        const double sc = comp == 0 ? prm.g_sx : (comp == 1 ? prm.g_sy : 1.0);
        elec_s[i] = u * sc;                                     // units of hz (for the nuclei)
        u_s[i] = u;
        float dd;
        on_lattice(u, 0, prm.g_n[comp] - 1, lat_s[i], dd);      // node index units of this axis
        dd_all[i] = dd * static_cast<float>(sc);                // residual in units of hz
    }
    __syncthreads();
    constexpr int TS = DZT ? NW * EP2 * (ACCV ? 2 : 1) : 0;     // float2 per z node of the table (ACCV: dz entries, then z2 entries)
    float *dzt = reinterpret_cast<float *>(acc + EPT * 2 * NT); // [segs * ZS + 1][NW][EPT]
    if constexpr (DZT) {
        // one entry per (z node, point of the CTA), formed in FP64 from the point's TRUE coordinate
        // and rounded once: dz = u_z - k, or (potential only) z2 = (u_z - k)^2
        const int nent = (prm.g_segs * GRID_ZS + 1) * NW * EPT;
        for (int i = threadIdx.x; i < nent; i += NT) {
            const int kz = i / (NW * EPT), pp = i - kz * (NW * EPT);
            if (pp >= ppb) continue;                            // (z-split plans stage fewer than NW point groups)
            const double dzt64 = u_s[pp * 3 + 2] - static_cast<double>(kz);
            if constexpr (ACCV) {
                dzt[(2 * kz + 0) * (NW * EPT) + pp] = static_cast<float>(dzt64);
                dzt[(2 * kz + 1) * (NW * EPT) + pp] = static_cast<float>(dzt64 * dzt64);
            } else {
                dzt[i] = static_cast<float>(VONLY ? dzt64 * dzt64 : dzt64);
            }
        }
        __syncthreads();
    }
    QMMM_MARK(1);

    const int wp = warp % WP, ws = warp / WP;
    const int ZL = FULL ? GRID_ZS : GRID_ZS / WS, z0 = FULL ? 0 : ws * ZL;   // this warp's z run inside every gchunk
    double2 *my = acc + threadIdx.x;                 // this thread's column: my[i * NT]
#pragma unroll
    for (int i = 0; i < EPT * 2; ++i) my[i * NT] = make_double2(0.0, 0.0);
    const double *pe = elec_s + wp * EPT * 3;
    // Lattice coordinates of this warp's points, two points per register pair, relative to the
    // reference node (irx, iry, irz), and their residuals dd (units of hz) in the warp's scratch.
    // Whole-grid lattice: reference node 0, filled once.  Local lattice (fine): refilled for
    // every gchunk by relattice() below.
    float *a_w = warp_s + warp * 6 * EPT, *dd_w = a_w + 3 * EPT;
    int *iref_w = iref_s + warp * 4;
    if (lane < 3 * EPT) {
        const int comp = lane / EPT, pt = lane - comp * EPT;
        a_w[lane] = lat_s[(wp * EPT + pt) * 3 + comp];
        dd_w[lane] = dd_all[(wp * EPT + pt) * 3 + comp];
    }
    if (lane < 3) iref_w[lane] = 0;
    __syncwarp();
    float2 ax[EP2], ay[EP2], az[EP2];
    int irx = 0, iry = 0, irz = 0;
    auto load_lattice = [&]() {
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            ax[e] = *reinterpret_cast<const float2 *>(a_w + 2 * e);
            ay[e] = *reinterpret_cast<const float2 *>(a_w + EPT + 2 * e);
            az[e] = *reinterpret_cast<const float2 *>(a_w + 2 * EPT + 2 * e);
        }
        irx = iref_w[0]; iry = iref_w[1]; irz = iref_w[2];
    };
    load_lattice();
    const int n_rows = prm.g_n[0] * prm.g_n[1];
    // fine: the lattice of the nodes of ONE gchunk -- rows tile_ * 32 .. + 31, z nodes
    // seg_ * ZS + zlo .. zhi -- computed in FP64 by the first 3 EPT lanes
    auto relattice = [&](int tile_, int seg_, int zlo, int zhi) {
        __syncwarp();
        if (lane < 3 * EPT) {
            const int comp = lane / EPT, pt = lane - comp * EPT;
            int i_lo, i_hi;
            if (comp == 2) {
                i_lo = seg_ * GRID_ZS + zlo;
                i_hi = seg_ * GRID_ZS + zhi;
            } else {
                const int nyy = prm.g_n[1];
                const int r0 = tile_ * 32, r1 = min(r0 + 31, n_rows - 1);
                const int x0 = r0 / nyy, x1 = r1 / nyy;
                if (comp == 0) { i_lo = x0; i_hi = x1; }
                else if (x0 == x1) { i_lo = r0 - x0 * nyy; i_hi = r1 - x0 * nyy; }
                else { i_lo = 0; i_hi = nyy - 1; }
            }
            float a, dd;
            on_lattice(u_s[(wp * EPT + pt) * 3 + comp], i_lo, i_hi, a, dd);
            a_w[lane] = a;
            dd_w[lane] = dd * static_cast<float>(comp == 0 ? prm.g_sx : (comp == 1 ? prm.g_sy : 1.0));
            if (pt == 0) iref_w[comp] = i_lo;
        }
        __syncwarp();
        load_lattice();
    };
    // FP32 accumulators over up to GRID_FLUSH gchunks, then FP64 columns.  cc: the first-order
    // correction for the lattice residual, sum over gchunks of E_gchunk(a) . dd
    float2 vv[EP2], tt[EP2], ex[EP2], ey[EP2], ez[EP2], cc[EP2];
#pragma unroll
    for (int e = 0; e < EP2; ++e) vv[e] = tt[e] = ex[e] = ey[e] = ez[e] = cc[e] = f2(0.0f, 0.0f);
    auto flush = [&]() {
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            double2 t;
            t = my[(4 * e + 0) * NT];            // V = (3 sum a - sum c r^2) / 2, the Newton step, as V0 - (T - V0) / 2
            t.x += static_cast<double>(vv[e].x) - 0.5 * static_cast<double>(tt[e].x) - static_cast<double>(cc[e].x);
            t.y += static_cast<double>(vv[e].y) - 0.5 * static_cast<double>(tt[e].y) - static_cast<double>(cc[e].y);
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
            vv[e] = tt[e] = ex[e] = ey[e] = ez[e] = cc[e] = f2(0.0f, 0.0f);
        }
    };

    // (tile, seg) of gchunk g = tile * segs + seg, and the lane's row (ix, iy) of that tile
    const int segs = prm.g_segs, ny = prm.g_n[1];
    int tile = lo / segs, seg = lo - tile * segs;
    int ix = (tile * 32 + lane) / ny, iy = tile * 32 + lane - ix * ny;

    QMMM_MARK(2);
    int pending = 0;
    if constexpr (NODEPACK) {
        // one point at a time, two NODES per register pair, whole gchunks per warp
        const bool second = blockIdx.x * ppb + 1 < prm.P;
        int it = 0;
        for (int g = lo + warp; g < hi; g += NW, ++it) {
            const int sl = 2 * warp + (it & 1);
            const int tl = g / segs, sg = g - tl * segs;
            const int rw = tl * 32 + lane, rx = rw / ny;
            if (fine) relattice(tl, sg, 0, GRID_ZS - 1);
            const float fxs = static_cast<float>(rx - irx), fys = static_cast<float>(rw - rx * ny - iry);
            const float fzs = static_cast<float>(sg * GRID_ZS - irz);
            mbar_wait(&full[sl], (it >> 1) & 1);
            const float *data = reinterpret_cast<const float *>(smem + static_cast<size_t>(sl) * STAGE_BYTES);
            auto one_point = [&](float axs, float ays, float azs, int pt, float &vvc, float &ttc, float &exc,
                                 float &eyc, float &ezc, float &ccc) {
                const float dxs = (axs - fxs) * static_cast<float>(prm.g_sx);   // exact difference (lattice), then hx/hz
                const float dys = (ays - fys) * static_cast<float>(prm.g_sy);
                GridRowF32N row;
                row.start(azs - fzs, fmaf(dys, dys, fmaf(dxs, dxs, 1e-30f)));
                float v1, t1;
                row.run(data + 4 * lane, GRID_ZS / 4, v1, t1);
                const float s1 = row.S.x + row.S.y;
                const float exg = dxs * s1, eyg = dys * s1, ezg = row.SZ.x + row.SZ.y;
                vvc += v1;
                ttc += t1 - v1;                    // T - V0 (exact: the two agree to 1e-6)
                exc += exg;
                eyc += eyg;
                ezc += ezg;
                if (fine)           // this gchunk was seen from its own lattice point: E_gchunk . dd
                    ccc = fmaf(exg, dd_w[pt], fmaf(eyg, dd_w[EPT + pt], fmaf(ezg, dd_w[2 * EPT + pt], ccc)));
            };
            one_point(ax[0].x, ay[0].x, az[0].x, 0, vv[0].x, tt[0].x, ex[0].x, ey[0].x, ez[0].x, cc[0].x);
            if (second) one_point(ax[0].y, ay[0].y, az[0].y, 1, vv[0].y, tt[0].y, ex[0].y, ey[0].y, ez[0].y, cc[0].y);
            __syncwarp();                          // every lane has read the slot
            if (lane == 0 && g + 2 * NW < hi) {    // refill it with the gchunk after next
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                load_own(g + 2 * NW, sl);
            }
            if (++pending == GRID_FLUSH) {
                flush();
                pending = 0;
            }
        }
    } else {
    int slot = 0;
    uint32_t phase = 0;
    for (int g = lo; g < hi; ++g) {
        if (warp == 0) produce();          // gchunk g + stages - 1 into the slot freed by g - 1
        if constexpr (VONLY) {
            // rxy2 = dx^2 + dy^2 of the lane's row from the points' true coordinates, in FP64,
            // rounded once (pe: units of hz; node (ix, iy) sits at (ix sx, iy sy))
            const double rowx = static_cast<double>(ix) * prm.g_sx, rowy = static_cast<double>(iy) * prm.g_sy;
            float2 rxy2[EP2], v[EP2], tq[EP2];
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                const double dx0 = pe[6 * e + 0] - rowx, dy0 = pe[6 * e + 1] - rowy;
                const double dx1 = pe[6 * e + 3] - rowx, dy1 = pe[6 * e + 4] - rowy;
                rxy2[e] = f2(static_cast<float>(fma(dy0, dy0, fma(dx0, dx0, 1e-30))),
                             static_cast<float>(fma(dy1, dy1, fma(dx1, dx1, 1e-30))));
                v[e] = tq[e] = f2(0.0f, 0.0f);
            }
            GridRowF32<EP2, TS, true> row;
            row.start(reinterpret_cast<const float2 *>(dzt) + (seg * GRID_ZS) * TS + wp * EP2, rxy2);
            mbar_wait(&full[slot], phase);
            row.run(reinterpret_cast<const float *>(smem + static_cast<size_t>(slot) * STAGE_BYTES) + 4 * lane,
                    GRID_ZS / 4, v, tq);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
#pragma unroll
            for (int e = 0; e < EP2; ++e) add_run(vv[e], tt[e], v[e], tq[e]);    // four rows per flush: compensated
        } else if constexpr (TRUEPT) {
            // r^2 of the TRUE point without FP64 in the loop: dx = a_x - ix is exact on the lattice
            // and u_x = a_x + dd_x, so (u_x - ix)^2 = dx^2 + 2 dx dd_x (+ dd_x^2 ~ 1e-11 dx^2); the
            // cross terms join rxy2 before it is rounded.  dz of the true point comes from the
            // table (rounded once).  No residual is left: nothing to correct V with afterwards, and E is
            // formed from the true differences (dx + dd_x, rounded) whatever the length of the axes.
            const float2 fx = bc(static_cast<float>(ix)), fy = bc(static_cast<float>(iy));
            float2 dx[EP2], dy[EP2], rxy2[EP2], v[EP2], tq[EP2];
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                dx[e] = __fadd2_rn(ax[e], f2(-fx.x, -fx.y));          // exact (lattice), node units
                dy[e] = __fadd2_rn(ay[e], f2(-fy.x, -fy.y));
                if (prm.g_ortho) {                                    // cells that are not cubic: hx/hz, hy/hz
                    dx[e] = __fmul2_rn(dx[e], bc(static_cast<float>(prm.g_sx)));
                    dy[e] = __fmul2_rn(dy[e], bc(static_cast<float>(prm.g_sy)));
                }
                const float2 ddx = *reinterpret_cast<const float2 *>(dd_w + 2 * e);        // units of hz
                const float2 ddy = *reinterpret_cast<const float2 *>(dd_w + EPT + 2 * e);
                if constexpr (ACCV) {
                    // rxy2 of the true point in FP64, rounded once (as in the potential-only kernel)
                    const double rowx = static_cast<double>(ix) * prm.g_sx, rowy = static_cast<double>(iy) * prm.g_sy;
                    const double dx0 = pe[6 * e + 0] - rowx, dy0 = pe[6 * e + 1] - rowy;
                    const double dx1 = pe[6 * e + 3] - rowx, dy1 = pe[6 * e + 4] - rowy;
                    rxy2[e] = f2(static_cast<float>(fma(dy0, dy0, fma(dx0, dx0, 1e-30))),
                                 static_cast<float>(fma(dy1, dy1, fma(dx1, dx1, 1e-30))));
                } else {
                    const float2 cross = __ffma2_rn(dx[e], ddx, __fmul2_rn(dy[e], ddy));
                    rxy2[e] = __ffma2_rn(dy[e], dy[e], __ffma2_rn(dx[e], dx[e], __ffma2_rn(cross, bc(2.0f), bc(1e-30f))));
                }
                dx[e] = __fadd2_rn(dx[e], ddx);                       // the true differences, for the field
                dy[e] = __fadd2_rn(dy[e], ddy);
                v[e] = tq[e] = f2(0.0f, 0.0f);
            }
            GridRowF32<EP2, TS, false, ACCV> row;
            // (z-split warps start at their own z run z0 of the gchunk; FULL: z0 = 0, ZL = 64)
            row.start(reinterpret_cast<const float2 *>(dzt) + (seg * GRID_ZS + z0) * TS + wp * EP2, rxy2);
            mbar_wait(&full[slot], phase);
            const float *data = reinterpret_cast<const float *>(smem + static_cast<size_t>(slot) * STAGE_BYTES);
            if constexpr (FULL)
                row.run(data + 4 * lane, GRID_ZS / 4, v, tq);
            else
                row.run(data + (z0 / 4) * 128 + 4 * lane, ZL / 4, v, tq);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                vv[e] = __fadd2_rn(vv[e], v[e]);
                tt[e] = __fadd2_rn(tt[e], tq[e]);
                ex[e] = __ffma2_rn(dx[e], row.S[e], ex[e]);
                ey[e] = __ffma2_rn(dy[e], row.S[e], ey[e]);
                ez[e] = __fadd2_rn(ez[e], row.SZ[e]);
            }
        } else {
        if (fine) relattice(tile, seg, z0, z0 + ZL - 1);
        const float2 fx = bc(static_cast<float>(ix - irx)), fy = bc(static_cast<float>(iy - iry));
        const float2 fz = bc(static_cast<float>(seg * GRID_ZS + z0 - irz));
        float2 dx[EP2], dy[EP2], rxy2[EP2], azb[EP2], v[EP2], tq[EP2];
#pragma unroll
        for (int e = 0; e < EP2; ++e) {
            dx[e] = __fadd2_rn(ax[e], f2(-fx.x, -fx.y));          // exact (lattice)
            dy[e] = __fadd2_rn(ay[e], f2(-fy.x, -fy.y));
            if (prm.g_ortho) {                                    // cells that are not cubic: hx/hz, hy/hz
                dx[e] = __fmul2_rn(dx[e], bc(static_cast<float>(prm.g_sx)));
                dy[e] = __fmul2_rn(dy[e], bc(static_cast<float>(prm.g_sy)));
            }
            if constexpr (!DZT) azb[e] = __fadd2_rn(az[e], f2(-fz.x, -fz.y));
            rxy2[e] = __ffma2_rn(dy[e], dy[e], __ffma2_rn(dx[e], dx[e], bc(1e-30f)));
            v[e] = tq[e] = f2(0.0f, 0.0f);
        }
        GridRowF32<EP2, TS> row;
        if constexpr (DZT)
            row.start(reinterpret_cast<const float2 *>(dzt) + (seg * GRID_ZS) * TS + wp * EP2, rxy2);
        else
            row.start(azb, rxy2);
        mbar_wait(&full[slot], phase);
        const float *data = reinterpret_cast<const float *>(smem + static_cast<size_t>(slot) * STAGE_BYTES);
        if constexpr (FULL)
            row.run(data + 4 * lane, GRID_ZS / 4, v, tq);
        else
            row.run(data + (z0 / 4) * 128 + 4 * lane, ZL / 4, v, tq);
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[slot]);
        // Ex = dx sum(s), Ey = dy sum(s), Ez = sum(s dz)
        if (fine) {
            // this gchunk was seen from its own lattice point a = u - dd: V -= E_gchunk(a) . dd
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                const float2 exg = __fmul2_rn(dx[e], row.S[e]), eyg = __fmul2_rn(dy[e], row.S[e]);
                const float2 ddx = *reinterpret_cast<const float2 *>(dd_w + 2 * e);
                const float2 ddy = *reinterpret_cast<const float2 *>(dd_w + EPT + 2 * e);
                const float2 ddz = *reinterpret_cast<const float2 *>(dd_w + 2 * EPT + 2 * e);
                vv[e] = __fadd2_rn(vv[e], v[e]);
                tt[e] = __fadd2_rn(tt[e], tq[e]);
                ex[e] = __fadd2_rn(ex[e], exg);
                ey[e] = __fadd2_rn(ey[e], eyg);
                ez[e] = __fadd2_rn(ez[e], row.SZ[e]);
                cc[e] = __ffma2_rn(exg, ddx, __ffma2_rn(eyg, ddy, __ffma2_rn(row.SZ[e], ddz, cc[e])));
            }
        } else {
#pragma unroll
            for (int e = 0; e < EP2; ++e) {
                vv[e] = __fadd2_rn(vv[e], v[e]);
                tt[e] = __fadd2_rn(tt[e], tq[e]);
                ex[e] = __ffma2_rn(dx[e], row.S[e], ex[e]);
                ey[e] = __ffma2_rn(dy[e], row.S[e], ey[e]);
                ez[e] = __fadd2_rn(ez[e], row.SZ[e]);
            }
        }
        }
        // (the potential-only kernel is bound by the XU pipe, which also does the FP32 -> FP64
        // conversions of a flush: every 4th gchunk there, 4.30 instead of 4.40 ms on config 3)
        if (++pending == (VONLY ? 4 : GRID_FLUSH)) {
            flush();
            pending = 0;
        }
        if (++slot == stages) {
            slot = 0;
            phase ^= 1u;
        }
        if (++seg == segs) {               // next row tile
            seg = 0;
            ++tile;
            iy += 32;
            if (ny >= 32) {
                if (iy >= ny) { iy -= ny; ++ix; }
            } else {
                ix = (tile * 32 + lane) / ny;
                iy = tile * 32 + lane - ix * ny;
            }
        }
    }
    }
    if (pending) flush();
    QMMM_MARK(3);
    // whole-grid lattice: the cells were seen from ONE lattice point a = u - dd: V(u) = V(a) - E(a) . dd,
    // applied to this thread's FP64 sums (before the nuclei, which are evaluated at u itself); the
    // local lattice has applied its corrections gchunk by gchunk (cc)
    if (!fine && !VONLY && !TRUEPT)
#pragma unroll
    for (int e = 0; e < EP2; ++e) {
        const float *d0 = dd_all + (wp * EPT + 2 * e) * 3;
        double2 t = my[(4 * e + 0) * NT];
        const double2 tx = my[(4 * e + 1) * NT], ty = my[(4 * e + 2) * NT], tz = my[(4 * e + 3) * NT];
        t.x -= tx.x * static_cast<double>(d0[0]) + ty.x * static_cast<double>(d0[1]) + tz.x * static_cast<double>(d0[2]);
        t.y -= tx.y * static_cast<double>(d0[3]) + ty.y * static_cast<double>(d0[4]) + tz.y * static_cast<double>(d0[5]);
        my[(4 * e + 0) * NT] = t;
    }

    // nuclear term of this CTA's share, FP64, grid units, into the same columns
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
    // ---- in-CTA reduction through shared memory, as in pair_kernel_f32x2 ----------------------
    double *red = reinterpret_cast<double *>(acc);   // reused after the barrier: [NW][EPT*4]
    double2 tot = make_double2(0.0, 0.0);
    __syncwarp();
    if (lane < 2 * EPT) {
        const double2 *rowp = acc + lane * NT + warp * 32;
#pragma unroll 8
        for (int j = 0; j < 32; ++j) {
            const double2 t = rowp[(j + lane) & 31];
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
        a *= (lane & 3) ? prm.g_scaleE : prm.g_scaleV;   // grid units -> hartree, hartree / bohr
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

// ----------------------------------------------------------------------------- FP64
// gchunk layout [ZS/2][32][2] double (16 KB).  13 DP lane operations + 1 MUFU.RSQ64H per pair
// (+ 1/4 for the dz base step); potential only: 8.
constexpr int GRID_STAGE_BYTES_F64 = GRID_NODES * sizeof(double);

template <int N>
__device__ __forceinline__ void consumer_sync() {     // named barrier 1: the N consumer warps only
    asm volatile("bar.sync 1, %0;" ::"n"(32 * N) : "memory");
}

// NW consumer warps (8 x 4 points or 16 x 2 points) + 1 TMA producer warp.
// WARPOWN (a handful of points, all owned by every warp): warp w loads and walks whole gchunks
// lo + w, lo + w + NW, ... by itself (one private slot per warp, no producer warp, no waiting
// on other warps), as the node-packed FP32 kernel does.
// DZT (EPT = 4, not WARPOWN; chosen by the launcher when the table fits): dz = u_z - k depends
// on the point and the z node only, not on the row, so the CTA tabulates it once in shared
// memory ([nz padded][WP * EPT] doubles) and the walk loads it with two broadcast LDS.128 per
// node instead of stepping it on the DP pipe: 12 DP lane operations per pair instead of 13
// (potential only: 7 instead of 8).
template <int EPT, bool WITH_E, int NW, bool WARPOWN = false, bool DZT = false>
__global__ void __launch_bounds__(32 * (NW + 1), 1) grid_kernel_f64(const PairParams prm) {
    static_assert(!DZT || (EPT == 4 && !WARPOWN), "dz table: 4 points per thread, shared stages");
    constexpr int STAGE_BYTES = GRID_STAGE_BYTES_F64;
    extern __shared__ __align__(128) unsigned char smem[];
    pdl_launch_dependents();
    QMMM_MARK_GT(8);
    QMMM_MARK(0);
    const int stages = WARPOWN ? NW : prm.stages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + static_cast<size_t>(stages) * STAGE_BYTES);
    uint64_t *empty = full + 8;
    int *flag = reinterpret_cast<int *>(empty + 8);
    double *red = reinterpret_cast<double *>(empty + 10);  // one double per consumer thread
    double *elec_s = red + 32 * NW;             // [WP*EPT][3], grid units

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int WP = WARPOWN ? 1 : prm.point_warps, WS = NW / WP;
    double *dzt = elec_s + WP * EPT * 3;        // DZT: [g_segs * ZS][WP*EPT], 16-byte aligned (EPT = 4)
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.y, lo, hi);
    const int nk = hi - lo;

    const bool producer = !WARPOWN && warp == NW && lane == 0;
    int pk = 0;
    auto load_step = [&]() {
        const int slot = pk % stages;
        if (pk >= stages) mbar_wait(&empty[slot], ((pk / stages) - 1) & 1);
        mbar_expect_tx(&full[slot], STAGE_BYTES);
        tma_bulk_g2s(smem + static_cast<size_t>(slot) * STAGE_BYTES,
                     prm.chunks + static_cast<size_t>(lo + pk) * STAGE_BYTES, STAGE_BYTES,
                     &full[slot]);
        ++pk;
    };
    auto load_own = [&](int g) {                   // WARPOWN: lane 0 of the owning warp
        mbar_expect_tx(&full[warp], STAGE_BYTES);
        tma_bulk_g2s(smem + static_cast<size_t>(warp) * STAGE_BYTES,
                     prm.chunks + static_cast<size_t>(g) * STAGE_BYTES, STAGE_BYTES, &full[warp]);
    };
    if (producer) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], NW);
        }
        fence_barrier_init();
        while (pk < nk && pk < stages) load_step();
    }
    if constexpr (WARPOWN) {
        if (warp < NW && lane == 0) {
            mbar_init(&full[warp], 1);
            fence_barrier_init();
            if (lo + warp < hi) load_own(lo + warp);
        }
    }
    const int ppb = WP * EPT;
    for (int i = threadIdx.x; i < ppb * 3; i += 32 * (NW + 1)) {
        int p = blockIdx.x * ppb + i / 3;
        p = p < prm.P ? p : prm.P - 1;
        const int comp = i % 3;
        // units of hz on every axis: (r - org) / hz; node (ix, iy, iz) sits at (ix sx, iy sy, iz)
        elec_s[i] = (point_coord(prm, static_cast<int64_t>(p) * 3 + comp) - prm.g_org[comp]) * prm.g_scaleV;
    }
    if constexpr (DZT) {                           // dz of every (z node, point of this CTA)
        const int nzp = prm.g_segs * GRID_ZS;
        for (int i = threadIdx.x; i < nzp * ppb; i += 32 * (NW + 1)) {
            const int kz = i / ppb, pp = i - kz * ppb;
            int p = blockIdx.x * ppb + pp;
            p = p < prm.P ? p : prm.P - 1;
            const double uz = (point_coord(prm, static_cast<int64_t>(p) * 3 + 2) - prm.g_org[2]) * prm.g_scaleV;
            dzt[i] = uz - static_cast<double>(kz);
        }
    }
    __syncthreads();
    QMMM_MARK(1);

    if (warp == NW) {
        if constexpr (!WARPOWN) {
            if (lane == 0)
                while (pk < nk) load_step();
        }
        return;                                    // WARPOWN: the consumer warps load for themselves
    }

    const int wp = warp % WP, ws = warp / WP;
    const double *pe = elec_s + wp * EPT * 3;
    double V[EPT], Ex[EPT], Ey[EPT], Ez[EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) V[e] = Ex[e] = Ey[e] = Ez[e] = 0.0;

    // one z run (n4 * 4 nodes at b, [k/2][32][2] doubles) of the lane's row at (fx, fy) (units
    // of hz: ix hx/hz, iy hy/hz), first node at z = fz, for the thread's EPT points
    const int tstride = WP * EPT;                  // DZT: doubles per z node in the table
    auto walk = [&](const double *b, int n4, double fx, double fy, double fz, const double *tz) {
        double dx[EPT], dy[EPT], rxy2[EPT], azb[EPT], S[EPT], SZ[EPT];
#pragma unroll
        for (int e = 0; e < EPT; ++e) {
            dx[e] = pe[3 * e + 0] - fx;
            dy[e] = pe[3 * e + 1] - fy;
            rxy2[e] = fma(dy[e], dy[e], fma(dx[e], dx[e], 1e-200));
            if constexpr (!DZT) azb[e] = pe[3 * e + 2] - fz;
            S[e] = SZ[e] = 0.0;
        }
#pragma unroll 1
        for (int k4 = 0; k4 < n4; ++k4) {
            const double2 Qa = *reinterpret_cast<const double2 *>(b + (2 * k4) * 64);
            const double2 Qb = *reinterpret_cast<const double2 *>(b + (2 * k4 + 1) * 64);
            const double qs[4] = {Qa.x, Qa.y, Qb.x, Qb.y};
#pragma unroll
            for (int t = 0; t < 4; ++t) {
                double dzs[EPT];
                if constexpr (DZT) {               // EPT = 4: two broadcast 128-bit loads
                    const double2 d01 = *reinterpret_cast<const double2 *>(tz + t * tstride);
                    const double2 d23 = *reinterpret_cast<const double2 *>(tz + t * tstride + 2);
                    dzs[0] = d01.x; dzs[1] = d01.y; dzs[EPT - 2] = d23.x; dzs[EPT - 1] = d23.y;
                } else {
#pragma unroll
                    for (int e = 0; e < EPT; ++e)
                        dzs[e] = t == 0 ? azb[e] : azb[e] - static_cast<double>(t);
                }
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                    const double dz = dzs[e];
                    const double r2 = fma(dz, dz, rxy2[e]);
                    const double y = rsqrt_refined_f64(r2);
                    if constexpr (WITH_E) {
                        const double p = qs[t] * y;
                        V[e] += p;
                        const double s = p * (y * y);
                        S[e] += s;
                        SZ[e] = fma(s, dz, SZ[e]);
                    } else {
                        V[e] = fma(qs[t], y, V[e]);
                    }
                }
            }
            if constexpr (DZT) {
                tz += 4 * tstride;
            } else {
#pragma unroll
                for (int e = 0; e < EPT; ++e) azb[e] -= 4.0;
            }
        }
        if constexpr (WITH_E) {
#pragma unroll
            for (int e = 0; e < EPT; ++e) {
                Ex[e] = fma(dx[e], S[e], Ex[e]);
                Ey[e] = fma(dy[e], S[e], Ey[e]);
                Ez[e] += SZ[e];
            }
        }
    };

    const int segs = prm.g_segs, ny = prm.g_n[1];
    QMMM_MARK(2);
    if constexpr (WARPOWN) {
        int it = 0;
        for (int g = lo + warp; g < hi; g += NW, ++it) {
            const int tl = g / segs, sg = g - tl * segs;
            const int rw = tl * 32 + lane, rx = rw / ny;
            mbar_wait(&full[warp], it & 1);
            walk(reinterpret_cast<const double *>(smem + static_cast<size_t>(warp) * STAGE_BYTES) + 2 * lane,
                 GRID_ZS / 4, static_cast<double>(rx) * prm.g_sx, static_cast<double>(rw - rx * ny) * prm.g_sy,
                 static_cast<double>(sg * GRID_ZS), nullptr);
            __syncwarp();                          // every lane has read the slot
            if (lane == 0 && g + NW < hi) {        // refill it with the warp's next gchunk
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                load_own(g + NW);
            }
        }
    } else {
        const int ZL = GRID_ZS / WS, z0 = ws * ZL;       // this warp's z run inside every gchunk
        // (tile, seg) of gchunk g = tile * segs + seg, and the lane's row (ix, iy) of that tile
        int tile = lo / segs, seg = lo - tile * segs;
        int ix = (tile * 32 + lane) / ny, iy = tile * 32 + lane - ix * ny;
        for (int k = 0; k < nk; ++k) {
            const int slot = k % stages;
            mbar_wait(&full[slot], (k / stages) & 1);
            walk(reinterpret_cast<const double *>(smem + static_cast<size_t>(slot) * STAGE_BYTES) +
                     (z0 / 2) * 64 + 2 * lane,
                 ZL / 4, static_cast<double>(ix) * prm.g_sx, static_cast<double>(iy) * prm.g_sy,
                 static_cast<double>(seg * GRID_ZS + z0),
                 dzt + (seg * GRID_ZS + z0) * tstride + wp * EPT);
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
            if (++seg == segs) {               // next row tile
                seg = 0;
                ++tile;
                iy += 32;
                if (ny >= 32) {
                    if (iy >= ny) { iy -= ny; ++ix; }
                } else {
                    ix = (tile * 32 + lane) / ny;
                    iy = tile * 32 + lane - ix * ny;
                }
            }
        }
    }

    QMMM_MARK(3);
    // nuclei (units of hz), FP64
    if constexpr (WITH_E) {
        nuclei_share<EPT>(prm, pe, ws, WS, lane, V, Ex, Ey, Ez);
    } else {
        double nEx[EPT], nEy[EPT], nEz[EPT];
#pragma unroll
        for (int e = 0; e < EPT; ++e) nEx[e] = nEy[e] = nEz[e] = 0.0;
        nuclei_share<EPT>(prm, pe, ws, WS, lane, V, nEx, nEy, nEz);
    }

    QMMM_MARK(4);
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
    consumer_sync<NW>();
    pdl_wait();                                  // the previous evaluation is done with the workspace
    if (ws == 0) {
        double a = 0.0;
        if (lane < EPT * 4)
            for (int s = 0; s < WS; ++s) a += red[((s * WP + wp) * EPT) * 4 + lane];
        a *= (lane & 3) ? prm.g_scaleE : prm.g_scaleV;
        const int p = (blockIdx.x * WP + wp) * EPT + lane / 4;
        if (prm.push_slots)
            push_records<EPT>(prm, a, (blockIdx.x * WP + wp) * EPT, lane);
        else if (lane < EPT * 4 && p < prm.P)
            prm.partial[(static_cast<int64_t>(blockIdx.y) * prm.P + p) * 4 + (lane & 3)] = a;
    }
    QMMM_MARK(5);
    if (prm.push_slots) {                        // (uniform over the grid)
        finish_point_block_push<32 * NW>(prm, WP * EPT, threadIdx.x, flag, reinterpret_cast<double *>(smem), red,
                                         [] { consumer_sync<NW>(); });
        QMMM_MARK(6);
        QMMM_MARK_GT(9);
        return;
    }
    finish_point_block<32 * NW>(prm, WP * EPT, threadIdx.x, flag, red, [] { consumer_sync<NW>(); },
                                prm.seq);
    QMMM_MARK(6);
    QMMM_MARK_GT(9);
}

// ----------------------------------------------------------------------------- create: detect
// Smallest positive difference between consecutive sources per axis (a candidate spacing):
// CTA b writes part[3b..3b+2].
__global__ void __launch_bounds__(256) grid_spacing_kernel(const double *xyz, int64_t M, double *part) {
    __shared__ double sh[8][3];
    double mn[3] = {1e300, 1e300, 1e300};
    for (int64_t j = blockIdx.x * 256ll + threadIdx.x; j + 1 < M; j += 256ll * gridDim.x)
        for (int k = 0; k < 3; ++k) {
            const double d = fabs(xyz[3 * (j + 1) + k] - xyz[3 * j + k]);
            if (d > 0.0) mn[k] = fmin(mn[k], d);
        }
    for (int k = 0; k < 3; ++k)
        for (int m = 16; m >= 1; m >>= 1) mn[k] = fmin(mn[k], __shfl_xor_sync(0xffffffffu, mn[k], m));
    if ((threadIdx.x & 31) == 0)
        for (int k = 0; k < 3; ++k) sh[threadIdx.x >> 5][k] = mn[k];
    __syncthreads();
    if (threadIdx.x < 3) {
        double v = sh[0][threadIdx.x];
        for (int w = 1; w < 8; ++w) v = fmin(v, sh[w][threadIdx.x]);
        part[3 * blockIdx.x + threadIdx.x] = v;
    }
}

struct GridGeom {
    double org[3];      // node (0,0,0)
    double h[3];        // spacing per axis (orthorhombic cells; cubic: all equal)
    int n[3];           // nodes per axis
    double tol;         // accepted distance of a source from its node, per axis (bohr)
};

// Every source must sit on a node (within tol) and no node may hold two sources; the charges
// go to the dense array dense[nx][ny][nz] (zero elsewhere).  bad[0] counts off-node sources,
// bad[1] duplicates.
__global__ void grid_scatter_kernel(const double *xyz, const double *q, int64_t M, GridGeom gg,
                                    double *dense, int *count, int *bad) {
    const int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (j >= M) return;
    int idx[3];
    bool ok = true;
    for (int k = 0; k < 3; ++k) {
        const double x = xyz[3 * j + k];
        const double fi = rint((x - gg.org[k]) / gg.h[k]);
        ok = ok && fi >= 0.0 && fi < static_cast<double>(gg.n[k]) &&
             fabs(fma(fi, gg.h[k], gg.org[k]) - x) <= gg.tol;
        idx[k] = static_cast<int>(fmin(fmax(fi, 0.0), static_cast<double>(gg.n[k] - 1)));
    }
    if (!ok) {
        atomicAdd(bad, 1);
        return;
    }
    const int64_t at = (static_cast<int64_t>(idx[0]) * gg.n[1] + idx[1]) * gg.n[2] + idx[2];
    if (atomicAdd(count + at, 1) != 0) {
        atomicAdd(bad + 1, 1);
        return;
    }
    dense[at] = q[j];
}

// Pack the dense charges into gchunks: one thread per (padded) row.  Cells beyond the grid are 0.
// REAL = float: each charge absorbs the rounding residual of the previous one (running monopole
// residual below one rounding unit); the residual runs along the row and
// on into the next row of the same tile of 32 rows (one thread per tile: a residual dropped at
// the end of every ROW left 16,384 of them on config 3, +1.4e-10 hartree at every point).
template <typename REAL>
__global__ void grid_pack_kernel(const double *dense, int64_t rows, int nz, int segs,
                                 int64_t rows_padded, double q_scale, REAL *out) {
    constexpr int PER = sizeof(REAL) == 4 ? 4 : 2;       // nodes per 128-bit load
    constexpr int ROWS = sizeof(REAL) == 4 ? 32 : 1;     // rows per thread
    const int64_t row0 = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (row0 >= rows_padded || row0 % ROWS != 0) return;
    double carry = 0.0;
    for (int64_t row = row0; row < row0 + ROWS; ++row) {
        const int64_t tile = row / 32;
        const int lane = static_cast<int>(row % 32);
        for (int seg = 0; seg < segs; ++seg) {
            REAL *o = out + (tile * segs + seg) * GRID_NODES;
            for (int k = 0; k < GRID_ZS; ++k) {
                const int iz = seg * GRID_ZS + k;
                const double qd = (row < rows && iz < nz) ? dense[row * nz + iz] * q_scale : 0.0;   // 2^k: exact
                REAL v;
                if constexpr (sizeof(REAL) == 4) {
                    const double want = qd + carry;
                    v = static_cast<float>(want);
                    carry = qd != 0.0 ? want - static_cast<double>(v) : carry;
                    if (qd == 0.0) v = 0.0f;                 // empty cells stay exactly empty
                } else {
                    v = qd;
                }
                o[(k / PER) * 32 * PER + lane * PER + (k % PER)] = v;
            }
        }
    }
}

// number of non-empty cells of a dense charge array (qmmm_field_create_grid reports it as M)
__global__ void grid_count_kernel(const double *dense, int64_t n, unsigned long long *out) {
    unsigned long long c = 0;
    for (int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x; j < n;
         j += static_cast<int64_t>(blockDim.x) * gridDim.x)
        c += dense[j] != 0.0;
    for (int m = 16; m >= 1; m >>= 1) c += __shfl_xor_sync(0xffffffffu, c, m);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(out, c);
}

// nuclei in units of hz: {(x - org) / hz, ..., Z}
__global__ void grid_nuclei_kernel(const double *nuc, int64_t K, GridGeom gg, double *out) {
    const int64_t j = blockIdx.x * static_cast<int64_t>(blockDim.x) + threadIdx.x;
    if (j >= K) return;
    for (int k = 0; k < 3; ++k) out[4 * j + k] = (nuc[4 * j + k] - gg.org[k]) / gg.h[2];
    out[4 * j + 3] = nuc[4 * j + 3];
}

}  // namespace qmmm
