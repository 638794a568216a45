/*
 * qmmm_field.h -- C ABI of the B200-native electrostatic potential / field library.
 *
 * Hot path of arxiv 1011.4687 ("Acceleration of a QM/MM-QMC simulation using GPU"):
 * the electrostatic potential that an environment's fixed charge-density cells and
 * nuclei produce at the QM electrons' positions,
 *
 *     V(r_i) = sum_{j<M} q_j / |r_i - R_j|  +  sum_{b<K} Z_b / |r_i - R_b|
 *                                              (Eq. 4; V = -U_ES)
 *     E(r_i) = -grad V(r_i) = sum_j q_j (r_i - R_j) / |r_i - R_j|^3   (north_star)
 *
 * an exact, open-boundary direct sum (no cutoff, no softening, no periodic images).
 * Atomic units (bohr, hartree, elementary charge).  The paper uploads the cell
 * positions / charges once per run and exchanges only r_new and U_ES per
 * Monte-Carlo step; that is the create / eval split below.
 *
 * Sign: the paper's U_ES (energy of an electron) is -V with q_j = -rho(r_m) dV for
 * the cells and +Z_b for the nuclei (readings 1-2).
 *
 * Precondition: no evaluation point coincides with a source (the paper has no
 * softening); a coincident pair yields IEEE inf/NaN.  Inputs are not scanned for
 * non-finite values.
 *
 * All entry points return a qmmm_status and never throw or abort; the message of
 * the last failure on the calling thread is available from qmmm_last_error().
 * Only sm_100 (B200) devices are supported; there is no CPU or other-GPU fallback.
 *
 * Determinism: identical inputs + same device + same library build give
 * bitwise-identical outputs (fixed CTA -> partial-slot mapping, fixed reduction
 * order, no floating-point atomics), independent of stream and earlier calls.
 */
#ifndef QMMM_FIELD_H
#define QMMM_FIELD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct qmmm_field qmmm_field;     /* opaque; owned by the library */

typedef enum {
    QMMM_OK = 0,
    QMMM_ERR_INVALID_ARG = 1,
    QMMM_ERR_ALLOC = 2,
    QMMM_ERR_CUDA = 3,
    QMMM_ERR_UNSUPPORTED_DEVICE = 4
} qmmm_status;

/* Arithmetic of the pairwise kernel (kernel in single or double,
 * everything around it in double).  I/O is FP64 in both modes.
 *   QMMM_FP64       : FP64 throughout (rel. error <= 1e-12 on V and E).
 *   QMMM_FP32_ACC64 : cell sources in FP32 arithmetic (MUFU rsqrt + one Newton
 *                     step, applied to the sum), running sums in FP64; nuclei always FP64
 *                     (per-point rel. error <= 1e-5 on V and on |E|, per-configuration
 *                     energy within 1e-5 hartree).  Conditions of the bound on |E|: the point
 *                     is at least two cell edges from every charged cell (one edge with the
 *                     lattice per work unit, qmmm_field_set_local_lattice), and the sum does
 *                     not cancel to less than about a hundredth of its terms (kappa <~ 100:
 *                     no FP32 arithmetic can do better than ~1e-7 x sum |q|/r^2).  E = NULL on
 *                     a grid runs a potential-only kernel (6 instead of 8 operations per pair)
 *                     whose row sums are compensated: on BASELINE config 3 its V is within
 *                     2.7e-8 hartree rms per point and 2.4e-6 hartree summed over all 16,384
 *                     points; the batched V + E kernel does the same by default (2.6e-8,
 *                     2.6e-6; qmmm_field_set_accurate_v). */
typedef enum { QMMM_FP64 = 0, QMMM_FP32_ACC64 = 1 } qmmm_precision;

/*
 * qmmm_field_create -- upload and pack one environment (once per run).
 *   src_xyz [M][3], src_q [M]   cell centres and cell CHARGES q_j (= -rho_j dV)
 *   nuc_xyz [K][3], nuc_Z [K]   nuclei, enter with charge +Z
 *   Each pointer may be a host pointer or a device pointer (detected); arrays are
 *   C-contiguous FP64.  M = 0 and/or K = 0 are valid (then the pointers may be NULL).
 *   max_points >= 1             largest W*N a later eval may pass (sizes the
 *                               per-CTA partials workspace).
 *   *out                        receives the handle.
 * Ownership: everything needed is copied; the caller may free its arrays on return.
 * The handle owns its device buffers.  Blocks until the packing has finished.
 * Errors: INVALID_ARG (NULL out, NULL array with nonzero count, M < 0, K < 0,
 * max_points < 1), UNSUPPORTED_DEVICE (current device is not compute capability
 * 10.x), ALLOC, CUDA.
 */
qmmm_status qmmm_field_create(const double *src_xyz, const double *src_q, int64_t M,
                              const double *nuc_xyz, const double *nuc_Z, int64_t K,
                              int64_t max_points, qmmm_field **out);

/*
 * qmmm_field_eval -- V and E at W*N evaluation points (once per step).
 *   elec_xyz  DEVICE [W*N][3] FP64    electron positions, W walkers x N electrons
 *   V         DEVICE [W*N]    FP64    out: potential (cells + nuclei)
 *   E         DEVICE [W*N][3] FP64    out: field; NULL = potential only
 *   prec      qmmm_precision
 *   stream    cudaStream_t (as void*); all work is enqueued on it, the call never
 *             synchronises or allocates, so it may be captured into a CUDA graph.  One eval in flight per handle (its workspace); for concurrent
 *             streams or host threads use qmmm_field_share.
 * Errors: INVALID_ARG (NULL handle/elec_xyz/V, W*N < 1 or > max_points, bad prec),
 * CUDA (launch failure).  Outputs are unspecified after an error.
 */
qmmm_status qmmm_field_eval(qmmm_field *h, const double *elec_xyz, int64_t W, int64_t N,
                            double *V, double *E, int prec, void *stream);

/*
 * qmmm_field_eval_energy -- the paper's own output (Eq. 4): the electrostatic
 * energy of each configuration's electrons in the environment's field,
 *     U_ES[w] = - sum_{i<N} V(r_{w,i})          (electrons carry charge -1),
 * without writing V or E back ("energy-fused variant").
 *   elec_xyz  DEVICE [W][N][3] FP64;   U  DEVICE [W] FP64 out;   prec, stream as eval.
 * The field is not formed in FP64 (potential-only kernel); the per-walker sum runs in a
 * fixed order (deterministic).  Two launches on `stream`, never synchronises.
 * Errors as qmmm_field_eval (U takes the place of V).
 */
qmmm_status qmmm_field_eval_energy(qmmm_field *h, const double *elec_xyz, int64_t W, int64_t N,
                                   double *U, int prec, void *stream);

/*
 * qmmm_field_eval_host -- the paper's per-step call: HOST buffers in and out;
 * returns when V_host (and E_host) hold the result.  Buffers may be pageable or pinned.
 *   W*N == 1  : served by a resident "move server": one cooperative kernel (one CTA per SM)
 *               that stays on the GPU, polls a pinned mailbox for r_new, evaluates, and
 *               writes {V, E} back -- no kernel launch, copy or synchronisation per move.
 *               It retires by itself after 2 ms without a request (and after 1 s in any
 *               case) and is restarted transparently; any other call on the handle retires
 *               it first.  While it is resident it occupies every SM, so there is at most
 *               one per device: when several handles make host-buffer calls at the same time
 *               (qmmm_field_share) a resident server is asked to yield and everybody uses the
 *               launch path below until the device is quiet again.  `stream` is not used.
 *               Environments with the grid-aware copy are served by the grid-aware server
 *               (every warp keeps its work units of charges in shared memory: configs[2]
 *               needs no source traffic at all per move), others -- and layout LIST -- by
 *               the source-list server.
 *   W*N <= 64 : one kernel launch on `stream`, no copies and no stream synchronisation: up to
 *               32 points travel as kernel parameters (more are read by the kernel from a
 *               pinned, device-mapped mailbox), and the results come back as one tagged
 *               record per point -- four self-validating 16-byte units {tag, V} {tag, Ex}
 *               {tag, Ey} {tag, Ez} -- written by the kernel straight into pinned host memory,
 *               which the call polls (or, for launch shapes the record collection does not
 *               cover, as V, E followed by a sequence number).
 *   otherwise : host->device copy, kernel, device->host copy on `stream`, synchronisation.
 * The launch paths and the source-list server give bitwise the result of qmmm_field_eval with
 * the same plan and layout; the grid-aware server splits the work units over its warps in its
 * own way and agrees to rounding (deterministic from call to call).
 * Same argument meaning and errors as qmmm_field_eval.
 */
qmmm_status qmmm_field_eval_host(qmmm_field *h, const double *elec_xyz_host, int64_t W,
                                 int64_t N, double *V_host, double *E_host, int prec,
                                 void *stream);

/*
 * qmmm_field_eval_move_host -- one single-electron move of the QMC loop (the
 * Metropolis step needs U_ES(r_new) - U_ES(r_old), Eq. 4): the potential and field
 * at r_new and their change from r_old, dV = V(r_new) - V(r_old) (the change of the electron's
 * electrostatic energy is -dV) and dE = E(r_new) - E(r_old), in one call with HOST buffers.
 *   r_old, r_new   HOST [3]       the electron's position before and after the proposed move
 *   V_old, E_old   HOST [1], [3]  V and E at r_old as a previous call returned them (V_new, E_new
 *                                 of the accepted move), or NULL: then r_old is evaluated too, in
 *                                 the SAME launch as r_new (one two-point evaluation, not two)
 *   V_new, E_new   HOST [1], [3]  out: V(r_new), E(r_new); E_new may be NULL (potential only:
 *                                 E_old and dE are then ignored)
 *   dV, dE         HOST [1], [3]  out: the differences; each may be NULL
 * With V_old (and E_old when E_new is wanted) this is the one-point call of qmmm_field_eval_host
 * -- the resident move server, 6-7 us per move on configs[2] -- plus a subtraction on the host;
 * without them it is the two-point launch path of qmmm_field_eval_host.  Accuracy: V and E as for
 * qmmm_field_eval; dV carries the absolute error of the two potentials (a difference of nearly
 * equal numbers), not a relative one.  Errors as qmmm_field_eval_host (the handle needs
 * max_points >= 2 for the two-point form).
 */
qmmm_status qmmm_field_eval_move_host(qmmm_field *h, const double *r_old, const double *r_new,
                                      const double *V_old, const double *E_old, double *V_new,
                                      double *E_new, double *dV, double *dE, int precision,
                                      void *stream);

/*
 * qmmm_field_eval_moves_host -- n successive single-configuration evaluations, the loop the
 * paper deploys (every Monte-Carlo step sends r_new and receives U_ES).  Step s
 * evaluates the N points elec_xyz_host[s][N][3] and writes V_host[s][N] (and E_host[s][N][3]
 * unless NULL) through the same per-move path as qmmm_field_eval_host with W = 1; the steps
 * are strictly sequential (step s+1 starts after the host has received step s), as in a
 * Metropolis walk where the next proposal depends on the last result.  *seconds (may be
 * NULL) receives the host wall-clock time of the whole loop.  Same errors as eval_host.
 */
qmmm_status qmmm_field_eval_moves_host(qmmm_field *h, const double *elec_xyz_host, int64_t n,
                                       int64_t N, double *V_host, double *E_host, int prec,
                                       void *stream, double *seconds);

/*
 * qmmm_field_eval_moves -- n INDEPENDENT single-configuration evaluations whose positions are
 * all known up front, on the device (BASELINE configs[2]: 1,000 evaluations along a given
 * random walk): move s evaluates the N points elec_xyz[s][N][3] (device) into V[s][N] and
 * E[s][N][3] (device; E may be NULL).  Equivalent to n calls of qmmm_field_eval with W = 1,
 * issued from C (no per-call binding cost) and always with overlapped launches
 * (qmmm_field_set_overlap): each move is its own kernel, move s + 1 starts while move s
 * finishes.  The FIRST move is launched with plain stream serialization, so elec_xyz may be
 * produced by whatever precedes the call on the stream; the later moves follow this library's
 * own kernels, which do not write elec_xyz.  Asynchronous on `stream`; capturable into a CUDA
 * graph.  Errors as qmmm_field_eval.
 */
qmmm_status qmmm_field_eval_moves(qmmm_field *h, const double *elec_xyz, int64_t n, int64_t N,
                                  double *V, double *E, int prec, void *stream);

/*
 * Grid-aware compact source format.  The paper's sources are "spatially
 * discretized cells": nodes of a regular grid.  When the cells are the nodes
 *     R(ix, iy, iz) = origin + (ix hx, iy hy, iz hz),   0 <= i_k < n[k]   (cubic or orthorhombic cells)
 * the library keeps a second copy that stores only the charges (4 B FP32 / 8 B FP64 per cell
 * instead of 16 / 32 B) and regenerates the coordinates from the indices.  Its kernels walk
 * the z rows of the grid, where dx, dy and dx^2 + dy^2 are row constants: 9 FP32 (13 FP64)
 * lane operations per pair instead of 14 (18).  Same V and E as the list kernels up to
 * rounding (FP64: node coordinates are origin + i*spacing, within 16 ulp of the listed
 * positions; tolerances as for the list).  Empty (masked) cells are zero charges.
 *
 * qmmm_field_create detects the structure by itself (every source must lie on a node within
 * 16 ulp of the largest coordinate, no node twice, at least half of the bounding grid
 * occupied, M >= 4096, cell edges within a factor 16 of each other); qmmm_field_create_grid takes the grid directly:
 *   origin [3]                  position of node (0,0,0), bohr (host pointer)
 *   spacing                     cell edge h > 0, bohr
 *   n [3]                       nodes per axis, 1..65536 each, at most 2e9 cells (host pointer)
 *   cell_q [n0][n1][n2]         cell CHARGES, C order (z fastest), host or device pointer;
 *                               0 = no cell there
 *   nuclei, max_points, out     as qmmm_field_create
 * A handle made by qmmm_field_create_grid has no source list (layout LIST is refused).  Precondition of the grid layout: no evaluation
 * point coincides with a node that carries charge (empty nodes are harmless).
 * Errors as qmmm_field_create.
 */
qmmm_status qmmm_field_create_grid(const double *origin, double spacing, const int64_t *n,
                                   const double *cell_q, const double *nuc_xyz,
                                   const double *nuc_Z, int64_t K, int64_t max_points,
                                   qmmm_field **out);
/* The same for orthorhombic cells: spacing [3] = (hx, hy, hz) (host pointer), nodes at
 * origin + (ix hx, iy hy, iz hz).  The row walk is unchanged (lengths are measured in units of
 * hz; dx, dy take the factors hx/hz, hy/hz once per row). */
qmmm_status qmmm_field_create_grid3(const double *origin, const double *spacing, const int64_t *n,
                                    const double *cell_q, const double *nuc_xyz,
                                    const double *nuc_Z, int64_t K, int64_t max_points,
                                    qmmm_field **out);

/* Which copy qmmm_field_eval uses.  AUTO (default): the grid kernels when the handle has a
 * grid with >= 2 work units (32 rows x 64 nodes) per slice and the batch is either a handful
 * of points (FP32 <= 2, FP64 <= 4: warp-private walks) or large enough to keep z runs of
 * >= 16 nodes per warp -- in practice one or two points, or a few dozen and more; otherwise
 * the list.  LIST / GRID force one (INVALID_ARG if the handle does not have that copy).
 * Sticky. */
typedef enum { QMMM_LAYOUT_AUTO = 0, QMMM_LAYOUT_LIST = 1, QMMM_LAYOUT_GRID = 2 } qmmm_layout;
qmmm_status qmmm_field_set_layout(qmmm_field *h, int layout);

typedef struct {
    int32_t present;             /* 1 if the handle has a grid copy */
    int32_t has_list;            /* 1 if the handle has a source list */
    int32_t layout;              /* qmmm_layout set by qmmm_field_set_layout */
    int32_t last_layout;         /* LIST or GRID: what the most recent eval used */
    int32_t n[3];                /* nodes per axis */
    int32_t reserved;
    double origin[3];            /* node (0,0,0), bohr */
    double spacing;              /* hz, bohr (= hx = hy for cubic cells) */
    int64_t n_gchunks;           /* work units of 32 rows x 64 z nodes (after padding) */
    int64_t bytes_fp32, bytes_fp64;
    double spacing3[3];          /* hx, hy, hz, bohr */
} qmmm_grid_info;
qmmm_status qmmm_field_get_grid_info(const qmmm_field *h, qmmm_grid_info *info);

/*
 * qmmm_field_share -- a second handle on the SAME environment for concurrent use.
 * The paper suggests OpenMP on the host code and one GPU shared by the node's MPI ranks
 * (PAPER.md:23, :242); one eval may be in flight per handle (its partials workspace, tickets
 * and mailboxes are per handle), so every host thread / stream gets its own handle.  The new
 * handle shares the parent's packed source copies (immutable after create; no copy, no
 * packing) and owns only its runtime buffers sized by max_points; plan, layout choice,
 * timing and the move server are per handle.  Handles may be destroyed in any order: the
 * source copies are freed with the last one.  Results are bitwise those of the parent.
 * Errors: INVALID_ARG (NULL argument, max_points < 1, current device differs from the
 * parent's), ALLOC, CUDA.
 */
qmmm_status qmmm_field_share(const qmmm_field *parent, int64_t max_points, qmmm_field **out);

/*
 * qmmm_sum_rank_partials -- the cross-device step of sharding by SOURCES (Eq. 5 of the paper,
 * PAPER.md:119-128, with one block B[m] per GPU): every rank evaluates all
 * points against its own cells, the per-rank partials {V, E} are gathered (NCCL all-gather of
 * 4 doubles per point), and this call adds them in RANK ORDER, out[i] = ((parts[0][i] +
 * parts[1][i]) + parts[2][i]) + ..., so that every rank holds bitwise the same sums (a tree
 * all-reduce would not fix the order).
 *   parts  DEVICE [R][n] FP64,  out  DEVICE [n] FP64 (may alias parts[0]),  1 <= R <= 65536.
 * Asynchronous on `stream`.  Errors: INVALID_ARG, CUDA (launch failure).
 */
qmmm_status qmmm_sum_rank_partials(const double *parts, int64_t R, int64_t n, double *out, void *stream);

/*
 * qmmm_field_min_distance -- debug helper, not part of the hot path (SURVEY.md 8(b) "r = 0"): the
 * smallest distance, in bohr, between the P evaluation points and the CHARGED sources of the
 * handle (cells with q != 0 and nuclei with Z != 0).  The evaluation has no softening and no
 * exclusion (PAPER.md:59 has none): a point on a source gives IEEE inf / NaN, and the FP32 bound
 * on |E| asks for a clearance of two cell edges (qmmm_precision above); this is the call that
 * checks such preconditions.  Brute force over all pairs in FP64, one kernel on `stream`, then a
 * stream synchronisation; allocates and frees 8 bytes of device memory.
 *   elec_xyz           DEVICE [P][3] FP64
 *   min_distance_host  HOST   [1]    out; +inf for an environment without charged sources
 * INVALID_ARG for NULL pointers or P < 1 (P is not limited by max_points).
 */
qmmm_status qmmm_field_min_distance(qmmm_field *h, const double *elec_xyz, int64_t P,
                                    double *min_distance_host, void *stream);

/*
 * FP32 grid kernels: granularity of the coordinate lattice.  The FP32 path keeps every
 * difference (point - node) EXACT by rounding the point's coordinates to a power-of-two lattice
 * and corrects V for the rounding residual to first order; E is evaluated at the lattice point
 * (relative error about 3 x residual / distance per cell).  With one lattice per grid axis the
 * residual is up to 2^-25 of the axis length in nodes: fine for axes of up to 128 nodes (all FP32
 * BASELINE configurations, whose points keep more than three cell edges from the cells; tested
 * at two), too coarse for long axes with points next to cells.  With a lattice per work unit
 * (32 rows x 64 z nodes) the residual is 2^-25 of the distance to THAT unit's farthest node,
 * i.e. a few 1e-6 nodes next to the point whatever the size of the grid, at about 8 % more time
 * (measured on configs[3]: 5.68 instead of 5.27 ms).  mode -1 (default): per work unit when an
 * axis has more than 128 nodes; 0: never; 1: always.  The source-list FP32 kernels always use a
 * lattice per 2,048-source block.  With it the FP32 tolerance on E holds for points at least
 * 1.2 cell edges from every charged cell (tested).  The kernels that tabulate dz per CTA
 * (evaluations of three points and more with the automatic plan, z axes of up to about 1,500
 * nodes: configs[1] and all batched BASELINE configurations) do not evaluate at a lattice
 * position at all -- they fold the residual into r^2 and into the differences -- so the
 * setting does not concern them.  Sticky; INVALID_ARG on another mode.
 */
qmmm_status qmmm_field_set_local_lattice(qmmm_field *h, int mode);

/*
 * FP32 grid kernels, batched V + E evaluations (every warp its own points, dz table: a few
 * hundred points and more per call): accuracy of V.  BASELINE.json's north star asks for the
 * total electrostatic energy sum_i V(r_i) within 1e-5 hartree; for a batch of 16,384 points
 * (configs[3]) that is 4e-12 of the sum, which plain FP32 arithmetic with FP64 accumulation of
 * row sums misses (3.1e-5: a common bias of +1.9e-9 hartree per point and 6.7e-8 rms).
 * enable != 0 (default): r^2 = rxy2 + z2 with rxy2 formed in FP64 per (point, row) and z2 from a
 * second per-CTA table, both rounded once, the last level of the FP32 row sums added with a
 * two-sum and the one below it pairwise (as in the potential-only kernel): 2.6e-8 rms, +1.6e-10
 * mean, 2.6e-6 over the batch (0.9e-6 ... 9.3e-6 over seven seeded batches of that size: 24-bit
 * r^2 leaves about 3.6e-6 +- 3.4e-6, so larger batches will exceed 1e-5), at 6 % more time
 * (configs[3]: 5.62 instead of 5.30 ms).  enable = 0: the faster kernel
 * (every per-configuration energy still within 2e-6 hartree).  E agrees between the two to FP32
 * rounding (1e-7 relative).  Used when both tables fit in shared memory beside a pipeline of at
 * least two stages (z axes of up to 192 nodes: every FP32 BASELINE configuration), else the
 * faster kernel runs (qmmm_field_info.last_accurate_v tells which one the last evaluation ran).
 * Sticky; shared handles inherit the parent's setting at qmmm_field_share.
 */
qmmm_status qmmm_field_set_accurate_v(qmmm_field *h, int enable);

/*
 * qmmm_field_eval_noalloc -- V and E (Eq. 4, and its field) for callers that
 * cannot allocate: code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc.  No handle (qmmm_field_create allocates): the environment is passed with every
 * call as it is, FP64, all pointers DEVICE pointers:
 *   src_xyz [M][3], src_q [M]   cells (charges q_j = -rho_j dV);   nuc_xyz [K][3], nuc_Z [K]  nuclei (+Z)
 *   elec_xyz [P][3]             evaluation points, 1 <= P <= QMMM_NOALLOC_MAX_POINTS
 *   V [P], E [P][3] (E may be NULL)   out
 * FP64 arithmetic throughout (relative error <= 1e-12 as QMMM_FP64), deterministic, one kernel
 * launch (plus a memset of a few hundred bytes) on `stream`, asynchronous.  The call makes NO
 * cudaMalloc / cudaFree / allocating library call: its scratch memory -- the per-slice partial
 * sums of Eq. 5-6 and the arrival tickets -- is a fixed file-scope __device__ array of 2 MiB +
 * 4 KiB that every GPU loading the library holds until the process exits.  The first call on a
 * device resolves that array's device address (cudaGetSymbolAddress, once per device); make
 * one call outside any graph capture first.
 * Sharing: every call of the process on a device uses the SAME array.  Calls that overlap on the
 * GPU (different streams or host threads with two calls in flight at once) race on it and give
 * wrong results: serialise them.  The array keeps the last call's contents; what must start at
 * zero (the tickets) is cleared on `stream` at the start of each call.
 * It is the plain formulation (sources read from the caller's arrays, no packed copy, no grid
 * detection): about half the FP64 rate of the handle-based list kernels (measured on B200, 4,096
 * points x 1.04 M cells: 0.40 against 0.86 T pair interactions per second; 1.20 T with the grid
 * kernels).  M = 0 and/or K = 0 are
 * valid.  Errors: INVALID_ARG (NULL where not allowed, negative M or K, P < 1, P beyond the
 * maximum -- the message names the limit), UNSUPPORTED_DEVICE, CUDA.
 */
#define QMMM_NOALLOC_MAX_POINTS 4096
qmmm_status qmmm_field_eval_noalloc(const double *src_xyz, const double *src_q, int64_t M,
                                    const double *nuc_xyz, const double *nuc_Z, int64_t K,
                                    const double *elec_xyz, int64_t P, double *V, double *E,
                                    void *stream);

/* qmmm_field_destroy -- frees the handle and its device buffers.  NULL is a no-op. */
qmmm_status qmmm_field_destroy(qmmm_field *h);

/* Launch plan of the pairwise kernel (Eq. 5-6: U = B[1]+...+B[N_B]).
 * 0 in a field of qmmm_field_set_plan means "choose automatically". */
typedef struct {
    int32_t points_per_thread;   /* register blocking: 1, 2, 4 or 8 electrons per thread */
    int32_t point_warps;         /* warps of a CTA that own different point groups: 1..16 (clamped) */
    int32_t slices;              /* N_B: CTAs the source sum is split over (per point block) */
    int32_t stages;              /* TMA pipeline depth (shared-memory stages), 2..8; reduced if it does not fit */
} qmmm_plan;

/* Override the automatic plan (testing partition independence, tuning).  Sticky
 * until changed; pass zeros to restore automatic choice.  INVALID_ARG on bad values. */
qmmm_status qmmm_field_set_plan(qmmm_field *h, const qmmm_plan *plan);

typedef struct {
    int64_t M, K, max_points;
    int64_t n_chunks;            /* 128-source chunks after padding */
    int64_t bytes_fp64, bytes_fp32, bytes_workspace;
    qmmm_plan last_plan;         /* plan used by the most recent eval */
    int32_t last_point_blocks;   /* grid.x of the most recent pair kernel (grid.y = slices) */
    int32_t last_launches;       /* kernels launched by the most recent eval */
    int32_t sm_count;
    int32_t last_dz_table;       /* 1: the most recent eval ran a grid kernel that tabulates dz in shared
                                  * memory (8 / 12 instead of 9 / 13 lane operations per pair) */
    int32_t device_errors;       /* nonzero: a kernel of this handle gave up a bounded wait (a cross-CTA
                                  * record never arrived; never expected) and wrote NaN results.  Read
                                  * without synchronising; the host-buffer calls return QMMM_ERR_CUDA. */
    int32_t last_local_lattice;  /* 1: the most recent eval ran the FP32 grid kernel with a coordinate
                                  * lattice per work unit (qmmm_field_set_local_lattice) */
    int32_t last_accurate_v;     /* 1: the most recent eval ran an FP32 grid kernel with the accurate-V
                                  * arithmetic (qmmm_field_set_accurate_v; also the potential-only kernel) */
    char last_kernel[192];       /* mangled name of the kernel the most recent evaluation launched (or of
                                  * the move server it started): which template instantiation ran */
} qmmm_field_info;

qmmm_status qmmm_field_get_info(const qmmm_field *h, qmmm_field_info *info);

/*
 * Per-kernel device timing for roofline measurements.  When enabled, eval records CUDA
 * events on its stream before and after the pair kernel (a few microseconds of overhead;
 * off by default).  qmmm_field_last_timing waits for the most recent eval to finish and
 * returns the kernel duration in milliseconds; *finalize_ms is always 0 (the cross-CTA sum
 * and the nuclear term are fused into the pair kernel: one launch per evaluation).
 * INVALID_ARG if timing is off or no eval has run.
 */
qmmm_status qmmm_field_set_timing(qmmm_field *h, int enable);

/*
 * Overlap of back-to-back evaluations on one stream (off by default).  The paper's use is a
 * long sequence of single-point evaluations, one per Monte-Carlo move; each is
 * a few microseconds, of which the launch, the prologue (barrier set-up, first bulk copies)
 * and the tail (fence, ticket, cross-CTA sum) are the larger part.  When enabled, eval
 * launches its kernel with programmatic stream serialization: it may START while the previous
 * kernel in the stream -- the previous evaluation -- is still running, does its prologue,
 * source walk and in-CTA reduction, and waits for the predecessor to finish (griddepcontrol)
 * only before it touches the partials workspace, the tickets or V / E.  Results are bitwise
 * the same as without overlap for the same launch plan.  The plans that change are the
 * few-point grid kernels (up to 64 points), which run 4-warp instead of
 * 8-warp CTAs so that several evaluations share an SM -- the period of a sequence is a CTA's
 * lifetime divided by the CTAs an SM holds -- i.e. another association of the same sums:
 * equal to rounding, and still deterministic from run to run.
 * Precondition while enabled: elec_xyz of an evaluation must not be written by the kernel that
 * immediately precedes the evaluation on the stream, WHATEVER that kernel is (this library's
 * previous evaluation, or a caller's kernel that proposes the next positions): the points are
 * read before the wait, and CUDA gives a programmatically launched kernel no visibility of its
 * predecessor's writes before that wait.  Put any other kernel (or an event) in between, or
 * leave overlap off for evaluations whose points the preceding kernel produces.  Ignored (plain
 * serialization) while timing is on and by the host-buffer paths.  Works inside CUDA-graph
 * capture.
 */
qmmm_status qmmm_field_set_overlap(qmmm_field *h, int enable);
qmmm_status qmmm_field_last_timing(qmmm_field *h, double *pair_ms, double *finalize_ms);

/*
 * qmmm_probe_peak -- same-run roofline denominators (north_star: "measured by a
 * microbenchmark in the same run").  Runs a register-only kernel of independent
 * dependent chains on every SM and reports the achieved rate.
 *   kind 0: FP32 FFMA, 1: FP64 DFMA, 2: MUFU.RSQ (FP32), 3: empty-kernel launch+sync,
 *        4: read bandwidth over a 33 MB buffer (resident in L2 after the warm-up pass),
 *        5: read bandwidth over a 537 MB buffer (HBM)   (the rooflines of the
 *           single-electron path, whose sources are 8-67 MB per evaluation)
 *   iters      inner iterations / passes over the buffer (0 = default)
 *   *rate      out: warp-lane operations per second (kind 0-2; an FMA counts 1),
 *              seconds per launch+sync (kind 3), or bytes per second (kind 4, 5)
 *   *seconds   out: device time of the timed launch (CUDA events), may be NULL
 * Synchronises the stream.  Kinds 4 and 5 allocate (and free) their buffer on the current
 * device.  Errors: INVALID_ARG (NULL rate, unknown kind), ALLOC, CUDA; qmmm_last_error() is set.
 */
qmmm_status qmmm_probe_peak(int kind, int iters, double *rate, double *seconds, void *stream);

/* Thread-local message of the last error returned on this thread ("" if none). */
const char *qmmm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* QMMM_FIELD_H */
