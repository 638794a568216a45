// qmmm_field.cu -- C ABI (include/qmmm_field.h) and host-side launch logic.
//
// create : upload + pack sources once ("required only once at the beginning
//          of a run"), FP64 SoA chunks and FP32 tile-local SoA chunks, nuclei FP64.
// eval   : ONE launch: pair kernel over (point blocks x source slices) -> per-slice partials
//          (Eq. 5-6) incl. the slice's share of the nuclei -> the last CTA
//          of each point block adds the slices in a fixed order and writes V, E.
// No torch types, no CPU fallback: every step of the path runs in the kernels of
// qmmm_kernels.cuh.
#include "qmmm_kernels.cuh"
#include "qmmm_grid.cuh"
#include "qmmm_server.cuh"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <ctime>
#include <climits>
#include <memory>
#include <mutex>
#include <new>
#include <string>

#include "../../include/qmmm_field.h"

using namespace qmmm;

namespace {

thread_local std::string g_last_error;

qmmm_status fail(qmmm_status st, const std::string &msg) {
    g_last_error = msg;
    return st;
}
qmmm_status cuda_fail(cudaError_t e, const char *what) {
    return fail(QMMM_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}
#define CUDA_TRY(expr)                                          \
    do {                                                        \
        cudaError_t _e = (expr);                                \
        if (_e != cudaSuccess) return cuda_fail(_e, #expr);     \
    } while (0)

}  // namespace
namespace qmmm {
void set_last_error(const char *msg) { g_last_error = msg ? msg : ""; }    // for qmmm_probe.cu
}
namespace {

int pow2_ceil(int64_t v) {
    int p = 1;
    while (p < v) p <<= 1;
    return p;
}
int gcd_int(int a, int b) {
    while (b) { int t = a % b; a = b; b = t; }
    return a;
}

constexpr int MAIL_POINTS = 64;   // eval_host uses the zero-copy mailbox up to this many points
constexpr int MAIL_REC_OFFSET = MAIL_POINTS * 8;   // doubles before the tagged answer records (4 KB: 64-byte aligned)

constexpr size_t stage_bytes(bool f32) {
    return STAGE_HDR + (f32 ? static_cast<size_t>(BLOCK_CHUNKS) * 4 * CHUNK * 4
                            : static_cast<size_t>(STAGE_CHUNKS_F64) * 4 * CHUNK * 8);
}
// FP32 packed kernel variants: (points per thread, consumer warps)
constexpr int F32X2_NW_EPT8 = 8, F32X2_NW_EPT4 = 16, F32X2_NW_EPT2 = 16;
int f32x2_warps(int ept) { return ept == 8 ? F32X2_NW_EPT8 : (ept == 4 ? F32X2_NW_EPT4 : F32X2_NW_EPT2); }
size_t pair_smem_bytes(bool f32, int stages, int ept, int wp) {
    if (f32 && ept == 8) return F32x2Layout<4, F32X2_NW_EPT8>::total(stages);
    if (f32 && ept == 4) return F32x2Layout<2, F32X2_NW_EPT4>::total(stages);
    if (f32 && ept == 2) return F32x2Layout<1, F32X2_NW_EPT2>::total(stages);
    return stages * stage_bytes(f32) + 18 * sizeof(uint64_t) +
           static_cast<size_t>(32) * COMPUTE_WARPS * sizeof(double) +
           static_cast<size_t>(wp) * ept * 3 * sizeof(double);
}

// FP32 grid kernel variants: (points per thread -> warps per CTA)
#ifndef QMMM_GRID_F32_MAXEPT
#define QMMM_GRID_F32_MAXEPT 4
#endif
#ifndef QMMM_GRID_NW_EPT4
#define QMMM_GRID_NW_EPT4 8
#endif
constexpr int GRID_NW_EPT8 = 8, GRID_NW_EPT4 = QMMM_GRID_NW_EPT4, GRID_NW_EPT2 = 16;
// FP64 grid kernel variants: 8 warps x 4 points, 16 warps x 2 (or 1) points
#ifndef QMMM_GRID_F64_MAXEPT
#define QMMM_GRID_F64_MAXEPT 4
#endif
#ifndef QMMM_GRID64_NW_EPT4
#define QMMM_GRID64_NW_EPT4 8
#endif
constexpr int GRID64_NW_EPT4 = QMMM_GRID64_NW_EPT4, GRID64_NW_EPT2 = 16, GRID64_NW_EPT1 = 16;
// a handful of points (one point group): every warp loads and walks whole gchunks of its own
#ifndef QMMM_GRID64_NW_WARPOWN
#define QMMM_GRID64_NW_WARPOWN 8
#endif
constexpr int GRID64_NW_WARPOWN = QMMM_GRID64_NW_WARPOWN;
bool grid_f64_warpown(int ept, int64_t P) { return P <= ept; }
// "Light" CTAs for overlapped few-point evaluations (qmmm_field_set_overlap).  With overlap,
// the CTAs of consecutive evaluations share the SMs and the steady-state period of a sequence
// is (lifetime of a CTA, waiting included) / (CTAs an SM holds), until the serial tail bounds
// it: smaller CTAs win although a single evaluation gets slower.  4 warps instead of 8
// (measured per overlapped evaluation, 1,000 replayed from one graph): config 2 FP32
// 5.7 -> 3.7 us, FP64 6.9 -> 3.6 us; config 1 FP64 13.8 -> 9.5 us (2 warps: 3.5 / 3.8 us).
constexpr int GRID64_NW_LIGHT = 4, GRID64_NW_WARPOWN_LIGHT = 4, GRID_NW_NODEPACK_LIGHT = 4;
bool grid_f64_light(bool overlap, int ept, int64_t P) {
    return overlap && (grid_f64_warpown(ept, P) || (ept == 4 && P <= 64));
}
int grid_f64_warps(int ept, int64_t P, bool light) {
    if (grid_f64_warpown(ept, P)) return light ? GRID64_NW_WARPOWN_LIGHT : GRID64_NW_WARPOWN;
    if (light) return GRID64_NW_LIGHT;
    return ept == 4 ? GRID64_NW_EPT4 : (ept == 2 ? GRID64_NW_EPT2 : GRID64_NW_EPT1);
}
// one or two points per evaluation: the node-packed kernel, 8 warps, two CTAs per SM
#ifndef QMMM_GRID_NW_NODEPACK
#define QMMM_GRID_NW_NODEPACK 8
#endif
constexpr int GRID_NW_NODEPACK = QMMM_GRID_NW_NODEPACK;
bool grid_f32_nodepack(int ept, int64_t P) { return ept == 2 && P <= 2; }
constexpr int GRID_NW_EPT4_LIGHT = 4;
bool grid_f32_light(bool overlap, int ept, int64_t P) {
    return overlap && (grid_f32_nodepack(ept, P) || (ept == 4 && P <= 64));
}
int grid_f32_warps(int ept, int64_t P, bool light) {
    if (grid_f32_nodepack(ept, P)) return light ? GRID_NW_NODEPACK_LIGHT : GRID_NW_NODEPACK;
    if (light && ept == 4) return GRID_NW_EPT4_LIGHT;
    return ept == 8 ? GRID_NW_EPT8 : (ept == 4 ? GRID_NW_EPT4 : GRID_NW_EPT2);
}
// dz table of the FP64 grid kernel (4 points per thread, shared stages): [z nodes padded to
// whole gchunks][points of the CTA] doubles; 0 when the variant has none
#ifndef QMMM_GRID_F64_DZT
#define QMMM_GRID_F64_DZT 1
#endif
#ifndef QMMM_GRID_F32_DZT
#define QMMM_GRID_F32_DZT 1
#endif
size_t grid_dzt_bytes(bool f32, int ept, int wp, int64_t P, int64_t g_segs, bool light) {
    if (f32) {      // 4 points per thread; every warp its own point group, or z-split warps: the same table
        if (!QMMM_GRID_F32_DZT || ept != 4 || g_segs > 4096) return 0;
        (void)wp;
        return light ? GridF32Layout<2, GRID_NW_EPT4_LIGHT>::dzt_bytes(static_cast<int>(g_segs))
                     : GridF32Layout<2, GRID_NW_EPT4>::dzt_bytes(static_cast<int>(g_segs));
    }
    if (!QMMM_GRID_F64_DZT || ept != 4 || grid_f64_warpown(ept, P)) return 0;
    return static_cast<size_t>(g_segs) * GRID_ZS * wp * ept * sizeof(double);
}
size_t grid_smem_bytes(bool f32, int stages, int ept, int wp, int64_t P, bool light) {
    if (f32 && ept == 8) return GridF32Layout<4, GRID_NW_EPT8>::total(stages);
    if (f32 && ept == 4)
        return light ? GridF32Layout<2, GRID_NW_EPT4_LIGHT>::total(stages) : GridF32Layout<2, GRID_NW_EPT4>::total(stages);
    if (f32 && grid_f32_nodepack(ept, P))       // warp-private pipelines: two slots per warp
        return light ? GridF32Layout<1, GRID_NW_NODEPACK_LIGHT>::total(2 * GRID_NW_NODEPACK_LIGHT)
                     : GridF32Layout<1, GRID_NW_NODEPACK>::total(2 * GRID_NW_NODEPACK);
    if (f32) return GridF32Layout<1, GRID_NW_EPT2>::total(stages);
    if (grid_f64_warpown(ept, P)) stages = grid_f64_warps(ept, P, light);   // one private slot per warp
    return static_cast<size_t>(stages) * GRID_STAGE_BYTES_F64 + 18 * sizeof(uint64_t) +
           static_cast<size_t>(32) * grid_f64_warps(ept, P, light) * sizeof(double) +
           static_cast<size_t>(wp) * ept * 3 * sizeof(double);
}

}  // namespace

// The packed source copies of one environment.  They are immutable after create and may be
// shared by several handles (qmmm_field_share): the last handle to go frees them.
struct SourceOwner {
    void *ptr[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    ~SourceOwner() {
        for (void *p : ptr)
            if (p) cudaFree(p);
    }
};

struct qmmm_field {
    std::shared_ptr<SourceOwner> keep;   // owns chunks64/32, origins, nuclei, gcells32/64, nuclei_u
    int64_t M = 0, K = 0, max_points = 0;
    int64_t n_chunks = 0, n_chunks64 = 0, n_blocks = 0;
    int device = 0, sm_count = 0;
    double *chunks64 = nullptr;    // [n_chunks64][4][128] double (cells, then nuclei)
    float *chunks32 = nullptr;     // [n_chunks][4][128] float (offsets from block origin, q)
    double *origins = nullptr;     // [n_blocks][4]
    double lattice = 1.0;          // FP32 coordinate quantum (power of two)
    double *nuclei = nullptr;      // [K][4]
    double *workspace = nullptr;   // partials [slices][P][4]
    int64_t workspace_doubles = 0;
    double *stage_elec = nullptr;  // eval_host staging: [max_points][3]
    double *stage_out = nullptr;   // eval_host staging: V [max_points] then E [max_points][3]
    qmmm_plan user_plan = {0, 0, 0, 0};
    qmmm_plan last_plan = {0, 0, 0, 0};
    int last_point_blocks = 0, last_launches = 0, last_dz_table = 0;
    bool timing = false, timed = false;
    bool overlap = false;          // qmmm_field_set_overlap: back-to-back evaluations may overlap
    bool overlap_now = false;      // ... and this evaluation is launched that way (not timed, no mailbox)
    cudaEvent_t ev[2] = {nullptr, nullptr};
    // per-move mailbox: pinned, device-mapped host memory (elec in; V, E and a sequence flag out)
    double *mail_h = nullptr, *mail_d = nullptr;   // [MAIL_POINTS*3 | MAIL_POINTS*4 | flag | pad | records MAIL_POINTS*8]
    bool last_mail_push = false;                   // the last mailbox evaluation answered with tagged records
    unsigned long long seq = 0;
    // resident move server (qmmm_server.cuh): serves single-point eval_host calls
    ServerMailbox *srv_mail_h = nullptr, *srv_mail_d = nullptr;
    ServerDevice *srv_dev = nullptr;
    cudaStream_t srv_stream = nullptr;
    bool srv_alive = false, srv_ok = true;     // srv_ok: cooperative launch available
    int srv_prec = -1;
    unsigned long long srv_launch_id = 0, srv_seq = 0;
    int *counters = nullptr;       // [max_points] arrival tickets of the point blocks (zero at rest)
    // push-model collection for overlapped few-point evaluations (qmmm_kernels.cuh): tagged records
    unsigned long long *push_slots = nullptr;      // [PUSH_MAX_RECORDS][8] words, zero at create
    unsigned long long push_seq = 0;               // tag of the last pushing evaluation
    // grid layout (qmmm_grid.cuh): present when the cells are nodes of a cubic grid
    bool has_list = true, has_grid = false;
    GridGeom grid = {{0, 0, 0}, {1.0, 1.0, 1.0}, {0, 0, 0}, 0.0};
    int64_t g_rows = 0, g_tiles = 0, g_segs = 0, n_g = 0;
    float *gcells32 = nullptr;     // [n_g][ZS/4][32][4]
    double *gcells64 = nullptr;    // [n_g][ZS/2][32][2]
    double *nuclei_u = nullptr;    // [K][4] nuclei in grid units
    int layout = QMMM_LAYOUT_AUTO, last_layout = QMMM_LAYOUT_LIST;
    double bb_lo[3] = {0, 0, 0}, bb_hi[3] = {0, 0, 0};   // bounding box of the cells
    double q_scale = 1.0;          // power of two applied to the cell charges of the FP32 copies
    int local_lattice = -1;        // FP32 grid kernel, lattice per gchunk: -1 automatic, 0 off, 1 on
    int last_local_lattice = 0;
    int accurate_v = 1;            // FP32 batched grid V + E kernel: accurate V (qmmm_field_set_accurate_v)
    int last_accurate_v = 0;
    const char *last_kernel = "";  // mangled name of the kernel the most recent evaluation ran
    // device error word (pinned, device-mapped): set by a kernel whose bounded wait gave up
    int *dev_err_h = nullptr, *dev_err_d = nullptr;
    // first evaluation of a qmmm_field_eval_moves sequence: launched WITHOUT programmatic
    // serialization, so that it orders after whatever produced the positions
    bool pdl_hold = false;
};

namespace {

// Automatic plan: enough (point block x source slice) CTAs to fill the
// SMs in whole waves; few points -> sources split across all warps and SMs.
qmmm_plan choose_plan(const qmmm_field *h, int64_t P, bool f32, bool grid = false) {
    qmmm_plan pl = h->user_plan;
    const int max_ept = f32 ? 8 : 4;
    // automatic choice: FP32 grid kernel 16 warps x 4 points (measured faster than 8 x 8)
    const int auto_ept = grid ? (f32 ? QMMM_GRID_F32_MAXEPT : QMMM_GRID_F64_MAXEPT) : max_ept;
    if (pl.points_per_thread == 0) pl.points_per_thread = std::min(auto_ept, pow2_ceil(P));
    pl.points_per_thread = std::min(pl.points_per_thread, max_ept);
    if (grid && f32) pl.points_per_thread = std::max(pl.points_per_thread, 2);   // packed pairs only
    const int64_t groups = (P + pl.points_per_thread - 1) / pl.points_per_thread;
    const bool light = grid && (f32 ? grid_f32_light(h->overlap_now, pl.points_per_thread, P)
                                    : grid_f64_light(h->overlap_now, pl.points_per_thread, P));
    const int nw = grid ? (f32 ? grid_f32_warps(pl.points_per_thread, P, light) : grid_f64_warps(pl.points_per_thread, P, light))
                        : ((f32 && pl.points_per_thread >= 2) ? f32x2_warps(pl.points_per_thread) : COMPUTE_WARPS);
    if (pl.point_warps == 0) {
        // as many point warps as there are groups, but keep at least 4 point blocks when the
        // points allow it: slices = SMs / 4 then, so every CTA streams a 4x longer source run
        // through its TMA ring and the last CTA adds 4x fewer partials per point
        int pw = std::min<int>(nw, pow2_ceil(groups));
        // (overlapped few-point evaluations: the SMs are filled by several evaluations in
        // flight, not by one, so a CTA takes as many point groups as it has warps)
        while (!light && pw > 1 && (groups + pw - 1) / pw < 4) pw >>= 1;
        pl.point_warps = pw;
    }
    if (pl.point_warps > nw) pl.point_warps = nw;
    const int64_t pb = (groups + pl.point_warps - 1) / pl.point_warps;
    if (pl.slices == 0 && light) {
        // Overlapped evaluations: fewer, longer CTAs -- a quarter of an SM count per evaluation
        // (measured, 200-1,000 evaluations replayed from one graph, with the push-model
        // collection: config 2 FP32 148 / 74 / 37 / 18 CTAs: 2.67 / 2.17 / 1.87 / 1.81 us, FP64
        // 2.58 / 2.24 / 2.22 / 2.28 us; config 1 FP32 74 / 36 / 18 CTAs: 3.42 / 3.00 / 2.91 us,
        // FP64 8.60 / 7.27 / 7.21 us); a single evaluation gets slower.
        pl.slices = static_cast<int>(std::max<int64_t>(1, (h->sm_count / 4) / pb));
    }
    if (pl.slices == 0) {
        const int g = gcd_int(static_cast<int>(pb % h->sm_count), h->sm_count);
        pl.slices = h->sm_count / g;       // pb * slices is a multiple of the SM count
        // Many waves: a CTA costs about 5 us of launch, pipeline fill, reduction and ticket
        // whatever its length, while a partly filled last wave costs less and less.  Halve
        // the slices (longer CTAs) as long as 32 or more waves remain.
        while (pl.slices > 1 && pb * ((pl.slices + 1) / 2) >= 32 * static_cast<int64_t>(h->sm_count))
            pl.slices = (pl.slices + 1) / 2;
    }
    const int64_t work_units = grid ? std::max<int64_t>(h->n_g, (h->K + 31) / 32)
                               : f32 ? std::max<int64_t>(h->n_chunks, (h->K + 31) / 32) : h->n_chunks64;
    pl.slices = static_cast<int>(std::max<int64_t>(1, std::min<int64_t>(pl.slices, work_units)));
    // the partials workspace bounds slices * P
    const int64_t cap = h->workspace_doubles / (4 * P);
    if (pl.slices > cap) pl.slices = static_cast<int>(std::max<int64_t>(1, cap));
    if (pl.stages == 0) {
        const bool bandwidth_bound = groups <= 2;
        if (!grid) pl.stages = f32 ? (pl.points_per_thread == 1 ? 6 : 4) : (bandwidth_bound ? 6 : 3);
    }
    if (grid && pl.stages == 0) pl.stages = 4;             // one gchunk (8 / 16 KB) per stage
    if (grid && f32 && grid_f32_nodepack(pl.points_per_thread, P)) {
        pl.point_warps = 1;                                // every warp walks whole gchunks of its own
        pl.stages = 2;                                     // two private slots per warp
    }
    if (grid && !f32 && grid_f64_warpown(pl.points_per_thread, P)) {
        pl.point_warps = 1;
        pl.stages = 1;                                     // one private slot per warp
    }
    return pl;
}

// AUTO layout: the grid kernels when the handle has a grid, the source-split warps of a CTA
// keep z runs of at least 16 nodes (at most 4 of them share a gchunk) and every slice gets at
// least two gchunks (32 rows x 64 nodes each); else the source list, whose kernels split the
// source range more finely (single points, a handful of points).
bool auto_uses_grid(const qmmm_field *h, int64_t P, bool f32) {
    if (!h->has_grid) return false;
    if (!h->has_list) return true;
    const qmmm_plan pl = choose_plan(h, P, f32, true);
    if (h->n_g < static_cast<int64_t>(2) * pl.slices) return false;
    if (f32 && grid_f32_nodepack(pl.points_per_thread, P)) return true;     // single-point walk
    if (!f32 && grid_f64_warpown(pl.points_per_thread, P)) return true;     // warp-private gchunks
    const int nw = f32 ? grid_f32_warps(pl.points_per_thread, P, grid_f32_light(h->overlap_now, pl.points_per_thread, P))
                       : grid_f64_warps(pl.points_per_thread, P, grid_f64_light(h->overlap_now, pl.points_per_thread, P));
    return nw / pl.point_warps <= 4;
}

// records (slices x P) the push-model collection of a handle can hold; the collecting CTA
// keeps slices x (points of a CTA) records of 32 bytes in its idle stage buffers
constexpr int64_t PUSH_MAX_RECORDS = 4096;
constexpr int64_t PUSH_MAX_CTA_RECORD_BYTES = 32768;   // and never more than the stage buffers hold

// One evaluation kernel launch.  prm.pdl: programmatic stream serialization -- the kernel may
// start while its predecessor in the stream is still running (qmmm_field_set_overlap; the
// kernels order themselves with griddepcontrol, qmmm_kernels.cuh).
constexpr int MAX_DEVICES = 64;
thread_local int g_device = 0;                    // device of the handle being evaluated (checked current)
thread_local const char *g_launched = "";         // mangled name of the kernel launched last on this thread

const char *kernel_name(const void *kern) {
    const char *name = nullptr;
    if (cudaFuncGetName(&name, kern) != cudaSuccess || !name) {
        cudaGetLastError();
        return "?";
    }
    return name;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (function, device): one record
// per device, shared by all host threads.
struct SmemConfig {
    std::atomic<size_t> bytes[MAX_DEVICES];
    SmemConfig() { for (auto &b : bytes) b.store(0); }
    template <typename K>
    cudaError_t ensure(K kern, size_t smem) {
        std::atomic<size_t> &cur = bytes[g_device];
        if (smem <= cur.load(std::memory_order_acquire)) return cudaSuccess;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             static_cast<int>(smem));
        if (e != cudaSuccess) return e;
        size_t seen = cur.load();
        while (seen < smem && !cur.compare_exchange_weak(seen, smem)) {}
        return cudaSuccess;
    }
};

cudaError_t launch_eval_kernel(void (*kern)(const PairParams), dim3 grid, unsigned threads, size_t smem,
                               cudaStream_t st, const PairParams &prm) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(threads);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = prm.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, prm);
}

template <typename REAL, int EPT, bool WITH_E = true>
cudaError_t launch_pair(const PairParams &prm, dim3 grid, size_t smem, cudaStream_t st) {
    auto kern = pair_kernel<REAL, EPT, WITH_E>;
    static SmemConfig configured;
    static const char *const name = kernel_name(reinterpret_cast<const void *>(kern));
    g_launched = name;
    cudaError_t e = configured.ensure(kern, smem);
    if (e != cudaSuccess) return e;
    return launch_eval_kernel(kern, grid, CTA_THREADS, smem, st, prm);
}

template <int EP2, int NW>
cudaError_t launch_pair_f32x2(const PairParams &prm, dim3 grid, size_t smem, cudaStream_t st) {
    auto kern = pair_kernel_f32x2<EP2, NW>;
    static SmemConfig configured;
    static const char *const name = kernel_name(reinterpret_cast<const void *>(kern));
    g_launched = name;
    cudaError_t e = configured.ensure(kern, smem);
    if (e != cudaSuccess) return e;
    return launch_eval_kernel(kern, grid, 32 * NW, smem, st, prm);
}

// FP64: pair_kernel<double, 1|2|4>.  FP32-acc64: the scalar kernel for one point per
// thread (bandwidth-bound), the packed f32x2 kernel for 2, 4 or 8.
cudaError_t launch_pair_ept(bool f32, int ept, const PairParams &prm, dim3 grid, size_t smem,
                            cudaStream_t st) {
    if (f32) {
        switch (ept) {
            case 1: return launch_pair<float, 1>(prm, grid, smem, st);
            case 2: return launch_pair_f32x2<1, F32X2_NW_EPT2>(prm, grid, smem, st);
            case 4: return launch_pair_f32x2<2, F32X2_NW_EPT4>(prm, grid, smem, st);
            case 8: return launch_pair_f32x2<4, F32X2_NW_EPT8>(prm, grid, smem, st);
        }
    } else if (prm.E) {
        switch (ept) {
            case 1: return launch_pair<double, 1>(prm, grid, smem, st);
            case 2: return launch_pair<double, 2>(prm, grid, smem, st);
            case 4: return launch_pair<double, 4>(prm, grid, smem, st);
        }
    } else {      // E == NULL: potential only (Eq. 4 is the potential alone)
        switch (ept) {
            case 1: return launch_pair<double, 1, false>(prm, grid, smem, st);
            case 2: return launch_pair<double, 2, false>(prm, grid, smem, st);
            case 4: return launch_pair<double, 4, false>(prm, grid, smem, st);
        }
    }
    return cudaErrorInvalidValue;
}

template <int EP2, int NW, bool NODEPACK = false, bool FULL = false, bool DZT = false, int FINE = -1,
          bool VONLY = false, bool ACCV = false>
cudaError_t launch_grid_f32(const PairParams &prm, dim3 grid, size_t smem, cudaStream_t st) {
    if constexpr (!NODEPACK && !FULL) {            // every warp its own point group: no z split
        if constexpr (EP2 == 2 && NW == GRID_NW_EPT4) {
            // E = NULL: the potential alone (Eq. 4), 6 instead of 8 operations per pair
            if (prm.point_warps == NW && prm.g_dzt && !prm.E)
                return launch_grid_f32<EP2, NW, false, true, true, 0, true>(prm, grid, smem, st);
            if (prm.point_warps == NW && prm.g_dzt && prm.g_accv)
                return launch_grid_f32<EP2, NW, false, true, true, 0, false, true>(prm, grid, smem, st);
        }
        if constexpr (EP2 == 2 && (NW == GRID_NW_EPT4 || NW == GRID_NW_EPT4_LIGHT)) {
            // (the dz-table kernels work from the point's true position: no lattice to refine)
            if (prm.point_warps == NW && prm.g_dzt)
                return launch_grid_f32<EP2, NW, false, true, true, 0>(prm, grid, smem, st);
        }
        if (prm.point_warps == NW)
            return prm.g_fine ? launch_grid_f32<EP2, NW, false, true, false, 1>(prm, grid, smem, st)
                              : launch_grid_f32<EP2, NW, false, true, false, 0>(prm, grid, smem, st);
        if constexpr (EP2 == 2 && !DZT && (NW == GRID_NW_EPT4 || NW == GRID_NW_EPT4_LIGHT)) {
            // few-point plans (z-split warps): the same table and true-point walk
            if (prm.g_dzt) return launch_grid_f32<EP2, NW, false, false, true>(prm, grid, smem, st);
        }
    }
    auto kern = grid_kernel_f32x2<EP2, NW, NODEPACK, FULL, DZT, FINE, VONLY, ACCV>;
    static SmemConfig configured;
    static const char *const name = kernel_name(reinterpret_cast<const void *>(kern));
    g_launched = name;
    cudaError_t e = configured.ensure(kern, smem);
    if (e != cudaSuccess) return e;
    return launch_eval_kernel(kern, grid, 32 * NW, smem, st, prm);
}
template <int EPT, bool WITH_E, int NW, bool WARPOWN = false, bool DZT = false>
cudaError_t launch_grid_f64(const PairParams &prm, dim3 grid, size_t smem, cudaStream_t st) {
    auto kern = grid_kernel_f64<EPT, WITH_E, NW, WARPOWN, DZT>;
    static SmemConfig configured;
    static const char *const name = kernel_name(reinterpret_cast<const void *>(kern));
    g_launched = name;
    cudaError_t e = configured.ensure(kern, smem);
    if (e != cudaSuccess) return e;
    return launch_eval_kernel(kern, grid, 32 * (NW + 1), smem, st, prm);
}
// Grid layout: FP32-acc64 packed kernel for 2, 4, 8 points per thread; FP64 for 1, 2, 4.
cudaError_t launch_grid_ept(bool f32, int ept, const PairParams &prm, dim3 grid, size_t smem,
                            cudaStream_t st) {
    if (f32) {
        switch (ept) {
            case 2:
                if (grid_f32_nodepack(2, prm.P))
                    return prm.g_light ? launch_grid_f32<1, GRID_NW_NODEPACK_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f32<1, GRID_NW_NODEPACK, true>(prm, grid, smem, st);
                return launch_grid_f32<1, GRID_NW_EPT2>(prm, grid, smem, st);
            case 4:
                if (prm.g_light) return launch_grid_f32<2, GRID_NW_EPT4_LIGHT>(prm, grid, smem, st);
                return launch_grid_f32<2, GRID_NW_EPT4>(prm, grid, smem, st);
            case 8: return launch_grid_f32<4, GRID_NW_EPT8>(prm, grid, smem, st);
        }
    } else if (prm.E) {
        switch (ept) {
            case 1:
                if (grid_f64_warpown(1, prm.P))
                    return prm.g_light ? launch_grid_f64<1, true, GRID64_NW_WARPOWN_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f64<1, true, GRID64_NW_WARPOWN, true>(prm, grid, smem, st);
                return launch_grid_f64<1, true, GRID64_NW_EPT1>(prm, grid, smem, st);
            case 2:
                if (grid_f64_warpown(2, prm.P))
                    return prm.g_light ? launch_grid_f64<2, true, GRID64_NW_WARPOWN_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f64<2, true, GRID64_NW_WARPOWN, true>(prm, grid, smem, st);
                return launch_grid_f64<2, true, GRID64_NW_EPT2>(prm, grid, smem, st);
            case 4:
                if (grid_f64_warpown(4, prm.P))
                    return prm.g_light ? launch_grid_f64<4, true, GRID64_NW_WARPOWN_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f64<4, true, GRID64_NW_WARPOWN, true>(prm, grid, smem, st);
                if (prm.g_light)
                    return prm.g_dzt ? launch_grid_f64<4, true, GRID64_NW_LIGHT, false, true>(prm, grid, smem, st)
                                     : launch_grid_f64<4, true, GRID64_NW_LIGHT>(prm, grid, smem, st);
                if (prm.g_dzt) return launch_grid_f64<4, true, GRID64_NW_EPT4, false, true>(prm, grid, smem, st);
                return launch_grid_f64<4, true, GRID64_NW_EPT4>(prm, grid, smem, st);
        }
    } else {
        switch (ept) {
            case 1:
                if (grid_f64_warpown(1, prm.P))
                    return prm.g_light ? launch_grid_f64<1, false, GRID64_NW_WARPOWN_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f64<1, false, GRID64_NW_WARPOWN, true>(prm, grid, smem, st);
                return launch_grid_f64<1, false, GRID64_NW_EPT1>(prm, grid, smem, st);
            case 2:
                if (grid_f64_warpown(2, prm.P))
                    return prm.g_light ? launch_grid_f64<2, false, GRID64_NW_WARPOWN_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f64<2, false, GRID64_NW_WARPOWN, true>(prm, grid, smem, st);
                return launch_grid_f64<2, false, GRID64_NW_EPT2>(prm, grid, smem, st);
            case 4:
                if (grid_f64_warpown(4, prm.P))
                    return prm.g_light ? launch_grid_f64<4, false, GRID64_NW_WARPOWN_LIGHT, true>(prm, grid, smem, st)
                                       : launch_grid_f64<4, false, GRID64_NW_WARPOWN, true>(prm, grid, smem, st);
                if (prm.g_light)
                    return prm.g_dzt ? launch_grid_f64<4, false, GRID64_NW_LIGHT, false, true>(prm, grid, smem, st)
                                     : launch_grid_f64<4, false, GRID64_NW_LIGHT>(prm, grid, smem, st);
                if (prm.g_dzt) return launch_grid_f64<4, false, GRID64_NW_EPT4, false, true>(prm, grid, smem, st);
                return launch_grid_f64<4, false, GRID64_NW_EPT4>(prm, grid, smem, st);
        }
    }
    return cudaErrorInvalidValue;
}

bool is_device_pointer(const void *p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// Returns a device pointer holding n doubles of src (copying when src is a host pointer).
cudaError_t to_device(const double *src, int64_t n, double **dev, bool *owned) {
    *owned = false;
    *dev = nullptr;
    if (n == 0) return cudaSuccess;
    if (is_device_pointer(src)) {
        *dev = const_cast<double *>(src);
        return cudaSuccess;
    }
    cudaError_t e = cudaMalloc(dev, n * sizeof(double));
    if (e != cudaSuccess) return e;
    *owned = true;
    return cudaMemcpy(*dev, src, n * sizeof(double), cudaMemcpyHostToDevice);
}


// Power of two 2^k with 2^k * max|q| in [0.5, 1) (1 when all charges are zero): the scale of the
// cell charges in the FP32 copies (PairParams::q_unscale).
cudaError_t charge_scale(const double *dq, int64_t n, double *scale) {
    *scale = 1.0;
    if (n <= 0) return cudaSuccess;
    unsigned long long *dmax = nullptr, hmax = 0;
    cudaError_t e = cudaMalloc(&dmax, sizeof(hmax));
    if (e == cudaSuccess) e = cudaMemset(dmax, 0, sizeof(hmax));
    if (e == cudaSuccess) {
        absmax_kernel<<<static_cast<unsigned>(std::min<int64_t>(1024, (n + 255) / 256)), 256>>>(dq, n, dmax);
        e = cudaMemcpy(&hmax, dmax, sizeof(hmax), cudaMemcpyDeviceToHost);
    }
    cudaFree(dmax);
    if (e != cudaSuccess) return e;
    double m;
    std::memcpy(&m, &hmax, 8);
    if (m > 0.0 && std::isfinite(m)) {
        int ex = 0;
        std::frexp(m, &ex);                       // m = f * 2^ex, 0.5 <= f < 1
        ex = std::max(-1000, std::min(1000, ex));
        *scale = std::ldexp(1.0, -ex);
    }
    return cudaSuccess;
}

// ------------------------------------------------------------------ grid layout (8(f)-1)
// Packs dense charges [nx][ny][nz] (device) into the FP32 and FP64 gchunk copies and converts
// the packed nuclei (h->nuclei) to grid units.
cudaError_t build_grid(qmmm_field *h, const double *ddense, const GridGeom &gg) {
    h->grid = gg;
    h->g_rows = static_cast<int64_t>(gg.n[0]) * gg.n[1];
    h->g_tiles = (h->g_rows + 31) / 32;
    h->g_segs = (gg.n[2] + GRID_ZS - 1) / GRID_ZS;
    h->n_g = h->g_tiles * h->g_segs;
    if (h->n_g < 1 || h->n_g > (int64_t(1) << 30)) return cudaErrorInvalidValue;
    const int64_t rows_padded = h->g_tiles * 32;
    cudaError_t e = cudaMalloc(&h->gcells32, h->n_g * GRID_NODES * sizeof(float));
    if (e == cudaSuccess) e = cudaMalloc(&h->gcells64, h->n_g * GRID_NODES * sizeof(double));
    if (e != cudaSuccess) return e;
    const unsigned nb = static_cast<unsigned>((rows_padded + 63) / 64);
    grid_pack_kernel<float><<<nb, 64>>>(ddense, h->g_rows, gg.n[2], static_cast<int>(h->g_segs),
                                        rows_padded, h->q_scale, h->gcells32);
    grid_pack_kernel<double><<<nb, 64>>>(ddense, h->g_rows, gg.n[2], static_cast<int>(h->g_segs),
                                         rows_padded, 1.0, h->gcells64);
    if (h->K > 0) {
        e = cudaMalloc(&h->nuclei_u, h->K * 4 * sizeof(double));
        if (e != cudaSuccess) return e;
        grid_nuclei_kernel<<<static_cast<unsigned>((h->K + 255) / 256), 256>>>(h->nuclei, h->K, gg,
                                                                              h->nuclei_u);
    }
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e == cudaSuccess) h->has_grid = true;
    return e;
}

// Are the cells nodes of a regular (orthorhombic) grid ("spatially discretized
// cell")?  Candidate spacing per axis from the smallest positive coordinate step between
// consecutive sources, node counts from the bounding box, then EVERY source is checked against its node (within a few
// ulp of the coordinates) and no node may hold two sources.  Anything else keeps the list.
cudaError_t detect_grid(qmmm_field *h, const double *dxyz, const double *dq, int64_t M) {
    if (M < 4096) return cudaSuccess;
    const int nb = static_cast<int>(std::min<int64_t>(256, (M + 255) / 256));
    double *dpart = nullptr;
    cudaError_t e = cudaMalloc(&dpart, 256 * 3 * sizeof(double));
    if (e != cudaSuccess) return e;
    double hpart[256 * 3];
    grid_spacing_kernel<<<nb, 256>>>(dxyz, M, dpart);
    e = cudaMemcpy(hpart, dpart, nb * 3 * sizeof(double), cudaMemcpyDeviceToHost);
    cudaFree(dpart);
    if (e != cudaSuccess) return e;
    GridGeom gg;
    double hcand[3], ext[3], maxabs = 0.0;
    int best = -1;
    for (int k = 0; k < 3; ++k) {
        hcand[k] = 1e300;
        for (int b = 0; b < nb; ++b) hcand[k] = std::min(hcand[k], hpart[3 * b + k]);
        ext[k] = h->bb_hi[k] - h->bb_lo[k];
        maxabs = std::max({maxabs, std::fabs(h->bb_lo[k]), std::fabs(h->bb_hi[k]), ext[k]});
        gg.org[k] = h->bb_lo[k];
        gg.n[k] = 1;
        if (ext[k] > 0.0) {
            if (!(hcand[k] < 1e299)) return cudaSuccess;
            const double nn = std::rint(ext[k] / hcand[k]) + 1.0;
            if (!(nn >= 2.0 && nn <= 65536.0)) return cudaSuccess;
            gg.n[k] = static_cast<int>(nn);
            if (best < 0 || gg.n[k] > gg.n[best]) best = k;
        }
    }
    if (best < 0) return cudaSuccess;
    // spacing per axis (orthorhombic cells; a flat axis takes the spacing of the finest one)
    for (int k = 0; k < 3; ++k)
        gg.h[k] = gg.n[k] > 1 ? ext[k] / (gg.n[k] - 1) : ext[best] / (gg.n[best] - 1);
    for (int k = 0; k < 3; ++k)             // cubic cells: one spacing, bit for bit
        if (std::fabs(gg.h[k] - gg.h[best]) <= 1e-14 * gg.h[best]) gg.h[k] = gg.h[best];
    gg.tol = 16.0 * 2.220446049250313e-16 * maxabs;
    const double total = static_cast<double>(gg.n[0]) * gg.n[1] * gg.n[2];
    if (total > 2.0 * static_cast<double>(M) + 65536.0 || total > 2.0e9) return cudaSuccess;   // too sparse
    {
        const double hmin = std::min({gg.h[0], gg.h[1], gg.h[2]}), hmax = std::max({gg.h[0], gg.h[1], gg.h[2]});
        if (hmax > 16.0 * hmin) return cudaSuccess;     // needle-shaped cells: keep the list
    }
    const int64_t ntot = static_cast<int64_t>(total);
    double *ddense = nullptr;
    int *dcount = nullptr;
    e = cudaMalloc(&ddense, ntot * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&dcount, (ntot + 2) * sizeof(int));
    if (e == cudaSuccess) e = cudaMemset(ddense, 0, ntot * sizeof(double));
    if (e == cudaSuccess) e = cudaMemset(dcount, 0, (ntot + 2) * sizeof(int));
    int bad[2] = {1, 1};
    if (e == cudaSuccess) {
        grid_scatter_kernel<<<static_cast<unsigned>((M + 255) / 256), 256>>>(dxyz, dq, M, gg, ddense,
                                                                            dcount + 2, dcount);
        e = cudaMemcpy(bad, dcount, sizeof(bad), cudaMemcpyDeviceToHost);
    }
    if (e == cudaSuccess && bad[0] == 0 && bad[1] == 0) e = build_grid(h, ddense, gg);
    cudaFree(ddense);
    cudaFree(dcount);
    if (e == cudaErrorMemoryAllocation) {      // no room for the extra copies: keep the list only
        cudaGetLastError();
        cudaFree(h->gcells32); h->gcells32 = nullptr;
        cudaFree(h->gcells64); h->gcells64 = nullptr;
        cudaFree(h->nuclei_u); h->nuclei_u = nullptr;
        h->has_grid = false;
        return cudaSuccess;
    }
    return e;
}

}  // namespace

namespace {

// Grid layout: cells as charges only, coordinates from the indices; everything in grid units.
void fill_grid_params(qmmm_field *h, PairParams &prm, bool f32) {
    prm.chunks = f32 ? reinterpret_cast<const char *>(h->gcells32)
                     : reinterpret_cast<const char *>(h->gcells64);
    prm.n_chunks = static_cast<int>(h->n_g);
    prm.nuc = h->nuclei_u;
    prm.K = static_cast<int>(h->K);
    for (int k = 0; k < 3; ++k) prm.g_org[k] = h->grid.org[k];
    for (int k = 0; k < 3; ++k) prm.g_inv_h[k] = 1.0 / h->grid.h[k];
    prm.g_sx = h->grid.h[0] / h->grid.h[2];        // exactly 1 for cubic cells
    prm.g_sy = h->grid.h[1] / h->grid.h[2];
    prm.g_ortho = (prm.g_sx != 1.0 || prm.g_sy != 1.0) ? 1 : 0;
    prm.g_scaleV = 1.0 / h->grid.h[2];
    prm.g_scaleE = 1.0 / (h->grid.h[2] * h->grid.h[2]);
    for (int k = 0; k < 3; ++k) prm.g_n[k] = h->grid.n[k];
    prm.g_segs = static_cast<int>(h->g_segs);
    // FP32: the whole-grid lattice quantum is 2^-24 of the axis (in nodes); beyond 128 nodes
    // the field of cells next to a point would lose accuracy (qmmm_grid.cuh, on_lattice)
    const int nmax = std::max({h->grid.n[0], h->grid.n[1], h->grid.n[2]});
    prm.g_fine = (f32 && (h->local_lattice == 1 || (h->local_lattice < 0 && nmax > 128))) ? 1 : 0;
    h->last_local_lattice = prm.g_fine;
}

// ------------------------------------------------------------------ resident move server
double now_seconds() {
    struct timespec t;
    clock_gettime(CLOCK_MONOTONIC, &t);
    return t.tv_sec + 1e-9 * t.tv_nsec;
}

// Host side of the request seqlock: seq_a, then r, then seq_b (program order = store order on x86).
void post_request(ServerMailbox *m, unsigned long long s, const double *r) {
    m->req[0] = s;
    std::atomic_thread_fence(std::memory_order_release);
    if (r)
        for (int i = 0; i < 3; ++i) {
            unsigned long long bits;
            std::memcpy(&bits, r + i, 8);
            m->req[1 + i] = bits;
        }
    std::atomic_thread_fence(std::memory_order_release);
    m->req[4] = s;
}

// One resident move server per device, and only while a single handle is making host-path
// evaluations there: a server occupies every SM, so the servers (and the launch-path kernels)
// of other handles on the same device would queue behind it for up to its lifetime.  A handle
// that finds another handle's server resident asks it to yield (request word 5; the leader
// retires after the move in flight), marks the device contended for a while, and uses the
// launch path; contended handles do not start servers.
struct DeviceServers {
    std::mutex mu;
    std::atomic<qmmm_field *> owner{nullptr};   // handle whose server is resident (or starting)
    qmmm_field *last_host = nullptr;    // handle of the most recent host-path evaluation
    double last_host_t = 0.0, contended_until = 0.0;
};
DeviceServers g_servers[MAX_DEVICES];
constexpr double CONTENDED_S = 0.05;

// Called by every evaluation that launches kernels: a resident server of ANOTHER handle on
// this device is asked to retire (its owner restarts it when the device is quiet again).
void yield_foreign_server(qmmm_field *h) {
    DeviceServers &ds = g_servers[h->device];
    qmmm_field *o = ds.owner.load(std::memory_order_acquire);
    if (o == nullptr || o == h) return;                      // re-checked under the lock
    std::lock_guard<std::mutex> lk(ds.mu);
    o = ds.owner.load();
    if (o && o != h && o->srv_mail_h) {
        o->srv_mail_h->req[5] = 1;
        ds.contended_until = now_seconds() + CONTENDED_S;
    }
}
// Host-path evaluation by h: two different handles within CONTENDED_S = contention.
void note_host_eval(qmmm_field *h) {
    DeviceServers &ds = g_servers[h->device];
    std::lock_guard<std::mutex> lk(ds.mu);
    const double t = now_seconds();
    if (ds.last_host && ds.last_host != h && t - ds.last_host_t < CONTENDED_S) ds.contended_until = t + CONTENDED_S;
    ds.last_host = h;
    ds.last_host_t = t;
}
void server_retired(qmmm_field *h) {
    DeviceServers &ds = g_servers[h->device];
    std::lock_guard<std::mutex> lk(ds.mu);
    if (ds.owner.load() == h) ds.owner = nullptr;
    h->srv_alive = false;
}
void forget_handle(qmmm_field *h) {              // destroy
    DeviceServers &ds = g_servers[h->device];
    std::lock_guard<std::mutex> lk(ds.mu);
    if (ds.owner.load() == h) ds.owner = nullptr;
    if (ds.last_host == h) ds.last_host = nullptr;
}

// Waits until the server launch `h->srv_launch_id` has retired, then joins its stream.
qmmm_status server_join(qmmm_field *h) {
    const double t0 = now_seconds();
    while (h->srv_mail_h->exited != h->srv_launch_id) {
        if (cudaStreamQuery(h->srv_stream) != cudaErrorNotReady) break;     // ended (or failed)
        if (now_seconds() - t0 > 10.0) return fail(QMMM_ERR_CUDA, "move server did not retire");
    }
    CUDA_TRY(cudaStreamSynchronize(h->srv_stream));
    server_retired(h);
    return QMMM_OK;
}

// Retires a running server (any other use of the handle's workspace must do this first).
qmmm_status server_stop(qmmm_field *h) {
    if (!h->srv_alive) return QMMM_OK;
    post_request(h->srv_mail_h, SERVER_EXIT, nullptr);
    qmmm_status st = server_join(h);
    post_request(h->srv_mail_h, h->srv_seq, nullptr);
    return st;
}

template <typename REAL>
cudaError_t server_launch(const ServerParams &sp, int slices, size_t smem, cudaStream_t st) {
    auto kern = move_server_kernel<REAL>;
    static SmemConfig configured;
    static const char *const name = kernel_name(reinterpret_cast<const void *>(kern));
    g_launched = name;
    cudaError_t e = configured.ensure(kern, smem);
    if (e != cudaSuccess) return e;
    void *args[] = {const_cast<ServerParams *>(&sp)};
    return cudaLaunchCooperativeKernel(reinterpret_cast<void *>(kern), dim3(1, slices),
                                       dim3(CTA_THREADS), args, smem, st);
}

template <bool F32>
cudaError_t server_grid_launch(const ServerParams &sp, int slices, size_t smem, cudaStream_t st) {
    auto kern = move_server_grid_kernel<F32>;
    static SmemConfig configured;
    static const char *const name = kernel_name(reinterpret_cast<const void *>(kern));
    g_launched = name;
    cudaError_t e = configured.ensure(kern, smem);
    if (e != cudaSuccess) return e;
    void *args[] = {const_cast<ServerParams *>(&sp)};
    return cudaLaunchCooperativeKernel(reinterpret_cast<void *>(kern), dim3(1, slices),
                                       dim3(32 * SERVER_GRID_NW), args, smem, st);
}

// Starts the server for `prec`; *usable = false when this problem cannot be served (the
// caller then uses the launch path).
qmmm_status server_start(qmmm_field *h, int prec, bool *usable) {
    const bool f32 = prec == QMMM_FP32_ACC64;
    *usable = false;
    // the grid-aware server when the handle has the compact copy (and LIST is not forced), else
    // the source-list server
    const bool grid = h->has_grid && h->layout != QMMM_LAYOUT_LIST;
    const int64_t n_chunks = grid ? h->n_g : (f32 ? h->n_chunks : h->n_chunks64);
    if (!h->srv_ok || n_chunks < 1 || h->timing || (!grid && !h->has_list)) return QMMM_OK;
    qmmm_plan pl = choose_plan(h, 1, f32);
    size_t smem = 0;
    if (grid) {
        pl.points_per_thread = 1;
        pl.point_warps = 1;
        pl.slices = static_cast<int>(std::min<int64_t>(h->sm_count, std::max<int64_t>(h->n_g, (h->K + 31) / 32)));
        pl.stages = f32 ? 2 : 1;
        smem = f32 ? ServerGridLayout<true>::total(pl.slices) : ServerGridLayout<false>::total(pl.slices);
        if (static_cast<int64_t>(pl.slices) * SLOT_WORDS > h->workspace_doubles) return QMMM_OK;
    } else {
        if (pl.points_per_thread != 1 || pl.point_warps != 1 || pl.slices > h->sm_count) return QMMM_OK;
    }
    const size_t extra = 128 + static_cast<size_t>(pl.slices) * 4 * sizeof(double);   // cmd, go, collected partials
    if (!grid) {
        smem = pair_smem_bytes(f32, pl.stages, 1, 1) + extra;
        while (smem > 227 * 1024 && pl.stages > 2) smem = pair_smem_bytes(f32, --pl.stages, 1, 1) + extra;
    }

    {
        // one resident server per device, and none while several handles make host-path calls
        DeviceServers &ds = g_servers[h->device];
        std::lock_guard<std::mutex> lk(ds.mu);
        qmmm_field *o = ds.owner.load();
        if (o && o != h) {
            if (o->srv_mail_h) o->srv_mail_h->req[5] = 1;
            ds.contended_until = now_seconds() + CONTENDED_S;
            return QMMM_OK;
        }
        if (now_seconds() < ds.contended_until) return QMMM_OK;
        ds.owner = h;
        h->srv_mail_h->req[5] = 0;
    }
    g_device = h->device;
    ServerParams sp;
    std::memset(&sp, 0, sizeof(sp));
    PairParams &prm = sp.pair;
    prm.partial = h->workspace;
    prm.P = 1;
    prm.n_chunks = static_cast<int>(n_chunks);
    prm.slices = pl.slices;
    prm.point_warps = 1;
    prm.stages = pl.stages;
    prm.q_unscale = f32 ? 1.0 / h->q_scale : 1.0;
    prm.counters = h->counters;
    prm.dev_err = h->dev_err_d;
    if (grid) {
        fill_grid_params(h, prm, f32);
    } else {
        prm.chunks = f32 ? reinterpret_cast<const char *>(h->chunks32)
                         : reinterpret_cast<const char *>(h->chunks64);
        prm.origins = h->origins;
        prm.lattice = h->lattice;
        prm.inv_lattice = 1.0 / h->lattice;
        prm.nuc = h->nuclei;
        prm.K = f32 ? static_cast<int>(h->K) : 0;
    }
    sp.mail = h->srv_mail_d;
    sp.dev = h->srv_dev;
    sp.start_seq = h->srv_seq;
    sp.launch_id = ++h->srv_launch_id;
    post_request(h->srv_mail_h, h->srv_seq, nullptr);
    ServerDevice init;
    std::memset(&init, 0, sizeof(init));
    for (int u = 0; u < 3; ++u) init.rec[2 * u] = h->srv_seq;       // tags of the last answered move
    {
        cudaError_t e0 = cudaMemcpy(h->srv_dev, &init, sizeof(init), cudaMemcpyHostToDevice);
        if (e0 == cudaSuccess)
            e0 = cudaMemset(h->workspace, 0, static_cast<size_t>(pl.slices) * SLOT_WORDS * 8);   // untagged slots
        if (e0 != cudaSuccess) {
            server_retired(h);
            return cuda_fail(e0, "move server set-up");
        }
    }
    cudaError_t e = grid ? (f32 ? server_grid_launch<true>(sp, pl.slices, smem, h->srv_stream)
                                : server_grid_launch<false>(sp, pl.slices, smem, h->srv_stream))
                         : (f32 ? server_launch<float>(sp, pl.slices, smem, h->srv_stream)
                                : server_launch<double>(sp, pl.slices, smem, h->srv_stream));
    if (e != cudaSuccess) {                    // e.g. the GPU is shared and cannot hold the grid
        cudaGetLastError();
        h->srv_ok = false;
        server_retired(h);
        return QMMM_OK;
    }
    h->srv_alive = true;
    h->last_kernel = g_launched;
    h->last_layout = grid ? QMMM_LAYOUT_GRID : QMMM_LAYOUT_LIST;
    h->srv_prec = prec;
    h->last_plan = pl;
    h->last_point_blocks = 1;
    h->last_launches = 0;
    *usable = true;
    return QMMM_OK;
}

// One move through the server.  *served = false: the caller must use the launch path.
qmmm_status server_move(qmmm_field *h, const double *r, double *V, double *E, int prec,
                        bool *served) {
    *served = false;
    if (h->srv_alive && h->srv_prec != prec) {
        qmmm_status st = server_stop(h);
        if (st != QMMM_OK) return st;
    }
    if (!h->srv_alive) {
        bool usable = false;
        qmmm_status st = server_start(h, prec, &usable);
        if (st != QMMM_OK) return st;
        if (!usable) return QMMM_OK;
    }
    ServerMailbox *m = h->srv_mail_h;
    const unsigned long long s = ++h->srv_seq;
    post_request(m, s, r);
    const double t0 = now_seconds();
    auto answered = [&]() { return m->ans[0] == s && m->ans[2] == s && m->ans[4] == s && m->ans[6] == s; };
    for (uint64_t spin = 1; !answered(); ++spin) {
        if (m->exited == h->srv_launch_id) {
            // the server retired (idle / lifetime) before taking this move: start a new one,
            // the request stays posted
            CUDA_TRY(cudaStreamSynchronize(h->srv_stream));
            server_retired(h);
            if (answered()) break;
            --h->srv_seq;                              // server_start reposts seq_req = srv_seq
            bool usable = false;
            qmmm_status st = server_start(h, prec, &usable);
            ++h->srv_seq;
            if (st != QMMM_OK) return st;
            if (!usable) return QMMM_OK;               // fall back to the launch path
            post_request(m, s, r);
        }
        if ((spin & 0xFFFFF) == 0 && now_seconds() - t0 > 10.0)
            return fail(QMMM_ERR_CUDA, "move server did not answer");
    }
    std::atomic_thread_fence(std::memory_order_acquire);
    unsigned long long bits[4] = {m->ans[1], m->ans[3], m->ans[5], m->ans[7]};
    std::atomic_thread_fence(std::memory_order_acquire);
    if (!answered())
        return fail(QMMM_ERR_CUDA, "move server: answer line changed while it was read");
    std::memcpy(V, &bits[0], 8);
    if (E) std::memcpy(E, &bits[1], 24);
    *served = true;
    return QMMM_OK;
}

}  // namespace

namespace {
// From here on the source copies are owned by a shared SourceOwner (qmmm_field_share).
void adopt_sources(qmmm_field *h) {
    h->keep = std::make_shared<SourceOwner>();
    void *p[7] = {h->chunks64, h->chunks32, h->origins, h->nuclei, h->gcells32, h->gcells64, h->nuclei_u};
    for (int i = 0; i < 7; ++i) h->keep->ptr[i] = p[i];
}

// Per-handle buffers that do not depend on the source format: partials workspace, tickets,
// mailboxes, move-server state, eval_host staging.
qmmm_status alloc_runtime(qmmm_field *h) {
#define RT_TRY(expr)                                                                       \
    do {                                                                                   \
        cudaError_t _e = (expr);                                                           \
        if (_e == cudaErrorMemoryAllocation)                                               \
            return fail(QMMM_ERR_ALLOC, std::string(#expr) + ": out of memory");           \
        if (_e != cudaSuccess) return cuda_fail(_e, #expr);                                \
    } while (0)
    // Partials workspace: slices * P * 4 doubles.  With P = h->max_points the automatic plan
    // uses at most sm_count slices; small P uses more slices but a smaller product.
    h->workspace_doubles =
        4 * std::max<int64_t>(static_cast<int64_t>(h->sm_count) * h->max_points, int64_t(1) << 16);
    RT_TRY(cudaMalloc(&h->workspace, h->workspace_doubles * sizeof(double)));
    RT_TRY(cudaMalloc(&h->counters, (h->max_points + 1) * sizeof(int)));      // + 1: mailbox `done`
    RT_TRY(cudaMemset(h->counters, 0, (h->max_points + 1) * sizeof(int)));
    RT_TRY(cudaMalloc(&h->push_slots, PUSH_MAX_RECORDS * PUSH_SLOT_WORDS * sizeof(unsigned long long)));
    RT_TRY(cudaMemset(h->push_slots, 0, PUSH_MAX_RECORDS * PUSH_SLOT_WORDS * sizeof(unsigned long long)));
    RT_TRY(cudaHostAlloc(&h->mail_h, (MAIL_REC_OFFSET + MAIL_POINTS * 8) * sizeof(double), cudaHostAllocMapped));
    std::memset(h->mail_h, 0, (MAIL_REC_OFFSET + MAIL_POINTS * 8) * sizeof(double));
    RT_TRY(cudaHostGetDevicePointer(&h->mail_d, h->mail_h, 0));
    RT_TRY(cudaHostAlloc(&h->srv_mail_h, sizeof(ServerMailbox), cudaHostAllocMapped));
    std::memset(h->srv_mail_h, 0, sizeof(ServerMailbox));
    RT_TRY(cudaHostGetDevicePointer(&h->srv_mail_d, h->srv_mail_h, 0));
    RT_TRY(cudaMalloc(&h->srv_dev, sizeof(ServerDevice)));
    RT_TRY(cudaStreamCreateWithFlags(&h->srv_stream, cudaStreamNonBlocking));
    {
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device);
        h->srv_ok = coop != 0;
    }
    RT_TRY(cudaHostAlloc(&h->dev_err_h, 64, cudaHostAllocMapped));
    std::memset(h->dev_err_h, 0, 64);
    RT_TRY(cudaHostGetDevicePointer(&h->dev_err_d, h->dev_err_h, 0));
    RT_TRY(cudaMalloc(&h->stage_elec, h->max_points * 3 * sizeof(double)));
    RT_TRY(cudaMalloc(&h->stage_out, h->max_points * 4 * sizeof(double)));
#undef RT_TRY
    return QMMM_OK;
}

}  // namespace

// =============================================================================== C ABI
extern "C" {

const char *qmmm_last_error(void) { return g_last_error.c_str(); }

qmmm_status qmmm_field_create(const double *src_xyz, const double *src_q, int64_t M,
                              const double *nuc_xyz, const double *nuc_Z, int64_t K,
                              int64_t max_points, qmmm_field **out) {
    if (!out) return fail(QMMM_ERR_INVALID_ARG, "create: out is NULL");
    *out = nullptr;
    if (M < 0 || K < 0) return fail(QMMM_ERR_INVALID_ARG, "create: negative M or K");
    if (max_points < 1 || max_points > INT_MAX)
        return fail(QMMM_ERR_INVALID_ARG, "create: max_points must be in [1, 2^31 - 1]");
    if (M > 0 && (!src_xyz || !src_q))
        return fail(QMMM_ERR_INVALID_ARG, "create: NULL source array with M > 0");
    if (K > 0 && (!nuc_xyz || !nuc_Z))
        return fail(QMMM_ERR_INVALID_ARG, "create: NULL nuclear array with K > 0");
    if (M > (int64_t(1) << 37)) return fail(QMMM_ERR_INVALID_ARG, "create: M too large");

    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(QMMM_ERR_UNSUPPORTED_DEVICE,
                    "create: device is sm_" + std::to_string(prop.major * 10 + prop.minor) +
                        ", this library is built for sm_100a (B200) only");

    qmmm_field *h = new (std::nothrow) qmmm_field();
    if (!h) return fail(QMMM_ERR_ALLOC, "create: host allocation failed");
    h->M = M; h->K = K; h->max_points = max_points;
    h->device = dev; h->sm_count = prop.multiProcessorCount;
    h->n_chunks = (M + CHUNK - 1) / CHUNK;                 // FP32 copy: cells only
    h->n_chunks64 = (M + K + CHUNK - 1) / CHUNK;           // FP64 copy: cells + nuclei
    h->n_blocks = (h->n_chunks + BLOCK_CHUNKS - 1) / BLOCK_CHUNKS;

    auto bail = [&](qmmm_status st) { qmmm_field_destroy(h); return st; };
#define CREATE_TRY(expr)                                                               \
    do {                                                                               \
        cudaError_t _e = (expr);                                                       \
        if (_e != cudaSuccess)                                                         \
            return bail(_e == cudaErrorMemoryAllocation                                \
                            ? fail(QMMM_ERR_ALLOC, std::string(#expr) + ": out of memory") \
                            : cuda_fail(_e, #expr));                                   \
    } while (0)

    {
        // device copies of the caller's arrays (no copy when they already are device pointers)
        double *dxyz = nullptr, *dq = nullptr, *dnxyz = nullptr, *dnz = nullptr;
        bool own[4] = {false, false, false, false};
        cudaError_t e = to_device(src_xyz, 3 * M, &dxyz, &own[0]);
        if (e == cudaSuccess) e = to_device(src_q, M, &dq, &own[1]);
        if (e == cudaSuccess) e = to_device(nuc_xyz, 3 * K, &dnxyz, &own[2]);
        if (e == cudaSuccess) e = to_device(nuc_Z, K, &dnz, &own[3]);
        const int T = 256;
        if (e == cudaSuccess) e = charge_scale(dq, M, &h->q_scale);
        if (e == cudaSuccess && M + K > 0) {
            // FP64 copy: cells then nuclei, one SoA chunk array (the nuclei are ordinary FP64 sources)
            const int64_t Mpad = h->n_chunks64 * CHUNK;
            e = cudaMalloc(&h->chunks64, Mpad * 4 * sizeof(double));
            if (e == cudaSuccess)
                pack_f64_kernel<<<static_cast<unsigned>((Mpad + T - 1) / T), T>>>(
                    dxyz, dq, M, dnxyz, dnz, K, Mpad, h->chunks64);
        }
        if (e == cudaSuccess && K > 0) {
            // FP32 path: the nuclei stay FP64, packed x, y, z, Z
            e = cudaMalloc(&h->nuclei, K * 4 * sizeof(double));
            if (e == cudaSuccess)
                pack_nuclei_kernel<<<static_cast<unsigned>((K + T - 1) / T), T>>>(dnxyz, dnz, K, h->nuclei);
        }
        if (e == cudaSuccess && M > 0) {
            e = cudaMalloc(&h->chunks32, h->n_chunks * CHUNK * 4 * sizeof(float));
            if (e == cudaSuccess) e = cudaMalloc(&h->origins, h->n_blocks * 4 * sizeof(double));
            double *dbb = nullptr;
            if (e == cudaSuccess) e = cudaMalloc(&dbb, 256 * 6 * sizeof(double));
            if (e == cudaSuccess) {
                // coordinate lattice of the FP32 copy: the largest extent of the cells' bounding
                // box fits in 2^24 quanta, so d = a - o is exact for every point inside the box
                const int nbb = static_cast<int>(std::min<int64_t>(256, (M + 255) / 256));
                double hbb[256 * 6];
                bbox_kernel<<<nbb, 256>>>(dxyz, M, dbb);
                e = cudaMemcpy(hbb, dbb, nbb * 6 * sizeof(double), cudaMemcpyDeviceToHost);
                double ext = 0.0;
                for (int k = 0; k < 3 && e == cudaSuccess; ++k) {
                    double lo = hbb[k], hi = hbb[3 + k];
                    for (int b = 1; b < nbb; ++b) {
                        lo = std::min(lo, hbb[6 * b + k]);
                        hi = std::max(hi, hbb[6 * b + 3 + k]);
                    }
                    h->bb_lo[k] = lo;
                    h->bb_hi[k] = hi;
                    ext = std::max(ext, hi - lo);
                }
                if (!(ext > 0.0) || !std::isfinite(ext)) ext = 1.0;
                int ex2 = 0;
                std::frexp(ext, &ex2);                       // ext = m * 2^ex2, 0.5 <= m < 1
                h->lattice = std::ldexp(1.0, ex2 - 24);
            }
            if (dbb) cudaFree(dbb);
            if (e == cudaSuccess) {
                origins_kernel<<<static_cast<unsigned>((h->n_blocks * 32 + T - 1) / T), T>>>(
                    dxyz, M, h->n_blocks, h->lattice, h->origins);
                pack_f32_kernel<<<static_cast<unsigned>((h->n_chunks + 63) / 64), 64>>>(
                    dxyz, dq, M, h->n_chunks, h->origins, h->lattice, h->q_scale, h->chunks32);
            }
        }
        if (e == cudaSuccess) e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaDeviceSynchronize();
        // grid-aware compact copies when the cells are nodes of a cubic grid (8(f)-1)
        if (e == cudaSuccess && M > 0) e = detect_grid(h, dxyz, dq, M);
        if (own[0]) cudaFree(dxyz);
        if (own[1]) cudaFree(dq);
        if (own[2]) cudaFree(dnxyz);
        if (own[3]) cudaFree(dnz);
        CREATE_TRY(e);
    }
    {
        qmmm_status rs = alloc_runtime(h);
        if (rs != QMMM_OK) return bail(rs);
    }
#undef CREATE_TRY
    adopt_sources(h);
    *out = h;
    return QMMM_OK;
}

qmmm_status qmmm_field_create_grid3(const double *origin, const double *spacing, const int64_t *n,
                                    const double *cell_q, const double *nuc_xyz,
                                    const double *nuc_Z, int64_t K, int64_t max_points,
                                    qmmm_field **out) {
    if (!out) return fail(QMMM_ERR_INVALID_ARG, "create_grid: out is NULL");
    *out = nullptr;
    if (!origin || !n || !cell_q || !spacing)
        return fail(QMMM_ERR_INVALID_ARG, "create_grid: NULL origin, spacing, n or cell_q");
    for (int k = 0; k < 3; ++k)
        if (!(spacing[k] > 0.0) || !std::isfinite(spacing[k]))
            return fail(QMMM_ERR_INVALID_ARG, "create_grid: spacing must be positive and finite");
    for (int k = 0; k < 3; ++k)
        if (n[k] < 1 || n[k] > 65536) return fail(QMMM_ERR_INVALID_ARG, "create_grid: n[k] must be in [1, 65536]");
    const double total = static_cast<double>(n[0]) * n[1] * n[2];
    if (total > 2.0e9) return fail(QMMM_ERR_INVALID_ARG, "create_grid: more than 2e9 cells");
    if (K < 0) return fail(QMMM_ERR_INVALID_ARG, "create_grid: negative K");
    if (max_points < 1 || max_points > INT_MAX)
        return fail(QMMM_ERR_INVALID_ARG, "create_grid: max_points must be in [1, 2^31 - 1]");
    if (K > 0 && (!nuc_xyz || !nuc_Z))
        return fail(QMMM_ERR_INVALID_ARG, "create_grid: NULL nuclear array with K > 0");

    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10)
        return fail(QMMM_ERR_UNSUPPORTED_DEVICE,
                    "create_grid: device is sm_" + std::to_string(prop.major * 10 + prop.minor) +
                        ", this library is built for sm_100a (B200) only");
    qmmm_field *h = new (std::nothrow) qmmm_field();
    if (!h) return fail(QMMM_ERR_ALLOC, "create_grid: host allocation failed");
    h->K = K; h->max_points = max_points;
    h->device = dev; h->sm_count = prop.multiProcessorCount;
    h->has_list = false;
    auto bail = [&](qmmm_status st) { qmmm_field_destroy(h); return st; };

    const int64_t ntot = static_cast<int64_t>(total);
    GridGeom gg;
    for (int k = 0; k < 3; ++k) {
        gg.org[k] = origin[k];
        gg.n[k] = static_cast<int>(n[k]);
        h->bb_lo[k] = origin[k];
        h->bb_hi[k] = origin[k] + (n[k] - 1) * spacing[k];
        gg.h[k] = spacing[k];
    }
    gg.tol = 0.0;
    double *dq = nullptr, *dnxyz = nullptr, *dnz = nullptr;
    unsigned long long *dcnt = nullptr, cnt = 0;
    bool own[3] = {false, false, false};
    cudaError_t e = to_device(cell_q, ntot, &dq, &own[0]);
    if (e == cudaSuccess) e = to_device(nuc_xyz, 3 * K, &dnxyz, &own[1]);
    if (e == cudaSuccess) e = to_device(nuc_Z, K, &dnz, &own[2]);
    if (e == cudaSuccess && K > 0) {
        e = cudaMalloc(&h->nuclei, K * 4 * sizeof(double));
        if (e == cudaSuccess)
            pack_nuclei_kernel<<<static_cast<unsigned>((K + 255) / 256), 256>>>(dnxyz, dnz, K, h->nuclei);
    }
    if (e == cudaSuccess) e = cudaMalloc(&dcnt, sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(dcnt, 0, sizeof(unsigned long long));
    if (e == cudaSuccess) {
        grid_count_kernel<<<1024, 256>>>(dq, ntot, dcnt);
        e = cudaMemcpy(&cnt, dcnt, sizeof(cnt), cudaMemcpyDeviceToHost);
    }
    if (e == cudaSuccess) e = charge_scale(dq, ntot, &h->q_scale);
    if (e == cudaSuccess) e = build_grid(h, dq, gg);
    cudaFree(dcnt);
    if (own[0]) cudaFree(dq);
    if (own[1]) cudaFree(dnxyz);
    if (own[2]) cudaFree(dnz);
    if (e == cudaErrorMemoryAllocation) return bail(fail(QMMM_ERR_ALLOC, "create_grid: out of device memory"));
    if (e != cudaSuccess) return bail(cuda_fail(e, "create_grid"));
    h->M = static_cast<int64_t>(cnt);            // non-empty cells
    {
        qmmm_status rs = alloc_runtime(h);
        if (rs != QMMM_OK) return bail(rs);
    }
    adopt_sources(h);
    *out = h;
    return QMMM_OK;
}

qmmm_status qmmm_field_create_grid(const double *origin, double spacing, const int64_t *n,
                                   const double *cell_q, const double *nuc_xyz,
                                   const double *nuc_Z, int64_t K, int64_t max_points,
                                   qmmm_field **out) {
    const double s3[3] = {spacing, spacing, spacing};
    return qmmm_field_create_grid3(origin, s3, n, cell_q, nuc_xyz, nuc_Z, K, max_points, out);
}

qmmm_status qmmm_field_share(const qmmm_field *parent, int64_t max_points, qmmm_field **out) {
    if (!out) return fail(QMMM_ERR_INVALID_ARG, "share: out is NULL");
    *out = nullptr;
    if (!parent || !parent->keep) return fail(QMMM_ERR_INVALID_ARG, "share: NULL or incomplete parent handle");
    if (max_points < 1 || max_points > INT_MAX)
        return fail(QMMM_ERR_INVALID_ARG, "share: max_points must be in [1, 2^31 - 1]");
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev != parent->device)
        return fail(QMMM_ERR_INVALID_ARG, "share: the current device is not the parent handle's device");
    qmmm_field *h = new (std::nothrow) qmmm_field();
    if (!h) return fail(QMMM_ERR_ALLOC, "share: host allocation failed");
    // the immutable part: source copies, their geometry and sizes
    h->keep = parent->keep;
    h->M = parent->M; h->K = parent->K; h->max_points = max_points;
    h->n_chunks = parent->n_chunks; h->n_chunks64 = parent->n_chunks64; h->n_blocks = parent->n_blocks;
    h->device = parent->device; h->sm_count = parent->sm_count;
    h->chunks64 = parent->chunks64; h->chunks32 = parent->chunks32; h->origins = parent->origins;
    h->lattice = parent->lattice; h->nuclei = parent->nuclei; h->q_scale = parent->q_scale;
    h->has_list = parent->has_list; h->has_grid = parent->has_grid; h->grid = parent->grid;
    h->g_rows = parent->g_rows; h->g_tiles = parent->g_tiles; h->g_segs = parent->g_segs; h->n_g = parent->n_g;
    h->gcells32 = parent->gcells32; h->gcells64 = parent->gcells64; h->nuclei_u = parent->nuclei_u;
    h->layout = parent->layout;
    h->local_lattice = parent->local_lattice;
    h->accurate_v = parent->accurate_v;
    for (int k = 0; k < 3; ++k) { h->bb_lo[k] = parent->bb_lo[k]; h->bb_hi[k] = parent->bb_hi[k]; }
    // its own mutable part: workspace, tickets, mailboxes, move server, staging, plan
    qmmm_status rs = alloc_runtime(h);
    if (rs != QMMM_OK) {
        qmmm_field_destroy(h);
        return rs;
    }
    *out = h;
    return QMMM_OK;
}

qmmm_status qmmm_field_set_layout(qmmm_field *h, int layout) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "set_layout: NULL handle");
    if (layout != QMMM_LAYOUT_AUTO && layout != QMMM_LAYOUT_LIST && layout != QMMM_LAYOUT_GRID)
        return fail(QMMM_ERR_INVALID_ARG, "set_layout: unknown layout");
    if (layout == QMMM_LAYOUT_GRID && !h->has_grid)
        return fail(QMMM_ERR_INVALID_ARG, "set_layout: this environment has no grid copy (the cells are not nodes of a cubic grid)");
    if (layout == QMMM_LAYOUT_LIST && !h->has_list)
        return fail(QMMM_ERR_INVALID_ARG, "set_layout: this environment was created from a grid and has no source list");
    server_stop(h);
    h->layout = layout;
    return QMMM_OK;
}

qmmm_status qmmm_field_get_grid_info(const qmmm_field *h, qmmm_grid_info *info) {
    if (!h || !info) return fail(QMMM_ERR_INVALID_ARG, "get_grid_info: NULL argument");
    std::memset(info, 0, sizeof(*info));
    info->present = h->has_grid ? 1 : 0;
    info->has_list = h->has_list ? 1 : 0;
    info->layout = h->layout;
    info->last_layout = h->last_layout;
    if (h->has_grid) {
        for (int k = 0; k < 3; ++k) {
            info->n[k] = h->grid.n[k];
            info->origin[k] = h->grid.org[k];
        }
        info->spacing = h->grid.h[2];
        for (int k = 0; k < 3; ++k) info->spacing3[k] = h->grid.h[k];
        info->n_gchunks = h->n_g;
        info->bytes_fp32 = h->n_g * GRID_NODES * 4;
        info->bytes_fp64 = h->n_g * GRID_NODES * 8;
    }
    return QMMM_OK;
}

qmmm_status qmmm_field_destroy(qmmm_field *h) {
    if (!h) return QMMM_OK;
    server_stop(h);
    forget_handle(h);
    if (h->dev_err_h) cudaFreeHost(h->dev_err_h);
    if (h->srv_stream) cudaStreamDestroy(h->srv_stream);
    if (h->srv_mail_h) cudaFreeHost(h->srv_mail_h);
    cudaFree(h->srv_dev);
    if (!h->keep) {                 // a handle that failed before its sources were adopted
        cudaFree(h->chunks64);
        cudaFree(h->chunks32);
        cudaFree(h->origins);
        cudaFree(h->nuclei);
        cudaFree(h->gcells32);
        cudaFree(h->gcells64);
        cudaFree(h->nuclei_u);
    }
    h->keep.reset();                // shared copies: freed with the last handle
    cudaFree(h->workspace);
    cudaFree(h->counters);
    cudaFree(h->push_slots);
    if (h->mail_h) cudaFreeHost(h->mail_h);
    cudaFree(h->stage_elec);
    cudaFree(h->stage_out);
    for (cudaEvent_t e : h->ev)
        if (e) cudaEventDestroy(e);
    delete h;
    return QMMM_OK;
}

qmmm_status qmmm_field_set_plan(qmmm_field *h, const qmmm_plan *plan) {
    if (!h || !plan) return fail(QMMM_ERR_INVALID_ARG, "set_plan: NULL argument");
    const int e = plan->points_per_thread, w = plan->point_warps;
    if (!(e == 0 || e == 1 || e == 2 || e == 4 || e == 8))
        return fail(QMMM_ERR_INVALID_ARG, "set_plan: points_per_thread must be 0,1,2,4,8");
    if (!(w == 0 || w == 1 || w == 2 || w == 4 || w == 8 || w == 16))
        return fail(QMMM_ERR_INVALID_ARG, "set_plan: point_warps must be 0,1,2,4,8,16");
    if (plan->slices < 0 || plan->slices > 65535)
        return fail(QMMM_ERR_INVALID_ARG, "set_plan: slices out of range");
    if (plan->stages != 0 && (plan->stages < 2 || plan->stages > 8))
        return fail(QMMM_ERR_INVALID_ARG, "set_plan: stages must be 0 or 2..8");
    server_stop(h);
    h->user_plan = *plan;
    return QMMM_OK;
}

qmmm_status qmmm_field_set_timing(qmmm_field *h, int enable) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "set_timing: NULL handle");
    if (enable && !h->ev[0])
        for (cudaEvent_t &e : h->ev) CUDA_TRY(cudaEventCreate(&e));
    server_stop(h);
    h->timing = enable != 0;
    h->timed = false;
    return QMMM_OK;
}

qmmm_status qmmm_field_set_local_lattice(qmmm_field *h, int mode) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "set_local_lattice: NULL handle");
    if (mode < -1 || mode > 1) return fail(QMMM_ERR_INVALID_ARG, "set_local_lattice: mode must be -1, 0 or 1");
    server_stop(h);
    h->local_lattice = mode;
    return QMMM_OK;
}

qmmm_status qmmm_field_set_accurate_v(qmmm_field *h, int enable) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "set_accurate_v: NULL handle");
    h->accurate_v = enable != 0;
    return QMMM_OK;
}

qmmm_status qmmm_field_set_overlap(qmmm_field *h, int enable) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "set_overlap: NULL handle");
    h->overlap = enable != 0;
    return QMMM_OK;
}

qmmm_status qmmm_field_last_timing(qmmm_field *h, double *pair_ms, double *finalize_ms) {
    if (!h || !pair_ms || !finalize_ms) return fail(QMMM_ERR_INVALID_ARG, "last_timing: NULL argument");
    if (!h->timing || !h->timed)
        return fail(QMMM_ERR_INVALID_ARG, "last_timing: timing is off or no eval has run");
    CUDA_TRY(cudaEventSynchronize(h->ev[1]));
    float a = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&a, h->ev[0], h->ev[1]));
    *pair_ms = a;
    *finalize_ms = 0.0;      // the cross-CTA sum is fused into the pair kernel
    return QMMM_OK;
}

qmmm_status qmmm_field_get_info(const qmmm_field *h, qmmm_field_info *info) {
    if (!h || !info) return fail(QMMM_ERR_INVALID_ARG, "get_info: NULL argument");
    std::memset(info, 0, sizeof(*info));
    info->M = h->M; info->K = h->K; info->max_points = h->max_points;
    info->n_chunks = h->n_chunks;
    info->bytes_fp64 = h->n_chunks64 * CHUNK * 4 * 8;
    info->bytes_fp32 = h->n_chunks * CHUNK * 4 * 4 + h->n_blocks * 32;
    info->bytes_workspace = h->workspace_doubles * 8;
    info->last_plan = h->last_plan;
    info->last_point_blocks = h->last_point_blocks;
    info->last_launches = h->last_launches;
    info->sm_count = h->sm_count;
    info->last_dz_table = h->last_dz_table;
    info->last_local_lattice = h->last_local_lattice;
    info->last_accurate_v = h->last_accurate_v;
    info->device_errors = h->dev_err_h ? *reinterpret_cast<volatile int *>(h->dev_err_h) : 0;
    std::strncpy(info->last_kernel, h->last_kernel ? h->last_kernel : "", sizeof(info->last_kernel) - 1);
    return QMMM_OK;
}

}  // extern "C"

namespace {
qmmm_status eval_impl(qmmm_field *h, const double *elec_xyz, int64_t W, int64_t N, double *V,
                      double *E, int prec, void *stream, unsigned long long *host_flag) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "eval: NULL handle");
    if (!elec_xyz || !V) return fail(QMMM_ERR_INVALID_ARG, "eval: NULL elec_xyz or V");
    if (W < 1 || N < 1 || W > h->max_points || N > h->max_points || W * N > h->max_points)
        return fail(QMMM_ERR_INVALID_ARG, "eval: W*N must be in [1, max_points]");
    if (prec != QMMM_FP64 && prec != QMMM_FP32_ACC64)
        return fail(QMMM_ERR_INVALID_ARG, "eval: unknown precision");
    const bool f32 = prec == QMMM_FP32_ACC64;
    const int P = static_cast<int>(W * N);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    {
        // launches, the shared-memory attribute and the handle's buffers belong to h->device
        int cur = -1;
        CUDA_TRY(cudaGetDevice(&cur));
        if (cur != h->device)
            return fail(QMMM_ERR_INVALID_ARG, "eval: the current device is not the handle's device");
        g_device = cur;
    }
    if (h->srv_alive) {                    // the resident server owns the workspace: retire it
        qmmm_status ss = server_stop(h);
        if (ss != QMMM_OK) return ss;
    }
    yield_foreign_server(h);               // another handle's resident server would hold every SM

    // overlapped launch (and the few-point plans that go with it): not between timing events,
    // not for the mailbox path, whose host reads V and E behind a flag
    h->overlap_now = h->overlap && !h->timing && !host_flag;
    const bool pdl_attr = h->overlap_now && !h->pdl_hold;
    const bool grid = h->layout == QMMM_LAYOUT_GRID ||
                      (h->layout == QMMM_LAYOUT_AUTO && auto_uses_grid(h, P, f32));
    qmmm_plan pl = choose_plan(h, P, f32, grid);
    const int64_t groups = (P + pl.points_per_thread - 1) / pl.points_per_thread;
    const int pb = static_cast<int>((groups + pl.point_warps - 1) / pl.point_warps);
    int launches = 0;
    const bool light = grid && (f32 ? grid_f32_light(h->overlap_now, pl.points_per_thread, P)
                                    : grid_f64_light(h->overlap_now, pl.points_per_thread, P));
    auto smem_of = [&](int stages) {
        return grid ? grid_smem_bytes(f32, stages, pl.points_per_thread, pl.point_warps, P, light)
                    : pair_smem_bytes(f32, stages, pl.points_per_thread, pl.point_warps);
    };
    size_t smem = smem_of(pl.stages);
    while (smem > 227 * 1024 && pl.stages > 2)           // a requested depth that does not fit is reduced
        smem = smem_of(--pl.stages);
    if (smem > 227 * 1024) return fail(QMMM_ERR_INVALID_ARG, "eval: plan exceeds shared memory");
    // grid kernels: dz table when it fits beside the stages (long z axes keep the stepped dz)
    const size_t dzt = grid ? grid_dzt_bytes(f32, pl.points_per_thread, pl.point_warps, P, h->g_segs, light) : 0;
    // (the FP32 kernel runs two CTAs per SM: half the budget each)
    const bool use_dzt = dzt > 0 && smem + dzt <= (f32 ? (light ? 56 : 110) : 200) * 1024;
    if (use_dzt) smem += dzt;
    // batched FP32 V + E kernel: accurate V (a z2 table beside the dz table) when both fit; the
    // pipeline gives up depth for it (2 stages instead of 4: +0.5 % time on config 3)
    bool use_accv = use_dzt && f32 && E && !light && h->accurate_v && pl.points_per_thread == 4 &&
                    pl.point_warps == GRID_NW_EPT4;
    if (use_accv) {
        int st = pl.stages;
        while (smem_of(st) + 2 * dzt > 110 * 1024 && st > 2) --st;
        if (smem_of(st) + 2 * dzt <= 110 * 1024) {
            pl.stages = st;
            smem = smem_of(st) + 2 * dzt;
        } else {
            use_accv = false;
        }
    }

    if (h->timing) CUDA_TRY(cudaEventRecord(h->ev[0], st));
    {
        PairParams prm;
        std::memset(&prm, 0, sizeof(prm));
        prm.elec = elec_xyz;
        prm.partial = h->workspace;
        prm.P = P;
        prm.slices = pl.slices;
        prm.point_warps = pl.point_warps;
        prm.stages = pl.stages;
        prm.V = V;
        prm.E = E;
        prm.counters = h->counters;
        prm.host_flag = host_flag;
        prm.seq = h->seq;
        prm.done = h->counters + h->max_points;
        // overlap with the previous evaluation on this stream (not with the timing events in
        // between, and not for the mailbox path, whose host reads V and E behind a flag)
        prm.q_unscale = f32 ? 1.0 / h->q_scale : 1.0;
        prm.pdl = pdl_attr ? 1 : 0;
        prm.dev_err = h->dev_err_d;
        // Few points, all CTAs of the launch resident together (at most
        // one per SM, so the collecting CTAs cannot keep the pushing ones from starting):
        // collect the CTA partials by tagged records instead of fence + ticket -- about 1 us
        // less per evaluation, and the serial tail that bounds the period of an overlapped
        // sequence.  Same summation order, bitwise the same result.  (Not for the mailbox
        // path, whose last CTA also publishes the host flag.)
        h->last_mail_push = false;
        if (host_flag && P <= INLINE_POINTS) {     // mailbox call: the points as kernel parameters
            std::memcpy(prm.pts, h->mail_h, static_cast<size_t>(P) * 3 * sizeof(double));
            prm.inline_pts = 1;
        }
        if (pl.points_per_thread <= 4 &&
            static_cast<int64_t>(pb) * pl.slices <= h->sm_count &&
            static_cast<int64_t>(pl.slices) * P <= PUSH_MAX_RECORDS &&
            static_cast<int64_t>(pl.slices) * pl.point_warps * pl.points_per_thread * 32 <=
                std::min<int64_t>(PUSH_MAX_CTA_RECORD_BYTES,
                                  static_cast<int64_t>(pl.stages) * (grid ? (f32 ? 8192 : 16384) : 32768))) {
            prm.push_slots = h->push_slots;
            prm.push_seq = ++h->push_seq;
            if (host_flag) {               // mailbox: the collecting CTAs answer with tagged records
                prm.host_flag = nullptr;
                prm.host_records = reinterpret_cast<unsigned long long *>(h->mail_d + MAIL_REC_OFFSET);
                h->last_mail_push = true;
            }
        }
        if (grid) {
            fill_grid_params(h, prm, f32);
            prm.g_dzt = use_dzt ? 1 : 0;
            prm.g_accv = use_accv ? 1 : 0;
            prm.g_light = light ? 1 : 0;
        } else {
            prm.chunks = f32 ? reinterpret_cast<const char *>(h->chunks32)
                             : reinterpret_cast<const char *>(h->chunks64);
            prm.origins = h->origins;
            prm.n_chunks = static_cast<int>(f32 ? h->n_chunks : h->n_chunks64);
            prm.lattice = h->lattice;
            prm.inv_lattice = 1.0 / h->lattice;
            prm.nuc = h->nuclei;
            prm.K = f32 ? static_cast<int>(h->K) : 0;     // FP64: nuclei are in the chunk array
        }
#ifdef QMMM_PHASE_TIMING
        prm.dbg = reinterpret_cast<long long *>(h->workspace + h->workspace_doubles - 16384);
#endif
        // point blocks vary fastest: the CTAs resident together read the same source slices,
        // so a slice is fetched from HBM once and then served from L2
        const dim3 grid_dim(pb, pl.slices);
        cudaError_t e = grid ? launch_grid_ept(f32, pl.points_per_thread, prm, grid_dim, smem, st)
                             : launch_pair_ept(f32, pl.points_per_thread, prm, grid_dim, smem, st);
        if (e != cudaSuccess) return cuda_fail(e, "pair_kernel launch");
        ++launches;
    }
    h->last_layout = grid ? QMMM_LAYOUT_GRID : QMMM_LAYOUT_LIST;
    h->last_kernel = g_launched;
    if (h->timing) {
        CUDA_TRY(cudaEventRecord(h->ev[1], st));
        h->timed = true;
    }

    h->last_plan = pl;
    h->last_point_blocks = pb;
    h->last_launches = launches;
    h->last_dz_table = use_dzt ? 1 : 0;
    // (potential-only evaluations of batched FP32 grids always run the compensated kernel)
    h->last_accurate_v = (use_accv || (use_dzt && f32 && !E && !light && pl.points_per_thread == 4 &&
                                       pl.point_warps == GRID_NW_EPT4)) ? 1 : 0;
    return QMMM_OK;
}
}  // namespace

extern "C" {

qmmm_status qmmm_field_eval(qmmm_field *h, const double *elec_xyz, int64_t W, int64_t N,
                            double *V, double *E, int prec, void *stream) {
    return eval_impl(h, elec_xyz, W, N, V, E, prec, stream, nullptr);
}

qmmm_status qmmm_field_eval_moves(qmmm_field *h, const double *elec_xyz, int64_t n, int64_t N,
                                  double *V, double *E, int prec, void *stream) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "eval_moves: NULL handle");
    if (n < 0) return fail(QMMM_ERR_INVALID_ARG, "eval_moves: n < 0");
    if (n > 0 && (!elec_xyz || !V)) return fail(QMMM_ERR_INVALID_ARG, "eval_moves: NULL elec_xyz or V");
    // independent evaluations (all positions are known up front): let them overlap
    const bool was = h->overlap;
    h->overlap = true;
    qmmm_status s = QMMM_OK;
    for (int64_t i = 0; i < n && s == QMMM_OK; ++i) {
        // the first move is launched with plain stream serialization (it reads elec_xyz, which
        // whatever precedes the call on the stream may have produced); moves 1.. overlap with
        // their predecessor, which is this library's own evaluation
        h->pdl_hold = i == 0;
        s = eval_impl(h, elec_xyz + i * N * 3, 1, N, V + i * N, E ? E + i * N * 3 : nullptr, prec, stream,
                      nullptr);
    }
    h->pdl_hold = false;
    h->overlap = was;
    return s;
}

qmmm_status qmmm_field_eval_energy(qmmm_field *h, const double *elec_xyz, int64_t W, int64_t N,
                                   double *U, int prec, void *stream) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "eval_energy: NULL handle");
    if (!U) return fail(QMMM_ERR_INVALID_ARG, "eval_energy: NULL U");
    // V goes to the handle's staging buffer (sized for max_points), E is not formed (FP64:
    // the potential-only kernel, Eq. 4 proper), then one small fixed-order sum per walker
    qmmm_status s = eval_impl(h, elec_xyz, W, N, h->stage_out, nullptr, prec, stream, nullptr);
    if (s != QMMM_OK) return s;
    walker_energy_kernel<<<static_cast<unsigned>((W + 7) / 8), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        h->stage_out, W, N, U);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "walker_energy_kernel launch");
    ++h->last_launches;
    return QMMM_OK;
}

qmmm_status qmmm_sum_rank_partials(const double *parts, int64_t R, int64_t n, double *out, void *stream) {
    if (!parts || !out) return fail(QMMM_ERR_INVALID_ARG, "sum_rank_partials: NULL pointer");
    if (R < 1 || R > 65536 || n < 0) return fail(QMMM_ERR_INVALID_ARG, "sum_rank_partials: need 1 <= R <= 65536, n >= 0");
    if (n == 0) return QMMM_OK;
    sum_rank_partials_kernel<<<static_cast<unsigned>((n + 255) / 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        parts, static_cast<int>(R), n, out);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "sum_rank_partials_kernel launch");
    return QMMM_OK;
}

qmmm_status qmmm_field_eval_host(qmmm_field *h, const double *elec_xyz_host, int64_t W,
                                 int64_t N, double *V_host, double *E_host, int prec,
                                 void *stream) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "eval_host: NULL handle");
    if (!elec_xyz_host || !V_host)
        return fail(QMMM_ERR_INVALID_ARG, "eval_host: NULL elec_xyz or V");
    if (W < 1 || N < 1 || W > h->max_points || N > h->max_points || W * N > h->max_points)
        return fail(QMMM_ERR_INVALID_ARG, "eval_host: W*N must be in [1, max_points]");
    const int64_t P = W * N;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    note_host_eval(h);
    auto device_error = [&]() -> bool { return *reinterpret_cast<volatile int *>(h->dev_err_h) != 0; };
    if (P == 1 && (prec == QMMM_FP64 || prec == QMMM_FP32_ACC64)) {
        // one point per call is the paper's own loop: served by the resident move server
        bool served = false;
        qmmm_status s = server_move(h, elec_xyz_host, V_host, E_host, prec, &served);
        if (s != QMMM_OK || served) return s;
    }
    if (P <= MAIL_POINTS) {
        // Per-move path ("r_new" in, U_ES out, every Monte-Carlo step): no
        // cudaMemcpy and no stream synchronisation.  The kernel reads the points from a
        // pinned, device-mapped mailbox, the CTA that finishes last writes V, E and then a
        // sequence number into it, and the host waits for that number.
        double *in_h = h->mail_h, *out_h = h->mail_h + MAIL_POINTS * 3;
        volatile unsigned long long *flag_h =
            reinterpret_cast<volatile unsigned long long *>(h->mail_h + MAIL_POINTS * 7);
        double *in_d = h->mail_d, *out_d = h->mail_d + MAIL_POINTS * 3;
        std::memcpy(in_h, elec_xyz_host, P * 3 * sizeof(double));
        ++h->seq;
        qmmm_status s = eval_impl(h, in_d, W, N, out_d, E_host ? out_d + P : nullptr, prec, stream,
                                  reinterpret_cast<unsigned long long *>(h->mail_d + MAIL_POINTS * 7));
        if (s != QMMM_OK) return s;
        if (h->last_mail_push) {
            // answered by tagged records {tag, V, Ex, Ey, Ez, tag}, one per point, written by the
            // collecting CTAs without fences: wait until every record carries this call's tag
            const volatile unsigned long long *rec =
                reinterpret_cast<const volatile unsigned long long *>(h->mail_h + MAIL_REC_OFFSET);
            const unsigned long long tag = h->push_seq;
            uint64_t spin = 1;
            for (int64_t p = 0; p < P; ++p) {
                const volatile unsigned long long *r = rec + p * 8;
                // four self-validating 16-byte units {tag, value}: each is one aligned 16-byte
                // store of the device, so a value is read after (and re-checked against) its tag
                auto complete = [&]() { return r[0] == tag && r[2] == tag && r[4] == tag && r[6] == tag; };
                for (;;) {
                    if (complete()) {
                        std::atomic_thread_fence(std::memory_order_acquire);
                        const unsigned long long bits[4] = {r[1], r[3], r[5], r[7]};
                        std::atomic_thread_fence(std::memory_order_acquire);
                        if (!complete()) continue;
                        std::memcpy(V_host + p, &bits[0], 8);
                        if (E_host) std::memcpy(E_host + 3 * p, &bits[1], 24);
                        break;
                    }
                    if ((++spin & 0xFFFF) == 0) {             // now and then: did the launch fail?
                        cudaError_t q = cudaStreamQuery(st);
                        if (q != cudaSuccess && q != cudaErrorNotReady) return cuda_fail(q, "eval_host: kernel");
                        if (q == cudaSuccess && !complete())
                            return fail(QMMM_ERR_CUDA, "eval_host: kernel finished without publishing its result");
                    }
                }
            }
            if (device_error())
                return fail(QMMM_ERR_CUDA, "eval_host: a cross-CTA collection timed out on the device (results are NaN)");
            return QMMM_OK;
        }
        for (uint64_t spin = 1; *flag_h != h->seq; ++spin) {
            if ((spin & 0xFFFF) == 0) {                   // now and then: did the launch fail?
                cudaError_t q = cudaStreamQuery(st);
                if (q != cudaSuccess && q != cudaErrorNotReady) return cuda_fail(q, "eval_host: kernel");
                if (q == cudaSuccess && *flag_h != h->seq)
                    return fail(QMMM_ERR_CUDA, "eval_host: kernel finished without publishing its result");
            }
        }
        std::atomic_thread_fence(std::memory_order_acquire);
        std::memcpy(V_host, out_h, P * sizeof(double));
        if (E_host) std::memcpy(E_host, out_h + P, P * 3 * sizeof(double));
        if (device_error())
            return fail(QMMM_ERR_CUDA, "eval_host: a cross-CTA collection timed out on the device (results are NaN)");
        return QMMM_OK;
    }
    CUDA_TRY(cudaMemcpyAsync(h->stage_elec, elec_xyz_host, P * 3 * sizeof(double),
                             cudaMemcpyHostToDevice, st));
    double *dV = h->stage_out, *dE = E_host ? h->stage_out + P : nullptr;
    qmmm_status s = eval_impl(h, h->stage_elec, W, N, dV, dE, prec, stream, nullptr);
    if (s != QMMM_OK) return s;
    // V and E are adjacent in the staging buffer: one device->host copy when both are wanted
    // and the host buffers are adjacent too, else two.
    if (E_host && E_host == V_host + P) {
        CUDA_TRY(cudaMemcpyAsync(V_host, dV, P * 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
    } else {
        CUDA_TRY(cudaMemcpyAsync(V_host, dV, P * sizeof(double), cudaMemcpyDeviceToHost, st));
        if (E_host)
            CUDA_TRY(cudaMemcpyAsync(E_host, dE, P * 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CUDA_TRY(cudaStreamSynchronize(st));
    if (device_error())
        return fail(QMMM_ERR_CUDA, "eval_host: a cross-CTA collection timed out on the device (results are NaN)");
    return QMMM_OK;
}

#ifdef QMMM_PHASE_TIMING
// Diagnostic build only: per-CTA phase clocks of the most recent packed-kernel launch.
qmmm_status qmmm_debug_phases(qmmm_field *h, long long *out, int n) {
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpy(out, h->workspace + h->workspace_doubles - 16384, n * sizeof(long long),
                        cudaMemcpyDeviceToHost));
    return QMMM_OK;
}
#endif

// ---- debug helper: smallest distance between the evaluation points and the charged sources ----
namespace {
constexpr int MIND_POINTS = 64;       // points per CTA (shared memory)
// Sources are enumerated from the FP64 list copy ([chunk][x, y, z, q][128], cells then nuclei) or,
// for handles without one, from the FP64 grid copy ([gchunk][ZS/2][32 rows][2]) plus the nuclei.
// Squared distances are >= 0, so their bit patterns order like unsigned integers: the minimum is
// taken with an integer atomic (order-independent, hence deterministic).
__global__ void __launch_bounds__(256) min_distance_kernel(const double *elec, int64_t P, const double *chunks64,
                                                           int64_t n_list, const double *gcells64, int64_t n_nodes,
                                                           qmmm::GridGeom gg, int g_segs, const double *nuclei,
                                                           int64_t K, unsigned long long *out) {
    __shared__ double pt[MIND_POINTS][3];
    const int64_t p0 = static_cast<int64_t>(blockIdx.x) * MIND_POINTS;
    const int np = static_cast<int>(P - p0 < MIND_POINTS ? P - p0 : MIND_POINTS);
    for (int i = threadIdx.x; i < np * 3; i += blockDim.x) pt[i / 3][i % 3] = elec[p0 * 3 + i];
    __syncthreads();
    double best = __longlong_as_double(0x7ff0000000000000ll);            // +inf
    auto visit = [&](double x, double y, double z) {
        for (int i = 0; i < np; ++i) {
            const double dx = pt[i][0] - x, dy = pt[i][1] - y, dz = pt[i][2] - z;
            const double d2 = fma(dz, dz, fma(dy, dy, dx * dx));
            best = d2 < best ? d2 : best;
        }
    };
    const int64_t stride = static_cast<int64_t>(gridDim.y) * blockDim.x;
    const int64_t first = static_cast<int64_t>(blockIdx.y) * blockDim.x + threadIdx.x;
    if (chunks64) {
        for (int64_t j = first; j < n_list; j += stride) {
            const double *c = chunks64 + (j / 128) * 512 + (j % 128);
            if (c[384] != 0.0) visit(c[0], c[128], c[256]);
        }
    } else {
        const int ny = gg.n[1];
        for (int64_t j = first; j < n_nodes; j += stride) {
            if (gcells64[j] == 0.0) continue;
            const int64_t c = j / qmmm::GRID_NODES;
            const int i = static_cast<int>(j % qmmm::GRID_NODES);
            const int64_t row = (c / g_segs) * 32 + (i / 2) % 32;
            const int iz = static_cast<int>(c % g_segs) * qmmm::GRID_ZS + 2 * (i / 64) + (i & 1);
            visit(gg.org[0] + gg.h[0] * static_cast<double>(row / ny), gg.org[1] + gg.h[1] * static_cast<double>(row % ny),
                  gg.org[2] + gg.h[2] * static_cast<double>(iz));
        }
        for (int64_t j = first; j < K; j += stride)
            if (nuclei[4 * j + 3] != 0.0) visit(nuclei[4 * j], nuclei[4 * j + 1], nuclei[4 * j + 2]);
    }
    for (int m = 16; m >= 1; m >>= 1) {
        const double o = __shfl_xor_sync(0xffffffffu, best, m);
        best = o < best ? o : best;
    }
    if ((threadIdx.x & 31) == 0) atomicMin(out, static_cast<unsigned long long>(__double_as_longlong(best)));
}
}  // namespace

qmmm_status qmmm_field_min_distance(qmmm_field *h, const double *elec_xyz, int64_t P, double *min_distance_host,
                                    void *stream) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "min_distance: NULL handle");
    if (!elec_xyz || !min_distance_host) return fail(QMMM_ERR_INVALID_ARG, "min_distance: NULL elec_xyz or result");
    if (P < 1) return fail(QMMM_ERR_INVALID_ARG, "min_distance: P must be >= 1");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned long long *out_d = nullptr, out_h = 0x7ff0000000000000ull;
    CUDA_TRY(cudaMalloc(&out_d, sizeof(out_h)));
    cudaError_t e = cudaMemcpyAsync(out_d, &out_h, sizeof(out_h), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && h->M + h->K > 0) {
        const bool list = h->has_list && h->chunks64;
        const int64_t n_list = h->n_chunks64 * 128, n_nodes = h->n_g * qmmm::GRID_NODES;
        const int64_t n_src = list ? n_list : n_nodes + h->K;
        const unsigned gx = static_cast<unsigned>((P + MIND_POINTS - 1) / MIND_POINTS);
        unsigned gy = static_cast<unsigned>(std::min<int64_t>((n_src + 255) / 256, std::max<int64_t>(1, 8 * h->sm_count / gx)));
        if (gy < 1) gy = 1;
        min_distance_kernel<<<dim3(gx, gy), 256, 0, st>>>(elec_xyz, P, list ? h->chunks64 : nullptr, n_list, h->gcells64,
                                                        n_nodes, h->grid, static_cast<int>(h->g_segs), h->nuclei, h->K, out_d);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&out_h, out_d, sizeof(out_h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(out_d);
    if (e != cudaSuccess) return cuda_fail(e, "min_distance");
    double d2;
    std::memcpy(&d2, &out_h, sizeof(d2));
    *min_distance_host = std::sqrt(d2);
    return QMMM_OK;
}

qmmm_status qmmm_field_eval_move_host(qmmm_field *h, const double *r_old, const double *r_new,
                                      const double *V_old, const double *E_old, double *V_new,
                                      double *E_new, double *dV, double *dE, int prec, void *stream) {
    if (!h) return fail(QMMM_ERR_INVALID_ARG, "eval_move_host: NULL handle");
    if (!r_old || !r_new || !V_new) return fail(QMMM_ERR_INVALID_ARG, "eval_move_host: NULL r_old, r_new or V_new");
    double Vo = 0.0, Eo[3] = {0.0, 0.0, 0.0};
    if (V_old && (!E_new || E_old)) {
        // the caller knows the old values: one point, the resident move server
        qmmm_status s = qmmm_field_eval_host(h, r_new, 1, 1, V_new, E_new, prec, stream);
        if (s != QMMM_OK) return s;
        Vo = *V_old;
        if (E_new) std::memcpy(Eo, E_old, sizeof(Eo));
    } else {
        // both points in one launch
        double pts[6], V2[2], E2[6];
        std::memcpy(pts, r_old, 3 * sizeof(double));
        std::memcpy(pts + 3, r_new, 3 * sizeof(double));
        qmmm_status s = qmmm_field_eval_host(h, pts, 1, 2, V2, E_new ? E2 : nullptr, prec, stream);
        if (s != QMMM_OK) return s;
        Vo = V2[0];
        *V_new = V2[1];
        if (E_new) {
            std::memcpy(Eo, E2, sizeof(Eo));
            std::memcpy(E_new, E2 + 3, 3 * sizeof(double));
        }
    }
    if (dV) *dV = *V_new - Vo;
    if (dE && E_new)
        for (int k = 0; k < 3; ++k) dE[k] = E_new[k] - Eo[k];
    return QMMM_OK;
}

qmmm_status qmmm_field_eval_moves_host(qmmm_field *h, const double *elec_xyz_host, int64_t n,
                                       int64_t N, double *V_host, double *E_host, int prec,
                                       void *stream, double *seconds) {
    if (n < 0) return fail(QMMM_ERR_INVALID_ARG, "eval_moves_host: n < 0");
    struct timespec t0, t1;
    clock_gettime(CLOCK_MONOTONIC, &t0);
    for (int64_t s = 0; s < n; ++s) {
        qmmm_status st = qmmm_field_eval_host(h, elec_xyz_host + s * N * 3, 1, N, V_host + s * N,
                                              E_host ? E_host + s * N * 3 : nullptr, prec, stream);
        if (st != QMMM_OK) return st;
    }
    clock_gettime(CLOCK_MONOTONIC, &t1);
    if (seconds) *seconds = (t1.tv_sec - t0.tv_sec) + 1e-9 * (t1.tv_nsec - t0.tv_nsec);
    return QMMM_OK;
}

}  // extern "C"
