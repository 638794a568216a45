// qmmm_server.cuh -- resident "move server" for the paper's deployed loop:
// every Monte-Carlo step the host sends ONE new electron position r_new and receives U_ES.
//
// A kernel launch costs ~10 us host-to-host on an idle GPU, as much as the evaluation itself
// (11 us at 2.08 M sources).  The server is launched once (cooperatively: one CTA per SM, all
// resident) and then serves moves from a pinned, device-mapped mailbox:
//
//   host   : writes {s, r, s} into the request line; spins until the answer line carries s
//   leader : one warp of CTA 0 polls the request line over PCIe (one transaction) and publishes
//            the move as three tagged 16-byte units {s, x} {s, y} {s, z} in device memory
//   all    : poll those units (L2), run their source slice exactly like pair_kernel<REAL,1> (TMA ring,
//            FP64 or FP32-acc64 pair math, in-CTA reduction)
//   all    : push their partial as one tagged record (four 16-byte units {s, value})
//   leader : collects the records, adds them in a fixed order and stores {s, V} {s, Ex}
//            {s, Ey} {s, Ez} to the answer line
//
// The producer warp prefetches the first ring stages of the NEXT move while the CTA waits
// (the sources do not depend on r), so a move starts on data that is already in shared memory.
// Every wait is bounded: the leader retires the server (cmd = EXIT) after IDLE_NS without a
// request, when the host posts EXIT, or after LIFE_NS; the host relaunches it transparently.
// Results are bitwise those of the launch path with the same partition.
#pragma once
#include "qmmm_kernels.cuh"
#include "qmmm_grid.cuh"

namespace qmmm {

struct ServerMailbox {                 // pinned host memory, device-mapped
    // request line, one 64-byte cache line, read by the device in ONE coalesced transaction:
    // the host writes seq_a, then r, then seq_b (x86 stores are ordered); the device accepts
    // a snapshot only when seq_a == seq_b (a seqlock), so r always belongs to that move
    volatile unsigned long long req[8];    // [0] seq_a  [1..3] r_new (as bits)  [4] seq_b; EXIT = retire
                                           // [5] yield: another handle wants the device -- retire
    // answer line: four self-validating 16-byte units {s, V} {s, Ex} {s, Ey} {s, Ez} (values as
    // bits), each written by the device with one aligned 16-byte store; the host takes the
    // answer when all four carry the move number s
    volatile unsigned long long ans[8];
    volatile unsigned long long exited;    // device -> host: launch id that has retired
    volatile unsigned long long pad[7];
};

struct ServerDevice {                  // device memory shared by the CTAs of the server
    // The published move: three self-validating 16-byte units {s, x} {s, y} {s, z} (s = move
    // number, or SERVER_EXIT; x, y, z = r_new as bits), each written by the leader with ONE
    // aligned 16-byte store and polled by the other CTAs with 16-byte loads until all three tags
    // agree and differ from the last move -- no fence on either side (round 1 wrote r_new, fenced,
    // then wrote the move number, and the readers fenced and loaded r_new after seeing the number:
    // two more L2 round trips per move).
    unsigned long long rec[8];
};

constexpr unsigned long long SERVER_EXIT = ~0ull;
constexpr long long SERVER_IDLE_NS = 2'000'000;        // retire after 2 ms without a request
constexpr long long SERVER_LIFE_NS = 1'000'000'000;    // and after 1 s in any case
constexpr long long SERVER_HARD_NS = 4'000'000'000;    // non-leaders give up (never expected)

struct ServerParams {
    PairParams pair;                       // P = 1, point_warps = 1; V/E/host_flag unused here
    ServerMailbox *mail;                   // device pointer of the mapped mailbox
    ServerDevice *dev;
    unsigned long long start_seq;          // moves <= start_seq are already answered
    unsigned long long launch_id;
};

__device__ __forceinline__ long long global_ns() {
    long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// Cross-CTA sum of one move, push model.  Every CTA stores its partial as one tagged 64-byte
// record of four self-validating 16-byte units {s, V} {s, Ex} {s, Ey} {s, Ez} (one aligned
// 16-byte store per lane, as push_records in qmmm_kernels.cuh) into its own slot -- no fence, no
// atomic ticket, and it is free for the next move at once.  The leader CTA collects: thread t
// polls slot t with four 16-byte volatile loads until all four tags carry s (move numbers only
// grow, so nothing is reset), the records go to shared memory, and the slices are added in
// exactly the order of finish_point_block (so the result is bitwise that of the launch path).
// Threads 0..3 then hold V, Ex, Ey, Ez and store {s, value} to the mapped answer line -- no
// system-scope fence (a PCIe round trip each) on the critical path.
constexpr int SLOT_WORDS = 8;              // 64-byte slots in the partials workspace

__device__ __forceinline__ void server_push(unsigned long long *slots, int lane, double acc,
                                            unsigned long long seq) {
    if (lane < 4)                          // lanes 0..3 hold V, Ex, Ey, Ez
        push_st_v2(slots + blockIdx.y * SLOT_WORDS + 2 * lane, seq,
                   static_cast<unsigned long long>(__double_as_longlong(acc)));
}

// Leader CTA only; all 256 consumer threads call it.  part_s: [slices][4] doubles of shared
// memory.  Returns false if a slot never arrived (hard timeout): the caller retires the server.
template <typename SYNC>
__device__ __forceinline__ bool server_collect(const PairParams &prm, ServerMailbox *mail,
                                               const unsigned long long *slots, int tid,
                                               double *part_s, double *scratch, int *flag, SYNC sync,
                                               unsigned long long seq, long long t_start) {
    constexpr int NT = 32 * COMPUTE_WARPS;
    if (tid == 0) *flag = 1;
    sync();
    for (int sl = tid; sl < prm.slices; sl += NT) {
        const unsigned long long *p = slots + sl * SLOT_WORDS;
        for (;;) {
            const push_u64x2 a = push_ld_v2(p), b = push_ld_v2(p + 2), c = push_ld_v2(p + 4), d = push_ld_v2(p + 6);
            if (a.x == seq && b.x == seq && c.x == seq && d.x == seq) {
                part_s[4 * sl + 0] = __longlong_as_double(static_cast<long long>(a.y));
                part_s[4 * sl + 1] = __longlong_as_double(static_cast<long long>(b.y));
                part_s[4 * sl + 2] = __longlong_as_double(static_cast<long long>(c.y));
                part_s[4 * sl + 3] = __longlong_as_double(static_cast<long long>(d.y));
                break;
            }
            if (global_ns() - t_start > SERVER_HARD_NS) { *flag = 0; break; }
        }
    }
    sync();
    if (!*flag) return false;
    const int G = NT / 4, v = tid & 3, g = tid >> 2;      // same association as finish_point_block
    double a[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    {
        int sidx = g;
        for (; sidx + 7 * G < prm.slices; sidx += 8 * G)
#pragma unroll
            for (int k = 0; k < 8; ++k) a[k] += part_s[4 * (sidx + k * G) + v];
#pragma unroll
        for (int k = 0; k < 8; ++k)                         // tail, compile-time indices
            if (sidx + k * G < prm.slices) a[k] += part_s[4 * (sidx + k * G) + v];
    }
    scratch[tid] = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
    sync();
    if (tid < 4) {
        double r = 0.0;
        for (int k = 0; k < G; ++k) r += scratch[k * 4 + tid];
        push_st_v2(const_cast<unsigned long long *>(mail->ans) + 2 * tid, seq,
                   static_cast<unsigned long long>(__double_as_longlong(r)));
    }
    return true;
}

// Warp 0 of every CTA waits here for the next move.  Leader CTA: polls the request line in pinned
// host memory, relays r_new through device memory and publishes the move number; the others
// poll that number.  Returns the move number (or SERVER_EXIT) in every lane; elec_s[0..2] = r_new.
__device__ __forceinline__ unsigned long long server_next_move(const ServerParams &sp, bool leader, int lane,
                                                               unsigned long long last, long long t_start,
                                                               double *elec_s) {
    unsigned long long c = 0, w = 0;
    if (leader) {
        // lanes 0..4 read the request line over PCIe in one transaction
        const long long t_idle = global_ns();
        for (;;) {
            w = lane < 6 ? sp.mail->req[lane] : 0ull;
            const unsigned long long a = __shfl_sync(0xffffffffu, w, 0);
            const unsigned long long b = __shfl_sync(0xffffffffu, w, 4);
            if (a == b && a != last) { c = a; break; }
            if (__shfl_sync(0xffffffffu, w, 5) != 0ull) {      // another handle wants the device
                c = SERVER_EXIT;
                break;
            }
            const long long now = __shfl_sync(0xffffffffu, global_ns(), 0);
            if (now - t_idle > SERVER_IDLE_NS || now - t_start > SERVER_LIFE_NS) {
                c = SERVER_EXIT;
                break;
            }
        }
        if (lane >= 1 && lane <= 3) {                        // lanes 1..3 hold x, y, z (as bits)
            if (c != SERVER_EXIT) elec_s[lane - 1] = __longlong_as_double(static_cast<long long>(w));
            push_st_v2(sp.dev->rec + 2 * (lane - 1), c, c != SERVER_EXIT ? w : 0ull);
        }
        __syncwarp();
    } else {
        push_u64x2 r = {0ull, 0ull};
        for (;;) {
            if (lane < 3) r = push_ld_v2(sp.dev->rec + 2 * lane);
            const unsigned long long t0 = __shfl_sync(0xffffffffu, r.x, 0), t1 = __shfl_sync(0xffffffffu, r.x, 1),
                                     t2 = __shfl_sync(0xffffffffu, r.x, 2);
            if (t0 == t1 && t1 == t2 && t0 != last) { c = t0; break; }
            const long long now = __shfl_sync(0xffffffffu, global_ns(), 0);
            if (now - t_start > SERVER_HARD_NS) {
                c = SERVER_EXIT;
                break;
            }
        }
        if (c != SERVER_EXIT && lane < 3) elec_s[lane] = __longlong_as_double(static_cast<long long>(r.y));
        __syncwarp();
    }
    return c;
}

// grid = (1, slices) with slices <= SM count, launched cooperatively (all CTAs resident).
template <typename REAL>
__global__ void __launch_bounds__(CTA_THREADS, 1) move_server_kernel(const ServerParams sp) {
    const PairParams &prm = sp.pair;
    constexpr bool F32 = sizeof(REAL) == 4;
    constexpr int CHUNK_BYTES = 4 * CHUNK * sizeof(REAL);
    constexpr int SC = F32 ? BLOCK_CHUNKS : STAGE_CHUNKS_F64;
    constexpr int STAGE_BYTES = STAGE_HDR + SC * CHUNK_BYTES;
    constexpr int WS = COMPUTE_WARPS;                        // one point: all warps split the sources

    extern __shared__ __align__(128) unsigned char smem[];
    const int stages = prm.stages;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + static_cast<size_t>(stages) * STAGE_BYTES);
    uint64_t *empty = full + 8;
    int *flag = reinterpret_cast<int *>(empty + 8);
    double *red = reinterpret_cast<double *>(empty + 10);    // [256]
    double *elec_s = red + 32 * COMPUTE_WARPS;               // [3]
    volatile unsigned long long *cmd_s = reinterpret_cast<volatile unsigned long long *>(elec_s + 4);
    volatile unsigned long long *go_s = cmd_s + 1;           // moves released to the producer, or EXIT
    double *part_s = elec_s + 8;                             // leader: [slices][4] collected partials
    unsigned long long *slots = reinterpret_cast<unsigned long long *>(prm.partial);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.y, lo, hi);
    int nsteps = 0;
    for (int c = lo; c < hi; c = stage_end<SC>(c, hi)) ++nsteps;
    const int npre = nsteps < stages ? nsteps : stages;      // steps prefetched before a move arrives

    if (threadIdx.x == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], COMPUTE_WARPS);
        }
        fence_barrier_init();
        *cmd_s = sp.start_seq;
        *go_s = 0;
    }
    __syncthreads();

    if (warp == COMPUTE_WARPS) {
        // ===================== producer warp ============================================
        if (lane == 0) {
            unsigned long long pk = 0, moves = 0;
            for (;;) {
                int pc = lo, step = 0;
                auto load_step = [&]() {
                    const int ce = stage_end<SC>(pc, hi);
                    const int slot = static_cast<int>(pk % stages);
                    if (pk >= static_cast<unsigned long long>(stages))
                        mbar_wait(&empty[slot], static_cast<uint32_t>((pk / stages) - 1) & 1u);
                    unsigned char *dst = smem + static_cast<size_t>(slot) * STAGE_BYTES;
                    const uint32_t bytes = static_cast<uint32_t>(ce - pc) * CHUNK_BYTES;
                    if constexpr (F32) {
                        mbar_expect_tx(&full[slot], bytes + 32);
                        tma_bulk_g2s(dst, prm.origins + 4 * (pc / SC), 32, &full[slot]);
                    } else {
                        mbar_expect_tx(&full[slot], bytes);
                    }
                    tma_bulk_g2s(dst + STAGE_HDR, prm.chunks + static_cast<size_t>(pc) * CHUNK_BYTES,
                                 bytes, &full[slot]);
                    pc = ce;
                    ++pk;
                    ++step;
                };
                while (step < npre) load_step();             // ahead of the next request
                ++moves;
                unsigned long long g;
                while ((g = *go_s) < moves) __nanosleep(40);
                if (g == SERVER_EXIT) break;
                while (step < nsteps) load_step();
            }
        }
        return;
    }

    // ========================= consumer warps ============================================
    const int ws = warp;
    unsigned long long k = 0, last = sp.start_seq, released = 0;
    const bool leader = blockIdx.y == 0;
    const long long t_start = global_ns();
    for (;;) {
        if (warp == 0) {
            const unsigned long long c = server_next_move(sp, leader, lane, last, t_start, elec_s);
            if (lane == 0) {
                *cmd_s = c;
                *go_s = c == SERVER_EXIT ? SERVER_EXIT : ++released;    // release the producer
            }
        }
        compute_warps_sync();
        const unsigned long long cmd = *cmd_s;
        if (cmd == SERVER_EXIT) {
            // drain the prefetched stages so that no bulk copy is in flight when the CTA ends
            for (int s = 0; s < npre; ++s, ++k)
                mbar_wait(&full[k % stages], static_cast<uint32_t>(k / stages) & 1u);
            break;
        }
        last = cmd;

        // ---- one evaluation of this CTA's slice, as pair_kernel<REAL, 1> -------------------
        double V[1] = {0.0}, Ex[1] = {0.0}, Ey[1] = {0.0}, Ez[1] = {0.0};
        const double px = elec_s[0], py = elec_s[1], pz = elec_s[2];
        for (int c = lo; c < hi; ++k) {
            const int ce = stage_end<SC>(c, hi);
            const int slot = static_cast<int>(k % stages);
            mbar_wait(&full[slot], static_cast<uint32_t>(k / stages) & 1u);
            const unsigned char *st = smem + static_cast<size_t>(slot) * STAGE_BYTES;
            const int nch = ce - c;
            if constexpr (F32) {
                const double *org = reinterpret_cast<const double *>(st);
                const double a0 = px - org[0], a1 = py - org[1], a2 = pz - org[2];
                float ddx, ddy, ddz;
                const float rx = lattice_round_local(a0, org[3], prm.lattice, prm.inv_lattice, ddx);
                const float ry = lattice_round_local(a1, org[3], prm.lattice, prm.inv_lattice, ddy);
                const float rz = lattice_round_local(a2, org[3], prm.lattice, prm.inv_lattice, ddz);
                float v32 = 0.f, ex32 = 0.f, ey32 = 0.f, ez32 = 0.f;
                const float *data = reinterpret_cast<const float *>(st + STAGE_HDR);
                for (int ch = ws; ch < nch; ch += WS) {
                    const float *b = data + ch * 4 * CHUNK + 4 * lane;
                    const float4 X = *reinterpret_cast<const float4 *>(b);
                    const float4 Y = *reinterpret_cast<const float4 *>(b + CHUNK);
                    const float4 Z = *reinterpret_cast<const float4 *>(b + 2 * CHUNK);
                    const float4 Q = *reinterpret_cast<const float4 *>(b + 3 * CHUNK);
                    pair_f32(rx, ry, rz, X.x, Y.x, Z.x, Q.x, v32, ex32, ey32, ez32);
                    pair_f32(rx, ry, rz, X.y, Y.y, Z.y, Q.y, v32, ex32, ey32, ez32);
                    pair_f32(rx, ry, rz, X.z, Y.z, Z.z, Q.z, v32, ex32, ey32, ez32);
                    pair_f32(rx, ry, rz, X.w, Y.w, Z.w, Q.w, v32, ex32, ey32, ez32);
                }
                const float corr = fmaf(ez32, ddz, fmaf(ey32, ddy, ex32 * ddx));
                V[0] += static_cast<double>(v32) - static_cast<double>(corr);
                Ex[0] += static_cast<double>(ex32);
                Ey[0] += static_cast<double>(ey32);
                Ez[0] += static_cast<double>(ez32);
            } else {
                const double *data = reinterpret_cast<const double *>(st + STAGE_HDR);
                for (int ch = ws; ch < nch; ch += WS) {
                    const double *b = data + ch * 4 * CHUNK + 2 * lane;
#pragma unroll
                    for (int half = 0; half < 2; ++half) {
                        const double2 X = *reinterpret_cast<const double2 *>(b + half * 64);
                        const double2 Y = *reinterpret_cast<const double2 *>(b + CHUNK + half * 64);
                        const double2 Z = *reinterpret_cast<const double2 *>(b + 2 * CHUNK + half * 64);
                        const double2 Q = *reinterpret_cast<const double2 *>(b + 3 * CHUNK + half * 64);
                        pair_f64(px, py, pz, X.x, Y.x, Z.x, Q.x, V[0], Ex[0], Ey[0], Ez[0]);
                        pair_f64(px, py, pz, X.y, Y.y, Z.y, Q.y, V[0], Ex[0], Ey[0], Ez[0]);
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[slot]);
            c = ce;
        }
        if constexpr (F32) {
            V[0] *= prm.q_unscale; Ex[0] *= prm.q_unscale; Ey[0] *= prm.q_unscale; Ez[0] *= prm.q_unscale;
            nuclei_share<1>(prm, elec_s, ws, WS, lane, V, Ex, Ey, Ez);
        }
        const double sV = warp_sum(V[0]), sEx = warp_sum(Ex[0]), sEy = warp_sum(Ey[0]), sEz = warp_sum(Ez[0]);
        if (lane == 0) {
            double *r = red + warp * 4;
            r[0] = sV; r[1] = sEx; r[2] = sEy; r[3] = sEz;
        }
        compute_warps_sync();
        if (warp == 0) {
            double acc = 0.0;
            if (lane < 4)
                for (int s = 0; s < WS; ++s) acc += red[s * 4 + lane];
            server_push(slots, lane, acc, cmd);
        }
        if (leader &&
            !server_collect(prm, sp.mail, slots, threadIdx.x, part_s, red, flag,
                            [] { compute_warps_sync(); }, cmd, t_start)) {
            // a slot never arrived (not expected): retire everybody
            if (threadIdx.x == 0) {
                for (int u = 0; u < 3; ++u) push_st_v2(sp.dev->rec + 2 * u, SERVER_EXIT, 0ull);
                *go_s = SERVER_EXIT;
            }
            compute_warps_sync();
            for (int s = 0; s < npre; ++s, ++k)
                mbar_wait(&full[k % stages], static_cast<uint32_t>(k / stages) & 1u);
            break;
        }
    }
    if (leader && threadIdx.x == 0) {
        __threadfence_system();
        sp.mail->exited = sp.launch_id;
    }
}

// ----------------------------------------------------------------------------- grid-aware server
// The same resident server for environments that have the grid-aware compact copy (charges
// only, qmmm_grid.cuh): 4 / 8 B per cell instead of 16 / 32 B, and the single-point walks of the
// grid kernels (FP32: two z nodes per register pair, GridRowF32N; FP64: the scalar row walk).
// Every warp owns the gchunks lo + w, lo + w + NW, ... of its CTA's slice and loads them itself
// into private slots (FP32 two, FP64 one): no producer warp, no waiting on other warps.  The
// assignment never changes, so a warp whose share fits its slots (configs[2]: 1,024 gchunks over
// 148 CTAs x 8 warps: at most one each) loads it ONCE when the server starts and serves every
// move from shared memory -- no source traffic at all per move; larger shares stream, with the
// first gchunks of the next move prefetched while the CTA waits for it.
// (Measured and rejected in round 2: 16 warps with half a gchunk -- 32 z nodes -- each.  The walk
// halves, but 512-thread barriers, the 16-warp reduction and the barrier around the 256-thread
// collection cost more: 6.52 / 7.14 us per move on configs[2] against 6.05 / 6.83 us.)
constexpr int SERVER_GRID_NW = 8;
template <bool F32>
struct ServerGridLayout {
    static constexpr int SLOTS = F32 ? 2 : 1;                       // per warp
    static constexpr int SLOT_BYTES = F32 ? GRID_NODES * 4 : GRID_NODES * 8;
    static constexpr int STAGE_BYTES = SERVER_GRID_NW * SLOTS * SLOT_BYTES;     // 128 KB
    static constexpr int NUC_STAGED = 64;                           // nuclei of the CTA's share kept in shared memory
    static constexpr int FIXED_BYTES = 16 * 8 /* barriers */ + 256 * 8 /* red / scratch */ + 8 * 8 /* r_new, cmd, flag */ +
                                       NUC_STAGED * 4 * 8 /* staged nuclei */;
    __host__ __device__ static constexpr size_t total(int slices) {
        return static_cast<size_t>(STAGE_BYTES) + FIXED_BYTES + static_cast<size_t>(slices) * 4 * sizeof(double);
    }
};

// prm: grid fields as for the grid kernels (chunks = gchunks, n_chunks = their number, nuc = nuclei
// in units of hz, g_*), P = 1; grid = (1, slices), slices <= SM count, launched cooperatively.
template <bool F32>
__global__ void __launch_bounds__(32 * SERVER_GRID_NW, 1) move_server_grid_kernel(const ServerParams sp) {
    using L = ServerGridLayout<F32>;
    constexpr int NW = SERVER_GRID_NW, NT = 32 * NW, S = L::SLOTS, SB = L::SLOT_BYTES;
    const PairParams &prm = sp.pair;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + L::STAGE_BYTES);          // [NW][S]
    double *red = reinterpret_cast<double *>(full + 16);                           // [256]
    double *elec_s = red + 256;                                                    // [3] r_new, bohr
    volatile unsigned long long *cmd_s = reinterpret_cast<volatile unsigned long long *>(elec_s + 4);
    int *flag = reinterpret_cast<int *>(elec_s + 6);
    double *nuc_s = elec_s + 8;                                                    // [NUC_STAGED][4]: this CTA's nuclei
    double *part_s = nuc_s + L::NUC_STAGED * 4;                                    // leader: [slices][4]
    unsigned long long *slots = reinterpret_cast<unsigned long long *>(prm.partial);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int lo, hi;
    slice_range(prm.n_chunks, prm.slices, blockIdx.y, lo, hi);
    const int cnt = hi - lo > warp ? (hi - lo - warp + NW - 1) / NW : 0;           // gchunks of this warp
    const int segs = prm.g_segs, ny = prm.g_n[1];
    unsigned char *my_slots = smem + static_cast<size_t>(warp) * S * SB;
    uint64_t *my_full = full + warp * S;
    uint32_t phase = 0, pending = 0;                     // bit per slot (warp-uniform)
    // Shares larger than the slots stream through them round robin: the n-th gchunk this warp
    // walks since the server started (its gchunk number n % cnt) sits in slot n % S, and the
    // slot is refilled at once with the gchunk that is walked S steps later.
    unsigned nrun = 0;
    auto load_into = [&](int i, int slot) {              // gchunk number i of this warp -> slot
        if (lane == 0) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            mbar_expect_tx(&my_full[slot], SB);
            tma_bulk_g2s(my_slots + static_cast<size_t>(slot) * SB,
                         prm.chunks + static_cast<size_t>(lo + warp + i * NW) * SB, SB, &my_full[slot]);
        }
        pending |= 1u << slot;
    };
    if (lane == 0) {
        for (int k = 0; k < S; ++k) mbar_init(&my_full[k], 1);
        fence_barrier_init();
    }
    if (threadIdx.x == 0) *cmd_s = sp.start_seq;
    __syncwarp();
    for (int i = 0; i < cnt && i < S; ++i) load_into(i, i);
    // the CTA's share of the nuclei never changes either: its first NUC_STAGED go to shared memory
    // once (a global load and its latency less per move), any more are read from global memory
    int klo, khi;
    slice_range(prm.K, prm.slices, blockIdx.y, klo, khi);
    const int kst = min(khi - klo, L::NUC_STAGED);
    for (int i = threadIdx.x; i < kst * 4; i += NT) nuc_s[i] = prm.nuc[4 * static_cast<int64_t>(klo) + i];
    __syncthreads();

    unsigned long long last = sp.start_seq;
    const bool leader = blockIdx.y == 0;
    const long long t_start = global_ns();
    const bool fine = F32 && prm.g_fine != 0;
    const int n_rows = prm.g_n[0] * prm.g_n[1];
    for (;;) {
        if (warp == 0) {
            const unsigned long long c = server_next_move(sp, leader, lane, last, t_start, elec_s);
            if (lane == 0) *cmd_s = c;
        }
        __syncthreads();
        const unsigned long long cmd = *cmd_s;
        if (cmd == SERVER_EXIT) {
            for (int k = 0; k < S; ++k)                  // no bulk copy may be in flight when the CTA ends
                if (pending & (1u << k)) mbar_wait(&my_full[k], (phase >> k) & 1u);
            break;
        }
        last = cmd;

        // the point in node units (u) and in units of hz (uh: the nuclei, the FP64 walk)
        double u[3], uh[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            u[k] = (elec_s[k] - prm.g_org[k]) * prm.g_inv_h[k];
            uh[k] = u[k] * (k == 0 ? prm.g_sx : (k == 1 ? prm.g_sy : 1.0));
        }
        double V = 0.0, Ex = 0.0, Ey = 0.0, Ez = 0.0;    // this thread's sums, grid units
        if constexpr (F32) {
            // lattice coordinates a (relative to the reference node ir) and residuals dd (units of hz)
            // of the point: lanes 0..2 compute one axis each, everybody gets all three
            float ax, ay, az, ddx, ddy, ddz;
            int irx, iry, irz;
            auto lattice = [&](int xl, int xh, int yl, int yh, int zl, int zh) {
                float a = 0.0f, dd = 0.0f;
                int il = 0;
                if (lane < 3) {
                    il = lane == 0 ? xl : (lane == 1 ? yl : zl);
                    on_lattice(u[lane], il, lane == 0 ? xh : (lane == 1 ? yh : zh), a, dd);
                    dd *= static_cast<float>(lane == 0 ? prm.g_sx : (lane == 1 ? prm.g_sy : 1.0));
                }
                ax = __shfl_sync(0xffffffffu, a, 0); ay = __shfl_sync(0xffffffffu, a, 1); az = __shfl_sync(0xffffffffu, a, 2);
                ddx = __shfl_sync(0xffffffffu, dd, 0); ddy = __shfl_sync(0xffffffffu, dd, 1); ddz = __shfl_sync(0xffffffffu, dd, 2);
                irx = __shfl_sync(0xffffffffu, il, 0); iry = __shfl_sync(0xffffffffu, il, 1); irz = __shfl_sync(0xffffffffu, il, 2);
            };
            if (!fine) lattice(0, prm.g_n[0] - 1, 0, prm.g_n[1] - 1, 0, prm.g_n[2] - 1);
            float vv = 0.0f, tt = 0.0f, ex = 0.0f, ey = 0.0f, ez = 0.0f, cc = 0.0f;
            int run = 0;
            auto flush = [&]() {
                V += 1.5 * static_cast<double>(vv) - 0.5 * static_cast<double>(tt) - static_cast<double>(cc);
                Ex += static_cast<double>(ex); Ey += static_cast<double>(ey); Ez += static_cast<double>(ez);
                vv = tt = ex = ey = ez = cc = 0.0f;
                run = 0;
            };
            for (int i = 0; i < cnt; ++i, ++nrun) {
                const int slot = cnt > S ? static_cast<int>(nrun % S) : i, g = lo + warp + i * NW;
                const int tl = g / segs, sg = g - tl * segs;
                const int rw = tl * 32 + lane, rx = rw / ny;
                if (fine) {                              // the lattice of THIS gchunk's nodes
                    const int r0 = tl * 32, r1 = min(r0 + 31, n_rows - 1), x0 = r0 / ny, x1 = r1 / ny;
                    lattice(x0, x1, x0 == x1 ? r0 - x0 * ny : 0, x0 == x1 ? r1 - x0 * ny : ny - 1,
                            sg * GRID_ZS, sg * GRID_ZS + GRID_ZS - 1);
                }
                if (pending & (1u << slot)) {
                    mbar_wait(&my_full[slot], (phase >> slot) & 1u);
                    phase ^= 1u << slot;
                    pending &= ~(1u << slot);
                }
                const float *data = reinterpret_cast<const float *>(my_slots + static_cast<size_t>(slot) * SB);
                const float dxs = (ax - static_cast<float>(rx - irx)) * static_cast<float>(prm.g_sx);   // exact, then hx/hz
                const float dys = (ay - static_cast<float>(rw - rx * ny - iry)) * static_cast<float>(prm.g_sy);
                GridRowF32N row;
                row.start(az - static_cast<float>(sg * GRID_ZS - irz), fmaf(dys, dys, fmaf(dxs, dxs, 1e-30f)));
                float v1, t1;
                row.run(data + 4 * lane, GRID_ZS / 4, v1, t1);
                const float s1 = row.S.x + row.S.y;
                const float exg = dxs * s1, eyg = dys * s1, ezg = row.SZ.x + row.SZ.y;
                vv += v1; tt += t1; ex += exg; ey += eyg; ez += ezg;
                if (fine) cc = fmaf(exg, ddx, fmaf(eyg, ddy, fmaf(ezg, ddz, cc)));
                __syncwarp();                            // every lane has read the slot
                if (cnt > S) load_into(i + S < cnt ? i + S : i + S - cnt, slot);   // (wraps to the next move)
                if (++run == GRID_FLUSH) flush();
            }
            if (run) flush();
            // whole-grid lattice: V(u) = V(a) - E(a) . dd (the local lattice did it gchunk by gchunk)
            if (!fine) V -= Ex * static_cast<double>(ddx) + Ey * static_cast<double>(ddy) + Ez * static_cast<double>(ddz);
            V *= prm.q_unscale; Ex *= prm.q_unscale; Ey *= prm.q_unscale; Ez *= prm.q_unscale;
        } else {
            for (int i = 0; i < cnt; ++i, ++nrun) {
                const int slot = cnt > S ? static_cast<int>(nrun % S) : i, g = lo + warp + i * NW;
                const int tl = g / segs, sg = g - tl * segs;
                const int rw = tl * 32 + lane, rx = rw / ny;
                if (pending & (1u << slot)) {
                    mbar_wait(&my_full[slot], (phase >> slot) & 1u);
                    phase ^= 1u << slot;
                    pending &= ~(1u << slot);
                }
                const double *b = reinterpret_cast<const double *>(my_slots + static_cast<size_t>(slot) * SB) + 2 * lane;
                const double dx = uh[0] - static_cast<double>(rx) * prm.g_sx;
                const double dy = uh[1] - static_cast<double>(rw - rx * ny) * prm.g_sy;
                const double rxy2 = fma(dy, dy, fma(dx, dx, 1e-200));
                double azb = uh[2] - static_cast<double>(sg * GRID_ZS), Sx = 0.0, SZ = 0.0;
#pragma unroll 1
                for (int k4 = 0; k4 < GRID_ZS / 4; ++k4) {
                    const double2 Qa = *reinterpret_cast<const double2 *>(b + (2 * k4) * 64);
                    const double2 Qb = *reinterpret_cast<const double2 *>(b + (2 * k4 + 1) * 64);
                    const double qs[4] = {Qa.x, Qa.y, Qb.x, Qb.y};
#pragma unroll
                    for (int t = 0; t < 4; ++t) {
                        const double dz = t == 0 ? azb : azb - static_cast<double>(t);
                        const double y = rsqrt_refined_f64(fma(dz, dz, rxy2));
                        const double p = qs[t] * y;
                        V += p;
                        const double sv = p * (y * y);
                        Sx += sv;
                        SZ = fma(sv, dz, SZ);
                    }
                    azb -= 4.0;
                }
                Ex = fma(dx, Sx, Ex);
                Ey = fma(dy, Sx, Ey);
                Ez += SZ;
                __syncwarp();
                if (cnt > S) load_into(i + S < cnt ? i + S : i + S - cnt, slot);
            }
        }
        // nuclei of this CTA's share (units of hz), FP64, thread-strided
        for (int j = threadIdx.x; j < khi - klo; j += NT) {
            const double *nu = j < kst ? nuc_s + 4 * j : prm.nuc + 4 * static_cast<int64_t>(klo + j);
            const double2 a = *reinterpret_cast<const double2 *>(nu);
            const double2 b2 = *reinterpret_cast<const double2 *>(nu + 2);
            pair_f64(uh[0], uh[1], uh[2], a.x, a.y, b2.x, b2.y, V, Ex, Ey, Ez);
        }
        const double sV = warp_sum(V), sEx = warp_sum(Ex), sEy = warp_sum(Ey), sEz = warp_sum(Ez);
        if (lane == 0) {
            double *r = red + warp * 4;
            r[0] = sV; r[1] = sEx; r[2] = sEy; r[3] = sEz;
        }
        __syncthreads();
        if (warp == 0) {
            double acc = 0.0;
            if (lane < 4) {
                for (int w = 0; w < NW; ++w) acc += red[w * 4 + lane];
                acc *= lane ? prm.g_scaleE : prm.g_scaleV;       // grid units -> hartree, hartree / bohr
            }
            server_push(slots, lane, acc, cmd);
        }
        __syncthreads();                                 // red is reused by the collection
        if (leader && !server_collect(prm, sp.mail, slots, threadIdx.x, part_s, red, flag,
                                      [] { __syncthreads(); }, cmd, t_start)) {
            if (threadIdx.x == 0) {                      // a slot never arrived (not expected): retire everybody
                for (int u = 0; u < 3; ++u) push_st_v2(sp.dev->rec + 2 * u, SERVER_EXIT, 0ull);
                if (prm.dev_err) *reinterpret_cast<volatile int *>(prm.dev_err) = 1;
            }
            for (int k = 0; k < S; ++k)
                if (pending & (1u << k)) mbar_wait(&my_full[k], (phase >> k) & 1u);
            break;
        }
    }
    if (leader && threadIdx.x == 0) {
        __threadfence_system();
        sp.mail->exited = sp.launch_id;
    }
}

}  // namespace qmmm
