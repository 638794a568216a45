// qmmm_server.cuh -- resident "move server" for the paper's deployed loop:
// every Monte-Carlo step the host sends ONE new electron position r_new and receives U_ES.
//
// A kernel launch costs ~10 us host-to-host on an idle GPU, as much as the evaluation itself
// (11 us at 2.08 M sources).  The server is launched once (cooperatively: one CTA per SM, all
// resident) and then serves moves from a pinned, device-mapped mailbox:
//
//   host   : writes {s, r, s} into the request line; spins until the answer line carries s
//   leader : one warp of CTA 0 polls the request line over PCIe (one transaction), copies r
//            to device memory, publishes s in cmd
//   all    : poll cmd (L2), run their source slice exactly like pair_kernel<REAL,1> (TMA ring,
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
    double elec[3];                        // r_new of the published move
    unsigned long long cmd;                // last published move number, or EXIT
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
                if (c != SERVER_EXIT && lane >= 1 && lane <= 3) {
                    const double v = __longlong_as_double(static_cast<long long>(w));
                    elec_s[lane - 1] = v;
                    sp.dev->elec[lane - 1] = v;
                    __threadfence();
                }
                __syncwarp();
                if (lane == 0) *reinterpret_cast<volatile unsigned long long *>(&sp.dev->cmd) = c;
            } else {
                for (;;) {
                    if (lane == 0) c = *reinterpret_cast<volatile unsigned long long *>(&sp.dev->cmd);
                    c = __shfl_sync(0xffffffffu, c, 0);
                    if (c != last) break;
                    const long long now = __shfl_sync(0xffffffffu, global_ns(), 0);
                    if (now - t_start > SERVER_HARD_NS) {
                        c = SERVER_EXIT;
                        break;
                    }
                }
                if (c != SERVER_EXIT) {
                    __threadfence();
                    if (lane < 3) elec_s[lane] = __ldcg(&sp.dev->elec[lane]);
                }
            }
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
                *reinterpret_cast<volatile unsigned long long *>(&sp.dev->cmd) = SERVER_EXIT;
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

}  // namespace qmmm
