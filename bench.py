#!/usr/bin/env python
"""bench.py -- pair-interactions/s of the QM/MM electrostatic potential + field hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl reference]

A "step" is one pass of the whole hot path (one fused launch: pair kernel incl. nuclei and the
cross-CTA sum) over one batch of synthetic evaluation points of the chosen BASELINE.json
configuration.  Rank 0 prints ONE JSON line.  See DESIGN.md "Measurement".

* value      : whole-job pair-interactions/s (G/s), inputs resident in HBM, per-step CUDA
               events on the launch stream, L2 flushed between steps, max over ranks.
* e2e        : same metric through qmmm_field_eval_host (the paper's per-step loop,
               PAPER.md:117): pinned HOST buffers, H2D + kernels + D2H + stream sync timed.
* roofline   : the pair kernel (events recorded by the library around its launch)
               against the FMA-lane rate measured by the library's microbenchmark in the
               same process ("bound": "alu").
* cpu_baseline: the CPU oracle as it stands on a bounded sample of the same workload.
* --impl reference : times the oracle (the only reference this tier has) on host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1011_4687_b200.workloads import CONFIG_SPECS, make_workload  # noqa: E402

METRIC = "pair-interactions/s"
UNIT = "Gpair/s"
# Algorithmic FMA-pipe lane operations per pair (DESIGN.md sections 5, 5b).  Source list, FP64:
# SURVEY.md 8(a), 18.  FP32: the Newton step is applied to the sum (V = (3 sum a - sum c r^2) / 2,
# one fma per pair), which leaves 3 sub, 3 for r^2, a, V0, y0^2, c, T, 3 fma for E = 14 (the
# per-pair step of SURVEY.md 8(a) costs 17).  Grid layout: dx, dy and dx^2 + dy^2 are constants
# of a z row: dz, r^2, a, V0, y0^2, c, sum c, sum c dz, T = 9 (FP32) or, with the per-pair cubic
# refinement, 13 (FP64).
# Grid kernels that tabulate dz = u_z - k in shared memory (it depends on the point and the z
# node only; qmmm_field_info.last_dz_table says whether the last launch did) load it instead of
# stepping it: one operation less, 8 (FP32) / 12 (FP64).
SLOTS = {("list", "fp32"): 14, ("list", "fp64"): 18, ("grid", "fp32"): 9, ("grid", "fp64"): 13}
# FP64 potential only (E = NULL).  List: 3 sub, 3 for r^2, 5 for the refinement, fma(q, y, V) = 12
# (round 1 printed 13; the SASS count of tests/test_sass_slots.py says 12).
SLOTS_V_ONLY = {"list": 12, "grid": 8}
SLOTS_V_ONLY_F32_GRID = 6                  # FP32 potential only, batched grid kernel: r^2, a, V0, y0^2, c, T
# Floating-point operations per pair of the same kernels (an fma counts 2), for readers who count
# flops (SURVEY.md 8(d) "eta_flop").  (layout, precision, dz table, potential only).  FP32 grid with
# the table, V + E: r^2 2 (1 when it is an add: accurate V), a 1, V0 1, y0^2 1, c 1, T 2, S 1, SZ 2 = 11;
# FP64 grid with the table: r^2 2, refinement 8, p 1, V 1, y^2 1, s 1, S 1, SZ 2 = 17.
FLOPS = {("list", "fp32", False, False): 21, ("list", "fp64", False, False): 27, ("list", "fp64", False, True): 19,
         ("grid", "fp32", False, False): 12, ("grid", "fp32", True, False): 11, ("grid", "fp32", True, True): 7,
         ("grid", "fp64", False, False): 18, ("grid", "fp64", True, False): 17,
         ("grid", "fp64", False, True): 12, ("grid", "fp64", True, True): 11}


def flops_for(layout, prec, info, v_only=False):
    key = (layout, prec, bool(info.get("last_dz_table")) and layout == "grid", bool(v_only))
    n = FLOPS.get(key, FLOPS.get((layout, prec, key[2], False)))
    if key == ("grid", "fp32", True, False) and info.get("last_accurate_v"):
        n -= 1                                   # accurate V: r^2 = rxy2 + z2 is an add, not an fma
    return n


def slots_for(layout, prec, info, v_only=False):
    """Algorithmic FMA-pipe lane operations per pair of the kernel the last launch ran."""
    n = SLOTS_V_ONLY[layout] if v_only else SLOTS[(layout, prec)]
    return n - 1 if (layout == "grid" and info.get("last_dz_table")) else n

KERNEL = {("list", "fp32"): "pair_kernel_f32x2", ("list", "fp64"): "pair_kernel<double>",
          ("grid", "fp32"): "grid_kernel_f32x2", ("grid", "fp64"): "grid_kernel_f64"}
DTYPE = {"fp32": "f32 (f64 accumulation)", "fp64": "f64"}
WORKLOAD_NAME = {i: f"configs[{i}] {s['name']}" for i, s in CONFIG_SPECS.items()}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index (0-4)")
    ap.add_argument("--precision", default=None, choices=["fp32", "fp64"])
    ap.add_argument("--layout", default="auto", choices=["auto", "list", "grid"],
                    help="source copy the kernels read: list of positions, or the grid-aware "
                         "compact format (auto: grid when the cells are grid nodes and the "
                         "batch has many points)")
    ap.add_argument("--potential-only", action="store_true",
                    help="E = NULL: the potential alone (PAPER.md Eq. 4 proper); fewer operations per pair")
    ap.add_argument("--fast-v", action="store_true",
                    help="qmmm_field_set_accurate_v(h, 0): the batched FP32 grid V + E kernel without the accurate-V "
                         "arithmetic (6 %% faster; misses the batch-total energy criterion, DESIGN.md section 6)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-sweep", action="store_true",
                    help="skip the per-config table (all five configs) at N=1")
    ap.add_argument("--cpu-sample-pairs", type=float, default=6e9,
                    help="pairs in the cpu_baseline sample (about 10-30 s of host time)")
    return ap.parse_args()


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks",
               0x100: "display_clock", 0x10: "sync_boost"}

    def __init__(self, index: int, period: float = 0.02):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        while not self._stop_evt.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                mask = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
                self.power.append(self.nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._stop_evt.set()
        if self.is_alive():
            self.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# ------------------------------------------------------------------------ oracle timing
def oracle_sample_rate(w, sample_pairs: float, seed: int = 99, nthreads: int = 0):
    """Times the CPU oracle (as it stands) on a seeded subsample of the evaluation points
    (nthreads = 0: all host cores this process may use)."""
    import oracle
    oracle.build()
    pts = w.elec_xyz.reshape(-1, 3)
    per_point = w.M + w.K
    n = int(max(1, min(len(pts), round(sample_pairs / per_point))))
    rng = np.random.default_rng(seed)
    idx = np.sort(rng.choice(len(pts), size=n, replace=False))
    sub = np.ascontiguousarray(pts[idx])
    t0 = time.perf_counter()
    # all host cores this process may use (torchrun sets OMP_NUM_THREADS=1 by default)
    res = oracle.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, sub,
                       nthreads=nthreads or len(os.sched_getaffinity(0)))
    dt = time.perf_counter() - t0
    pairs = n * per_point
    return dict(pairs=pairs, seconds=dt, rate=pairs / dt, threads=res.threads, n_points=n,
                n_total=len(pts))


def run_reference(args):
    """--impl reference: the oracle on host cores, same metric/config; rank 0 only."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    w = make_workload(args.config)
    prec = args.precision or w.precisions[0]
    # each step: a bounded sample sized so warmup+steps finish within a few minutes
    per_step_pairs = min(args.cpu_sample_pairs / 4, 1.5e9)
    for _ in range(args.warmup):
        oracle_sample_rate(w, per_step_pairs / 8)
    times, pairs, threads, npts = [], 0, 1, 0
    for s in range(args.steps):
        r = oracle_sample_rate(w, per_step_pairs, seed=1000 + s)
        times.append(r["seconds"]); pairs += r["pairs"]; threads = r["threads"]; npts = r["n_points"]
    total = sum(times)
    value = pairs / total / 1e9
    sample = f"{npts} of {w.P} evaluation points per step x all {w.M}+{w.K} sources"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOAD_NAME[args.config], "precision": "fp64 (oracle)",
                   "M": w.M, "K": w.K, "W": w.W, "N": w.N,
                   "note": "CPU oracle (plain FP64 Kahan double loop), bounded sample per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------ GPU arm
class L2Flusher:
    """Writes a buffer larger than the 126 MB L2 between timed steps."""

    def __init__(self, torch, nbytes=256 << 20):
        self.buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        self.k = 0

    def __call__(self):
        self.k = (self.k + 1) & 0x7F
        self.buf.fill_(self.k)


def probe_peaks(B):
    ffma, _ = B.qmmm_probe_peak(0)
    dfma, _ = B.qmmm_probe_peak(1)
    mufu, _ = B.qmmm_probe_peak(2)
    return {"ffma_lane_ops_per_s": ffma, "dfma_lane_ops_per_s": dfma, "mufu_lane_ops_per_s": mufu}


def probe_memory_and_launch(B):
    """SURVEY.md 8(d) "Timing protocol": empty-kernel launch + sync latency and the read
    bandwidth over a 33 MB (L2-resident) and a 537 MB (HBM) buffer, same process."""
    launch_s, _ = B.qmmm_probe_peak(3)
    l2, _ = B.qmmm_probe_peak(4)
    hbm, _ = B.qmmm_probe_peak(5)
    out = {"empty_launch_plus_sync_us": launch_s * 1e6, "l2_read_GBps_33MB": l2 / 1e9,
           "hbm_read_GBps_537MB": hbm / 1e9}
    # Floor of the per-move host path (r_new in, U_ES out, every step): 1,000
    # sequential single-point moves through the resident move server against an environment of
    # ONE cell -- request written by the host, answer visible to the host, next to no evaluation
    # in between: what the pinned-mailbox round trip over PCIe costs by itself.
    one_xyz = np.array([[7.0, 0.0, 0.0]]); one_q = np.array([-0.5])
    h1 = B.qmmm_field_create(one_xyz, one_q, None, None, 1)
    try:
        rng = np.random.default_rng(5)
        walk = np.ascontiguousarray(rng.normal(size=(1000, 3)) * 0.5)
        hV = np.zeros(1000); hE = np.zeros((1000, 3))
        for prec in ("fp32", "fp64"):
            B.qmmm_field_eval_moves_host(h1, walk[:50], 50, 1, hV, hE, prec)
            secs = B.qmmm_field_eval_moves_host(h1, walk, 1000, 1, hV, hE, prec)
            out[f"host_move_round_trip_us_one_cell_{prec}"] = secs * 1e6 / 1000
    finally:
        B.qmmm_field_destroy(h1)
    mp = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(mp):
        try:
            out["measured_peaks_hbm_GBps"] = json.load(open(mp))["hbm_gbs"]
        except Exception:
            pass
    return out


def time_steps(torch, B, h, batches, W, N, prec, steps, warmup, flush, stream, want_E=True):
    """Per-step CUDA events on the launch stream; returns (step_ms list, pair_ms list)."""
    P = W * N
    V = torch.empty(P, dtype=torch.float64, device="cuda")
    E = torch.empty((P, 3), dtype=torch.float64, device="cuda") if want_E else None
    for i in range(warmup):
        B.qmmm_field_eval(h, batches[i % len(batches)], W, N, V, E, prec, stream)
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
           for _ in range(steps)]
    pair_ms = []
    for i in range(steps):
        if flush is not None:
            flush()
        evs[i][0].record(stream)
        B.qmmm_field_eval(h, batches[i % len(batches)], W, N, V, E, prec, stream)
        evs[i][1].record(stream)
        pair_ms.append(B.qmmm_field_last_timing(h)[0])      # waits for this eval
    torch.cuda.synchronize()
    return [a.elapsed_time(b) for a, b in evs], pair_ms, (V, E)


def sweep_all_configs(torch, B, peaks, main_cfg, main_result, mem=None):
    """Per-config table (N=1): ms per evaluation, Gpair/s and FMA-pipe fraction for every
    BASELINE.json configuration and precision; config 2 also as the QMC host loop."""
    out = []
    stream = torch.cuda.current_stream()
    flush = L2Flusher(torch)
    for idx in sorted(CONFIG_SPECS):
        w = make_workload(idx)
        W, N = (1, 1) if w.sequential else (w.W, w.N)
        P = W * N
        h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, P)
        try:
            pts = torch.from_numpy(w.elec_xyz.reshape(-1, 3)).cuda()
            batches = [pts[i:i + 1].contiguous() for i in range(8)] if w.sequential else [pts]
            has_grid = B.qmmm_field_get_grid_info(h)["present"]
            # the automatic layout, then the other one for comparison where a grid copy exists
            runs = [(prec, "auto") for prec in w.precisions]
            if has_grid and not w.sequential:
                runs += [(prec, "other") for prec in w.precisions]
            for prec, which in runs:
                reps = 5 if idx >= 3 else 30
                B.qmmm_field_set_layout(h, "auto")
                B.qmmm_field_set_timing(h, True)
                if which == "other":
                    used = [r["layout"] for r in out if r["config"] == idx and r["precision"] == prec][0]
                    B.qmmm_field_set_layout(h, "list" if used == "grid" else "grid")
                step_ms, pair_ms, _ = time_steps(torch, B, h, batches, W, N, prec, reps, 3, flush, stream)
                layout = B.qmmm_field_get_grid_info(h)["last_layout"]
                pairs = P * (w.M + w.K)
                peak = peaks["ffma_lane_ops_per_s" if prec == "fp32" else "dfma_lane_ops_per_s"]
                info = B.qmmm_field_get_info(h)
                slots = slots_for(layout, prec, info)
                row = {"config": idx, "name": w.name, "precision": prec, "layout": layout,
                       "layout_choice": "auto" if which == "auto" else "forced",
                       "points": P, "M": w.M,
                       "K": w.K, "pairs_per_eval": pairs,
                       "ms_per_eval_median": float(np.median(step_ms)),
                       "ms_per_eval_min": float(np.min(step_ms)),
                       "pair_kernel_ms_median": float(np.median(pair_ms)),
                       "gpairs_per_s": pairs / np.median(step_ms) / 1e6,
                       "slots_per_pair": slots, "dz_table": bool(info["last_dz_table"]),
                       "fma_pipe_frac": pairs * slots / (np.median(step_ms) * 1e-3) / peak,
                       "plan": info["last_plan"]}
                if w.sequential:
                    # (i) 1,000 back-to-back evaluations, positions resident on the device
                    B.qmmm_field_set_timing(h, False)
                    V = torch.empty(1, dtype=torch.float64, device="cuda")
                    E = torch.empty((1, 3), dtype=torch.float64, device="cuda")
                    walk = [pts[i:i + 1].contiguous() for i in range(len(pts))]
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    torch.cuda.synchronize()
                    e0.record(stream)
                    for p in walk:
                        B.qmmm_field_eval(h, p, 1, 1, V, E, prec, stream)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    row["us_per_eval_1000_back_to_back"] = e0.elapsed_time(e1) * 1e3 / len(walk)
                    # (i') the same 1,000 launches captured once in a CUDA graph and replayed: no
                    # host launch cost per evaluation (the Python / ctypes call is ~12 us)
                    gr = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(gr):
                        for p in walk:
                            B.qmmm_field_eval(h, p, 1, 1, V, E, prec)
                    gr.replay()
                    torch.cuda.synchronize()
                    cs = torch.cuda.current_stream()
                    e0.record(cs)
                    gr.replay()
                    e1.record(cs)
                    torch.cuda.synchronize()
                    row["us_per_eval_1000_cuda_graph"] = e0.elapsed_time(e1) * 1e3 / len(walk)
                    del gr
                    # (i'') the same graph with overlapped evaluations (qmmm_field_set_overlap:
                    # programmatic dependent launch, evaluation n + 1 starts while n finishes)
                    B.qmmm_field_set_overlap(h, True)
                    gr = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(gr):
                        for p in walk:
                            B.qmmm_field_eval(h, p, 1, 1, V, E, prec)
                    gr.replay()
                    torch.cuda.synchronize()
                    e0.record(cs)
                    gr.replay()
                    e1.record(cs)
                    torch.cuda.synchronize()
                    row["us_per_eval_1000_cuda_graph_overlap"] = e0.elapsed_time(e1) * 1e3 / len(walk)
                    del gr
                    B.qmmm_field_set_overlap(h, False)
                    # (i-3) no graph: ONE library call (qmmm_field_eval_moves) issues the 1,000
                    # overlapped launches from C
                    nm = len(pts)
                    Vm = torch.empty(nm, dtype=torch.float64, device="cuda")
                    Em = torch.empty((nm, 3), dtype=torch.float64, device="cuda")
                    B.qmmm_field_eval_moves(h, pts, nm, 1, Vm, Em, prec, stream)
                    torch.cuda.synchronize()
                    e0.record(stream)
                    B.qmmm_field_eval_moves(h, pts, nm, 1, Vm, Em, prec, stream)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    row["us_per_eval_1000_eval_moves_call"] = e0.elapsed_time(e1) * 1e3 / nm
                    # (ii) the QMC loop of PAPER.md:117: r_new in (24 B), U out (32 B), every move;
                    # the loop itself runs inside the library (qmmm_field_eval_moves_host)
                    hp = np.ascontiguousarray(w.elec_xyz.reshape(-1, 3))
                    hV = np.zeros(len(hp)); hE = np.zeros((len(hp), 3))
                    B.qmmm_field_eval_moves_host(h, hp[:50], 50, 1, hV, hE, prec, stream)
                    secs = B.qmmm_field_eval_moves_host(h, hp, len(hp), 1, hV, hE, prec, stream)
                    row["us_per_eval_host_loop"] = secs * 1e6 / len(hp)
                    if layout == "grid":        # charges only, empty cells included
                        gi = B.qmmm_field_get_grid_info(h)
                        bytes_eval = gi["bytes_fp32" if prec == "fp32" else "bytes_fp64"]
                    else:
                        bytes_eval = w.M * (16 if prec == "fp32" else 32)
                    row["source_bytes_per_eval"] = bytes_eval
                    row["source_GBps_back_to_back"] = bytes_eval / (row["us_per_eval_1000_back_to_back"] * 1e-6) / 1e9
                    row["source_GBps_cuda_graph"] = bytes_eval / (row["us_per_eval_1000_cuda_graph"] * 1e-6) / 1e9
                    row["source_GBps_cuda_graph_overlap"] = bytes_eval / (row["us_per_eval_1000_cuda_graph_overlap"] * 1e-6) / 1e9
                    if mem:
                        # the single-electron path is bound by source bandwidth and latency, not by
                        # the FMA pipe: its rates against the measured read bandwidths
                        for k in ("back_to_back", "cuda_graph", "cuda_graph_overlap"):
                            row[f"frac_of_l2_read_bw_{k}"] = row[f"source_GBps_{k}"] / mem["l2_read_GBps_33MB"]
                            row[f"frac_of_hbm_read_bw_{k}"] = row[f"source_GBps_{k}"] / mem["hbm_read_GBps_537MB"]
                        row["source_bytes_fit_l2"] = bool(bytes_eval < 100e6)
                        row["empty_launch_plus_sync_us"] = mem["empty_launch_plus_sync_us"]
                        # the host loop against its floor (the same loop on a one-cell environment)
                        row["us_per_eval_host_loop_floor"] = mem[f"host_move_round_trip_us_one_cell_{prec}"]
                        row["us_per_eval_host_loop_above_floor"] = (row["us_per_eval_host_loop"]
                                                                    - mem[f"host_move_round_trip_us_one_cell_{prec}"])
                if not w.sequential and idx <= 1:
                    # launch-free figure for the small configurations (an evaluation is of the
                    # size of one kernel launch): 200 evaluations captured once in a CUDA graph
                    # and replayed, sources warm in L2 as in a running QMC job
                    B.qmmm_field_set_timing(h, False)
                    V = torch.empty(P, dtype=torch.float64, device="cuda")
                    E = torch.empty((P, 3), dtype=torch.float64, device="cuda")
                    gr = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(gr):
                        for _ in range(200):
                            B.qmmm_field_eval(h, pts, W, N, V, E, prec)
                    gr.replay()
                    torch.cuda.synchronize()
                    cs = torch.cuda.current_stream()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(cs)
                    gr.replay()
                    e1.record(cs)
                    torch.cuda.synchronize()
                    us = e0.elapsed_time(e1) * 1e3 / 200
                    row["us_per_eval_200_cuda_graph"] = us
                    row["fma_pipe_frac_cuda_graph"] = pairs * slots / (us * 1e-6) / peak
                    del gr
                    # the same with overlapped evaluations (programmatic dependent launch)
                    B.qmmm_field_set_overlap(h, True)
                    gr = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(gr):
                        for _ in range(200):
                            B.qmmm_field_eval(h, pts, W, N, V, E, prec)
                    gr.replay()
                    torch.cuda.synchronize()
                    e0.record(cs)
                    gr.replay()
                    e1.record(cs)
                    torch.cuda.synchronize()
                    B.qmmm_field_set_overlap(h, False)
                    us = e0.elapsed_time(e1) * 1e3 / 200
                    info_o = B.qmmm_field_get_info(h)       # the overlapped plan (light CTAs) and its kernel
                    slots_o = slots_for(layout, prec, info_o)
                    row["us_per_eval_200_cuda_graph_overlap"] = us
                    row["slots_per_pair_overlap"] = slots_o
                    row["plan_overlap"] = info_o["last_plan"]
                    row["fma_pipe_frac_cuda_graph_overlap"] = pairs * slots_o / (us * 1e-6) / peak
                    del gr
                out.append(row)
                if prec == "fp32" and not w.sequential and idx == 3 and layout == "grid":
                    # FP32 potential only (E = NULL): the paper's own computation, Eq. 4; the batched
                    # grid kernel needs 6 FMA-pipe operations + 1 MUFU per pair: the XU pipe bounds it
                    B.qmmm_field_set_timing(h, True)
                    step_ms, pair_ms, _ = time_steps(torch, B, h, batches, W, N, prec, reps, 3, flush,
                                                     stream, want_E=False)
                    info = B.qmmm_field_get_info(h)
                    out.append({"config": idx, "name": w.name, "precision": "fp32 potential-only",
                                "layout": layout, "layout_choice": "auto" if which == "auto" else "forced",
                                "points": P, "M": w.M, "K": w.K, "pairs_per_eval": pairs,
                                "ms_per_eval_median": float(np.median(step_ms)),
                                "pair_kernel_ms_median": float(np.median(pair_ms)),
                                "gpairs_per_s": pairs / np.median(step_ms) / 1e6,
                                "slots_per_pair": SLOTS_V_ONLY_F32_GRID,
                                "fma_pipe_frac": pairs * SLOTS_V_ONLY_F32_GRID / (np.median(step_ms) * 1e-3) / peak,
                                "xu_pipe_frac": pairs / (np.median(step_ms) * 1e-3) / peaks["mufu_lane_ops_per_s"],
                                "kernel_symbol": info.get("last_kernel", ""), "plan": info["last_plan"]})
                    # V + E without the accurate-V arithmetic (qmmm_field_set_accurate_v(h, 0)): the
                    # kernel of rounds 1-2 before the batch-total criterion was met
                    B.qmmm_field_set_accurate_v(h, False)
                    step_ms, pair_ms, _ = time_steps(torch, B, h, batches, W, N, prec, reps, 3, flush, stream)
                    info = B.qmmm_field_get_info(h)
                    B.qmmm_field_set_accurate_v(h, True)
                    out.append({"config": idx, "name": w.name, "precision": "fp32, accurate_v off",
                                "layout": layout, "layout_choice": "auto" if which == "auto" else "forced",
                                "points": P, "M": w.M, "K": w.K, "pairs_per_eval": pairs,
                                "ms_per_eval_median": float(np.median(step_ms)),
                                "pair_kernel_ms_median": float(np.median(pair_ms)),
                                "gpairs_per_s": pairs / np.median(step_ms) / 1e6,
                                "slots_per_pair": slots,
                                "fma_pipe_frac": pairs * slots / (np.median(step_ms) * 1e-3) / peak,
                                "xu_pipe_frac": pairs / (np.median(step_ms) * 1e-3) / peaks["mufu_lane_ops_per_s"],
                                "kernel_symbol": info.get("last_kernel", ""), "plan": info["last_plan"]})
                if prec == "fp64" and not w.sequential and idx in (1, 4):
                    # potential only (E = NULL): the paper's own computation, Eq. 4; 12 (list) or
                    # 8 (grid; 7 with the dz table) DP slots
                    B.qmmm_field_set_timing(h, True)
                    step_ms, pair_ms, _ = time_steps(torch, B, h, batches, W, N, prec, reps, 3, flush,
                                                     stream, want_E=False)
                    layout = B.qmmm_field_get_grid_info(h)["last_layout"]
                    info = B.qmmm_field_get_info(h)
                    vslots = slots_for(layout, prec, info, v_only=True)
                    out.append({"config": idx, "name": w.name, "precision": "fp64 potential-only",
                                "layout": layout, "layout_choice": "auto" if which == "auto" else "forced",
                                "points": P, "M": w.M, "K": w.K, "pairs_per_eval": pairs,
                                "ms_per_eval_median": float(np.median(step_ms)),
                                "ms_per_eval_min": float(np.min(step_ms)),
                                "pair_kernel_ms_median": float(np.median(pair_ms)),
                                "gpairs_per_s": pairs / np.median(step_ms) / 1e6,
                                "fma_pipe_frac": pairs * vslots / (np.median(step_ms) * 1e-3) / peak,
                                "slots_per_pair": vslots, "dz_table": bool(info["last_dz_table"]),
                                "plan": info["last_plan"]})
        finally:
            B.qmmm_field_destroy(h)
        del w
    return out


def run_ours(args):
    import torch
    rank, world, local = dist_env()
    torch.cuda.set_device(local % max(1, torch.cuda.device_count()))
    dist = None
    if world > 1:
        import torch.distributed as dist
        # QMMM_BENCH_BACKEND=gloo lets the multi-rank control flow be exercised on a box with
        # fewer GPUs than ranks (ranks then share a device; they never wait on one another)
        backend = os.environ.get("QMMM_BENCH_BACKEND", "nccl")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
    from paper_1011_4687_b200 import binding as B     # raises if the CUDA library is missing
    from paper_1011_4687_b200.workloads import draw_points

    w = make_workload(args.config)
    prec = args.precision or w.precisions[0]
    W, N = (1, 1) if w.sequential else (w.W, w.N)
    P = W * N
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # the environment is replicated on every GPU; each rank evaluates its own walkers
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, P)
    B.qmmm_field_set_layout(h, args.layout)
    B.qmmm_field_set_timing(h, True)
    if args.fast_v:
        B.qmmm_field_set_accurate_v(h, False)
    n_batches = 4
    host_batches = [draw_points(args.config, W, N, seed=1 + 97 * rank + b).reshape(-1, 3)
                    for b in range(n_batches)]
    batches = [torch.from_numpy(b).cuda() for b in host_batches]
    flush = L2Flusher(torch)
    peaks0 = probe_peaks(B)

    # ---- device-resident timing -------------------------------------------------------
    sampler = ClockSampler(torch.cuda.current_device())
    barrier()
    sampler.start()
    step_ms, pair_ms, _ = time_steps(torch, B, h, batches, W, N, prec, args.steps, args.warmup,
                                     flush, stream, want_E=not args.potential_only)
    barrier()
    clocks = sampler.stop()
    peaks1 = probe_peaks(B)
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    pairs_step_rank = P * (w.M + w.K)
    value = world * pairs_step_rank * args.steps / (total_ms * 1e-3) / 1e9
    info = B.qmmm_field_get_info(h)
    layout = B.qmmm_field_get_grid_info(h)["last_layout"]

    # ---- end to end: host buffers through the C ABI -----------------------------------
    B.qmmm_field_set_timing(h, False)
    pin_in = [torch.from_numpy(b.copy()).pin_memory() for b in host_batches]
    pin_out = torch.zeros(P * 4, dtype=torch.float64).pin_memory()
    hV, hE = pin_out[:P], (None if args.potential_only else pin_out[P:].reshape(P, 3))
    for i in range(args.warmup):
        B.qmmm_field_eval_host(h, pin_in[i % n_batches], W, N, hV, hE, prec, stream)
    barrier()
    t0 = time.perf_counter()
    for i in range(args.steps):
        B.qmmm_field_eval_host(h, pin_in[i % n_batches], W, N, hV, hE, prec, stream)
    barrier()
    e2e_s = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(e2e_s, op=dist.ReduceOp.MAX)
    e2e_value = world * pairs_step_rank * args.steps / float(e2e_s.item()) / 1e9

    if rank == 0:
        peak_key = "ffma_lane_ops_per_s" if prec == "fp32" else "dfma_lane_ops_per_s"
        peak_lane = 0.5 * (peaks0[peak_key] + peaks1[peak_key])
        pair_s = float(np.mean(pair_ms)) * 1e-3
        if args.potential_only and prec == "fp32":
            # only the batched grid kernel has an FP32 potential-only variant (template arguments
            # <.., VONLY = true, ACCV = false>: its symbol ends in ...ELb1ELb0EEEv...); every other
            # FP32 path runs its V + E kernel with E = NULL
            v_kernel = "ELb1ELb0EEEvNS_10PairParamsE" in info.get("last_kernel", "") and "grid_kernel_f32x2" in info.get("last_kernel", "")
            slots = SLOTS_V_ONLY_F32_GRID if v_kernel else slots_for(layout, prec, info)
        else:
            slots = slots_for(layout, prec, info, v_only=args.potential_only)
        achieved = P * w.M * slots * 2 / pair_s / 1e12
        peak_tf = 2 * peak_lane / 1e12
        # DRAM bytes per pair-kernel launch from the committed ncu capture (profiles/), if any
        def lookup_traffic(key):
            tpath = os.path.join(ROOT, "profiles", "pair_kernel_traffic.csv")
            if os.path.exists(tpath):
                for ln in open(tpath):
                    f = ln.strip().split(",")
                    if len(f) >= 3 and f[0] == key:
                        return float(f[1]), f[2]
            return None, None
        traffic, traffic_file = lookup_traffic(f"config{args.config}_{prec}_{layout}")
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": DTYPE[prec], "data": "synthetic",
            "config": {"workload": WORKLOAD_NAME[args.config], "precision": prec, "M": w.M,
                       "M_nominal": w.M_nominal, "K": w.K, "W": W, "N": N,
                       "pairs_per_step_per_gpu": pairs_step_rank,
                       "parallelism": f"walkers sharded x{world}, sources replicated, no collective",
                       "layout": layout, "outputs": "V only (E = NULL)" if args.potential_only else "V and E",
                       "accurate_v": "off (--fast-v)" if args.fast_v else ("on (library default): batched FP32 grid V + E kernel with the z2 table, FP64-formed rxy2 "
                                      "and compensated row sums -- the batch's total energy within 1e-5 hartree of the oracle's "
                                      "(tests/test_grid_gpu.py::test_config3_grid_fp32_full_energy); the sweep row "
                                      "'fp32, accurate_v off' times the faster kernel") if prec == "fp32" else "n/a (FP64)",
                       "l2": "flushed between timed steps (256 MB write)", "plan": info["last_plan"],
                       "point_blocks": info["last_point_blocks"]},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": P * 24,
                    "d2h_bytes_per_step": P * (8 if args.potential_only else 32)},
            "gpu_launches": info["last_launches"] * args.steps,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak_tf, "unit": "TFLOP/s",
                         "frac": achieved / peak_tf, "traffic": traffic,
                         "kernel": KERNEL[(layout, prec)], "kernel_symbol": info.get("last_kernel", ""),
                         "kernel_ms": pair_s * 1e3,
                         "slots_per_pair": slots, "dz_table": bool(info.get("last_dz_table")),
                         # the same launch against SURVEY.md 8(d)'s fixed per-pair figure (17 FP32 /
                         # 18 FP64 slots: list of positions, per-pair refinement); above 1 when the
                         # kernel needs fewer operations than that formulation
                         "frac_at_survey_slots": P * w.M * (17 if prec == "fp32" else 18) / pair_s / peak_lane,
                         # the flop-counting view (SURVEY.md 8(d) eta_flop): the kernel's own flops per
                         # pair (an fma = 2) and, for FP32, the survey's fixed 24, over 2 x the lane rate
                         "flops_per_pair": flops_for(layout, prec, info, v_only=args.potential_only),
                         "eta_flop": P * w.M * flops_for(layout, prec, info, v_only=args.potential_only) / pair_s / (2 * peak_lane),
                         "eta_flop_at_survey_24": (P * w.M * 24 / pair_s / (2 * peak_lane)) if prec == "fp32" else None,
                         # one MUFU (RSQ / RSQ64H) per pair against the measured MUFU rate: the
                         # co-limiter of the FP32 grid kernel
                         "xu_frac": P * w.M / pair_s / (0.5 * (peaks0["mufu_lane_ops_per_s"] + peaks1["mufu_lane_ops_per_s"])),
                         "definition": "pairs x slots x 2 / pair-kernel time vs 2 x FMA lane rate of "
                                       "the same-run microbenchmark (qmmm_probe_peak)",
                         "peak_source": "measured, same process (mean of before/after)",
                         "peak_nominal_tflops": 148 * (128 if prec == "fp32" else 64) * 2 * 1.965e-3,
                         "mufu_lane_ops_per_s": peaks1["mufu_lane_ops_per_s"],
                         "probe_before": peaks0, "probe_after": peaks1},
        }
        if traffic is not None:
            line["roofline"]["traffic_source"] = (f"ncu --set full capture profiles/{traffic_file}; looked up "
                                                  "(profiles/pair_kernel_traffic.csv), not measured in this run")
        if world == 1:
            cb = oracle_sample_rate(w, args.cpu_sample_pairs)
            line["cpu_baseline"] = {
                "value": cb["rate"] / 1e9, "unit": UNIT, "cores": cb["threads"], "kind": "oracle",
                "sample": f"{cb['n_points']} of {cb['n_total']} evaluation points x all "
                          f"{w.M}+{w.K} sources ({cb['pairs']:.3g} pairs, {cb['seconds']:.1f} s)"}
            # the same oracle on ONE core (SURVEY.md 8(d) "CPU baseline" (b)): 1 % of the points, the
            # rate scales linearly in the points; the paper's speed-ups are quoted per one core
            c1 = oracle_sample_rate(w, 0.01 * P * (w.M + w.K), seed=98, nthreads=1)
            line["cpu_baseline_one_core"] = {
                "value": c1["rate"] / 1e9, "unit": UNIT, "cores": c1["threads"], "kind": "oracle",
                "sample": f"{c1['n_points']} of {c1['n_total']} evaluation points (1 %) x all {w.M}+{w.K} "
                          f"sources ({c1['pairs']:.3g} pairs, {c1['seconds']:.1f} s); rate is per pair, "
                          f"so it carries over to the full batch"}
            line["paper_context"] = {
                "paper_gpu_vs_one_cpu_core": {"sp": 23.6, "dp": 11.0,
                                              "what": "GTX 275 vs one Core i7 920 core, whole QMC run incl. upload "
                                                      "(PAPER.md:13, :165); another machine and a whole program: context only"},
                "this_run_gpu_vs_one_cpu_core": {"precision": prec, "ratio": value / (c1["rate"] / 1e9),
                                                 "what": "this kernel path (device-resident) vs the FP64 oracle on one "
                                                         "host core of this box"}}
            mem = probe_memory_and_launch(B)
            line["probes"] = mem
            if not args.no_sweep:
                B.qmmm_field_destroy(h)
                h = None
                del batches
                line["configs"] = sweep_all_configs(torch, B, peaks1, args.config, line, mem)
                # configs[4] in FP64 is the roofline case of the FP64 kernels: its
                # own block, from the sweep's row (same process, same DFMA probe)
                for r in line["configs"]:
                    if r["config"] == 4 and r["precision"] == "fp64" and r["layout_choice"] == "auto":
                        ach = r["pairs_per_eval"] * r["slots_per_pair"] * 2 / (r["pair_kernel_ms_median"] * 1e-3) / 1e12
                        pk = 2 * peaks1["dfma_lane_ops_per_s"] / 1e12
                        line["roofline_fp64"] = {
                            "workload": WORKLOAD_NAME[4], "bound": "alu", "achieved": ach, "peak": pk,
                            "unit": "TFLOP/s", "frac": ach / pk, "kernel": KERNEL[(r["layout"], "fp64")],
                            "kernel_ms": r["pair_kernel_ms_median"], "slots_per_pair": r["slots_per_pair"],
                            "dz_table": r["dz_table"], "gpairs_per_s": r["gpairs_per_s"],
                            "frac_at_survey_slots": r["pairs_per_eval"] * 18 / (r["pair_kernel_ms_median"] * 1e-3)
                                                    / peaks1["dfma_lane_ops_per_s"],
                            "traffic": lookup_traffic(f"config4_fp64_{r['layout']}")[0],
                            "traffic_source": "ncu --set full capture under profiles/ (pair_kernel_traffic.csv); looked up",
                            "peak_source": "measured DFMA lane rate, same process (qmmm_probe_peak)"}
                    if (r["config"] == args.config and r["precision"] == "fp32, accurate_v off"
                            and r["layout_choice"] == "auto" and prec == "fp32"):
                        # the same workload with qmmm_field_set_accurate_v(h, 0): the faster kernel that
                        # misses the batch-total energy criterion (context for roofline.frac)
                        line["roofline"]["accurate_v_off"] = {
                            "frac": r["fma_pipe_frac"], "gpairs_per_s": r["gpairs_per_s"],
                            "kernel_ms": r["pair_kernel_ms_median"], "kernel_symbol": r["kernel_symbol"]}
        print(json.dumps(line), flush=True)
    if h is not None:
        B.qmmm_field_destroy(h)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
