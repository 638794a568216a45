"""Per-phase clock table of single evaluations (diagnostic build of the library).

    python -m paper_1011_4687_b200.phase_table [--out DIR]

Builds a QMMM_PHASE_TIMING variant of the library (every evaluation kernel then records
clock64 / globaltimer at its phase boundaries per CTA; the regular build has none of this),
runs BASELINE.json configs[1] (32 points) and configs[2] (1 point) in both precisions with the
automatic plan, and prints for each: the kernel span, the median / maximum time of every phase
over the CTAs, and the period of the same evaluation replayed serially from a CUDA graph.
This is where the time of a FEW-POINT evaluation goes.
"""
from __future__ import annotations

import argparse
import ctypes
import os
import sys
import tempfile

import numpy as np

NAMES = ["prologue: barriers, first bulk copies, points staged", "row / lattice setup",
         "source walk (waits for the bulk copies included)", "nuclear term (FP64)",
         "in-CTA reduction, partial pushed", "cross-CTA collection (collecting CTAs) / exit"]


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=None, help="directory for the diagnostic library (default: a temp dir)")
    args = ap.parse_args()
    from . import build as _b
    out_dir = args.out or tempfile.mkdtemp(prefix="qmmm_diag_")
    lib_path = os.path.join(out_dir, "libqmmm_field_phases.so")
    _b.build(force=True, defines=["QMMM_PHASE_TIMING"], out=lib_path)
    os.environ["QMMM_FIELD_LIB"] = lib_path
    import torch
    from . import binding as B
    from .workloads import make_workload
    lib = B._lib
    lib.qmmm_debug_phases.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int]
    clk_ghz = torch.cuda.get_device_properties(0).clock_rate / 1e6 if hasattr(torch.cuda.get_device_properties(0), "clock_rate") else 1.965

    def table(h, n_cta, label):
        buf = np.zeros(n_cta * 10, dtype=np.int64)
        assert lib.qmmm_debug_phases(h, buf.ctypes.data, buf.size) == 0
        m = buf.reshape(n_cta, 10)
        d = np.diff(m[:, :7], axis=1) / clk_ghz / 1e3                  # us per phase and CTA
        span = (m[:, 9].max() - m[:, 8].min()) / 1e3                   # globaltimer ns -> us
        skew = (m[:, 8].max() - m[:, 8].min()) / 1e3
        print(f"## {label}\n\n{n_cta} CTAs; kernel span (first CTA start to last CTA end) {span:.2f} us; "
              f"CTA start skew {skew:.2f} us\n")
        print("| phase | median us | max us |\n|---|---|---|")
        for k, nm in enumerate(NAMES):
            print(f"| {nm} | {np.median(d[:, k]):.2f} | {d[:, k].max():.2f} |")
        whole = (m[:, 6] - m[:, 0]) / clk_ghz / 1e3
        print(f"| whole CTA | {np.median(whole):.2f} | {whole.max():.2f} |")

    for cfg, npts in ((1, 32), (2, 1)):
        w = make_workload(cfg)
        pts = torch.from_numpy(w.elec_xyz.reshape(-1, 3)[:npts].copy()).cuda()
        h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, npts)
        V = torch.zeros(npts, dtype=torch.float64, device="cuda")
        E = torch.zeros((npts, 3), dtype=torch.float64, device="cuda")
        try:
            for prec in ("fp32", "fp64"):
                for _ in range(5):
                    B.qmmm_field_eval(h, pts, 1, npts, V, E, prec)
                torch.cuda.synchronize()
                info = B.qmmm_field_get_info(h)
                n_cta = info["last_point_blocks"] * info["last_plan"]["slices"]
                pairs = npts * (w.M + w.K)
                table(h, n_cta, f"configs[{cfg}] {prec}, {npts} point(s) x {w.M} cells + {w.K} nuclei "
                                f"({pairs:.3g} pairs); plan {info['last_plan']}; kernel `{info['last_kernel']}`")
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    for _ in range(200):
                        B.qmmm_field_eval(h, pts, 1, npts, V, E, prec)
                g.replay()
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(); g.replay(); e1.record()
                torch.cuda.synchronize()
                print(f"\n200 evaluations replayed serially from one CUDA graph: "
                      f"{e0.elapsed_time(e1) * 1e3 / 200:.2f} us per evaluation (this diagnostic build)\n")
        finally:
            B.qmmm_field_destroy(h)


if __name__ == "__main__":
    main()
