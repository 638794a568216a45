"""Every evaluation-kernel instantiation the library contains is launched at least once here and
its result compared with the CPU oracle.

The launch logic chooses among a few dozen template instantiations (pair_kernel*, grid_kernel_*,
move_server_kernel) by layout, precision, point count, plan, overlap and E / no E; a variant that
only an odd combination selects could be wrong unnoticed.  qmmm_field_info.last_kernel names the
instantiation an evaluation launched (mangled symbol); the set seen here must equal the set of
kernel symbols in the built library (read from the .so with nm), so adding an instantiation
without a recipe below fails this test.
"""
import os
import re
import subprocess

import numpy as np
import pytest

from paper_1011_4687_b200.workloads import make_workload
from parity_check import check

pytestmark = pytest.mark.gpu

TOL = {"fp64": 1e-12, "fp32": 1e-5}
FAMILIES = ("pair_kernel", "pair_kernel_f32x2", "grid_kernel_f32x2", "grid_kernel_f64", "move_server_kernel",
            "move_server_grid_kernel")


def exported_kernels(lib_path):
    out = subprocess.run(["nm", lib_path], capture_output=True, text=True, check=True).stdout
    names = set()
    for ln in out.splitlines():
        f = ln.split()
        if len(f) == 3 and f[2].startswith("_ZN4qmmm") and re.match(r"_ZN4qmmm\d+(%s)I" % "|".join(FAMILIES), f[2]) \
                and f[2].endswith(("PairParamsE", "ServerParamsE")):
            names.add(f[2])
    return names


def demangle(names):
    try:
        r = subprocess.run(["c++filt"], input="\n".join(sorted(names)), capture_output=True, text=True)
        return r.stdout.split("\n")
    except Exception:
        return sorted(names)


def long_axis_grid(rng, nz=600):
    """A 9 x 8 x nz grid: the dz table of the batched kernels does not fit (stepped dz)."""
    n, h = (9, 8, nz), 0.25
    origin = np.array([-1.0, -0.9, -0.5 * h * (nz - 1)])
    centre = origin + 0.5 * h * (np.array(n) - 1)
    q = -rng.random(n) * 1e-2
    idx = np.stack(np.meshgrid(*[np.arange(k) for k in n], indexing="ij"), axis=-1)
    pos = origin + h * idx
    q[np.linalg.norm(pos - centre, axis=-1) < 1.6] = 0.0
    keep = q != 0.0
    return (origin, h, n, np.ascontiguousarray(q), np.ascontiguousarray(pos[keep]), np.ascontiguousarray(q[keep]), centre)


def test_every_kernel_instantiation_runs_and_agrees_with_the_oracle(oracle_mod):
    import torch
    from paper_1011_4687_b200 import binding as B
    exported = exported_kernels(B.LIB_PATH)
    assert len(exported) >= 40, exported
    seen = {}
    rng = np.random.default_rng(42)

    w = make_workload(1)
    P0 = 72
    base = rng.normal(size=(P0, 3)) * 0.8
    ref_all = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, base, want_abs=True)

    class Sub:                                   # the oracle's result restricted to the first n points
        def __init__(self, r, n):
            self.V, self.E, self.absV, self.absE = r.V[:n], r.E[:n], r.absV[:n], r.absE[:n]

    def evaluate(h, pts, ref, layout, prec, plan, overlap, want_E, tag):
        B.qmmm_field_set_layout(h, layout)
        B.qmmm_field_set_plan(h, **plan)
        B.qmmm_field_set_overlap(h, overlap)
        n = len(pts)
        d = torch.from_numpy(np.ascontiguousarray(pts)).cuda()
        V = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
        E = torch.full((n, 3), float("nan"), dtype=torch.float64, device="cuda") if want_E else None
        B.qmmm_field_eval(h, d, 1, n, V, E, prec)
        torch.cuda.synchronize()
        name = B.qmmm_field_get_info(h)["last_kernel"]
        try:
            check(ref, V.cpu().numpy(), E.cpu().numpy() if want_E else None, TOL[prec])
        except AssertionError as exc:
            raise AssertionError(f"{tag} -> {name}: {exc}") from None
        seen.setdefault(name, tag)

    # ---- config 1's environment (64^3 grid + list): list kernels, grid kernels with the dz table
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, P0)
    try:
        for prec in ("fp64", "fp32"):
            for want_E in (True, False):
                for overlap in (False, True):
                    for n in (1, 2, 4, 24, P0):
                        for ppt in (0, 1, 2, 4, 8):
                            for pw in (0, 1, 16):
                                if ppt == 8 and prec == "fp64":
                                    continue
                                plan = dict(points_per_thread=ppt, point_warps=pw)
                                for layout in ("list", "grid"):
                                    if layout == "list" and (overlap or pw == 16):
                                        continue        # the list kernels have no overlap / FULL variants
                                    evaluate(h, base[:n], Sub(ref_all, n), layout, prec, plan, overlap, want_E,
                                             f"cfg1 {layout} {prec} n={n} ppt={ppt} pw={pw} ov={overlap} E={want_E}")
        # the batched FP32 V + E kernel without the accurate-V arithmetic (qmmm_field_set_accurate_v)
        B.qmmm_field_set_accurate_v(h, False)
        for n in (24, P0):
            evaluate(h, base[:n], Sub(ref_all, n), "grid", "fp32", dict(points_per_thread=4, point_warps=16), False, True,
                     f"cfg1 grid fp32 n={n} ppt=4 pw=16 accurate_v off")
        B.qmmm_field_set_accurate_v(h, True)
        # the move servers (single-point host calls): grid-aware on this handle, source list when forced
        for layout in ("auto", "list"):
            for prec in ("fp64", "fp32"):
                B.qmmm_field_set_layout(h, layout)
                B.qmmm_field_set_plan(h)
                for i in range(3):
                    v = np.zeros(1); e = np.zeros((1, 3))
                    B.qmmm_field_eval_host(h, np.ascontiguousarray(base[i:i + 1]), 1, 1, v, e, prec)
                    name = B.qmmm_field_get_info(h)["last_kernel"]
                    sub = Sub(ref_all, i + 1)
                    sub.V, sub.E, sub.absV, sub.absE = sub.V[i:], sub.E[i:], sub.absV[i:], sub.absE[i:]
                    check(sub, v, e, TOL[prec])
                seen.setdefault(name, f"move server {layout} {prec}")
    finally:
        B.qmmm_field_destroy(h)

    # ---- long z axes.  1,700 nodes: no dz table fits, the batched kernels step dz.  130 nodes: the
    # table fits and the FP32 kernels use the lattice per work unit (more than 128 nodes).
    for nz in (1700, 130):
        origin, hh, n3, dense, pos, q, centre = long_axis_grid(rng, nz)
        pts = centre + rng.normal(size=(P0, 3)) * 0.3
        pts = centre + (pts - centre) * np.minimum(1.0, 0.9 / np.linalg.norm(pts - centre, axis=1))[:, None]
        ref_long = oracle_mod.field(pos, q, np.zeros((0, 3)), np.zeros(0), pts, want_abs=True)
        h = B.qmmm_field_create_grid(origin, hh, n3, dense, None, None, P0)
        try:
            for prec in ("fp64", "fp32"):
                for want_E in (True, False):
                    for overlap in (False, True):
                        for local in ((-1, 0) if prec == "fp32" else (-1,)):
                            B.qmmm_field_set_local_lattice(h, local)
                            for n in (24, P0):
                                for ppt, pw in ((4, 0), (4, 8), (4, 4), (4, 1), (2, 16), (8, 8)):
                                    if ppt == 8 and prec == "fp64":
                                        continue
                                    if local == 0 and prec == "fp32" and want_E:
                                        continue        # whole-grid lattice forced on an axis of more than 128 nodes:
                                                        # E is out of tolerance by design (include/qmmm_field.h)
                                    evaluate(h, pts[:n], Sub(ref_long, n), "grid", prec,
                                             dict(points_per_thread=ppt, point_warps=pw), overlap, want_E,
                                             f"nz={nz} {prec} n={n} ppt={ppt} pw={pw} ov={overlap} E={want_E} local={local}")
            if nz == 130:
                # light CTAs (overlap) with the dz table beside a shallow pipeline, lattice per work unit
                B.qmmm_field_set_local_lattice(h, -1)
                evaluate(h, pts[:24], Sub(ref_long, 24), "grid", "fp32",
                         dict(points_per_thread=4, point_warps=4, stages=2), True, True,
                         "nz=130 fp32 n=24 ppt=4 pw=4 stages=2 ov=True E=True local=-1")
        finally:
            B.qmmm_field_destroy(h)

    missing = exported - set(seen)
    extra = set(seen) - exported
    print(f"{len(seen)} kernel instantiations launched:")
    for name, tag in sorted(seen.items()):
        print(f"  {name}  <- {tag}")
    assert not extra, f"launched kernels that nm does not list: {demangle(extra)}"
    assert not missing, "instantiations in the library that no recipe here launches:\n  " + "\n  ".join(demangle(missing))
