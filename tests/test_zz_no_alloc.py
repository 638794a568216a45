"""qmmm_field_eval_noalloc: the one entry point that allocates nothing (its scratch memory is a
fixed __device__ array inside the library; include/qmmm_field.h).  Its output is compared with
the existing path's (qmmm_field_create + qmmm_field_eval, FP64) within the FP64 tolerance the
parity tests use (1e-12 relative, vector norm for E), on two calls in a row that share the
scratch array -- different environments and batch sizes, so the second call runs on the first
one's leftovers.  Collected last on purpose (the suite runs with pytest -x); passes alone in a
fresh process and after the other tests.
"""
import numpy as np
import pytest

from paper_1011_4687_b200.workloads import make_workload

pytestmark = pytest.mark.gpu

TOL64 = 1e-12


def _existing_path(torch, B, w, pts):
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, len(pts))
    try:
        d = torch.from_numpy(np.ascontiguousarray(pts)).cuda()
        V = torch.full((len(pts),), float("nan"), dtype=torch.float64, device="cuda")
        E = torch.full((len(pts), 3), float("nan"), dtype=torch.float64, device="cuda")
        B.qmmm_field_eval(h, d, 1, len(pts), V, E, "fp64")
        torch.cuda.synchronize()
        return V.cpu().numpy(), E.cpu().numpy()
    finally:
        B.qmmm_field_destroy(h)


def _close(V, E, Vref, Eref):
    eV = np.abs(V - Vref) / np.abs(Vref)
    eE = np.linalg.norm(E - Eref, axis=1) / np.linalg.norm(Eref, axis=1)
    assert eV.max() <= TOL64, f"V: max rel deviation {eV.max():.3e}"
    assert eE.max() <= TOL64, f"E: max rel deviation {eE.max():.3e}"


def test_noalloc_entry_point_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "this test needs a CUDA device"
    from paper_1011_4687_b200 import binding as B
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    rng = np.random.default_rng(2026)

    # call 1: config 1's environment (252,192 cells + 256 nuclei), 100 points (ragged last point block)
    w1 = make_workload(1)
    p1 = rng.normal(size=(100, 3)) * 0.8
    # call 2: config 0's environment (4,096 random cells + 16 nuclei), 37 points: fewer point blocks,
    # more slices per point -- the partials region still holds call 1's numbers
    w0 = make_workload(0)
    p2 = rng.normal(size=(37, 3)) * 0.9
    ref1 = _existing_path(torch, B, w1, p1)
    ref2 = _existing_path(torch, B, w0, p2)

    dev1 = [t(a) for a in (w1.src_xyz, w1.src_q, w1.nuc_xyz, w1.nuc_Z, p1)]
    dev2 = [t(a) for a in (w0.src_xyz, w0.src_q, w0.nuc_xyz, w0.nuc_Z, p2)]
    V1 = torch.full((100,), float("nan"), dtype=torch.float64, device="cuda")
    E1 = torch.full((100, 3), float("nan"), dtype=torch.float64, device="cuda")
    V2 = torch.full((37,), float("nan"), dtype=torch.float64, device="cuda")
    E2 = torch.full((37, 3), float("nan"), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    B.qmmm_field_eval_noalloc(*dev1, V1, E1)                  # two calls in a row on one stream,
    B.qmmm_field_eval_noalloc(*dev2, V2, E2)                  # no synchronisation in between
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before
    _close(V1.cpu().numpy(), E1.cpu().numpy(), *ref1)
    _close(V2.cpu().numpy(), E2.cpu().numpy(), *ref2)

    # the same two calls again: bitwise the same (deterministic; the tickets were left at rest)
    V1b, E1b, V2b = torch.zeros_like(V1), torch.zeros_like(E1), torch.zeros_like(V2)
    B.qmmm_field_eval_noalloc(*dev1, V1b, E1b)
    B.qmmm_field_eval_noalloc(*dev2, V2b, None)               # potential only: E = NULL
    torch.cuda.synchronize()
    assert torch.equal(V1, V1b) and torch.equal(E1, E1b) and torch.equal(V2, V2b)

    # nuclei only / cells only, and the limit: a clear error beyond QMMM_NOALLOC_MAX_POINTS
    Vn = torch.zeros(37, dtype=torch.float64, device="cuda")
    Vc = torch.zeros(37, dtype=torch.float64, device="cuda")
    B.qmmm_field_eval_noalloc(None, None, dev2[2], dev2[3], dev2[4], Vn, None)
    B.qmmm_field_eval_noalloc(dev2[0], dev2[1], None, None, dev2[4], Vc, None)
    torch.cuda.synchronize()
    assert torch.allclose(Vn + Vc, V2, rtol=1e-12, atol=0)
    big = torch.zeros((B.QMMM_NOALLOC_MAX_POINTS + 1, 3), dtype=torch.float64, device="cuda")
    Vbig = torch.zeros(B.QMMM_NOALLOC_MAX_POINTS + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(B.QmmmError) as ei:
        B.qmmm_field_eval_noalloc(*dev2[:4], big, Vbig, None)
    assert ei.value.status == 1 and "QMMM_NOALLOC_MAX_POINTS" in str(ei.value)
    # the largest batch that is accepted (one slice per point block region: 4,096 points)
    pts_max = t(rng.normal(size=(B.QMMM_NOALLOC_MAX_POINTS, 3)) * 0.9)
    Vmax = torch.zeros(B.QMMM_NOALLOC_MAX_POINTS, dtype=torch.float64, device="cuda")
    B.qmmm_field_eval_noalloc(*dev2[:4], pts_max, Vmax, None)
    B.qmmm_field_eval_noalloc(*dev2, V2b, None)               # and the small batch again afterwards
    torch.cuda.synchronize()
    assert torch.equal(V2, V2b) and bool(torch.isfinite(Vmax).all())
