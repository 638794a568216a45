"""Out-of-bounds writes, hunted without compute-sanitizer (closed on this GPU pool: SURVEY.md
section 4 T4 asked for memcheck).  Every output of every device entry point
is a slice from the INTERIOR of a larger buffer filled with a sentinel; after the call the guard
zones on both sides must still hold the sentinel bit for bit, and the interior must be fully
written (no sentinel left).  Ragged point counts (tails of point blocks, of warps, of the
points-per-thread groups), both layouts, both precisions, E / no E, and the entry points
qmmm_field_eval, _eval_moves, _eval_energy and _eval_noalloc.  Inputs sit between guards too:
a kernel reading past them would not be caught, but the clamped tail loads are exercised with
NaN-poisoned neighbours, which would surface in the results (checked finite).
"""
import numpy as np
import pytest

from paper_1011_4687_b200.workloads import make_workload

pytestmark = pytest.mark.gpu

SENTINEL = 1.2345678901234567e300
GUARD = 512                                     # doubles on each side


def guarded(torch, n):
    """(whole buffer, interior view of n doubles)"""
    buf = torch.full((GUARD + n + GUARD,), SENTINEL, dtype=torch.float64, device="cuda")
    return buf, buf[GUARD:GUARD + n]


def guards_intact(buf, n):
    return bool((buf[:GUARD] == SENTINEL).all()) and bool((buf[GUARD + n:] == SENTINEL).all())


def poisoned_points(torch, pts):
    """The points between NaN guards: a read past either end poisons the result."""
    n = pts.size
    buf = torch.full((GUARD + n + GUARD,), float("nan"), dtype=torch.float64, device="cuda")
    buf[GUARD:GUARD + n] = torch.from_numpy(np.ascontiguousarray(pts).reshape(-1)).cuda()
    return buf, buf[GUARD:GUARD + n].view(-1, 3)


@pytest.mark.parametrize("layout", ["list", "grid"])
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_outputs_stay_inside_their_buffers(layout, precision):
    import torch
    from paper_1011_4687_b200 import binding as B
    w = make_workload(1)
    rng = np.random.default_rng(31)
    sizes = [1, 2, 3, 4, 5, 7, 8, 9, 15, 16, 17, 31, 32, 33, 63, 64, 65, 100, 127, 129, 257]
    Pmax = max(sizes)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, Pmax)
    try:
        B.qmmm_field_set_layout(h, layout)
        for overlap in (False, True):
            B.qmmm_field_set_overlap(h, overlap)
            for P in sizes:
                pts = rng.normal(size=(P, 3)) * 0.8
                keep, d = poisoned_points(torch, pts)
                for want_E in (True, False):
                    vb, V = guarded(torch, P)
                    eb, Ef = guarded(torch, 3 * P)
                    B.qmmm_field_eval(h, d, 1, P, V, Ef.view(P, 3) if want_E else None, precision)
                    torch.cuda.synchronize()
                    tag = (layout, precision, overlap, P, want_E)
                    assert guards_intact(vb, P) and guards_intact(eb, 3 * P), tag
                    assert bool(torch.isfinite(V).all()) and not bool((V == SENTINEL).any()), tag
                    if want_E:
                        assert bool(torch.isfinite(Ef).all()) and not bool((Ef == SENTINEL).any()), tag
                    else:
                        assert bool((Ef == SENTINEL).all()), tag           # E = NULL: nothing written at all
        B.qmmm_field_set_overlap(h, False)
        # n moves of N points each (overlapped launches from C), and per-walker energies
        for n, N in ((7, 1), (5, 3), (3, 33)):
            pts = rng.normal(size=(n * N, 3)) * 0.8
            keep, d = poisoned_points(torch, pts)
            vb, V = guarded(torch, n * N)
            eb, Ef = guarded(torch, 3 * n * N)
            B.qmmm_field_eval_moves(h, d, n, N, V, Ef.view(n * N, 3), precision)
            ub, U = guarded(torch, n)
            B.qmmm_field_eval_energy(h, d, n, N, U, precision)
            torch.cuda.synchronize()
            assert guards_intact(vb, n * N) and guards_intact(eb, 3 * n * N) and guards_intact(ub, n), (n, N)
            assert bool(torch.isfinite(V).all()) and bool(torch.isfinite(Ef).all()) and bool(torch.isfinite(U).all())
            assert not bool((V == SENTINEL).any()) and not bool((U == SENTINEL).any())
            # U[w] = -sum_i V(r_wi): the two entry points agree
            assert torch.allclose(U, -V.view(n, N).sum(1), rtol=1e-6 if precision == "fp32" else 1e-12, atol=0)
    finally:
        B.qmmm_field_destroy(h)


def test_noalloc_outputs_stay_inside_their_buffers():
    import torch
    from paper_1011_4687_b200 import binding as B
    w = make_workload(0)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    src = [t(a) for a in (w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z)]
    rng = np.random.default_rng(32)
    for P in (1, 7, 8, 9, 100, 1000):
        pts = rng.normal(size=(P, 3)) * 0.9
        keep, d = poisoned_points(torch, pts)
        vb, V = guarded(torch, P)
        eb, Ef = guarded(torch, 3 * P)
        B.qmmm_field_eval_noalloc(*src, d, V, Ef.view(P, 3))
        torch.cuda.synchronize()
        assert guards_intact(vb, P) and guards_intact(eb, 3 * P), P
        assert bool(torch.isfinite(V).all()) and bool(torch.isfinite(Ef).all()), P
        assert not bool((V == SENTINEL).any()) and not bool((Ef == SENTINEL).any()), P


def test_min_distance_helper_against_brute_force():
    """qmmm_field_min_distance (debug helper, SURVEY.md 8(b) "r = 0"): the smallest distance between
    the points and the CHARGED sources -- source-list handles (cells and nuclei; pads and empty
    cells do not count), grid-only handles (qmmm_field_create_grid), ragged point counts, a point
    placed on a cell, and an environment without sources -- against numpy."""
    import torch
    from paper_1011_4687_b200 import binding as B
    rng = np.random.default_rng(77)

    def brute(pts, *sources):
        best = np.inf
        for xyz, q in sources:
            keep = np.asarray(q) != 0.0
            if keep.any():
                d = np.linalg.norm(pts[:, None, :] - np.asarray(xyz)[keep][None, :, :], axis=2)
                best = min(best, float(d.min()))
        return best

    for idx in (0, 1):
        w = make_workload(idx)
        h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, 8)
        try:
            for P in (1, 5, 64, 65, 200):                       # P is not limited by max_points
                pts = rng.normal(size=(P, 3)) * 1.5
                got = B.qmmm_field_min_distance(h, torch.from_numpy(pts).cuda())
                want = brute(pts, (w.src_xyz, w.src_q), (w.nuc_xyz, w.nuc_Z))
                assert abs(got - want) <= 1e-12 * want, (idx, P, got, want)
            pts = rng.normal(size=(7, 3))
            pts[3] = w.src_xyz[np.flatnonzero(w.src_q)[11]]      # a point ON a charged cell
            assert B.qmmm_field_min_distance(h, torch.from_numpy(pts).cuda()) == 0.0
        finally:
            B.qmmm_field_destroy(h)
    # grid-only handle: 20 x 13 x 70 nodes with empty cells, orthorhombic spacing, 3 nuclei
    n, hh, origin = (20, 13, 70), np.array([0.3, 0.25, 0.2]), np.array([-3.0, -1.5, -7.0])
    dense = -rng.random(n) * 1e-2
    dense[rng.random(n) > 0.6] = 0.0
    idx3 = np.stack(np.meshgrid(*[np.arange(k) for k in n], indexing="ij"), axis=-1)
    pos = (origin + hh * idx3).reshape(-1, 3)
    nuc = rng.normal(size=(3, 3)) * 2.0
    Z = np.array([1.0, 0.0, 8.0])                                # a nucleus of charge 0 does not count
    h = B.qmmm_field_create_grid(origin, tuple(hh), n, np.ascontiguousarray(dense), nuc, Z, 4)
    try:
        assert not B.qmmm_field_get_grid_info(h)["has_list"]
        for P in (1, 33, 130):
            pts = rng.normal(size=(P, 3)) * 2.0
            got = B.qmmm_field_min_distance(h, torch.from_numpy(pts).cuda())
            want = brute(pts, (pos, dense.reshape(-1)), (nuc, Z))
            assert abs(got - want) <= 1e-12 * want, (P, got, want)
    finally:
        B.qmmm_field_destroy(h)
    h = B.qmmm_field_create(None, None, None, None, 4)           # nothing to be near to
    try:
        assert B.qmmm_field_min_distance(h, torch.zeros((3, 3), dtype=torch.float64, device="cuda")) == np.inf
        with pytest.raises(B.QmmmError):
            B.qmmm_field_min_distance(h, torch.zeros((0, 3), dtype=torch.float64, device="cuda"))
    finally:
        B.qmmm_field_destroy(h)
