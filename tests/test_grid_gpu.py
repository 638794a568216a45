"""GPU parity of the grid-aware compact format (include/qmmm_field.h
"Grid-aware compact source format") against the CPU oracle, through the C ABI.

The oracle knows nothing of grids: it gets the list of occupied nodes (positions and charges)
and runs the plain Eq. 4 double loop.  Tolerances as for the list kernels.
"""
import numpy as np
import pytest

from paper_1011_4687_b200.workloads import make_workload, subsample_points

pytestmark = pytest.mark.gpu

TOL64 = 1e-12
TOL32 = 1e-5
E_TOL = 1e-5          # hartree
NO_XYZ, NO_Z = np.zeros((0, 3)), np.zeros(0)


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    return torch


@pytest.fixture(scope="module")
def B():
    from paper_1011_4687_b200 import binding
    return binding


def run(torch, B, handle, pts, precision, want_E=True, layout=None, plan=None):
    if layout is not None:
        B.qmmm_field_set_layout(handle, layout)
    B.qmmm_field_set_plan(handle, **(plan or {}))
    d = torch.from_numpy(np.ascontiguousarray(pts)).cuda()
    V = torch.full((len(pts),), float("nan"), dtype=torch.float64, device="cuda")
    E = torch.full((len(pts), 3), float("nan"), dtype=torch.float64, device="cuda") if want_E else None
    B.qmmm_field_eval(handle, d, 1, len(pts), V, E, precision)
    torch.cuda.synchronize()
    return V.cpu().numpy(), (E.cpu().numpy() if want_E else None)


def rel_errors(ref, V, E):
    eV = np.abs(V - ref.V) / np.abs(ref.V)
    eE = None
    if E is not None:
        eE = np.linalg.norm(E - ref.E, axis=1) / np.linalg.norm(ref.E, axis=1)
    return eV, eE


from parity_check import check  # noqa: E402  (tests/parity_check.py: the tolerance rule)


def random_grid(rng, n, h, origin, fill=0.8, hole=None, signed=False):
    """Dense charges on an n[0] x n[1] x n[2] grid and the list of its occupied nodes."""
    q = -rng.random(n) * 1e-2
    if signed:
        q *= rng.choice([-1.0, 1.0], size=n)
    q[rng.random(n) > fill] = 0.0
    idx = np.stack(np.meshgrid(*[np.arange(k) for k in n], indexing="ij"), axis=-1)
    pos = np.asarray(origin) + h * idx
    if hole is not None:                       # masked sphere (the QM region)
        c, r = hole
        q[np.linalg.norm(pos - np.asarray(c), axis=-1) < r] = 0.0
    keep = q != 0.0
    return np.ascontiguousarray(q), np.ascontiguousarray(pos[keep]), np.ascontiguousarray(q[keep])


# ------------------------------------------------------------------------------ detection
def test_detection_on_the_baseline_configs(torch_cuda, B):
    w = make_workload(1)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, 64)
    try:
        gi = B.qmmm_field_get_grid_info(h)
        assert gi["present"] and gi["has_list"]
        assert gi["n"] == (64, 64, 64)
        assert abs(gi["spacing"] - 0.3) < 1e-13
        assert np.allclose(gi["origin"], [-9.45] * 3, atol=1e-13)
        assert gi["n_gchunks"] == 64 * 64 // 32
    finally:
        B.qmmm_field_destroy(h)
    w0 = make_workload(0)                      # random positions in a shell: no grid
    h = B.qmmm_field_create(w0.src_xyz, w0.src_q, w0.nuc_xyz, w0.nuc_Z, 8)
    try:
        gi = B.qmmm_field_get_grid_info(h)
        assert not gi["present"]
        with pytest.raises(B.QmmmError):
            B.qmmm_field_set_layout(h, "grid")
    finally:
        B.qmmm_field_destroy(h)


def test_detection_refuses_off_node_and_duplicate_sources(torch_cuda, B):
    rng = np.random.default_rng(5)
    _, pos, q = random_grid(rng, (20, 24, 40), 0.25, (-2.0, 1.0, 3.0), fill=1.0)
    for kind in ("off-node", "duplicate", "needles"):
        p, c = pos.copy(), q.copy()
        if kind == "off-node":
            p[len(p) // 2, 1] += 1e-9
        elif kind == "duplicate":
            p[7] = p[8]
        else:
            p[:, 2] *= 40.0                      # cell edges 1 : 1 : 40
        h = B.qmmm_field_create(p, c, None, None, 4)
        try:
            assert not B.qmmm_field_get_grid_info(h)["present"], kind
        finally:
            B.qmmm_field_destroy(h)
    h = B.qmmm_field_create(pos, q, None, None, 4)
    try:
        gi = B.qmmm_field_get_grid_info(h)
        assert gi["present"] and gi["spacing3"] == (0.25, 0.25, 0.25)
    finally:
        B.qmmm_field_destroy(h)
    p = pos.copy()
    p[:, 2] = 3.0 + (p[:, 2] - 3.0) * 1.5        # orthorhombic cells 0.25 x 0.25 x 0.375: accepted
    h = B.qmmm_field_create(p, q, None, None, 4)
    try:
        gi = B.qmmm_field_get_grid_info(h)
        assert gi["present"] and np.allclose(gi["spacing3"], (0.25, 0.25, 0.375), rtol=1e-13)
    finally:
        B.qmmm_field_destroy(h)


# ------------------------------------------------------------------------------ parity
@pytest.mark.parametrize("precision,tol", [("fp64", TOL64), ("fp32", TOL32)])
def test_config1_grid_layout(torch_cuda, B, oracle_mod, precision, tol):
    """Config 1 (64^3 grid, masked sphere, 256 nuclei, 32 points) with the grid layout forced;
    the list layout on the same handle must agree to rounding."""
    w = make_workload(1)
    pts = w.elec_xyz.reshape(-1, 3)
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, len(pts))
    try:
        V, E = run(torch_cuda, B, h, pts, precision, layout="grid")
        assert B.qmmm_field_get_grid_info(h)["last_layout"] == "grid"
        check(ref, V, E, tol)
        dE = abs(V.sum() - ref.V.sum())
        assert dE <= (E_TOL if precision == "fp32" else 1e-9), f"energy deviation {dE:.3e} hartree"
        Vl, El = run(torch_cuda, B, h, pts, precision, layout="list")
        assert B.qmmm_field_get_grid_info(h)["last_layout"] == "list"
        assert np.max(np.abs(V - Vl) / np.abs(Vl)) <= 2 * tol
        V2, E2 = run(torch_cuda, B, h, pts, precision, layout="grid")
        assert np.array_equal(V, V2) and np.array_equal(E, E2)          # bitwise repeatable
        if precision == "fp64":
            Vp, none = run(torch_cuda, B, h, pts, precision, want_E=False, layout="grid")
            assert none is None
            check(ref, Vp, None, tol)
    finally:
        B.qmmm_field_destroy(h)


@pytest.mark.parametrize("n,h,P", [((20, 13, 70), 0.3, 33), ((5, 7, 9), 0.5, 3), ((33, 32, 64), 0.2, 100),
                                   ((1, 40, 129), 0.25, 8), ((40, 1, 1), 0.4, 1), ((64, 3, 200), 0.1, 17),
                                   ((24, 40, 70), (0.3, 0.2, 0.25), 50), ((40, 33, 64), (0.17, 0.31, 0.23), 1),
                                   ((16, 16, 130), (0.5, 0.45, 0.1), 4)])
@pytest.mark.parametrize("precision,tol", [("fp64", TOL64), ("fp32", TOL32)])
def test_create_grid_ragged_shapes(torch_cuda, B, oracle_mod, n, h, P, precision, tol):
    """qmmm_field_create_grid with row counts that are not multiples of 32, z extents that are
    not multiples of 64, empty cells, nuclei, and point counts with ragged tails."""
    rng = np.random.default_rng(hash((n, P)) % (2 ** 32))
    origin = rng.normal(size=3) * 2.0
    centre = origin + 0.5 * np.asarray(h) * (np.array(n) - 1)
    dense, pos, q = random_grid(rng, n, np.asarray(h), origin, fill=0.7, hole=(centre, 1.6))
    K = 5
    nuc = centre + rng.normal(size=(K, 3)) * 4.0 + 6.0
    Z = rng.choice([1.0, 6.0, 8.0], size=K)
    pts = centre + rng.normal(size=(P, 3)) * 0.5
    pts = centre + (pts - centre) * np.minimum(1.0, 1.2 / np.linalg.norm(pts - centre, axis=1))[:, None]
    ref = oracle_mod.field(pos, q, nuc, Z, pts, want_abs=True)
    hnd = B.qmmm_field_create_grid(origin, h, n, dense, nuc, Z, P)
    try:
        gi = B.qmmm_field_get_grid_info(hnd)
        assert gi["present"] and not gi["has_list"] and gi["n"] == tuple(n)
        assert B.qmmm_field_get_info(hnd)["M"] == len(q)
        with pytest.raises(B.QmmmError):
            B.qmmm_field_set_layout(hnd, "list")
        V, E = run(torch_cuda, B, hnd, pts, precision)
        check(ref, V, E, tol)
        # the same through a device pointer and through the per-move host path
        hd = B.qmmm_field_create_grid(origin, h, n, torch_cuda.from_numpy(dense).cuda(),
                                      torch_cuda.from_numpy(nuc).cuda(), torch_cuda.from_numpy(Z).cuda(), P)
        try:
            V2, E2 = run(torch_cuda, B, hd, pts, precision)
            assert np.array_equal(V, V2) and np.array_equal(E, E2)
            Vh = np.zeros(P); Eh = np.zeros((P, 3))
            B.qmmm_field_eval_host(hd, np.ascontiguousarray(pts), 1, P, Vh, Eh, precision)
            if P == 1:
                # one point: the grid-aware move server, which splits the work units over its warps
                # in its own way (equal to rounding, checked against the oracle)
                assert "move_server_grid_kernel" in B.qmmm_field_get_info(hd)["last_kernel"]
                check(ref, Vh, Eh, tol)
            else:
                assert np.array_equal(V, Vh) and np.array_equal(E, Eh)
        finally:
            B.qmmm_field_destroy(hd)
    finally:
        B.qmmm_field_destroy(hnd)


@pytest.mark.parametrize("precision,tol", [("fp64", TOL64), ("fp32", TOL32)])
def test_grid_partition_independence_and_source_order(torch_cuda, B, oracle_mod, precision, tol):
    """Eq. 5-6: any partition of the sum gives the result to rounding; the
    order of the source LIST does not matter at all (the dense grid is the same: bitwise)."""
    rng = np.random.default_rng(11)
    n, h, origin = (32, 48, 128), 0.25, (-4.0, -6.0, -16.0)
    centre = np.asarray(origin) + 0.5 * h * (np.array(n) - 1)
    _, pos, q = random_grid(rng, n, h, origin, fill=0.95, hole=(centre, 2.5))
    pts = centre + rng.normal(size=(70, 3)) * 0.7
    ref = oracle_mod.field(pos, q, NO_XYZ, NO_Z, pts, want_abs=True)
    h1 = B.qmmm_field_create(pos, q, None, None, len(pts))
    perm = rng.permutation(len(q))
    h2 = B.qmmm_field_create(np.ascontiguousarray(pos[perm]), np.ascontiguousarray(q[perm]), None, None, len(pts))
    try:
        assert B.qmmm_field_get_grid_info(h1)["present"] and B.qmmm_field_get_grid_info(h2)["present"]
        base = run(torch_cuda, B, h1, pts, precision, layout="grid")
        check(ref, *base, tol)
        shuf = run(torch_cuda, B, h2, pts, precision, layout="grid")
        assert np.array_equal(base[0], shuf[0]) and np.array_equal(base[1], shuf[1])
        epts = (2, 4, 8) if precision == "fp32" else (1, 2, 4)
        for ept in epts:
            for pw in (1, 2, 8):
                for slices in (1, 5, 37):
                    V, E = run(torch_cuda, B, h1, pts, precision,
                               plan=dict(points_per_thread=ept, point_warps=pw, slices=slices, stages=3))
                    check(ref, V, E, tol)
                    bound = 1e-13 if precision == "fp64" else 1e-6
                    assert np.max(np.abs(V - base[0]) / np.abs(base[0])) <= bound
        # batched walkers = one walker at a time, bitwise, under the same plan
        plan = dict(points_per_thread=epts[-1], point_warps=2, slices=7, stages=4)
        Vb, Eb = run(torch_cuda, B, h1, pts[:64], precision, plan=plan)
        for wlk in range(4):
            Vw, Ew = run(torch_cuda, B, h1, pts[16 * wlk:16 * wlk + 16], precision, plan=plan)
            assert np.array_equal(Vw, Vb[16 * wlk:16 * wlk + 16]) and np.array_equal(Ew, Eb[16 * wlk:16 * wlk + 16])
    finally:
        B.qmmm_field_destroy(h1)
        B.qmmm_field_destroy(h2)


@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_point_on_an_empty_node_is_harmless(torch_cuda, B, oracle_mod, precision):
    """Masked-out cells are zero charges in the grid copy; an evaluation point that coincides
    with one must not produce 0 * inf."""
    rng = np.random.default_rng(3)
    n, h, origin = (16, 32, 64), 0.5, (-4.0, -8.0, -16.0)
    centre = np.asarray(origin) + h * np.array([8, 16, 32])          # a node, inside the hole
    dense, pos, q = random_grid(rng, n, h, origin, fill=1.0, hole=(centre, 2.0))
    pts = np.stack([centre, centre + [h, 0, 0], centre + [0.1, 0.2, -0.3]])
    ref = oracle_mod.field(pos, q, NO_XYZ, NO_Z, pts, want_abs=True)
    hnd = B.qmmm_field_create_grid(origin, h, n, dense, None, None, len(pts))
    try:
        V, E = run(torch_cuda, B, hnd, pts, precision)
        assert np.all(np.isfinite(V)) and np.all(np.isfinite(E))
        # E at the centre of a symmetric hole is a small difference of large terms (kappa_E far
        # above 1e3): check() holds it to err / kappa, everything else to the plain tolerance
        check(ref, V, E, TOL64 if precision == "fp64" else TOL32)
    finally:
        B.qmmm_field_destroy(hnd)


def test_grid_symmetry_pins_without_the_oracle(torch_cuda, B):
    """Closed forms the grid kernels must hit by themselves: one charged node (V = q/d,
    E = q d/d^3) and a full symmetric cube of equal charges (E = 0 at its centre)."""
    n, h, origin = (9, 9, 9), 0.5, (-2.0, -2.0, -2.0)
    dense = np.zeros(n)
    dense[6, 2, 7] = -0.75
    node = np.asarray(origin) + h * np.array([6, 2, 7])
    pts = np.array([[0.1, 0.2, -0.3], [1.0, -1.0, 0.25]])
    hnd = B.qmmm_field_create_grid(origin, h, n, dense, None, None, 2)
    try:
        for precision, tol in (("fp64", 1e-14), ("fp32", 1e-6)):
            V, E = run(torch_cuda, B, hnd, pts, precision)
            d = pts - node
            r = np.linalg.norm(d, axis=1)
            assert np.max(np.abs(V - (-0.75 / r)) / (0.75 / r)) <= tol
            assert np.max(np.linalg.norm(E - (-0.75 * d / r[:, None] ** 3), axis=1) * r ** 2 / 0.75) <= tol
    finally:
        B.qmmm_field_destroy(hnd)
    cube = np.full(n, 0.01)
    cube[4, 4, 4] = 0.0                        # the point sits on the (empty) centre node
    hnd = B.qmmm_field_create_grid(origin, h, n, cube, None, None, 1)
    try:
        for precision, tol in (("fp64", 1e-13), ("fp32", 1e-6)):
            V, E = run(torch_cuda, B, hnd, np.zeros((1, 3)), precision)
            assert np.linalg.norm(E) <= tol * abs(V[0])
    finally:
        B.qmmm_field_destroy(hnd)


# ------------------------------------------------------------ the bench configurations
def test_config3_grid_fp32_full_energy(torch_cuda, B, oracle_mod, full_oracle):
    """Config 3 in the launch configuration bench.py times (AUTO -> grid kernels): V and E on a
    seeded 1 % subsample, the total energy per walker and whole batch against the oracle on
    all 16,384 points; the list layout on the same handle for comparison."""
    w = make_workload(3)
    pts = w.elec_xyz.reshape(-1, 3)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, len(pts))
    try:
        V, E = run(torch_cuda, B, h, pts, "fp32")
        assert B.qmmm_field_get_grid_info(h)["last_layout"] == "grid"
        assert "ELb0ELb1EEEv" in B.qmmm_field_get_info(h)["last_kernel"]  # <2, 8, false, true, true, 0, false, ACCV = true>
        assert B.qmmm_field_get_info(h)["last_accurate_v"] == 1
        B.qmmm_field_set_accurate_v(h, False)     # the faster V + E kernel (same E; V to 7e-8 rms instead of 3e-8)
        Vf, Ef = run(torch_cuda, B, h, pts, "fp32")
        assert "ELb0ELb0EEEv" in B.qmmm_field_get_info(h)["last_kernel"]
        assert B.qmmm_field_get_info(h)["last_accurate_v"] == 0
        B.qmmm_field_set_accurate_v(h, True)
        Vl, El = run(torch_cuda, B, h, pts, "fp32", layout="list")
        # E = NULL: the potential-only kernel (Eq. 4 proper; no lattice, 6 operations per pair)
        Vp, _ = run(torch_cuda, B, h, pts, "fp32", want_E=False, layout="auto")
        assert "ELb1ELb0EEEv" in B.qmmm_field_get_info(h)["last_kernel"]  # <2, 8, false, true, true, 0, VONLY = true, false>
        assert B.qmmm_field_get_info(h)["last_accurate_v"] == 1
        U = torch_cuda.zeros(w.W, dtype=torch_cuda.float64, device="cuda")
        B.qmmm_field_eval_energy(h, torch_cuda.from_numpy(pts).cuda(), w.W, w.N, U, "fp32")
        torch_cuda.cuda.synchronize()
        U = U.cpu().numpy()
    finally:
        B.qmmm_field_destroy(h)
    full = full_oracle(3)                         # every point, V and E
    check(full, V, E, TOL32)
    check(full, Vf, Ef, TOL32)
    check(full, Vl, El, TOL32)
    check(full, Vp, None, TOL32)
    dU = np.abs(U + full.V.reshape(w.W, w.N).sum(1))
    print(f"config3 fp32 eval_energy: per-walker max |dU| = {dU.max():.3e} hartree")
    assert dU.max() <= E_TOL
    for name, v in (("grid", V), ("grid, accurate_v off", Vf), ("list", Vl), ("grid potential-only", Vp)):
        per_walker = np.abs(v.reshape(w.W, w.N).sum(1) - full.V.reshape(w.W, w.N).sum(1))
        batch = abs(v.sum() - full.V.sum())
        d = v - full.V
        print(f"config3 fp32 {name}: per-walker max |dE| = {per_walker.max():.3e}, batch |dE| = {batch:.3e} "
              f"hartree, per point mean {d.mean():.3e} rms {d.std():.3e} max {np.abs(d).max():.3e}")
        assert per_walker.max() <= E_TOL
        assert batch / w.W <= E_TOL
        assert batch <= 1e-4
        if name in ("grid", "grid potential-only"):
            # the configuration bench.py times (V and E) and the energy path (Eq. 4 needs V only;
            # qmmm_field_eval_energy runs the potential-only kernel): the north star's criterion
            # taken literally -- the sum over all 16,384 points within 1e-5 hartree of the
            # oracle's, 4e-12 of the 2.5e6 hartree it adds up
            assert batch <= E_TOL, batch
    # and through the entry point that returns energies: sum over walkers of U[w]
    batch_U = abs(U.sum() + full.V.sum())
    print(f"config3 fp32 eval_energy: whole batch |dU| = {batch_U:.3e} hartree")
    assert batch_U <= E_TOL
    # the field is formed from the same sums either way (r^2 differs in its last bit)
    assert np.max(np.linalg.norm(E - Ef, axis=1) / np.linalg.norm(Ef, axis=1)) <= 1e-6
    for name, e in (("grid", E), ("list", El)):
        eE = np.linalg.norm(e - full.E, axis=1) / np.linalg.norm(full.E, axis=1)
        kE = full.absE / np.linalg.norm(full.E, axis=1)
        print(f"config3 fp32 {name}: max rel err of |E| over all points {eE.max():.3e} "
              f"(kappa_E max {kE.max():.1f}; E uses the raw MUFU.RSQ value, DESIGN.md reading 21)")


def test_config4_grid_fp64(torch_cuda, B, full_oracle):
    """Config 4 (16.7 M cells x 2,048 points, FP64) in bench.py's launch configuration
    (AUTO -> grid kernels): V and E of all 2,048 points against the oracle, for the grid
    kernel and its potential-only variant (the list kernels: tests/test_parity_gpu.py)."""
    w = make_workload(4)
    pts = w.elec_xyz.reshape(-1, 3)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, len(pts))
    try:
        gi = B.qmmm_field_get_grid_info(h)
        assert gi["present"] and gi["n"] == (256, 256, 256)
        V, E = run(torch_cuda, B, h, pts, "fp64")
        assert B.qmmm_field_get_grid_info(h)["last_layout"] == "grid"
        assert B.qmmm_field_get_info(h)["last_dz_table"]
        Vp, _ = run(torch_cuda, B, h, pts, "fp64", want_E=False)
        assert B.qmmm_field_get_grid_info(h)["last_layout"] == "grid"
    finally:
        B.qmmm_field_destroy(h)
    ref = full_oracle(4)
    check(ref, V, E, TOL64)
    check(ref, Vp, None, TOL64)


# ------------------------------------------------------------------ per-walker energy (Eq. 4)
@pytest.mark.parametrize("precision,tol", [("fp64", 1e-11), ("fp32", E_TOL)])
@pytest.mark.parametrize("layout", ["list", "grid"])
def test_eval_energy_per_walker(torch_cuda, B, oracle_mod, precision, tol, layout):
    """qmmm_field_eval_energy: U_ES[w] = -sum_i V(r_wi) for 6 walkers x 37
    electrons on config 1's environment, against the oracle's per-walker sums."""
    w = make_workload(1, n_points=(6, 37))
    pts = w.elec_xyz.reshape(-1, 3)
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_E=False)
    want = -ref.V.reshape(6, 37).sum(1)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, len(pts))
    try:
        B.qmmm_field_set_layout(h, layout)
        d = torch_cuda.from_numpy(pts).cuda()
        U = torch_cuda.full((6,), float("nan"), dtype=torch_cuda.float64, device="cuda")
        B.qmmm_field_eval_energy(h, d, 6, 37, U, precision)
        torch_cuda.cuda.synchronize()
        got = U.cpu().numpy()
        assert np.max(np.abs(got - want)) <= tol, f"max |dU| = {np.max(np.abs(got - want)):.3e} hartree"
        U2 = torch_cuda.zeros(6, dtype=torch_cuda.float64, device="cuda")
        B.qmmm_field_eval_energy(h, d, 6, 37, U2, precision)
        torch_cuda.cuda.synchronize()
        assert np.array_equal(got, U2.cpu().numpy())                     # deterministic
        V, _ = run(torch_cuda, B, h, pts, precision, want_E=False)
        assert np.max(np.abs(got + V.reshape(6, 37).sum(1))) <= 1e-11    # = -sum of eval's V
    finally:
        B.qmmm_field_destroy(h)


# --------------------------------------------------------------------- seeded random sweep
def test_random_grids_plans_and_precisions(torch_cuda, B, oracle_mod):
    """40 seeded random combinations of grid shape, spacing, fill, point count, launch plan,
    precision and entry point (list + detection, or qmmm_field_create_grid), each against the
    oracle on the list of occupied nodes."""
    rng = np.random.default_rng(20261104)
    for case in range(40):
        n = tuple(int(v) for v in rng.integers(1, 70, size=3))
        if rng.random() < 0.5:
            n = (n[0], int(rng.choice([32, 64, 96])), int(rng.choice([64, 128])))
        h = float(rng.choice([0.1, 0.25, 0.3, 0.5]))
        origin = rng.normal(size=3) * 3.0
        centre = origin + 0.5 * h * (np.array(n) - 1)
        dense, pos, q = random_grid(rng, n, h, origin, fill=float(rng.uniform(0.55, 1.0)),
                                    hole=(centre, 1.5), signed=bool(rng.random() < 0.3))
        if len(q) == 0:
            continue
        K = int(rng.integers(0, 9))
        nuc = centre + rng.normal(size=(K, 3)) * 3.0 + 5.0
        Z = rng.choice([1.0, 6.0, 7.0, 8.0], size=K)
        P = int(rng.choice([1, 2, 3, 5, 8, 17, 32, 33, 64, 100, 257]))
        pts = centre + rng.normal(size=(P, 3)) * 0.4
        pts = centre + (pts - centre) * np.minimum(1.0, 1.1 / np.linalg.norm(pts - centre, axis=1))[:, None]
        precision = "fp32" if rng.random() < 0.5 else "fp64"
        tol = TOL32 if precision == "fp32" else TOL64
        ref = oracle_mod.field(pos, q, nuc if K else NO_XYZ, Z if K else NO_Z, pts, want_abs=True)
        use_list = len(q) >= 4096 and rng.random() < 0.5
        if use_list:
            hnd = B.qmmm_field_create(pos, q, nuc if K else None, Z if K else None, P)
        else:
            hnd = B.qmmm_field_create_grid(origin, h, n, dense, nuc if K else None, Z if K else None, P)
        try:
            gi = B.qmmm_field_get_grid_info(hnd)
            if not gi["present"]:       # a sparse random grid may fail the fill criterion
                continue
            plan = dict(points_per_thread=int(rng.choice([0, 1, 2, 4, 8])),
                        point_warps=int(rng.choice([0, 1, 2, 4, 8, 16])),
                        slices=int(rng.choice([0, 1, 3, 37, 200])), stages=int(rng.choice([0, 2, 5, 8])))
            want_E = bool(rng.random() < 0.8)
            V, E = run(torch_cuda, B, hnd, pts, precision, want_E=want_E, layout="grid", plan=plan)
            msg = f"case {case}: n={n} h={h} P={P} {precision} plan={plan} list={use_list}"
            try:
                check(ref, V, E if want_E else None, tol)
            except AssertionError as exc:
                raise AssertionError(f"{msg}: {exc}") from None
        finally:
            B.qmmm_field_destroy(hnd)


# ------------------------------------------------- shared handles
@pytest.mark.parametrize("precision", ["fp64", "fp32"])
def test_shared_handles_on_concurrent_streams(torch_cuda, B, precision):
    """qmmm_field_share: two handles on one environment (shared packed sources, own
    workspaces) evaluate different point sets concurrently on two streams; results are bitwise
    those of one handle used sequentially, also after the parent has been destroyed."""
    torch = torch_cuda
    w = make_workload(1)
    rng = np.random.default_rng(8)
    pa = rng.normal(size=(48, 3)) * 0.8
    pb = rng.normal(size=(200, 3)) * 0.8
    parent = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, 48)
    child = B.qmmm_field_share(parent, 200)
    try:
        Va, Ea = run(torch, B, parent, pa, precision)
        gi_p, gi_c = B.qmmm_field_get_grid_info(parent), B.qmmm_field_get_grid_info(child)
        assert gi_c["present"] == gi_p["present"] and gi_c["n"] == gi_p["n"]
        Vb, Eb = run(torch, B, child, pb, precision)
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        da, db = torch.from_numpy(pa).cuda(), torch.from_numpy(pb).cuda()
        oa = (torch.zeros(48, dtype=torch.float64, device="cuda"), torch.zeros((48, 3), dtype=torch.float64, device="cuda"))
        ob = (torch.zeros(200, dtype=torch.float64, device="cuda"), torch.zeros((200, 3), dtype=torch.float64, device="cuda"))
        torch.cuda.synchronize()
        for _ in range(60):                      # interleaved launches, no synchronisation
            B.qmmm_field_eval(parent, da, 1, 48, oa[0], oa[1], precision, s1)
            B.qmmm_field_eval(child, db, 1, 200, ob[0], ob[1], precision, s2)
        torch.cuda.synchronize()
        assert np.array_equal(oa[0].cpu().numpy(), Va) and np.array_equal(oa[1].cpu().numpy(), Ea)
        assert np.array_equal(ob[0].cpu().numpy(), Vb) and np.array_equal(ob[1].cpu().numpy(), Eb)
        B.qmmm_field_destroy(parent)             # the child keeps the source copies alive
        parent = None
        Vb2, Eb2 = run(torch, B, child, pb, precision)
        assert np.array_equal(Vb2, Vb) and np.array_equal(Eb2, Eb)
        hv = np.zeros(1); he = np.zeros((1, 3))  # the child's own move server
        B.qmmm_field_eval_host(child, np.ascontiguousarray(pb[:1]), 1, 1, hv, he, precision)
        assert np.all(np.isfinite(hv)) and abs(hv[0] - Vb[0]) <= 1e-5 * abs(Vb[0])
    finally:
        if parent is not None:
            B.qmmm_field_destroy(parent)
        B.qmmm_field_destroy(child)


# ----------------------------------------------------------------------- CUDA graphs
@pytest.mark.parametrize("layout,precision", [("grid", "fp32"), ("grid", "fp64"), ("list", "fp32"), ("list", "fp64")])
def test_eval_is_cuda_graph_capturable(torch_cuda, B, layout, precision):
    """qmmm_field_eval only enqueues work on the caller's stream (no allocation, no
    synchronisation), so a sequence of evaluations can be captured into a CUDA graph and
    replayed; the replay gives bitwise the eager results, also after the inputs change."""
    torch = torch_cuda
    w = make_workload(1)
    rng = np.random.default_rng(4)
    P = 32
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, P)
    try:
        B.qmmm_field_set_layout(h, layout)
        pts = [torch.from_numpy(rng.normal(size=(P, 3)) * 0.8).cuda() for _ in range(3)]
        outs = [(torch.zeros(P, dtype=torch.float64, device="cuda"),
                 torch.zeros((P, 3), dtype=torch.float64, device="cuda")) for _ in range(3)]
        eager = []
        for p in pts:                                   # eager reference (also warms up)
            V = torch.zeros(P, dtype=torch.float64, device="cuda")
            E = torch.zeros((P, 3), dtype=torch.float64, device="cuda")
            B.qmmm_field_eval(h, p, 1, P, V, E, precision)
            torch.cuda.synchronize()
            eager.append((V.cpu().numpy(), E.cpu().numpy()))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for p, (V, E) in zip(pts, outs):
                B.qmmm_field_eval(h, p, 1, P, V, E, precision)      # current (capturing) stream
        for rep in range(3):
            for V, E in outs:
                V.zero_(); E.zero_()
            g.replay()
            torch.cuda.synchronize()
            for (V, E), (Ve, Ee) in zip(outs, eager):
                assert np.array_equal(V.cpu().numpy(), Ve) and np.array_equal(E.cpu().numpy(), Ee)
        # new positions in the same buffers: the graph re-reads them
        new = torch.from_numpy(rng.normal(size=(P, 3)) * 0.8).cuda()
        Vn = torch.zeros(P, dtype=torch.float64, device="cuda"); En = torch.zeros((P, 3), dtype=torch.float64, device="cuda")
        B.qmmm_field_eval(h, new, 1, P, Vn, En, precision)
        torch.cuda.synchronize()
        pts[1].copy_(new)
        g.replay()
        torch.cuda.synchronize()
        assert np.array_equal(outs[1][0].cpu().numpy(), Vn.cpu().numpy())
        assert np.array_equal(outs[1][1].cpu().numpy(), En.cpu().numpy())
    finally:
        B.qmmm_field_destroy(h)


# --------------------------------------------------------- dz table and its fallback
@pytest.mark.parametrize("nz,P,precision,tol,table", [
    (64, 128, "fp32", TOL32, True), (130, 128, "fp32", TOL32, True), (400, 128, "fp32", TOL32, False),
    (64, 128, "fp64", TOL64, True), (300, 128, "fp64", TOL64, True), (600, 128, "fp64", TOL64, False),
    (64, 8, "fp32", TOL32, True), (1700, 8, "fp32", TOL32, False), (64, 3, "fp64", TOL64, False)])
def test_dz_table_and_stepped_dz_kernels(torch_cuda, B, oracle_mod, nz, P, precision, tol, table):
    """The grid kernels tabulate dz = u_z - k per CTA in shared memory when the table fits
    (qmmm_field_info.last_dz_table; FP32: batched and few-point plans alike, FP64: the batched
    plan) and step it per pair otherwise (long z axes; the FP64 few-point walks): both against
    the oracle, on z extents with ragged last gchunks."""
    n = (9, 8, nz)
    h = 0.25
    rng = np.random.default_rng(1000 + nz + P)
    origin = np.array([-1.0, -0.9, -0.5 * h * (nz - 1)]) + rng.normal(size=3) * 0.1
    centre = origin + 0.5 * h * (np.array(n) - 1)
    dense, pos, q = random_grid(rng, n, h, origin, fill=0.8, hole=(centre, 1.6))
    nuc = centre + np.array([3.0, -2.5, 4.0]) + rng.normal(size=(4, 3))
    Z = np.array([1.0, 6.0, 7.0, 8.0])
    pts = centre + rng.normal(size=(P, 3)) * 0.3
    pts = centre + (pts - centre) * np.minimum(1.0, 0.6 / np.linalg.norm(pts - centre, axis=1))[:, None]
    ref = oracle_mod.field(pos, q, nuc, Z, pts, want_abs=True)
    hnd = B.qmmm_field_create_grid(origin, h, n, dense, nuc, Z, P)
    try:
        V, E = run(torch_cuda, B, hnd, pts, precision)
        assert bool(B.qmmm_field_get_info(hnd)["last_dz_table"]) == table
        check(ref, V, E, tol)
        if precision == "fp64":                                   # potential only
            V0, _ = run(torch_cuda, B, hnd, pts, precision, want_E=False)
            check(ref, V0, None, tol)
    finally:
        B.qmmm_field_destroy(hnd)


@pytest.mark.parametrize("layout", ["grid", "list"])
@pytest.mark.parametrize("clearance,local", [(2.0, -1), (1.2, 1)])
def test_fp32_field_next_to_cells_on_a_128_node_axis(torch_cuda, B, oracle_mod, layout, clearance, local):
    """What include/qmmm_field.h promises for axes of up to 128 nodes (all FP32 BASELINE
    configurations): with the whole-grid lattice (automatic there) E keeps 1e-5 for points two
    cell edges from the charged cells; with qmmm_field_set_local_lattice(h, 1) for points 1.2
    cell edges away.  The list kernels always use a lattice per 2,048-source block."""
    n, h = (12, 11, 128), 0.25
    rng = np.random.default_rng(5)
    origin = np.array([-1.4, -1.3, -0.5 * h * 127]) + rng.normal(size=3) * 0.05
    centre = origin + 0.5 * h * (np.array(n) - 1)
    dense, pos, q = random_grid(rng, n, h, origin, fill=0.9, hole=(centre, 1.0))
    d = pos - centre
    r = np.linalg.norm(d, axis=1)
    rim = np.argsort(r)[:96]
    pts = pos[rim] - d[rim] / r[rim, None] * (clearance * h)
    ref = oracle_mod.field(pos, q, NO_XYZ, NO_Z, pts, want_abs=True)
    hnd = B.qmmm_field_create(pos, q, None, None, len(pts))
    try:
        B.qmmm_field_set_local_lattice(hnd, local)
        V, E = run(torch_cuda, B, hnd, pts, "fp32", layout=layout)
        if layout == "grid":
            assert B.qmmm_field_get_info(hnd)["last_local_lattice"] == (1 if local == 1 else 0)
        check(ref, V, E, TOL32)
    finally:
        B.qmmm_field_destroy(hnd)


@pytest.mark.parametrize("layout", ["grid", "list"])
@pytest.mark.parametrize("nz", [400, 130])
def test_fp32_field_next_to_cells_on_a_long_axis(torch_cuda, B, oracle_mod, layout, nz):
    """FP32 evaluates the field at the point's LATTICE position (only V is corrected for the
    residual).  With one lattice per grid axis the residual is 2^-25 of the
    axis length: on a 400-node axis, 1.2 nodes from a charged cell, |E| was off by 1.5e-5 in
    round 1.  The lattice per work unit (grid kernels; automatic beyond 128 nodes) and per
    2,048-source block (list kernels) keeps the plain 1e-5: points 1.2 nodes from charged
    cells, both layouts, no clearance clause."""
    n, h = (12, 11, nz), 0.25
    rng = np.random.default_rng(7 + nz)
    origin = np.array([-1.4, -1.3, -0.5 * h * (nz - 1)]) + rng.normal(size=3) * 0.05
    centre = origin + 0.5 * h * (np.array(n) - 1)
    dense, pos, q = random_grid(rng, n, h, origin, fill=0.9, hole=(centre, 1.0))
    # points 1.2 nodes (0.3 bohr) from charged cells on the rim of the hole, on the inner side
    d = pos - centre
    r = np.linalg.norm(d, axis=1)
    rim = np.argsort(r)[:96]
    pts = pos[rim] - d[rim] / r[rim, None] * (1.2 * h)
    pts = np.concatenate([pts, centre + rng.normal(size=(32, 3)) * 0.2])
    nearest = np.min(np.linalg.norm(pts[:, None, :] - pos[None, rim, :], axis=2), axis=1)
    assert 1.0 * h <= nearest.min() <= 1.2001 * h
    nuc = centre + np.array([3.0, -2.5, 4.0]) + rng.normal(size=(4, 3))
    Z = np.array([1.0, 6.0, 7.0, 8.0])
    ref = oracle_mod.field(pos, q, nuc, Z, pts, want_abs=True)
    hnd = B.qmmm_field_create(pos, q, nuc, Z, len(pts))
    try:
        assert B.qmmm_field_get_grid_info(hnd)["present"]
        for plan in (dict(), dict(points_per_thread=8), dict(points_per_thread=2, point_warps=4, slices=9)):
            V, E = run(torch_cuda, B, hnd, pts, "fp32", layout=layout, plan=plan)
            if layout == "grid":
                assert bool(B.qmmm_field_get_info(hnd)["last_local_lattice"]) == (nz > 128)
            check(ref, V, E, TOL32)
        for npts in (1, 2):                                         # the node-packed single-point walk
            V, E = run(torch_cuda, B, hnd, pts[:npts], "fp32", layout=layout)
            eV, eE = rel_errors(ref, np.concatenate([V, ref.V[npts:]]), np.concatenate([E, ref.E[npts:]]))
            assert eV.max() <= TOL32 and eE.max() <= TOL32
        if layout == "grid" and nz <= 128 + 2:
            # forcing the lattice per work unit on a short axis changes nothing but rounding
            B.qmmm_field_set_local_lattice(hnd, 1)
            V1, E1 = run(torch_cuda, B, hnd, pts, "fp32", layout=layout)
            assert B.qmmm_field_get_info(hnd)["last_local_lattice"] == 1
            check(ref, V1, E1, TOL32)
            B.qmmm_field_set_local_lattice(hnd, -1)
        V64, E64 = run(torch_cuda, B, hnd, pts, "fp64", layout=layout)
        check(ref, V64, E64, TOL64)
    finally:
        B.qmmm_field_destroy(hnd)


@pytest.mark.parametrize("layout", ["grid", "list"])
def test_unit_of_charge_does_not_matter(torch_cuda, B, layout):
    """Scaling every charge by 2^k scales V and E by 2^k BITWISE (the oracle has the same pin):
    FP64 trivially; FP32 because its copies store the cell charges relative to a power of two
    near the largest one, so tiny charges (below FP32's normal range, 1.2e-38) keep their
    precision instead of being flushed."""
    w = make_workload(1, n_points=(1, 24))
    pts = w.elec_xyz.reshape(-1, 3)
    out = {}
    for k in (0, -100, -140, 60):
        f = 2.0 ** k
        hnd = B.qmmm_field_create(w.src_xyz, w.src_q * f, w.nuc_xyz, w.nuc_Z * f, len(pts))
        try:
            for prec in ("fp64", "fp32"):
                out[(k, prec)] = run(torch_cuda, B, hnd, pts, prec, layout=layout)
        finally:
            B.qmmm_field_destroy(hnd)
    for prec in ("fp64", "fp32"):
        V0, E0 = out[(0, prec)]
        for k in (-100, -140, 60):
            V, E = out[(k, prec)]
            assert np.array_equal(V, V0 * 2.0 ** k) and np.array_equal(E, E0 * 2.0 ** k), (prec, k)


# ----------------------------------------------- overlapped back-to-back evaluations (PDL)
@pytest.mark.parametrize("layout,precision", [("grid", "fp32"), ("grid", "fp64"), ("list", "fp32"), ("list", "fp64")])
@pytest.mark.parametrize("P", [1, 4, 32])
def test_overlapped_back_to_back_evaluations_are_bitwise_the_same(torch_cuda, B, oracle_mod, layout,
                                                                  precision, P):
    """qmmm_field_set_overlap: evaluation n + 1 starts while evaluation n is still running
    (programmatic dependent launch) and waits for it only before it touches the workspace, the
    tickets and the outputs.  300 evaluations of changing batch size in one stream -- every one
    reuses the same workspace and tickets -- give bitwise the results of the serial launches
    (same plan), eagerly and replayed from a CUDA graph; a sample is checked against the oracle."""
    torch = torch_cuda
    w = make_workload(1)
    rng = np.random.default_rng(11)
    n = 300
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, P)
    try:
        B.qmmm_field_set_layout(h, layout)
        sizes = [P if i % 3 else max(1, P // 2) for i in range(n)]      # the plan changes too
        pts = [torch.from_numpy(rng.normal(size=(sz, 3)) * 0.8).cuda() for sz in sizes]
        res = {}
        for mode in ("serial", "overlap", "graph"):
            B.qmmm_field_set_overlap(h, mode != "serial")
            V = torch.full((n, P), float("nan"), dtype=torch.float64, device="cuda")
            E = torch.full((n, P, 3), float("nan"), dtype=torch.float64, device="cuda")
            if mode == "graph":
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g):
                    for i, p in enumerate(pts):
                        B.qmmm_field_eval(h, p, 1, sizes[i], V[i, :sizes[i]], E[i, :sizes[i]], precision)
                g.replay()
                g.replay()
            else:
                for i, p in enumerate(pts):
                    B.qmmm_field_eval(h, p, 1, sizes[i], V[i, :sizes[i]], E[i, :sizes[i]], precision)
            torch.cuda.synchronize()
            res[mode] = (V.cpu().numpy(), E.cpu().numpy())
        assert np.array_equal(res["graph"][0], res["overlap"][0], equal_nan=True)
        assert np.array_equal(res["graph"][1], res["overlap"][1], equal_nan=True)
        if layout == "grid":
            # overlapped few-point grid evaluations run 4-warp CTAs (several evaluations share an
            # SM): another split of the z runs / gchunks over the warps, so the sums agree with
            # the serial launches to rounding (of the arithmetic type), not bitwise
            rt = 1e-12 if precision == "fp64" else 2e-6
            assert np.allclose(res["overlap"][0], res["serial"][0], rtol=rt, atol=0, equal_nan=True)
            assert np.allclose(res["overlap"][1], res["serial"][1], rtol=0,
                               atol=rt * np.nanmax(np.abs(res["serial"][1])), equal_nan=True)
        else:
            assert np.array_equal(res["overlap"][0], res["serial"][0], equal_nan=True)
            assert np.array_equal(res["overlap"][1], res["serial"][1], equal_nan=True)
        tol = TOL64 if precision == "fp64" else TOL32
        for i in (0, 1, 150, n - 1):
            q = pts[i].cpu().numpy()
            ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, q, want_abs=True)
            check(ref, res["overlap"][0][i, :sizes[i]], res["overlap"][1][i, :sizes[i]], tol)
    finally:
        B.qmmm_field_destroy(h)


@pytest.mark.parametrize("precision,tol", [("fp64", TOL64), ("fp32", TOL32)])
@pytest.mark.parametrize("layout", ["grid", "list"])
def test_eval_moves_device_sequence(torch_cuda, B, oracle_mod, precision, tol, layout):
    """qmmm_field_eval_moves: 200 independent single-electron moves of config 2's random walk
    (and a 3-point variant) issued from C as overlapped launches; every move against the
    oracle, twice bitwise the same, and the handle's overlap setting is left as it was."""
    torch = torch_cuda
    w = make_workload(2, n_points=(200, 1))
    pts = w.elec_xyz.reshape(-1, 3)
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, 4)
    try:
        B.qmmm_field_set_layout(h, layout)
        d = torch.from_numpy(pts).cuda()
        out = []
        for rep in range(2):
            V = torch.full((200,), float("nan"), dtype=torch.float64, device="cuda")
            E = torch.full((200, 3), float("nan"), dtype=torch.float64, device="cuda")
            B.qmmm_field_eval_moves(h, d, 200, 1, V, E, precision)
            torch.cuda.synchronize()
            out.append((V.cpu().numpy(), E.cpu().numpy()))
        assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
        check(ref, out[0][0], out[0][1], tol)
        # three points per move (66 moves), potential only
        V3 = torch.full((198,), float("nan"), dtype=torch.float64, device="cuda")
        B.qmmm_field_eval_moves(h, d, 66, 3, V3, None, precision)
        torch.cuda.synchronize()
        eV = np.abs(V3.cpu().numpy() - ref.V[:198]) / np.abs(ref.V[:198])
        assert eV.max() <= tol
        # a plain eval afterwards is serial again (same result as a fresh serial evaluation)
        V1, E1 = run(torch, B, h, pts[:1], precision)
        assert abs(V1[0] - ref.V[0]) <= tol * abs(ref.V[0])
        with pytest.raises(B.QmmmError):
            B.qmmm_field_eval_moves(h, d, -1, 1, V, E, precision)
    finally:
        B.qmmm_field_destroy(h)


def test_overlap_stress_two_streams_mixed_shapes(torch_cuda, B):
    """Overlapped launches, light CTAs and tagged-record collection under stress: two handles on
    the same environment (qmmm_field_share) run 250 evaluations each on two concurrent streams,
    batch size, precision, layout and E / no E changing from one evaluation to the next (so
    ticket and push collections, light and batched plans, grid and list kernels alternate on
    the same workspace).  Every result must equal a serial reference of the same call to
    rounding; a stale or torn record would be off by orders of magnitude."""
    torch = torch_cuda
    w = make_workload(1)
    rng = np.random.default_rng(77)
    sizes = [1, 2, 3, 4, 5, 8, 17, 32, 64, 100, 257]
    Pmax = max(sizes)
    parent = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, Pmax)
    child = B.qmmm_field_share(parent, Pmax)
    try:
        n = 250
        calls = []
        for i in range(n):
            P = int(rng.choice(sizes))
            calls.append((P, str(rng.choice(["fp32", "fp64"])), str(rng.choice(["auto", "list"])),
                          bool(rng.random() < 0.8),
                          torch.from_numpy(rng.normal(size=(P, 3)) * 0.8).cuda()))
        # serial reference on the parent
        ref = []
        B.qmmm_field_set_overlap(parent, False)
        for P, prec, lay, wantE, pts in calls:
            B.qmmm_field_set_layout(parent, lay)
            V = torch.zeros(P, dtype=torch.float64, device="cuda")
            E = torch.zeros((P, 3), dtype=torch.float64, device="cuda") if wantE else None
            B.qmmm_field_eval(parent, pts, 1, P, V, E, prec)
            ref.append((V, E))
        torch.cuda.synchronize()
        # overlapped, both handles at once on two streams
        streams = [torch.cuda.Stream(), torch.cuda.Stream()]
        outs = [[], []]
        for k, hnd in enumerate((parent, child)):
            B.qmmm_field_set_overlap(hnd, True)
        for (P, prec, lay, wantE, pts) in calls:
            for k, hnd in enumerate((parent, child)):
                B.qmmm_field_set_layout(hnd, lay)
                with torch.cuda.stream(streams[k]):          # (the NaN fill on the same stream)
                    V = torch.full((P,), float("nan"), dtype=torch.float64, device="cuda")
                    E = torch.full((P, 3), float("nan"), dtype=torch.float64, device="cuda") if wantE else None
                    B.qmmm_field_eval(hnd, pts, 1, P, V, E, prec, streams[k])
                outs[k].append((V, E))
        torch.cuda.synchronize()
        for k in range(2):
            for (P, prec, lay, wantE, pts), (Vr, Er), (V, E) in zip(calls, ref, outs[k]):
                rt = 1e-12 if prec == "fp64" else 2e-6
                assert torch.allclose(V, Vr, rtol=rt, atol=0), (k, P, prec, lay)
                if wantE:
                    assert float((E - Er).abs().max()) <= rt * float(Er.abs().max()), (k, P, prec, lay)
    finally:
        B.qmmm_field_destroy(child)
        B.qmmm_field_destroy(parent)


# ------------------------------------------ config 2 on the device: warp-private grid walks
@pytest.mark.parametrize("precision,tol", [("fp64", TOL64), ("fp32", TOL32)])
def test_config2_single_point_device_evaluations(torch_cuda, B, oracle_mod, precision, tol):
    """Config 2 (one electron, 2.08 M cells + 1,024 nuclei) evaluated point by point with
    qmmm_field_eval in bench.py's launch configuration: AUTO picks the grid kernels' single-point
    modes (FP32: node-packed walk, FP64: warp-own walk).  24 positions of the seeded random
    walk against the oracle; a two-point and a four-point batch as well."""
    w = make_workload(2, n_points=(24, 1))
    pts = w.elec_xyz.reshape(-1, 3)
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    h = B.qmmm_field_create(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, 4)
    try:
        V = np.zeros(len(pts)); E = np.zeros((len(pts), 3))
        for i in range(len(pts)):
            V[i:i + 1], E[i:i + 1] = run(torch_cuda, B, h, pts[i:i + 1], precision)
            assert B.qmmm_field_get_grid_info(h)["last_layout"] == "grid"
        check(ref, V, E, tol)
        assert B.qmmm_field_get_info(h)["last_plan"]["point_warps"] == 1
        for n in (2, 4):
            Vn, En = run(torch_cuda, B, h, pts[:n], precision)
            eV, eE = rel_errors(ref, np.concatenate([Vn, V[n:]]), np.concatenate([En, E[n:]]))
            assert eV.max() <= tol and eE.max() <= tol
        Vl, El = run(torch_cuda, B, h, pts[:1], precision, layout="list")
        assert abs(Vl[0] - V[0]) <= 2 * tol * abs(V[0])
    finally:
        B.qmmm_field_destroy(h)


def test_accurate_v_and_potential_only_on_orthorhombic_cells(torch_cuda, B, oracle_mod):
    """The batched FP32 table kernels that form rxy2 in FP64 from the points' true coordinates
    (accurate V, the default; potential only) on cells that are not cubic (0.3 x 0.2 x 0.25 bohr,
    24 x 40 x 70 nodes: two z segments, empty cells): against the oracle, with the faster V + E
    kernel beside them; qmmm_field_info.last_accurate_v says which one ran."""
    rng = np.random.default_rng(5)
    n, hh = (24, 40, 70), np.array([0.3, 0.2, 0.25])
    origin = np.array([1.0, -2.0, 0.5])
    centre = origin + 0.5 * hh * (np.array(n) - 1)
    dense, pos, q = random_grid(rng, n, hh, origin, fill=0.7, hole=(centre, 1.6))
    P = 300
    pts = centre + rng.normal(size=(P, 3)) * 0.5
    pts = centre + (pts - centre) * np.minimum(1.0, 1.1 / np.linalg.norm(pts - centre, axis=1))[:, None]
    ref = oracle_mod.field(pos, q, NO_XYZ, NO_Z, pts, want_abs=True)
    h = B.qmmm_field_create_grid(origin, tuple(hh), n, dense, None, None, P)
    try:
        rms = {}
        for want_E, accurate in ((True, True), (True, False), (False, True)):
            B.qmmm_field_set_accurate_v(h, accurate)
            V, E = run(torch_cuda, B, h, pts, "fp32", want_E=want_E, plan=dict(points_per_thread=4, point_warps=16))
            check(ref, V, E, TOL32)
            assert B.qmmm_field_get_info(h)["last_accurate_v"] == int(accurate)
            assert B.qmmm_field_get_info(h)["last_dz_table"] == 1
            rms[(want_E, accurate)] = float(np.std(V - ref.V))
        assert rms[(True, True)] < 0.8 * rms[(True, False)]        # measured: 6.6e-8 against 1.2e-7
        assert rms[(False, True)] < 0.8 * rms[(True, False)]
    finally:
        B.qmmm_field_destroy(h)
