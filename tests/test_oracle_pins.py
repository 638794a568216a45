"""Pins for the CPU oracle (oracle/qmmm_oracle.c) against things other than itself.

The paper prints no worked numeric example of Eq. 4, so the oracle
is pinned by closed forms, exact symmetric cases, invariants, multiprecision brute
force and an independent library restatement (SURVEY.md 8(c) "What pins each part").
Each test names the mistake it would catch.
"""
import math

import numpy as np
import pytest

from paper_1011_4687_b200.workloads import make_workload

EMPTY3 = np.zeros((0, 3))
EMPTY = np.zeros(0)


def norm_err(a, b):
    return np.linalg.norm(a - b, axis=-1) / np.linalg.norm(b, axis=-1)


# ---------------------------------------------------------------- single term
def test_single_term_value_sign_direction(oracle_mod):
    """V = q/d, E = q d_vec/d^3: catches a wrong sign, a swapped r_i/R_j, r^2 vs r^3."""
    R = np.array([[1.0, -2.0, 0.5]])
    q = np.array([-0.75])
    r = np.array([[3.0, 1.0, -1.5]])
    d = r[0] - R[0]
    dn = math.sqrt(float(d @ d))
    res = oracle_mod.field(R, q, EMPTY3, EMPTY, r)
    assert res.V[0] == pytest.approx(q[0] / dn, rel=4e-16)
    np.testing.assert_allclose(res.E[0], q[0] * d / dn ** 3, rtol=1e-15)
    # positive charge: potential positive, field points away from the source
    res = oracle_mod.field(R, -q, EMPTY3, EMPTY, r)
    assert res.V[0] > 0 and float(res.E[0] @ d) > 0


def test_nuclei_enter_with_plus_Z(oracle_mod):
    """Eq. 4: nuclei are a second list with charge +Z; same as appending them to the
    source list (bitwise, same order).  Catches a dropped or sign-flipped nuclear term."""
    w = make_workload(0)
    a = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz)
    b = oracle_mod.field(np.vstack([w.src_xyz, w.nuc_xyz]), np.concatenate([w.src_q, w.nuc_Z]),
                         EMPTY3, EMPTY, w.elec_xyz)
    assert np.array_equal(a.V, b.V) and np.array_equal(a.E, b.E)
    only_nuc = oracle_mod.field(EMPTY3, EMPTY, w.nuc_xyz, w.nuc_Z, w.elec_xyz)
    assert np.all(only_nuc.V > 0)


def test_empty_lists_give_zero(oracle_mod):
    res = oracle_mod.field(EMPTY3, EMPTY, EMPTY3, EMPTY, np.ones((3, 3)))
    assert np.all(res.V == 0) and np.all(res.E == 0)


# ---------------------------------------------------------- closed forms
def _shell_quadrature(a, n_theta=32, n_phi=64):
    """Product quadrature on the sphere of radius a: Gauss-Legendre in cos(theta) x
    equispaced phi; weights sum to 1 (integrates spherical harmonics exactly up to
    degree ~ min(2 n_theta - 1, n_phi - 1))."""
    x, wgt = np.polynomial.legendre.leggauss(n_theta)
    phi = (np.arange(n_phi) + 0.5) * (2 * np.pi / n_phi)
    ct, ph = np.meshgrid(x, phi, indexing="ij")
    st = np.sqrt(1 - ct ** 2)
    pts = a * np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=-1).reshape(-1, 3)
    wts = np.repeat(wgt / (2.0 * n_phi), n_phi)
    return pts, wts


def test_uniform_shell_closed_form(oracle_mod):
    """Newton's shell theorem: outside V = Q/r, E = Q r_vec/r^3; inside V = Q/a, E = 0.
    A many-term machine-precision pin of both V and E."""
    a, Q = 2.0, -3.5
    pts, wts = _shell_quadrature(a)
    outside = np.array([[3.0, 2.0, 1.0], [0.0, 0.0, 5.0], [-2.5, 2.5, 1.2]])
    res = oracle_mod.field(pts, Q * wts, EMPTY3, EMPTY, outside)
    rn = np.linalg.norm(outside, axis=1)
    np.testing.assert_allclose(res.V, Q / rn, rtol=2e-14)
    np.testing.assert_allclose(res.E, Q * outside / rn[:, None] ** 3, rtol=0, atol=3e-14)
    inside = np.array([[0.5, -0.4, 0.3], [0.0, 0.0, 0.0]])
    res = oracle_mod.field(pts, Q * wts, EMPTY3, EMPTY, inside)
    np.testing.assert_allclose(res.V, Q / a, rtol=2e-14)
    np.testing.assert_allclose(res.E, 0.0, atol=3e-14)


def test_ring_on_axis_and_cube_centre(oracle_mod):
    """n equal charges on a ring, point on the axis: V = Q/sqrt(a^2+z^2),
    E_z = Q z/(a^2+z^2)^{3/2}, E_x = E_y = 0.  Cube corners, centre: E = 0."""
    n, a, z, Q = 64, 1.5, 0.8, 2.0
    ang = np.arange(n) * 2 * np.pi / n
    ring = np.stack([a * np.cos(ang), a * np.sin(ang), np.zeros(n)], axis=1)
    res = oracle_mod.field(ring, np.full(n, Q / n), EMPTY3, EMPTY, [[0.0, 0.0, z]])
    s2 = a * a + z * z
    assert res.V[0] == pytest.approx(Q / math.sqrt(s2), rel=1e-15)
    assert res.E[0, 2] == pytest.approx(Q * z / s2 ** 1.5, rel=1e-15)
    assert abs(res.E[0, 0]) < 1e-15 and abs(res.E[0, 1]) < 1e-15
    cube = np.array([[sx, sy, sz] for sx in (-1, 1) for sy in (-1, 1) for sz in (-1, 1)], float)
    res = oracle_mod.field(cube, np.ones(8), EMPTY3, EMPTY, [[0.0, 0.0, 0.0]])
    assert res.V[0] == pytest.approx(8 / math.sqrt(3), rel=1e-15)
    assert np.all(np.abs(res.E[0]) < 1e-15)


def test_gaussian_cloud_closed_form(oracle_mod):
    """Semantics of q = rho dV (reading 1): a normalised s-Gaussian on a
    grid gives V = erf(sqrt(alpha) r)/r and
    E_r = erf(sqrt(alpha) r)/r^2 - 2 sqrt(alpha/pi) exp(-alpha r^2)/r outside the cloud.
    Quadrature-limited pin; also discriminates erf from 1."""
    alpha, h, n = 1.0, 0.2, 81                      # grid +-8 bohr
    ax = (np.arange(n) - (n - 1) / 2) * h
    X, Y, Z = np.meshgrid(ax, ax, ax, indexing="ij")
    pts = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    q = (alpha / np.pi) ** 1.5 * np.exp(-alpha * (pts ** 2).sum(1)) * h ** 3
    for rvec, tolV, tolE in (([2.7, 2.7, 2.7], 1e-10, 1e-9), ([1.5, 1.5, 1.3], 1e-4, 5e-4)):
        rvec = np.array(rvec)
        r = float(np.linalg.norm(rvec))
        res = oracle_mod.field(pts, q, EMPTY3, EMPTY, rvec[None])
        V_ref = math.erf(math.sqrt(alpha) * r) / r
        Er = math.erf(math.sqrt(alpha) * r) / r ** 2 \
            - 2 * math.sqrt(alpha / math.pi) * math.exp(-alpha * r * r) / r
        assert res.V[0] == pytest.approx(V_ref, rel=tolV)
        np.testing.assert_allclose(res.E[0], Er * rvec / r, rtol=tolE)
    # the second point (r = 2.49, quadrature error 3e-5) must tell erf(2.49) = 0.99957
    # from 1, i.e. a Gaussian cloud from a point charge
    assert abs(V_ref - 1 / r) / V_ref > 4e-4


# ----------------------------------------------- independent arithmetic / code
def test_summation_vs_fsum(oracle_mod):
    """Kahan result vs math.fsum (exactly rounded) of the oracle's own terms:
    pins the summation, not the terms."""
    w = make_workload(0)
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz, want_abs=True)
    for i in range(w.P):
        t = oracle_mod.potential_terms(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z,
                                       w.elec_xyz.reshape(-1, 3)[i])
        exact = math.fsum(t)
        assert abs(res.V[i] - exact) <= 2 ** -52 * abs(exact)
        assert res.absV[i] == pytest.approx(math.fsum(np.abs(t)), rel=1e-15)



def test_absolute_sums_absV_absE_are_pinned(oracle_mod):
    """The oracle's condition-number sums absV = sum_j |q_j|/r_ij and absE = sum_j |q_j|/r_ij^2
    (SURVEY.md 8(c) "Error metrics") scale every kappa-aware GPU assertion, so they are pinned
    like V itself: one source (closed form |q|/d and |q|/d^2: catches dividing by r once
    instead of twice, a signed instead of an absolute term), and on config 0 against the
    exactly rounded math.fsum of terms formed here with numpy from the positions (not from the
    oracle's own term routine), and against 50-digit mpmath on a mixed-sign tiny case."""
    R = np.array([[1.0, -2.0, 0.5]])
    r = np.array([[3.0, 1.0, -1.5]])
    d2 = float(((r[0] - R[0]) ** 2).sum())
    for q in (-0.75, 0.75):
        res = oracle_mod.field(R, np.array([q]), EMPTY3, EMPTY, r, want_abs=True)
        assert res.absV[0] == pytest.approx(0.75 / math.sqrt(d2), rel=4e-16)
        assert res.absE[0] == pytest.approx(0.75 / d2, rel=4e-16)
    # one cell and one nucleus of opposite sign: the absolute sums add, V and E cancel partly
    res = oracle_mod.field(R, np.array([-2.0]), np.array([[1.0, -2.0, 2.5]]), np.array([2.0]), r,
                           want_abs=True)
    d2n = float(((r[0] - np.array([1.0, -2.0, 2.5])) ** 2).sum())
    assert res.absV[0] == pytest.approx(2.0 / math.sqrt(d2) + 2.0 / math.sqrt(d2n), rel=4e-16)
    assert res.absE[0] == pytest.approx(2.0 / d2 + 2.0 / d2n, rel=4e-16)
    assert abs(res.V[0]) < res.absV[0] and np.linalg.norm(res.E[0]) < res.absE[0]

    w = make_workload(0)
    pts = w.elec_xyz.reshape(-1, 3)
    allx = np.vstack([w.src_xyz, w.nuc_xyz])
    allq = np.abs(np.concatenate([w.src_q, w.nuc_Z]))
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    for i in range(w.P):
        r2 = ((pts[i] - allx) ** 2).sum(1)
        assert res.absV[i] == pytest.approx(math.fsum(allq / np.sqrt(r2)), rel=4e-15)
        assert res.absE[i] == pytest.approx(math.fsum(allq / r2), rel=4e-15)

    import mpmath as mp
    mp.mp.dps = 50
    rng = np.random.default_rng(12)
    src = rng.uniform(-6, 6, (48, 3)); src = src[np.linalg.norm(src, axis=1) > 2.5]
    q = rng.normal(size=len(src))
    pts = rng.uniform(-1, 1, (3, 3))
    res = oracle_mod.field(src, q, EMPTY3, EMPTY, pts, want_abs=True)
    for i, p in enumerate(pts):
        aV = mp.mpf(0); aE = mp.mpf(0)
        for Rj, qj in zip(src, q):
            r2 = sum((mp.mpf(float(p[k])) - mp.mpf(float(Rj[k]))) ** 2 for k in range(3))
            aV += abs(mp.mpf(float(qj))) / mp.sqrt(r2)
            aE += abs(mp.mpf(float(qj))) / r2
        assert res.absV[i] == pytest.approx(float(aV), rel=1e-15)
        assert res.absE[i] == pytest.approx(float(aE), rel=1e-15)


def _mp_field(src_xyz, src_q, nuc_xyz, nuc_Z, pts):
    import mpmath as mp
    mp.mp.dps = 50
    allx = np.vstack([src_xyz, nuc_xyz])
    allq = np.concatenate([src_q, nuc_Z])
    V, E = [], []
    for r in pts:
        v = mp.mpf(0)
        e = [mp.mpf(0)] * 3
        rr = [mp.mpf(float(c)) for c in r]
        for R, q in zip(allx, allq):
            d = [rr[k] - mp.mpf(float(R[k])) for k in range(3)]
            r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2]
            inv = 1 / mp.sqrt(r2)
            v += mp.mpf(float(q)) * inv
            g = mp.mpf(float(q)) * inv / r2
            e = [e[k] + g * d[k] for k in range(3)]
        V.append(v)
        E.append(e)
    return V, E


def test_mpmath_brute_force_tiny(oracle_mod):
    """50-digit brute force on 4 points x (64 sources + 4 nuclei) with mixed signs:
    oracle within a few ulp x kappa.  Certifies the 1e-12 budget."""
    rng = np.random.default_rng(11)
    src = rng.uniform(-6, 6, (64, 3)); src = src[np.linalg.norm(src, axis=1) > 2.5]
    q = rng.normal(size=len(src))
    nuc = rng.uniform(3, 6, (4, 3)); Z = np.array([1.0, 6.0, 7.0, 8.0])
    pts = rng.uniform(-1, 1, (4, 3))
    res = oracle_mod.field(src, q, nuc, Z, pts, want_abs=True)
    V, E = _mp_field(src, q, nuc, Z, pts)
    for i in range(len(pts)):
        assert abs(res.V[i] - float(V[i])) <= 4e-16 * res.absV[i]
        ee = np.array([float(x) for x in E[i]])
        assert np.linalg.norm(res.E[i] - ee) <= 8e-16 * res.absE[i]


def test_mpmath_config0_and_golden(oracle_mod):
    """Config 0 (8 x 4,112): oracle vs 50-digit brute force, and vs the stored golden
    (tests/golden/config0_oracle.txt, written by tests/golden/make_config0_golden.py
    from the oracle only)."""
    import os
    w = make_workload(0)
    pts = w.elec_xyz.reshape(-1, 3)
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    V, E = _mp_field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts[:2])
    for i in range(2):
        assert abs(res.V[i] - float(V[i])) <= 4e-16 * res.absV[i]
        ee = np.array([float(x) for x in E[i]])
        assert np.linalg.norm(res.E[i] - ee) <= 8e-16 * res.absE[i]
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "config0_oracle.txt"))
    # generator transcendental functions may differ by an ulp across machines
    np.testing.assert_allclose(res.V, gold[:, 0], rtol=1e-12)
    assert np.all(norm_err(res.E, gold[:, 1:4]) < 1e-11)


def test_scipy_restatement(oracle_mod):
    """Independent code path: scipy cdist -> (q / D).sum (pairwise summation)."""
    from scipy.spatial.distance import cdist
    w = make_workload(1, n_points=(1, 4))
    pts = w.elec_xyz.reshape(-1, 3)
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts)
    allx = np.vstack([w.src_xyz, w.nuc_xyz]); allq = np.concatenate([w.src_q, w.nuc_Z])
    D = cdist(pts, allx)
    V = (allq[None] / D).sum(1)
    d = pts[:, None, :] - allx[None, :, :]
    E = (allq[None, :, None] * d / D[:, :, None] ** 3).sum(1)
    np.testing.assert_allclose(res.V, V, rtol=1e-12)
    assert np.all(norm_err(res.E, E) < 1e-11)


# ------------------------------------------------------------- invariants
def test_superposition_and_pow2_scaling(oracle_mod):
    w = make_workload(0)
    pts = w.elec_xyz.reshape(-1, 3)
    full = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    a = oracle_mod.field(w.src_xyz[:1500], w.src_q[:1500], EMPTY3, EMPTY, pts)
    b = oracle_mod.field(w.src_xyz[1500:], w.src_q[1500:], w.nuc_xyz, w.nuc_Z, pts)
    assert np.all(np.abs(a.V + b.V - full.V) <= 4e-16 * full.absV)
    assert np.all(np.linalg.norm(a.E + b.E - full.E, axis=1) <= 4e-16 * full.absE)
    s = oracle_mod.field(w.src_xyz, w.src_q * 8.0, w.nuc_xyz, w.nuc_Z * 8.0, pts)
    assert np.array_equal(s.V, full.V * 8.0) and np.array_equal(s.E, full.E * 8.0)


def test_permutation_of_sources(oracle_mod):
    """Eq. 7 == Eq. 8: term order changes rounding only."""
    w = make_workload(0)
    pts = w.elec_xyz.reshape(-1, 3)
    base = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    perm = np.random.default_rng(5).permutation(w.M)
    res = oracle_mod.field(w.src_xyz[perm], w.src_q[perm], w.nuc_xyz, w.nuc_Z, pts)
    assert np.all(np.abs(res.V - base.V) <= 4e-16 * base.absV)
    assert np.all(np.linalg.norm(res.E - base.E, axis=1) <= 4e-16 * base.absE)


def test_translation_on_dyadic_lattice_is_bitwise(oracle_mod):
    """All coordinates multiples of 2^-20, shifted by a lattice vector: every
    difference r_i - R_j is bit-identical, so V and E are too.  Catches any use of
    absolute coordinates."""
    rng = np.random.default_rng(7)
    snap = lambda a: np.round(a * 2 ** 20) / 2 ** 20
    src = snap(rng.uniform(4, 9, (500, 3)) * rng.choice([-1, 1], (500, 3)))
    q = rng.normal(size=500)
    nuc = snap(rng.uniform(4, 9, (5, 3))); Z = np.array([1.0, 6, 7, 8, 1])
    pts = snap(rng.uniform(-2, 2, (6, 3)))
    shift = np.array([37.0, -12.5, 3.0 + 2 ** -10])
    a = oracle_mod.field(src, q, nuc, Z, pts)
    b = oracle_mod.field(src + shift, q, nuc + shift, Z, pts + shift)
    assert np.array_equal(a.V, b.V) and np.array_equal(a.E, b.E)


def test_rotation_by_90_degrees(oracle_mod):
    """(x,y,z) -> (-y,x,z): V equal, E rotates with the system.  Catches a
    transposed / mis-indexed coordinate."""
    w = make_workload(0)
    rot = lambda a: np.stack([-a[:, 1], a[:, 0], a[:, 2]], axis=1)
    pts = w.elec_xyz.reshape(-1, 3)
    a = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    b = oracle_mod.field(rot(w.src_xyz), w.src_q, rot(w.nuc_xyz), w.nuc_Z, rot(pts))
    assert np.all(np.abs(a.V - b.V) <= 8e-16 * a.absV)
    assert np.all(np.linalg.norm(rot(a.E) - b.E, axis=1) <= 8e-16 * a.absE)
    # asymmetric system: the three components really differ
    assert abs(a.E[0, 0] - a.E[0, 1]) > 1e-6


def test_field_is_minus_gradient_of_potential(oracle_mod):
    """E = -grad V by a 4th-order central difference of the oracle's own V."""
    w = make_workload(0)
    pts = w.elec_xyz.reshape(-1, 3)[:4]
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts)
    h = 2e-3
    grad = np.zeros((len(pts), 3))
    for k in range(3):
        e = np.zeros(3); e[k] = h
        Vs = [oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts + m * e, want_E=False).V
              for m in (-2, -1, 1, 2)]
        grad[:, k] = (Vs[0] - 8 * Vs[1] + 8 * Vs[2] - Vs[3]) / (12 * h)
    assert np.all(norm_err(-grad, res.E) < 2e-9)


def test_mean_value_property_and_gauss_law(oracle_mod):
    """Away from the sources V is harmonic: its average over a small sphere equals
    its value at the centre; the flux of E through a sphere is 4 pi x (enclosed
    charge).  Both by the same product quadrature."""
    w = make_workload(0)
    c = np.array([0.3, -0.2, 0.1])
    sph, wts = _shell_quadrature(1.0, 24, 48)
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, sph + c)
    centre = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, c[None])
    assert float(wts @ res.V) == pytest.approx(centre.V[0], rel=1e-13)
    flux = 4 * np.pi * float(wts @ (res.E * sph).sum(1))           # radius 1
    assert abs(flux) < 1e-11                                        # no charge inside r < 1.4
    # sphere of radius 40 about the origin encloses every charge (all within r < 10);
    # harmonics of degree l decay like (10/40)^l, far below the quadrature's degree
    big, wb = _shell_quadrature(40.0, 48, 96)
    res = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, big)
    flux = 4 * np.pi * 40.0 * float(wb @ (res.E * big).sum(1))
    assert flux == pytest.approx(4 * np.pi * (w.src_q.sum() + w.nuc_Z.sum()), rel=1e-12)


def test_thread_count_independent(oracle_mod):
    w = make_workload(0)
    a = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz, nthreads=1)
    b = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz, nthreads=3)
    assert np.array_equal(a.V, b.V) and np.array_equal(a.E, b.E)
