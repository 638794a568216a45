"""The arithmetic identity behind the compensated row sums of the FP32 grid kernels
(paper_1011_4687_b200/csrc/qmmm_grid.cuh, GridRowF32::run and add_run), checked
in IEEE float32 on the CPU with numpy -- no GPU, no oracle, none of the library's code.

The kernels sum a row of 64 terms a_k (V0) and c_k r_k^2 (T) as a tree 4 -> 16 -> 64 and return
V = V0 - D / 2 with D = T - V0 (the Newton step applied to the sum).  Where the last level is
compensated they keep, for every add s = fl(v + x), the error term er = (s - v) - x and fold
2 er into D.  What this test pins:

* the fast two-sum is exact whenever |v| >= |x| (always from the third 16-node sum on): s - er ==
  v + x in exact arithmetic, so the compensated V equals the exactly summed 16-node sums; where
  the second sum is the larger one the error term may itself round (half an ulp of that sum,
  in a minority of rows);
* T16 - V16 is exact (Sterbenz) when the two agree to a factor of two, as they do to 1e-6;
* on slowly varying same-sign terms -- the shape of a row's terms -- the plain last level is
  off by rounding errors of the size the error terms account for, and the compensated value is
  closer to the exact sum than the plain one by construction.
"""
from fractions import Fraction

import numpy as np

f32 = np.float32


def seq(values):
    s = values[0]
    for x in values[1:]:
        s = f32(s + x)
    return s


def row_terms(rng, n=64):
    """Same-sign, slowly varying terms like q / r along a grid row, and their Newton partners."""
    z = np.arange(n) - rng.uniform(0, n)
    rxy2 = rng.uniform(4.0, 400.0)
    q = -rng.uniform(0.5, 1.0) * 1e-3
    r2 = (rxy2 + z * z).astype(f32)
    y0 = (f32(1.0) / np.sqrt(r2.astype(np.float64))).astype(f32)
    y0 = (y0 * (f32(1.0) + rng.uniform(-2e-7, 2e-7, n).astype(f32))).astype(f32)     # a seed, not the exact value
    a = (f32(q) * y0).astype(f32)
    c = (a * (y0 * y0).astype(f32)).astype(f32)
    t = (c.astype(np.float64) * r2.astype(np.float64))                               # fma: exact product, rounded in the sum
    return a, t


def tree_16(a, t):
    """The two lower levels (4 -> 16) in float32: four nodes one after the other (t through an fma
    chain), the four 4-node sums pairwise."""
    v16, t16 = [], []
    for g in range(0, len(a), 16):
        vs, ts = [], []
        for k in range(g, g + 16, 4):
            vs.append(seq([a[k], a[k + 1], a[k + 2], a[k + 3]]))
            acc = f32(t[k])
            for j in range(k + 1, k + 4):
                acc = f32(np.float64(acc) + t[j])                                    # fma(c, r2, acc): one rounding
            ts.append(acc)
        v16.append(f32(f32(vs[0] + vs[1]) + f32(vs[2] + vs[3])))                    # pairwise, as the compensated kernels
        t16.append(f32(f32(ts[0] + ts[1]) + f32(ts[2] + ts[3])))
    return v16, t16


def test_two_sum_last_level_returns_the_exact_sum_of_the_16_node_sums():
    rng = np.random.default_rng(11)
    worse = inexact_rows = 0
    for _ in range(300):
        a, t = row_terms(rng)
        v16, t16 = tree_16(a, t)
        # the kernel's compensated level: v, d in float32
        v, d = f32(0.0), f32(0.0)
        all_exact = True
        for x, tx in zip(v16, t16):
            d16 = f32(tx - x)
            assert Fraction(float(d16)) == Fraction(float(tx)) - Fraction(float(x))      # Sterbenz: exact
            s = f32(v + x)
            bb = f32(s - v)
            er = f32(bb - x)
            if abs(v) >= abs(x) or v == 0:
                assert Fraction(float(s)) - Fraction(float(er)) == Fraction(float(v)) + Fraction(float(x))
            else:                 # second partial sum with the smaller term first: er is itself rounded
                all_exact &= Fraction(float(s)) - Fraction(float(er)) == Fraction(float(v)) + Fraction(float(x))
            v = s
            d = f32(d + f32(f32(2.0) * er + d16))
        V_comp = float(v) - 0.5 * float(d)
        # what it should equal: the exact sum of the 16-node sums, Newton step applied
        V0 = sum(Fraction(float(x)) for x in v16)
        T = sum(Fraction(float(x)) for x in t16)
        V_exact = float(V0 - (T - V0) / 2)
        # the plain last level
        vp, tp = seq(v16), seq(t16)
        V_plain = 1.5 * float(vp) - 0.5 * float(tp)
        ulp = float(np.spacing(f32(abs(V_exact))))
        # d's own rounding only -- or, where the one two-sum outside the exact regime was inexact,
        # half an ulp of the SECOND 16-node sum (at most half an ulp of the row sum, when that
        # group holds most of the row)
        inexact_rows += not all_exact
        assert abs(V_comp - V_exact) <= (0.02 if all_exact else 0.51) * ulp, (V_comp, V_exact, ulp)
        assert abs(V_plain - V_exact) <= 2.5 * ulp
        worse += abs(V_plain - V_exact) > abs(V_comp - V_exact)
    assert worse >= 200           # the plain level is off by a good fraction of an ulp in most rows
    assert inexact_rows <= 90     # a minority (16 % here): the second 16-node sum is the larger one and its error term rounds
