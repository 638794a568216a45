"""DESIGN.md reading 21: the FP32 kernels apply the Newton step of the reciprocal square root
to the SUM instead of to every pair,

    q y1 = q y0 (3 - r^2 y0^2) / 2 = (3 a - c r^2) / 2,   a = q y0,  c = q y0^3
    =>  V = sum q y1 = (3 sum a - sum c r^2) / 2.

This file checks the arithmetic of that reading on the CPU with numpy only (no product code,
no oracle code): the identity itself, the quadratic convergence it inherits from Newton's
method, and why the compact per-pair form y0 (3 - r^2 y0^2) / 2 cannot be used in FP32."""
import numpy as np


def seeded_problem(n=200_000, seed=7):
    rng = np.random.default_rng(seed)
    r2 = rng.uniform(150.0, 9000.0, n)                  # grid units squared, as on config 3
    q = -rng.uniform(0.0, 1e-3, n)
    eps = rng.uniform(-1.2e-7, 1.2e-7, n) + 5.5e-9      # a MUFU-like seed: ~2^-23, small mean bias
    y0 = (1.0 + eps) / np.sqrt(r2)
    return r2, q, y0


def test_identity_and_quadratic_convergence_in_exact_arithmetic():
    r2, q, y0 = seeded_problem()
    v_true = np.sum(q / np.sqrt(r2))
    v_raw = np.sum(q * y0)
    a, c = q * y0, q * y0 ** 3
    v_sum = 0.5 * (3.0 * np.sum(a) - np.sum(c * r2))
    v_pair = np.sum(q * (y0 * (3.0 - r2 * y0 * y0) * 0.5))
    assert abs(v_sum - v_pair) <= 1e-15 * abs(v_true)              # the same value
    assert abs(v_raw - v_true) / abs(v_true) > 3e-9                # the raw seed is biased
    assert abs(v_sum - v_true) / abs(v_true) < 1e-13               # -1.5 eps^2


def test_fp32_sum_form_keeps_the_correction_the_compact_pair_form_rounds_it_away():
    r2, q, y0 = seeded_problem()
    v_true = np.sum(q / np.sqrt(r2))
    f = np.float32
    r2f, qf, y0f = r2.astype(f), q.astype(f), y0.astype(f)
    # inputs as the kernel sees them (FP32), exact reference for those inputs
    v_ref = np.sum(qf.astype(np.float64) / np.sqrt(r2f.astype(np.float64)))
    a = qf * y0f
    c = a * (y0f * y0f)
    t = (c.astype(np.float64) * r2f.astype(np.float64)).astype(f)   # fma(c, r2, T): the product is exact
    v_sum = 0.5 * (3.0 * np.sum(a.astype(np.float64)) - np.sum(t.astype(np.float64)))
    compact = (y0f * (f(3.0) - (r2f * y0f) * y0f)) * f(0.5)         # every step rounded to FP32
    v_compact = np.sum((qf * compact).astype(np.float64))
    err_sum = abs(v_sum - v_ref) / abs(v_ref)
    err_compact = abs(v_compact - v_ref) / abs(v_ref)
    assert err_sum < 1e-9, err_sum                                  # unbiased: per-pair roundings average out
    assert err_compact > 3 * err_sum                                # the bracket ~2 has an ulp of 2.4e-7
    assert abs(v_ref - v_true) / abs(v_true) < 1e-7                 # (input rounding is a separate matter)
