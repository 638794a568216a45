"""The tolerance rule of the GPU parity tests, shared by the test files."""
import numpy as np


def check(ref, V, E, tol):
    """plain relative tolerance on V and on the vector norm of E.  Only a point
    whose sum is ill-conditioned beyond kappa = 1e3 (kappa_V = sum|q|/r / |V|, kappa_E =
    sum|q|/r^2 / |E|) is instead held to err / kappa <= a few rounding units of the arithmetic:
    1e-15 (9 x 2^-53) in FP64, 1.2e-7 (2 x 2^-24) in FP32 -- a relative tolerance on a sum that
    cancels to a thousandth of its terms is not meaningful, and no arithmetic can sum terms
    that a few of them dominate to better than its own rounding unit times sum|term|.
    No tolerance is scaled by kappa below 1e3."""
    esc = 1e-15 if tol < 1e-9 else 1.2e-7
    with np.errstate(divide="ignore", invalid="ignore"):
        errV = np.abs(V - ref.V) / np.abs(ref.V)
        kV = ref.absV / np.abs(ref.V)
        okV = (errV <= tol) | ((kV > 1e3) & (np.abs(V - ref.V) <= esc * ref.absV))
    bad = np.flatnonzero(~okV)
    assert bad.size == 0, (f"V: {bad.size} point(s) over {tol:g}; worst rel err {np.nanmax(errV[bad]):.3e} "
                           f"at kappa_V {kV[bad][np.nanargmax(errV[bad])]:.1f} (kappa escape only above 1e3, "
                           f"err/kappa <= {esc:g})")
    if E is not None:
        nE = np.linalg.norm(ref.E, axis=1)
        dE = np.linalg.norm(E - ref.E, axis=1)
        with np.errstate(divide="ignore", invalid="ignore"):
            errE = dE / nE
            kE = ref.absE / nE
            okE = (errE <= tol) | ((kE > 1e3) & (dE <= esc * ref.absE))
        bad = np.flatnonzero(~okE)
        assert bad.size == 0, (f"E: {bad.size} point(s) over {tol:g}; worst rel err {np.nanmax(errE[bad]):.3e} "
                               f"at kappa_E {kE[bad][np.nanargmax(errE[bad])]:.1f} (kappa escape only above 1e3, "
                               f"err/kappa <= {esc:g})")
    return float(np.nanmax(errV))
