"""The tolerance rule of the GPU parity tests, shared by the test files."""
import numpy as np


def check(ref, V, E, tol):
    """plain relative tolerance on V and on the vector norm of E.  Only a point
    whose sum is ill-conditioned beyond kappa = 1e3 (kappa_V = sum|q|/r / |V|, kappa_E =
    sum|q|/r^2 / |E|) is instead held to err / kappa <= tol * 1e-3 (1e-15 in FP64, 1e-8 in
    FP32: a relative tolerance on a sum that cancels to a thousandth of its terms is not
    meaningful).  No tolerance is scaled by kappa below 1e3."""
    with np.errstate(divide="ignore", invalid="ignore"):
        errV = np.abs(V - ref.V) / np.abs(ref.V)
        kV = ref.absV / np.abs(ref.V)
        okV = (errV <= tol) | ((kV > 1e3) & (np.abs(V - ref.V) <= tol * 1e-3 * ref.absV))
    bad = np.flatnonzero(~okV)
    assert bad.size == 0, (f"V: {bad.size} point(s) over {tol:g}; worst rel err {np.nanmax(errV[bad]):.3e} "
                           f"at kappa_V {kV[bad][np.nanargmax(errV[bad])]:.1f} (kappa escape only above 1e3, "
                           f"err/kappa <= {tol * 1e-3:g})")
    if E is not None:
        nE = np.linalg.norm(ref.E, axis=1)
        dE = np.linalg.norm(E - ref.E, axis=1)
        with np.errstate(divide="ignore", invalid="ignore"):
            errE = dE / nE
            kE = ref.absE / nE
            okE = (errE <= tol) | ((kE > 1e3) & (dE <= tol * 1e-3 * ref.absE))
        bad = np.flatnonzero(~okE)
        assert bad.size == 0, (f"E: {bad.size} point(s) over {tol:g}; worst rel err {np.nanmax(errE[bad]):.3e} "
                               f"at kappa_E {kE[bad][np.nanargmax(errE[bad])]:.1f} (kappa escape only above 1e3, "
                               f"err/kappa <= {tol * 1e-3:g})")
    return float(np.nanmax(errV))
