"""Seeded synthetic workloads with the shape of the paper's benchmark system.

The paper measures on one private data set (glycine trimer, fragment fr1:
M = 268,782 density cells, 19 MM atoms) that is not
available.  The five configurations of BASELINE.json ``configs`` (restated in
SURVEY.md section 8(d)) stand in for it: a QM region at the origin surrounded by a
discretised environment electron density of H/C/N/O nuclei.

This module only *generates inputs* (positions, charges, evaluation points).  It
contains none of the method's arithmetic (no 1/r sums) and is shared by the
oracle-side tests, the CUDA-side tests and ``bench.py``: both sides consume the
same FP64 arrays.

Recipe (readings 15-19 of SURVEY.md 8(c)):

* RNG: ``numpy.random.default_rng(seed)`` (PCG64), seed = config index.
  Draw order: nuclei positions -> Z -> alpha -> (config 0 only) source positions
  -> evaluation points.
* Density: rho(r) = sum_k w_k (alpha_k/pi)^{3/2} exp(-alpha_k |r - C_k|^2), one
  normalised s-Gaussian per nucleus centred on it, alpha_k ~ U[0.5, 2] bohr^-2,
  w_k = 1 (``neutral=True``: w_k = Z_k).
* Cell charge q_j = -rho(R_j) * dV (electrons are negative); nuclei carry +Z.
* Grid configs: nodes (i - (n-1)/2) h per axis, nodes with r < r_mask dropped
  (compacted list, C order, z fastest).
* Electrons: N(0, sigma^2) per axis, redrawn until r < r_clip (rejection).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional, Tuple

import numpy as np

__all__ = ["Workload", "make_workload", "CONFIG_SPECS", "subsample_points", "draw_points"]


@dataclass
class Workload:
    """One seeded problem instance (all arrays FP64, C-contiguous)."""

    index: int
    name: str
    src_xyz: np.ndarray          # [M][3] bohr
    src_q: np.ndarray            # [M] cell charges (q_j = -rho_j dV)
    nuc_xyz: np.ndarray          # [K][3]
    nuc_Z: np.ndarray            # [K] nuclear charges (+Z)
    elec_xyz: np.ndarray         # [W][N][3] evaluation points
    precisions: Tuple[str, ...]  # which paths BASELINE.json times on it
    M_nominal: int               # grid nodes before masking
    sequential: bool = False     # config 2: W = evaluations in sequence, N = 1
    meta: dict = field(default_factory=dict)

    @property
    def M(self) -> int:
        return int(self.src_q.shape[0])

    @property
    def K(self) -> int:
        return int(self.nuc_Z.shape[0])

    @property
    def W(self) -> int:
        return int(self.elec_xyz.shape[0])

    @property
    def N(self) -> int:
        return int(self.elec_xyz.shape[1])

    @property
    def P(self) -> int:
        return self.W * self.N

    @property
    def pairs_per_eval(self) -> int:
        """Pair interactions of one field evaluation (sequential: one point)."""
        pts = self.N if self.sequential else self.P
        return pts * (self.M + self.K)


# index -> specification
CONFIG_SPECS = {
    0: dict(name="tiny-fp64", kind="shell", M=4096, K=16, W=1, N=8,
            shell=(4.0, 10.0), sigma=1.0, r_clip=3.0, precisions=("fp64",)),
    1: dict(name="single-configuration", kind="grid", grid=(64, 64, 64), h=0.3,
            r_mask=4.0, K=256, W=1, N=32, sigma=1.0, r_clip=3.0,
            precisions=("fp64", "fp32")),
    2: dict(name="single-electron-move", kind="grid", grid=(128, 128, 128), h=0.25,
            r_mask=4.0, K=1024, W=1000, N=1, walk_sigma=0.2, r_clip=3.0,
            precisions=("fp32", "fp64"), sequential=True),
    3: dict(name="batched-walkers", kind="grid", grid=(128, 128, 64), h=0.3,
            r_mask=4.0, K=512, W=256, N=64, sigma=1.5, r_clip=3.0,
            precisions=("fp32",)),
    4: dict(name="large-environment", kind="grid", grid=(256, 256, 256), h=0.2,
            r_mask=5.0, K=4096, W=16, N=128, sigma=1.5, r_clip=4.0,
            precisions=("fp64",)),
}


def _shell_points(rng: np.random.Generator, n: int, a: float, b: float) -> np.ndarray:
    """n points uniform in VOLUME in the shell a < r < b (reading 18)."""
    v = rng.standard_normal((n, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    u = rng.random(n)
    r = np.cbrt(u * (b ** 3 - a ** 3) + a ** 3)
    return v * r[:, None]


def _box_minus_sphere(rng: np.random.Generator, n: int, half: np.ndarray,
                      r_mask: float) -> np.ndarray:
    """n points uniform in the box [-half, half] outside the sphere r < r_mask."""
    out = np.empty((n, 3))
    filled = 0
    while filled < n:
        c = (rng.random((n - filled, 3)) * 2.0 - 1.0) * half
        c = c[np.linalg.norm(c, axis=1) >= r_mask]
        out[filled:filled + len(c)] = c
        filled += len(c)
    return out


def _clipped_gaussian(rng: np.random.Generator, n: int, sigma: float,
                      r_clip: float) -> np.ndarray:
    """n points N(0, sigma^2) per axis, each redrawn until r < r_clip (reading 17)."""
    out = np.empty((n, 3))
    filled = 0
    while filled < n:
        c = rng.standard_normal((n - filled, 3)) * sigma
        c = c[np.linalg.norm(c, axis=1) < r_clip]
        out[filled:filled + len(c)] = c
        filled += len(c)
    return out


def _random_walk(rng: np.random.Generator, n: int, step_sigma: float,
                 r_clip: float) -> np.ndarray:
    """Gaussian random walk from the origin; a step is redrawn until r < r_clip."""
    out = np.empty((n, 3))
    pos = np.zeros(3)
    for i in range(n):
        while True:
            trial = pos + rng.standard_normal(3) * step_sigma
            if np.linalg.norm(trial) < r_clip:
                break
        pos = trial
        out[i] = pos
    return out


def _density_at_points(pts: np.ndarray, centres: np.ndarray, alpha: np.ndarray,
                       w: np.ndarray, chunk: int = 4096) -> np.ndarray:
    """rho at arbitrary points (config 0 and spot checks); plain evaluation."""
    rho = np.zeros(len(pts))
    norm = w * (alpha / np.pi) ** 1.5
    for s in range(0, len(pts), chunk):
        d2 = ((pts[s:s + chunk, None, :] - centres[None, :, :]) ** 2).sum(-1)
        rho[s:s + chunk] = (np.exp(-alpha[None, :] * d2) * norm[None, :]).sum(1)
    return rho


def _density_on_grid(axes, centres, alpha, w) -> np.ndarray:
    """rho on a tensor grid.  Each s-Gaussian is separable, exp(-a|r-C|^2) =
    ex(x) ey(y) ez(z), so rho[:, :, iz] = EX^T diag(norm * EZ[:, iz]) EY; per z slab
    only Gaussians with exp(-alpha dz^2) >= 1e-20 are kept (dropped terms are
    below 1e-20 of a Gaussian's peak)."""
    x, y, z = axes
    norm = w * (alpha / np.pi) ** 1.5
    ex = np.exp(-alpha[:, None] * (x[None, :] - centres[:, 0:1]) ** 2)
    ey = np.exp(-alpha[:, None] * (y[None, :] - centres[:, 1:2]) ** 2)
    ez = np.exp(-alpha[:, None] * (z[None, :] - centres[:, 2:3]) ** 2) * norm[:, None]
    rho = np.empty((len(x), len(y), len(z)))
    for iz in range(len(z)):
        sel = ez[:, iz] >= 1e-20 * norm
        rho[:, :, iz] = (ex[sel] * ez[sel, iz][:, None]).T @ ey[sel]
    return rho


def make_workload(index: int, seed: Optional[int] = None, neutral: bool = False,
                  n_points: Optional[Tuple[int, int]] = None) -> Workload:
    """Build configuration ``index`` (0-4).  ``n_points=(W, N)`` overrides the
    evaluation-point count (used by tests to shrink a case); everything drawn
    before the evaluation points is unaffected by it."""
    spec = CONFIG_SPECS[index]
    seed = index if seed is None else seed
    rng = np.random.default_rng(seed)
    K = spec["K"]
    W, N = n_points if n_points is not None else (spec["W"], spec["N"])

    if spec["kind"] == "shell":
        a, b = spec["shell"]
        nuc_xyz = _shell_points(rng, K, a, b)
    else:
        nx, ny, nz = spec["grid"]
        h = spec["h"]
        axes = [(np.arange(n) - (n - 1) / 2.0) * h for n in (nx, ny, nz)]
        half = np.array([ax[-1] for ax in axes])
        nuc_xyz = _box_minus_sphere(rng, K, half, spec["r_mask"])
    nuc_Z = rng.choice(np.array([1.0, 6.0, 7.0, 8.0]), size=K)
    alpha = rng.uniform(0.5, 2.0, size=K)
    w = nuc_Z.copy() if neutral else np.ones(K)

    if spec["kind"] == "shell":
        M_nominal = spec["M"]
        src_xyz = _shell_points(rng, M_nominal, a, b)
        dV = (4.0 * np.pi / 3.0) * (b ** 3 - a ** 3) / M_nominal
        rho = _density_at_points(src_xyz, nuc_xyz, alpha, w)
    else:
        M_nominal = nx * ny * nz
        dV = h ** 3
        rho3 = _density_on_grid(axes, nuc_xyz, alpha, w)
        X, Y, Z = np.meshgrid(*axes, indexing="ij")
        keep = (X * X + Y * Y + Z * Z) >= spec["r_mask"] ** 2   # reading 16: dropped
        src_xyz = np.stack([X[keep], Y[keep], Z[keep]], axis=1)
        rho = rho3[keep]
        del rho3, X, Y, Z, keep
    src_q = -rho * dV

    if spec.get("sequential"):
        elec = _random_walk(rng, W * N, spec["walk_sigma"], spec["r_clip"])
    else:
        elec = _clipped_gaussian(rng, W * N, spec["sigma"], spec["r_clip"])
    elec_xyz = np.ascontiguousarray(elec.reshape(W, N, 3))

    return Workload(
        index=index, name=spec["name"],
        src_xyz=np.ascontiguousarray(src_xyz), src_q=np.ascontiguousarray(src_q),
        nuc_xyz=np.ascontiguousarray(nuc_xyz), nuc_Z=np.ascontiguousarray(nuc_Z),
        elec_xyz=elec_xyz, precisions=spec["precisions"], M_nominal=M_nominal,
        sequential=bool(spec.get("sequential", False)),
        meta=dict(seed=seed, dV=dV, alpha=alpha, neutral=neutral,
                  h=spec.get("h"), grid=spec.get("grid"), r_mask=spec.get("r_mask")),
    )


def subsample_points(P: int, fraction: float, seed: int) -> np.ndarray:
    """Seeded, sorted subsample of point indices (config 3 parity: 1 %)."""
    rng = np.random.default_rng(seed)
    n = max(1, int(round(P * fraction)))
    return np.sort(rng.choice(P, size=n, replace=False))


def draw_points(index: int, W: int, N: int, seed: int) -> np.ndarray:
    """Another seeded batch of evaluation points [W][N][3] with configuration ``index``'s
    distribution (bench.py: a different batch per step / per rank; the environment is not
    redrawn)."""
    spec = CONFIG_SPECS[index]
    rng = np.random.default_rng([seed, index, 0x9E3779B9])
    if spec.get("sequential"):
        pts = _random_walk(rng, W * N, spec["walk_sigma"], spec["r_clip"])
    else:
        pts = _clipped_gaussian(rng, W * N, spec["sigma"], spec["r_clip"])
    return np.ascontiguousarray(pts.reshape(W, N, 3))
