"""Host-side checks of the seeded input generators (no method arithmetic here)."""
import numpy as np
import pytest

from paper_1011_4687_b200.workloads import CONFIG_SPECS, make_workload, subsample_points


def test_config0_shape_and_constraints():
    w = make_workload(0)
    assert (w.M, w.K, w.W, w.N) == (4096, 16, 1, 8)
    rs = np.linalg.norm(w.src_xyz, axis=1)
    assert rs.min() > 4.0 and rs.max() < 10.0
    rn = np.linalg.norm(w.nuc_xyz, axis=1)
    assert rn.min() > 4.0 and rn.max() < 10.0
    assert np.linalg.norm(w.elec_xyz.reshape(-1, 3), axis=1).max() < 3.0
    assert set(np.unique(w.nuc_Z)) <= {1.0, 6.0, 7.0, 8.0}
    assert np.all(w.src_q < 0)                      # q_j = -rho_j dV
    # dV = shell volume / M (SURVEY.md 8(c) reading 18)
    assert w.meta["dV"] == pytest.approx(4 * np.pi / 3 * (1000 - 64) / 4096)
    assert w.pairs_per_eval == 8 * (4096 + 16)


@pytest.mark.parametrize("idx,M_actual", [(1, 252_192), (3, 1_038_624)])
def test_grid_configs_masked_counts(idx, M_actual):
    """Masked-node counts of SURVEY.md 8(d) (nodes with r < r_mask dropped)."""
    w = make_workload(idx, n_points=(1, 4))
    spec = CONFIG_SPECS[idx]
    assert w.M == M_actual and w.M_nominal == int(np.prod(spec["grid"]))
    assert np.linalg.norm(w.src_xyz, axis=1).min() >= spec["r_mask"]
    # total electron count of the environment: one electron per Gaussian, minus
    # what falls in the masked sphere / outside the box
    assert 0.5 * w.K < -w.src_q.sum() <= w.K
    # C order, z fastest: first two kept nodes differ in z by h
    assert w.src_xyz[1, 2] - w.src_xyz[0, 2] == pytest.approx(spec["h"])


def test_determinism_and_point_override():
    a = make_workload(1, n_points=(1, 4))
    b = make_workload(1, n_points=(2, 8))
    assert np.array_equal(a.src_q, b.src_q) and np.array_equal(a.nuc_xyz, b.nuc_xyz)
    c = make_workload(1, n_points=(1, 4))
    assert np.array_equal(a.elec_xyz, c.elec_xyz)


def test_random_walk_confined():
    w = make_workload(2, n_points=(50, 1))
    p = w.elec_xyz.reshape(-1, 3)
    assert w.sequential and np.linalg.norm(p, axis=1).max() < 3.0
    steps = np.diff(p, axis=0)
    assert 0.1 < steps.std() < 0.3


def test_subsample_points():
    idx = subsample_points(16384, 0.01, seed=3)
    assert len(idx) == 164 and len(np.unique(idx)) == 164 and idx.max() < 16384
    assert np.array_equal(idx, subsample_points(16384, 0.01, seed=3))
