import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (B200); run with -m gpu")


@pytest.fixture(scope="session")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.fixture(scope="session")
def full_oracle(oracle_mod):
    """The oracle on EVERY evaluation point of a BASELINE configuration (V, E and the
    condition-number sums), computed once per session and shared by the parity files:
    config 3 is 1.7e10 pairs, config 4 3.4e10 (about 8 s / 17 s on the GPU box's 16 cores)."""
    from paper_1011_4687_b200.workloads import make_workload
    cache = {}

    def get(cfg):
        if cfg not in cache:
            w = make_workload(cfg)
            pts = w.elec_xyz.reshape(-1, 3)
            cache[cfg] = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
        return cache[cfg]
    return get
