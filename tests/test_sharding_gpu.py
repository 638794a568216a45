"""The multi-GPU sharding code over the CUDA path (PAPER.md:203-205,
Table V): two ranks over gloo, each with its own handle of the CUDA library, sharing the one
GPU of this box.  They never wait on one another's kernels (walker sharding has no data-path
collective; source sharding gathers partials once).  Results against the single-rank oracle.
Throughput of two ranks serialised on one device says nothing and is not asserted."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_1011_4687_b200.workloads import make_workload
from parity_check import check

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOL = {"fp64": 1e-12, "fp32": 1e-5}


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _torchrun(nproc, script_and_args, env=None, timeout=900):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port())] + script_and_args
    return subprocess.run(cmd, capture_output=True, text=True, timeout=timeout, cwd=ROOT,
                          env=dict(os.environ, **(env or {})))


def test_two_ranks_walker_and_source_sharding_over_the_cuda_path(tmp_path, oracle_mod):
    W, N = 5, 13                                     # uneven walker split: 3 + 2
    out = _torchrun(2, [os.path.join(ROOT, "tests", "shard_worker.py"), str(tmp_path), str(W), str(N)])
    assert out.returncode == 0, out.stderr[-4000:]
    w = make_workload(1, n_points=(W, N))
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz.reshape(-1, 3), want_abs=True)
    for prec in ("fp64", "fp32"):
        got = {}
        for kind in ("walk", "src"):
            for r in range(2):
                V = np.load(tmp_path / f"{kind}_{prec}_V{r}.npy")
                E = np.load(tmp_path / f"{kind}_{prec}_E{r}.npy")
                check(ref, V.reshape(-1), E.reshape(-1, 3), TOL[prec])
                got[(kind, r)] = (V, E)
            # the gathered / summed result is bitwise the same on both ranks
            assert np.array_equal(got[(kind, 0)][0], got[(kind, 1)][0])
            assert np.array_equal(got[(kind, 0)][1], got[(kind, 1)][1])
        assert got[("walk", 0)][0].shape == (W, N) and got[("walk", 0)][1].shape == (W, N, 3)


def test_bench_two_ranks_prints_the_contract_line():
    out = _torchrun(2, [os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2", "--warmup", "3",
                        "--no-sweep", "--config", "1"],
                    env={"QMMM_BENCH_BACKEND": "gloo"})
    assert out.returncode == 0, out.stderr[-4000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.strip().startswith("{")]
    assert len(lines) == 1, out.stdout
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["steps"] == 2 and d["warmup"] == 3
    assert d["metric"] == "pair-interactions/s" and d["unit"] == "Gpair/s" and d["scaling"] == "weak"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["gpu_launches"] > 0
    assert d["e2e"]["value"] > 0 and d["e2e"]["h2d_bytes_per_step"] > 0
    assert "roofline" in d and "clocks" in d and d["config"]["workload"].startswith("configs[1]")
    assert "cpu_baseline" not in d                   # rank 0 at N = 1 only
