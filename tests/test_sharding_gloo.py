"""Multi-rank host logic on CPU (gloo, world_size 2): walkers are sharded, sources are
replicated, and the gathered result equals the single-rank result (
PAPER.md:203-205).  The per-rank evaluation is the oracle here (test infrastructure): this
test covers the sharding / gather plumbing, not the kernels."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_1011_4687_b200.sharding import eval_sharded, eval_source_sharded, source_shard, walker_shard
from paper_1011_4687_b200.workloads import make_workload


def test_walker_shard_covers_disjoint_balanced():
    for W in (0, 1, 5, 16, 256, 257):
        for world in (1, 2, 3, 8):
            blocks = [walker_shard(W, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and sum(c for _, c in blocks) == W
            for (s0, c0), (s1, _) in zip(blocks, blocks[1:]):
                assert s0 + c0 == s1
            counts = [c for _, c in blocks]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        walker_shard(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank_main(rank, world, port, W, N, out_dir):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = make_workload(0, n_points=(W, N))

        def evaluate(pts):
            r = oracle.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts.numpy().reshape(-1, 3))
            return (torch.from_numpy(r.V).reshape(pts.shape[0], N),
                    torch.from_numpy(r.E).reshape(pts.shape[0], N, 3))

        V, E = eval_sharded(evaluate, torch.from_numpy(w.elec_xyz), rank, world)
        np.save(os.path.join(out_dir, f"V{rank}.npy"), V.numpy())
        np.save(os.path.join(out_dir, f"E{rank}.npy"), E.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("W,N", [(5, 3), (2, 4), (1, 2)])
def test_gloo_world2_gather_equals_single_rank(tmp_path, oracle_mod, W, N):
    world = 2
    mp.spawn(_rank_main, args=(world, _free_port(), W, N, str(tmp_path)), nprocs=world, join=True)
    w = make_workload(0, n_points=(W, N))
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, w.elec_xyz.reshape(-1, 3))
    for r in range(world):
        V = np.load(tmp_path / f"V{r}.npy")
        E = np.load(tmp_path / f"E{r}.npy")
        assert V.shape == (W, N) and E.shape == (W, N, 3)
        assert np.array_equal(V.reshape(-1), ref.V)          # same oracle, same points: bitwise
        assert np.array_equal(E.reshape(-1, 3), ref.E)


def _rank_main_sources(rank, world, port, P, out_dir):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = make_workload(0, n_points=(1, P))
        lo, cnt = source_shard(w.M, rank, world)
        nuc_xyz = w.nuc_xyz if rank == 0 else w.nuc_xyz[:0]       # the nuclei live on rank 0
        nuc_Z = w.nuc_Z if rank == 0 else w.nuc_Z[:0]

        def evaluate_local(pts):
            r = oracle.field(w.src_xyz[lo:lo + cnt], w.src_q[lo:lo + cnt], nuc_xyz, nuc_Z, pts.numpy())
            return torch.from_numpy(r.V), torch.from_numpy(r.E)

        V, E = eval_source_sharded(evaluate_local, torch.from_numpy(w.elec_xyz.reshape(-1, 3)), rank, world)
        np.save(os.path.join(out_dir, f"sV{rank}.npy"), V.numpy())
        np.save(os.path.join(out_dir, f"sE{rank}.npy"), E.numpy())
    finally:
        dist.destroy_process_group()


def test_gloo_world2_source_sharding_fixed_order_sum(tmp_path, oracle_mod):
    """Eq. 5-6 across ranks: each rank sums its own cells, the partials are
    added in rank order.  Every rank gets bitwise the same result; it equals the single-rank
    oracle to a few ulp x kappa (only the association of the sum differs)."""
    world, P = 2, 6
    mp.spawn(_rank_main_sources, args=(world, _free_port(), P, str(tmp_path)), nprocs=world, join=True)
    w = make_workload(0, n_points=(1, P))
    pts = w.elec_xyz.reshape(-1, 3)
    ref = oracle_mod.field(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, pts, want_abs=True)
    V0, E0 = np.load(tmp_path / "sV0.npy"), np.load(tmp_path / "sE0.npy")
    V1, E1 = np.load(tmp_path / "sV1.npy"), np.load(tmp_path / "sE1.npy")
    assert np.array_equal(V0, V1) and np.array_equal(E0, E1)          # identical on all ranks
    assert np.all(np.abs(V0 - ref.V) <= 8 * np.finfo(float).eps * ref.absV)
    assert np.all(np.linalg.norm(E0 - ref.E, axis=1) <= 8 * np.finfo(float).eps * ref.absE)
    # the partition itself: contiguous, disjoint, complete
    blocks = [source_shard(w.M, r, world) for r in range(world)]
    assert blocks[0][0] == 0 and blocks[0][1] + blocks[1][1] == w.M and blocks[1][0] == blocks[0][1]
