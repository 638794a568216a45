"""One rank of tests/test_sharding_gpu.py (launched with torch.distributed.run, gloo backend;
the ranks share GPU 0 and never wait on one another's kernels).  Each rank owns a handle of the
CUDA library and runs the sharding helpers over it; rank r writes its results to out_dir."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1011_4687_b200 import binding as B  # noqa: E402
from paper_1011_4687_b200.sharding import eval_sharded, eval_source_sharded, source_shard  # noqa: E402
from paper_1011_4687_b200.workloads import make_workload  # noqa: E402


def main(out_dir, W, N):
    rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
    torch.cuda.set_device(0)
    dist.init_process_group("gloo")
    try:
        w = make_workload(1, n_points=(W, N))
        elec = torch.from_numpy(w.elec_xyz).cuda()
        # (1) walkers sharded, sources replicated, gather of V and E
        with B.FieldEvaluator(w.src_xyz, w.src_q, w.nuc_xyz, w.nuc_Z, W * N) as ev:
            for prec in ("fp64", "fp32"):
                V, E = eval_sharded(lambda pts: ev.eval(pts, prec), elec, rank, world)
                np.save(os.path.join(out_dir, f"walk_{prec}_V{rank}.npy"), V.cpu().numpy())
                np.save(os.path.join(out_dir, f"walk_{prec}_E{rank}.npy"), E.cpu().numpy())
        # (2) sources sharded (Eq. 5 across ranks): rank 0 also owns the nuclei
        lo, cnt = source_shard(w.M, rank, world)
        nx = w.nuc_xyz if rank == 0 else None
        nz = w.nuc_Z if rank == 0 else None
        with B.FieldEvaluator(np.ascontiguousarray(w.src_xyz[lo:lo + cnt]),
                              np.ascontiguousarray(w.src_q[lo:lo + cnt]), nx, nz, W * N) as ev:
            pts = elec.reshape(-1, 3).contiguous()
            for prec in ("fp64", "fp32"):
                V, E = eval_source_sharded(lambda p: ev.eval(p, prec), pts, rank, world)
                np.save(os.path.join(out_dir, f"src_{prec}_V{rank}.npy"), V.cpu().numpy())
                np.save(os.path.join(out_dir, f"src_{prec}_E{rank}.npy"), E.cpu().numpy())
        torch.cuda.synchronize()
    finally:
        dist.destroy_process_group()


if __name__ == "__main__":
    main(sys.argv[1], int(sys.argv[2]), int(sys.argv[3]))
