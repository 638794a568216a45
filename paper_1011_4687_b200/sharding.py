"""Sharding across GPUs.

By walkers (the paper's own scaling, Table V: independent walkers on MPI
ranks, one GPU each, no communication in the data path): every rank holds a replica of the
environment (<= 802 MB for the largest configuration) and evaluates a contiguous block of
walkers.  There is NO collective in the hot path; the only communication is the optional
gather of the results (4 doubles per point).

By sources (Eq. 5-6 across devices: U = B[1] + ... + B[N_B] with one block
per GPU), for environments that do not fit one GPU: every rank holds a contiguous range of the
cells (the nuclei go to rank 0), evaluates ALL points against it, and the per-rank partial
{V, E} are exchanged once (4 doubles per point) and added in RANK ORDER on every rank, so the
result is deterministic and identical on all ranks (a tree all-reduce would not fix the order).

Communication is ``torch.distributed`` (NCCL on GPUs, gloo in the CPU tests).  This module
holds none of the method's arithmetic beyond that fixed-order sum of partials: the evaluation
itself is the callable passed in (on a GPU: ``FieldEvaluator.eval``).
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import torch


def walker_shard(W: int, rank: int, world: int) -> Tuple[int, int]:
    """(first walker, number of walkers) of ``rank``: contiguous, balanced to within one,
    the first ``W % world`` ranks take the extra walker."""
    if world < 1 or not (0 <= rank < world) or W < 0:
        raise ValueError("walker_shard: need 0 <= rank < world and W >= 0")
    base, extra = divmod(W, world)
    count = base + (1 if rank < extra else 0)
    start = rank * base + min(rank, extra)
    return start, count


def eval_sharded(evaluate: Callable, elec_xyz: torch.Tensor, rank: int, world: int,
                 gather: bool = True, group=None):
    """Evaluate ``elec_xyz`` [W, N, 3] with the walkers split over ``world`` ranks.

    ``evaluate(pts [w, N, 3]) -> (V [w, N], E [w, N, 3])`` runs on this rank's walkers only.
    With ``gather`` every rank receives the full V [W, N] and E [W, N, 3] (rank order = walker
    order, so the result is identical to a single-rank evaluation); without it the local
    block and its walker range are returned.
    """
    W, N = int(elec_xyz.shape[0]), int(elec_xyz.shape[1])
    start, count = walker_shard(W, rank, world)
    if count > 0:
        V_loc, E_loc = evaluate(elec_xyz[start:start + count].contiguous())
    else:
        V_loc = elec_xyz.new_zeros((0, N))
        E_loc = elec_xyz.new_zeros((0, N, 3))
    if not gather or world == 1:
        return (V_loc, E_loc) if world == 1 else (V_loc, E_loc, (start, count))

    import torch.distributed as dist
    # uneven blocks: pad every block to the largest one, gather, then drop the padding
    cmax = -(-W // world)
    buf = elec_xyz.new_zeros((cmax, N, 4))
    buf[:count, :, 0] = V_loc
    buf[:count, :, 1:] = E_loc
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf, group=group)
    parts = [out[r][:walker_shard(W, r, world)[1]] for r in range(world)]
    full = torch.cat(parts, dim=0)
    return full[..., 0].contiguous(), full[..., 1:].contiguous()


def source_shard(M: int, rank: int, world: int) -> Tuple[int, int]:
    """(first cell, number of cells) of ``rank``: contiguous, balanced to within one."""
    return walker_shard(M, rank, world)


def eval_source_sharded(evaluate_local: Callable, elec_xyz: torch.Tensor, rank: int, world: int,
                        group=None):
    """V, E at ``elec_xyz`` [P, 3] from an environment whose cells are split over the ranks.

    ``evaluate_local(pts [P, 3]) -> (V [P], E [P, 3])`` is this rank's partial: the sum over
    ITS cells (rank 0 also owns the nuclei).  Every rank returns the full sums, bitwise the
    same on all ranks: the partials are gathered and added in rank order 0, 1, 2, ...
    """
    V_loc, E_loc = evaluate_local(elec_xyz)
    if world == 1:
        return V_loc, E_loc
    import torch.distributed as dist
    P = int(elec_xyz.shape[0])
    buf = elec_xyz.new_empty((P, 4))
    buf[:, 0] = V_loc
    buf[:, 1:] = E_loc
    out = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(out, buf, group=group)
    if buf.is_cuda:
        # the fixed-order sum is a call of the library (qmmm_sum_rank_partials), not arithmetic here
        from . import binding as B
        parts = torch.stack(out, dim=0).contiguous()
        total = torch.empty_like(buf)
        B.qmmm_sum_rank_partials(parts, total)
    else:
        # CPU tensors (the gloo plumbing test, whose per-rank evaluator is the oracle): same order
        total = out[0].clone()
        for r in range(1, world):          # fixed order: deterministic, identical everywhere
            total += out[r]
    return total[:, 0].contiguous(), total[:, 1:].contiguous()
