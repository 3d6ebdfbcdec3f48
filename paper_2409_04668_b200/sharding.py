"""Host-side sharding of a run over ranks: histories are independent, so every rank takes a
contiguous range of history ids (whole statistical batches) with the full problem and private tallies; the only
exchange is one sum-reduction of the raw tally accumulators and ledgers at the end.  Pure bookkeeping -- no
transport arithmetic here."""
from __future__ import annotations

import numpy as np


def shard_range(n_total: int, world: int, rank: int, n_batches: int | None = None):
    """(first_history_id, n_histories[, n_batches]) of `rank`.  With n_batches the split is by whole batches
    (batch size n_total / n_batches), earlier ranks taking the remainder."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad world/rank")
    if n_batches is None:
        base, rem = divmod(n_total, world)
        n = base + (1 if rank < rem else 0)
        first = rank * base + min(rank, rem)
        return first, n
    if n_total % n_batches:
        raise ValueError("n_batches must divide n_total")
    hb = n_total // n_batches
    base, rem = divmod(n_batches, world)
    nb = base + (1 if rank < rem else 0)
    first_b = rank * base + min(rank, rem)
    return first_b * hb, nb * hb, nb


def all_reduce_tallies(sum_, sumsq, ledger, group=None):
    """Sum-reduce raw accumulators over the process group (gloo on CPU tensors, nccl on CUDA tensors)."""
    import torch
    import torch.distributed as dist

    out = []
    for a in (sum_, sumsq, ledger):
        t = a if isinstance(a, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
        out.append(t if isinstance(a, torch.Tensor) else t.numpy())
    return tuple(out)


def all_reduce_state(problem, group=None, device=None):
    """The one exchange of a domain-replicated run: export the handle's accumulators as one
    fp64 vector, sum it over the ranks (NCCL when `device` is a CUDA device, gloo on the host otherwise) and import
    the sum back, so that every rank's tallies_get / counters_get answer for the whole job.  `problem` is anything with
    state_size / state_export / state_import (paper_2409_04668_b200.Problem)."""
    import torch
    import torch.distributed as dist

    n = problem.state_size()
    buf = torch.empty(n, dtype=torch.float64, device=device if device is not None else "cpu")
    problem.state_export(buf)
    # whenever a process group exists, one-rank groups included: a one-rank sum is the identity, and it is the one way to
    # put ncclAllReduce on the exported device buffer where a second GPU does not exist (tests/test_gpu_vr.py)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=group)
    problem.state_import(buf)
    return buf
