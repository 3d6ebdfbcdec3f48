"""Host logic of the multi-rank path: history-range sharding and the tally reduction,
exercised with world_size 2 on the gloo backend; the per-rank runs are the oracle's (CPU)."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def merge_statistics(sum_, sumsq, n_hist, n_batches):
    """mean / sdev from reduced accumulators, written out here for the check: the product computes them
    inside mcdc_tallies_get after mcdc_state_import."""
    hb = n_hist / n_batches
    mean = sum_ / n_hist
    if n_batches > 1:
        var = (sumsq / (hb * hb) / n_batches - mean * mean) / (n_batches - 1)
        sdev = np.sqrt(np.maximum(var, 0.0))
    else:
        sdev = np.zeros_like(mean)
    return mean, sdev


def test_shard_range_partitions_exactly():
    from paper_2409_04668_b200.sharding import shard_range
    for n, w in ((10, 3), (7, 7), (1000003, 8), (5, 8)):
        got = [shard_range(n, w, r) for r in range(w)]
        assert got[0][0] == 0 and sum(c for _, c in got) == n
        for (f0, c0), (f1, _) in zip(got, got[1:]):
            assert f1 == f0 + c0
    parts = [shard_range(1000, 3, r, n_batches=10) for r in range(3)]
    assert [p[2] for p in parts] == [4, 3, 3] and [p[0] for p in parts] == [0, 400, 700]
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import Oracle
    from paper_2409_04668_b200.sharding import all_reduce_tallies, shard_range
    from workloads import configs as W

    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N, B = 4000, 8
    p = W.config1_slab(n_histories=N, n_batches=B)
    first, n, nb = shard_range(N, world, rank, n_batches=B)
    o = Oracle(p)
    o.run(n, p.seed, n_batches=nb, first_history_id=first)
    s, q2 = o.tally_sums()
    c = o.counters()
    ledger = np.array([c[k] for k in ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost")])
    s, q2, ledger = all_reduce_tallies(s.copy(), q2.copy(), ledger)
    mean, sdev = merge_statistics(s, q2, N, B)
    if rank == 0:
        q.put((mean, sdev, ledger))
    dist.destroy_process_group()


def test_two_rank_run_equals_the_single_rank_run():
    from oracle import Oracle
    from workloads import configs as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    mean, sdev, ledger = q.get(timeout=120)
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    N, B = 4000, 8
    p = W.config1_slab(n_histories=N, n_batches=B)
    o = Oracle(p); o.run(N, p.seed, n_batches=B)
    m1, s1 = o.tallies()
    assert np.allclose(mean, m1, rtol=1e-13, atol=0) and np.allclose(sdev, s1, rtol=1e-9, atol=1e-18)
    c = o.counters()
    assert ledger[0] == c["source"] and ledger[2] == c["capture"] and ledger[5] == c["census_final"]
    assert ledger[0] + ledger[1] == ledger[2:].sum()


class _OracleState:
    """Stands in for paper_2409_04668_b200.Problem on a box without a GPU: the same state vector layout
    (include/mcdc.h mcdc_state_*), filled from an oracle run."""

    def __init__(self, p, first, n, nb):
        from oracle import Oracle
        self.p = p
        self.o = Oracle(p)
        self.o.run(n, p.seed, n_batches=nb, first_history_id=first)
        self.vec = None

    def state_size(self):
        return 2 * self.p.n_bins + 2 * self.p.n_census + 20

    def state_export(self, t):
        s, q = self.o.tally_sums(); w, n = self.o.census(); c = self.o.counters()
        led = [c[k] for k in ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "vr_gain", "vr_loss")]
        cnt = [c[k] for k in ("histories", "segments", "collisions", "surf_hits", "census_events", "children", "lost_n", "pc_removed", "pc_added")]
        v = np.concatenate([s.ravel(), q.ravel(), w, n.astype(np.float64), led, np.array(cnt, dtype=np.float64),
                            [c["histories"], c["batches"]]])
        t.copy_(__import__("torch").from_numpy(v))

    def state_import(self, t):
        self.vec = t.numpy().copy()


def _worker_state(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_2409_04668_b200.sharding import all_reduce_state, shard_range
    from workloads import configs as W

    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    N, B = 3000, 6
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    first, n, nb = shard_range(N, world, rank, n_batches=B)
    h = _OracleState(p, first, n, nb)
    all_reduce_state(h)                                   # host buffer -> gloo
    q.put((rank, h.vec))
    dist.destroy_process_group()


def test_all_reduce_state_gives_every_rank_the_whole_job():
    from oracle import Oracle
    from workloads import configs as W
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker_state, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    got = dict(q.get(timeout=180) for _ in range(2))
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    assert np.array_equal(got[0], got[1])                 # every rank holds the same reduced state
    N, B = 3000, 6
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    o = Oracle(p); o.run(N, p.seed, n_batches=B)
    v = got[0]; nb_ = p.n_bins; K = p.n_census
    mean, sdev = merge_statistics(v[:nb_], v[nb_:2 * nb_], v[-2], v[-1])
    m1, s1 = o.tallies()
    assert v[-2] == N and v[-1] == B
    assert np.allclose(mean, m1.ravel(), rtol=1e-13, atol=0) and np.allclose(sdev, s1.ravel(), rtol=1e-9, atol=1e-18)
    w, n = o.census(); c = o.counters()
    assert np.array_equal(v[2 * nb_ + K:2 * nb_ + 2 * K], n.astype(np.float64))
    assert v[2 * nb_ + 2 * K] == c["source"] and v[2 * nb_ + 2 * K + 9 + 1] == c["segments"]
