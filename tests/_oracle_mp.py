"""The oracle run as independent processes over disjoint history-id ranges (whole statistical batches) with the raw
accumulators added afterwards.  Pin E5 (tests/test_oracle_transport.py: schedule independence, split ranges) says the
sums are those of the single run; histories are independent.  Test infrastructure: calls only oracle/."""
from __future__ import annotations

import multiprocessing as mp
import os

import numpy as np

COUNTER_KEYS = ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "histories", "segments",
                "collisions", "surf_hits", "census_events", "children", "lost_n", "batches")


def _part(args):
    name, kw, seed, first, n, nb, collision = args
    from oracle import Oracle
    from workloads import configs as W
    p = W.get_config(name, **kw)
    o = Oracle(p)
    if collision:
        o.enable_collision_tally(True)
    o.run(n, seed, n_batches=nb, first_history_id=first)
    s, q = o.tally_sums()
    w, c = o.census()
    cnt = o.counters()
    out = {"sum": s, "sumsq": q, "pop_w": w, "pop_n": c, "counters": {k: cnt[k] for k in COUNTER_KEYS}}
    o.close()
    return out


def oracle_sums(name, n_histories, n_batches, seed=None, nproc=None, **kw):
    """Sum / sumsq / census / counters of `n_histories` histories of get_config(name) in `n_batches` batches, computed
    by `nproc` oracle processes (default: all cores), each taking a contiguous range of whole batches."""
    from workloads import configs as W
    kw = dict(kw, n_histories=n_histories, n_batches=n_batches)
    p = W.get_config(name, **kw)
    seed = p.seed if seed is None else seed
    nproc = max(1, min(nproc or (os.cpu_count() or 1), n_batches))
    hb = n_histories // n_batches
    assert hb * n_batches == n_histories
    # more, smaller parts than processes: the last parts then balance the load
    n_parts = min(n_batches, 4 * nproc)
    bounds = [round(i * n_batches / n_parts) for i in range(n_parts + 1)]
    jobs = [(name, kw, seed, bounds[i] * hb, (bounds[i + 1] - bounds[i]) * hb, bounds[i + 1] - bounds[i], False)
            for i in range(n_parts) if bounds[i + 1] > bounds[i]]
    ctx = mp.get_context("spawn")
    tot = None
    with ctx.Pool(nproc) as pool:
        for r in pool.imap_unordered(_part, jobs):
            if tot is None:
                tot = r
            else:
                for k in ("sum", "sumsq", "pop_w", "pop_n"):
                    tot[k] = tot[k] + r[k]
                for k in COUNTER_KEYS:
                    tot["counters"][k] += r["counters"][k]
    tot["problem"] = p
    tot["nproc"] = nproc
    return tot


def mean_sdev(sum_, sumsq, n_hist, n_batches):
    """SURVEY.md A.9 written out: mean = sum / N; with m_b = S_b / (N/B): sdev = sqrt((sum m_b^2 / B - mean^2) / (B - 1))."""
    hb = n_hist / n_batches
    mean = sum_ / n_hist
    if n_batches > 1:
        var = (sumsq / (hb * hb) / n_batches - mean * mean) / (n_batches - 1)
        sdev = np.sqrt(np.maximum(var, 0.0))
    else:
        sdev = np.zeros_like(mean)
    return mean, sdev
