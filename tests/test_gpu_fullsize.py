"""GPU parity at the BASELINE sizes, in the launch configuration bench.py times (north_star: "oracle-matching tallies
on all 5 configs ... every tally bin within |z| <= 4 of the combined standard error, and the integrated flux within
1e-3 relative").  The oracle side is the oracle run as one process per host core over disjoint history ranges with the
sums added (tests/_oracle_mp.py, held to the single run by tests/test_oracle_parallel.py and pin E5).  Because both
sides follow the same trajectories the bins agree to summation-order rounding; the tests assert the official bar AND
that tighter one."""
import numpy as np
import pytest

from _oracle_mp import COUNTER_KEYS, mean_sdev, oracle_sums

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(1500)]


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2409_04668_b200 as M
    M.lib()
    return M


@pytest.mark.parametrize("name", ["config1", "config1a", "config2", "config3"])
def test_full_size_tallies_match_the_oracle_bin_by_bin(M, name):
    from workloads import configs as W
    p = W.get_config(name)                                # BASELINE size: 1e6 / 1e6 / 1e7 / 1e7 histories, 100 batches
    N, B = p.n_histories, p.n_batches
    assert N == {"config1": 10 ** 6, "config1a": 10 ** 6, "config2": 10 ** 7, "config3": 10 ** 7}[name]
    g = M.Problem(p)
    g.run()
    cg = g.counters()
    mg, sg = g.tallies()
    wg, ng = g.census()
    g.close()
    tot = oracle_sums(name, N, B)
    co = tot["counters"]
    # integer event totals: equal unless a history's decision flipped on a 1e-16 tie (north_star: >= 99.999 % of
    # histories bit-exact); the ledger balance itself is exact
    for k in COUNTER_KEYS:
        assert abs(cg[k] - co[k]) <= 1e-6 * max(1.0, co[k]), (k, cg[k], co[k])
    assert cg["histories"] == N and cg["batches"] == B
    assert cg["source"] + cg["production"] == cg["capture"] + cg["fission_abs"] + cg["leak"] + cg["census_final"] + cg["lost"]
    assert np.abs(ng.astype(np.int64) - tot["pop_n"].astype(np.int64)).max() <= max(2, 1e-6 * tot["pop_n"].max())
    mo, so = mean_sdev(tot["sum"], tot["sumsq"], N, B)
    mo = mo.reshape(mg.shape); so = so.reshape(mg.shape)
    scale = np.abs(mo).max()
    # the official bar
    err = np.sqrt(so ** 2 + sg ** 2) + 1e-12 * scale
    z = np.abs(mg - mo) / err
    assert z.max() <= 4.0, (name, z.max())
    assert mg.sum() == pytest.approx(mo.sum(), rel=1e-3)
    # what shared trajectories allow: summation order only (a flipped history moves single bins by ~1/N)
    bad = np.abs(mg - mo) > 1e-7 * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale
    assert bad.mean() <= 1e-5, (name, bad.sum())
    assert mg.sum() == pytest.approx(mo.sum(), rel=1e-9)
    assert np.allclose(sg, so, rtol=1e-4, atol=1e-9 * scale)


def test_config4_1e8_histories_across_launches_sampled_against_the_oracle(M):
    """Config 4 at 1e8 histories run as four launches of 2.5e7 (sub-batches): exact ledger, per-history event counts
    summing to the counters, and histories on both sides of every launch boundary recomputed one by one by the oracle."""
    from oracle import Oracle
    from workloads import configs as W
    N, B, sub = 10 ** 8, 100, 25_000_000
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    g = M.Problem(p, max_histories_per_subbatch=sub, max_batches_in_flight=25, async_only=True)
    g.run(record_history_events=True)
    c = g.counters()
    ev = g.history_events()
    assert c["histories"] == N and c["batches"] == B and c["lost_n"] == 0
    assert c["kernel_launches"] == 8                      # 4 x (k_warp + k_closeout)
    assert c["source"] + c["production"] == c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"]
    assert c["segments"] == c["collisions"] + c["surf_hits"] + c["census_events"]
    tot = ev.sum(axis=0, dtype=np.uint64)
    assert tot[0] == c["collisions"] and tot[1] == c["surf_hits"] and tot[2] == c["children"] and tot[3] == c["census_events"]
    w, n = g.census()
    assert n.sum() == c["census_events"] and w[-1] == c["census_final"]
    o = Oracle(p)
    for first in (0, sub - 300, 2 * sub - 300, 3 * sub - 300, N - 600):
        o.reset()
        o.run(600, p.seed, n_batches=1, first_history_id=first, record_history_events=True)
        assert np.array_equal(o.history_events(), ev[first:first + 600]), first
    # the mean track length per history against the full-size config-3 run is covered by the 1e7 test; here: the
    # per-history rates are those of the 1e7 run to statistical accuracy
    mean, sdev = g.tallies()
    assert np.all(mean >= 0) and np.all(np.isfinite(sdev))
    assert c["segments"] / N == pytest.approx(38.3, rel=0.01) and c["children"] / N == pytest.approx(1.04, rel=0.02)
    g.close()


def test_config4_1e9_histories_ledger_and_launch_plan(M):
    """1e9 histories as device-sized sub-batches (4 launches of 2.5e8, 32-bit in-launch history ids): exact weight
    balance and counter identities at the full size of BASELINE config 4."""
    from workloads import configs as W
    N, B, sub = 10 ** 9, 100, 250_000_000
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    g = M.Problem(p, max_histories_per_subbatch=sub, max_batches_in_flight=25, async_only=True)
    g.run()
    c = g.counters()
    assert c["histories"] == N and c["batches"] == B and c["lost_n"] == 0 and c["kernel_launches"] == 8
    assert c["source"] == N
    assert c["source"] + c["production"] == c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"]
    assert c["segments"] == c["collisions"] + c["surf_hits"] + c["census_events"]
    w, n = g.census()
    assert n.sum() == c["census_events"] and w[-1] == c["census_final"]
    assert c["segments"] / N == pytest.approx(38.3, rel=0.005)
    mean, sdev = g.tallies()
    assert np.all(mean >= 0) and np.all(sdev >= 0) and mean.sum() > 0
    g.close()
