"""The parallel-oracle helper of the full-size GPU tests is itself held to the single oracle run (pin E5: history
ranges may be simulated in any split and summed)."""
import numpy as np

from _oracle_mp import COUNTER_KEYS, mean_sdev, oracle_sums


def test_parallel_oracle_equals_the_single_run():
    from oracle import Oracle
    from workloads import configs as W
    N, B = 6000, 12
    tot = oracle_sums("config3", N, B, nproc=3)
    p = W.get_config("config3", n_histories=N, n_batches=B)
    o = Oracle(p)
    o.run(N, p.seed, n_batches=B)
    s, q = o.tally_sums()
    # batches are whole in every part: S_b, hence sum S_b^2, are the same numbers added in another order
    assert np.allclose(tot["sum"], s, rtol=1e-13, atol=0) and np.allclose(tot["sumsq"], q, rtol=1e-13, atol=0)
    c = o.counters()
    for k in COUNTER_KEYS:
        assert tot["counters"][k] == c[k], k
    w, n = o.census()
    assert np.array_equal(tot["pop_n"], n) and np.array_equal(tot["pop_w"], w)
    m, sd = mean_sdev(tot["sum"], tot["sumsq"], N, B)
    m1, s1 = o.tallies()
    assert np.allclose(m, m1, rtol=1e-13, atol=0) and np.allclose(sd, s1, rtol=1e-9, atol=1e-18)
