"""Pins for the oracle's variance-reduction rows (DESIGN.md Appendix G): implicit capture,
weight roulette and the population control at census.  What fixes them: (G-a) a pure absorber loses its whole weight
at the first collision either way, so implicit capture must reproduce the analog run bit for bit; (G-b) the techniques
are unbiased, so the infinite-medium closed forms N(t) = N0 exp(-0.1 t) and its per-bin integral still hold; (G-c) the
weight ledger closes (source + production + vr_gain = capture + fission_abs + leak + census_final + lost + vr_loss);
(G-d) the weight after n collisions of a non-multiplying medium is (Sigma_s/Sigma_t)^n exactly; (G-e) the control
makes floor or ceil of w/w_t copies with the right mean, conserves the weight in expectation and holds the population
at the target; (G-f) none of it depends on the processing order."""
import numpy as np
import pytest

from oracle import Oracle, draws
from workloads import configs as W

LAM = 0.1


def _residual(c):
    gain = c["source"] + c["production"] + c["vr_gain"]
    loss = c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"] + c["lost"] + c["vr_loss"]
    return (gain - loss) / gain


def test_Ga_pure_absorber_implicit_capture_equals_analog_bitwise():
    p = W.get_config("config1a", n_histories=20000, n_batches=10)
    a = Oracle(p); a.run(p.n_histories, p.seed, n_batches=10, record_history_events=True)
    b = Oracle(p); b.set_technique(implicit_capture=True)
    b.run(p.n_histories, p.seed, n_batches=10, record_history_events=True)
    sa, qa = a.tally_sums(); sb, qb = b.tally_sums()
    assert np.array_equal(sa, sb) and np.array_equal(qa, qb)
    assert np.array_equal(a.history_events(), b.history_events())
    ca, cb = a.counters(), b.counters()
    assert ca["capture"] == cb["capture"] and ca["leak"] == cb["leak"] and cb["vr_gain"] == 0.0


@pytest.mark.parametrize("tech", [dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0),
                                  dict(population_control=True),
                                  dict(implicit_capture=True, wr_threshold=0.25, wr_survive=0.5, population_control=True)])
def test_Gb_Gc_unbiased_infinite_medium_and_ledger(tech):
    p = W.config0_infinite_medium(n_histories=40000, n_batches=20)
    o = Oracle(p); o.set_technique(**tech)
    o.run(p.n_histories, p.seed, n_batches=p.n_batches)
    k = np.arange(20)
    exact = (np.exp(-LAM * k) - np.exp(-LAM * (k + 1))) / LAM
    mean, sdev = o.tallies()
    mean, sdev = mean.ravel(), sdev.ravel()
    z = (mean - exact) / sdev
    assert np.abs(z).max() < 4.0, z
    # the whole-run flux integral: sum of the bins, error from the batch sums
    assert abs(mean.sum() - exact.sum()) < 4.0 * np.sqrt((sdev ** 2).sum()) * 3.0
    w, n = o.census()
    popex = np.exp(-LAM * np.arange(1, 21))
    assert np.all(np.abs(w / p.n_histories - popex) < 6.0 * np.maximum(sdev, 1e-3) + 1e-3)
    c = o.counters()
    assert abs(_residual(c)) < 1e-12
    if tech.get("implicit_capture"):
        assert not np.array_equal(w, n.astype(float))         # weights are no longer 1
    if tech.get("wr_threshold"):
        assert c["vr_gain"] > 0.0 and c["vr_loss"] > 0.0
        # roulette is fair: weight created and removed agree within the noise of the game
        assert abs(c["vr_gain"] - c["vr_loss"]) < 0.05 * (c["vr_gain"] + c["vr_loss"]) + 50.0


def test_Gd_weight_after_n_collisions_is_a_power_of_the_scattering_ratio():
    """Non-multiplying infinite medium, implicit capture, no roulette: nothing ever dies before the final census and
    the weight at the end is 0.7^(collisions of that history) -- per history, exactly."""
    p = W.config0_infinite_medium(n_histories=3000, n_batches=10)
    p.sigma_s = np.array([[[0.7]]]); p.sigma_c = np.array([[0.3]]); p.sigma_f = np.array([[0.0]]); p.nu = np.array([[0.0]])
    o = Oracle(p); o.set_technique(implicit_capture=True)
    o.run(p.n_histories, p.seed, n_batches=10, record_history_events=True)
    # (G-b) unbiased: the flux per time bin is the integral of exp(-Sigma_c v t)
    k = np.arange(20)
    exact = (np.exp(-0.3 * k) - np.exp(-0.3 * (k + 1))) / 0.3
    mean, sdev = o.tallies()
    assert np.abs((mean.ravel() - exact) / sdev.ravel()).max() < 4.0
    ev = o.history_events()
    c = o.counters()
    assert c["children"] == 0 and c["leak"] == 0.0 and c["census_events"] == 20 * p.n_histories
    expect = np.sort(0.7 ** ev[:, 0].astype(np.float64))
    assert c["census_final"] == pytest.approx(expect.sum(), rel=1e-12)
    assert c["capture"] == pytest.approx(p.n_histories - expect.sum(), rel=1e-12)
    w, n = o.census()
    assert n[-1] == p.n_histories and w[-1] == pytest.approx(c["census_final"], rel=1e-13)
    # expected weight at t: exp(-Sigma_c v t)
    assert w[-1] / p.n_histories == pytest.approx(np.exp(-0.3 * 20.0), rel=0.08)


def test_Ge_population_control_unit():
    p = W.config0_infinite_medium(n_histories=100, n_batches=1)
    o = Oracle(p)
    rng = np.random.default_rng(5)
    n = 20000
    w = rng.uniform(0.05, 3.0, n)
    key = rng.integers(1, 2 ** 63, n, dtype=np.uint64); ctr = rng.integers(0, 50, n).astype(np.uint32)
    target = 15000
    n_out, w_t = o.population_control(w, key, ctr, target)
    W_fix = np.floor(w * 2.0 ** 40).sum() / 2.0 ** 40
    assert w_t == W_fix / target
    ratio = w / w_t
    assert np.all((n_out == np.floor(ratio)) | (n_out == np.floor(ratio) + 1))
    # the draw is the particle's own next draw: n = floor(ratio + xi)
    for i in range(0, n, 997):
        xi = draws(int(key[i]), int(ctr[i]), 1)[0]
        assert n_out[i] == int(np.floor(ratio[i] + xi))
    # unbiased: sum of copies = sum of ratios within the noise of n Bernoulli trials
    frac = ratio - np.floor(ratio)
    assert abs(n_out.sum() - ratio.sum()) < 4.0 * np.sqrt((frac * (1 - frac)).sum())
    assert abs(n_out.sum() - target) < 4.0 * np.sqrt((frac * (1 - frac)).sum())
    # order independence: any permutation of the bank gives the same copies
    perm = rng.permutation(n)
    n2, w_t2 = o.population_control(w[perm], key[perm], ctr[perm], target)
    assert w_t2 == w_t and np.array_equal(n2, n_out[perm])


def test_Ge_population_is_held_at_the_target():
    p = W.config0_infinite_medium(n_histories=20000, n_batches=4)
    o = Oracle(p); o.set_technique(population_control=True)
    o.run(p.n_histories, p.seed, n_batches=4)
    wa, na = o.census_after(); w, n = o.census()
    hb = p.n_histories // 4
    assert na[-1] == 0 and np.all(np.abs(na[:-1].astype(float) / 4 - hb) < 5.0 * np.sqrt(hb))
    # the control conserves the weight up to its own noise, census by census
    assert np.all(np.abs(wa[:-1] - w[:-1]) < 5.0 * np.sqrt(w[:-1] * (w[:-1] / na[:-1])))
    # without it the analog population decays as exp(-0.1 t): at the last census 13.5 % are left
    assert n[-1] > 0.7 * p.n_histories * np.exp(-LAM)        # arrivals of the last step: one step of decay from hb
    c = o.counters()
    assert c["pc_removed"] == 0 and c["pc_added"] > 0        # a decaying population is only ever split (w / w_t >= 1)
    custom = Oracle(p); custom.set_technique(population_control=True, pc_target=1000)
    custom.run(p.n_histories, p.seed, n_batches=4)
    assert np.all(np.abs(custom.census_after()[1][:-1].astype(float) / 4 - 1000) < 5.0 * np.sqrt(1000))
    assert custom.counters()["pc_removed"] > 0               # 5000 arrivals rouletted down to 1000 at the first census


@pytest.mark.parametrize("name,N", [("config0", 4000), ("config3", 1000)])
def test_Gf_schedule_independence_with_all_techniques(name, N):
    p = W.get_config(name, n_histories=N, n_batches=4)
    tech = dict(implicit_capture=True, wr_threshold=0.3, wr_survive=0.6, population_control=True)
    base = Oracle(p); base.set_technique(**tech); base.run(N, p.seed, n_batches=4, record_history_events=True)
    ev0 = base.history_events(); s0, _ = base.tally_sums(); c0 = base.counters()
    for kw in (dict(bank_fifo=True), dict(reverse_histories=True)):
        o = Oracle(p); o.set_technique(**tech); o.run(N, p.seed, n_batches=4, record_history_events=True, **kw)
        assert np.array_equal(o.history_events(), ev0)
        s, _ = o.tally_sums()
        assert np.abs(s - s0).max() <= 1e-12 * np.abs(s0).max()
        c = o.counters()
        for key in ("collisions", "surf_hits", "census_events", "children", "pc_removed", "pc_added"):
            assert c[key] == c0[key]
        assert c["capture"] == pytest.approx(c0["capture"], rel=1e-12)
    assert abs(_residual(c0)) < 1e-12
