"""Pins for the oracle's collision-estimator tally (the paper's Fig. 3; SURVEY.md 8(f) NEXT-4;
DESIGN.md Appendix I).  (I-a) one group, Sigma_t = 1, unit weights, every collision inside the mesh: the tally summed
over all bins is the number of collisions, exactly, and every time bin follows the infinite-medium closed form;
(I-b) a pure-absorber beam collides once, at x = v t: the bin (x, t) pattern and the per-bin expectation
exp(-x_i) - exp(-x_i+1) are closed forms; (I-c) it estimates the same flux as the track-length tally, group by group;
(I-d) sites outside the mesh or the time grid score nothing."""
import numpy as np
import pytest

from oracle import Oracle
from workloads import configs as W


def test_Ia_sum_is_the_collision_count_and_bins_follow_the_closed_form():
    p = W.config0_infinite_medium(n_histories=40000, n_batches=20)
    o = Oracle(p); o.enable_collision_tally()
    o.run(p.n_histories, p.seed, n_batches=p.n_batches)
    mc, sc = o.collision_tallies()
    c = o.counters()
    assert mc.sum() * p.n_histories == pytest.approx(c["collisions"], rel=1e-13)
    k = np.arange(20)
    exact = (np.exp(-0.1 * k) - np.exp(-0.1 * (k + 1))) / 0.1
    assert np.abs((mc.ravel() - exact) / sc.ravel()).max() < 4.0
    mt, st = o.tallies()
    assert np.abs((mc - mt).ravel() / np.sqrt(sc ** 2 + st ** 2).ravel()).max() < 4.0
    # off by default: a fresh handle leaves the collision tally at zero and the track-length tally unchanged
    q = Oracle(p); q.run(p.n_histories, p.seed, n_batches=p.n_batches)
    assert np.array_equal(q.tallies()[0], mt) and q.collision_tallies()[0].sum() == 0.0


def test_Ib_pure_absorber_beam_bins():
    N = 200_000
    p = W.get_config("config1a", n_histories=N, n_batches=10)
    o = Oracle(p); o.enable_collision_tally()
    o.run(N, p.seed, n_batches=10)
    mc, _ = o.collision_tallies()                         # [t][g][z][y][x] = [50][1][1][1][100]
    a = mc[:, 0, 0, 0, :] * N                             # collisions per (t-bin, x-bin) / Sigma_t (= 1 where x < 10)
    xe = np.linspace(0.0, 30.0, 101); te = p.time_edges
    # the beam flies at v = 1 from x = 0 at t = 0: a collision at x happens at t = x
    nz = np.argwhere(a > 0)
    for it, ix in nz:
        assert max(xe[ix], te[it]) <= min(xe[ix + 1], te[it + 1]) + 1e-12
    per_x = a.sum(axis=0)
    n_in = 30                                             # x < 9 cm (region 0), t < 10 s holds all of them
    expect = N * (np.exp(-xe[:n_in]) - np.exp(-xe[1:n_in + 1]))
    sig = np.sqrt(np.maximum(expect, 1.0))
    assert np.all(np.abs(per_x[:n_in] - expect) < 4.5 * sig)
    assert per_x[:n_in].sum() == pytest.approx(o.counters()["collisions"], abs=N * np.exp(-9.0) + 5)


def test_Ic_same_flux_as_the_track_length_tally_group_by_group():
    p = W.infinite_medium_multigroup(material=0, n_histories=60000, n_batches=20, t_end=2e-7)
    o = Oracle(p); o.enable_collision_tally()
    o.run(p.n_histories, p.seed, n_batches=p.n_batches)
    mc, sc = o.collision_tallies(); mt, st = o.tallies()
    err = np.sqrt(sc ** 2 + st ** 2)
    # compare where the collision estimator has Gaussian statistics: at least 100 expected collisions in the bin
    # (the slowest groups move 0.04 cm in the whole time range and collide a handful of times in 60 000 histories)
    events = mt * p.n_histories * p.sigma_t[0][None, :, None, None, None]
    ok = events >= 100.0
    assert ok.sum() >= 60
    assert np.abs((mc - mt)[ok] / err[ok]).max() < 4.5
    gt, gc = mt.sum(axis=(0, 2, 3, 4)), mc.sum(axis=(0, 2, 3, 4))
    assert np.allclose(gc[:5], gt[:5], rtol=0.03)
    assert not np.allclose(gc, gt, rtol=1e-6)             # a different estimator, not a copy
    # the rare groups: Poisson counts around Sigma_t x track length
    n_col = gc[5:] * p.n_histories * p.sigma_t[0][5:]
    n_exp = gt[5:] * p.n_histories * p.sigma_t[0][5:]
    assert np.all(np.abs(n_col - n_exp) < 4.5 * np.sqrt(n_exp) + 1.0)


def test_Id_sites_outside_mesh_or_time_grid_score_nothing():
    p = W.stress_geometry(n_histories=30000, n_batches=6, covering_mesh=False)   # the mesh clips the geometry
    o = Oracle(p); o.enable_collision_tally()
    o.run(p.n_histories, p.seed, n_batches=6)
    mc, _ = o.collision_tallies(); mt, _ = o.tallies()
    assert mc.sum() > 0
    assert np.all(mc[mt == 0.0] == 0.0)                   # no collision score in a bin no track ever crossed
    full = W.stress_geometry(n_histories=30000, n_batches=6, covering_mesh=True)
    f = Oracle(full); f.enable_collision_tally(); f.run(full.n_histories, full.seed, n_batches=6)
    assert f.collision_tallies()[0].sum() > mc.sum()      # the clipped mesh lost the sites outside it
