"""Pins for the oracle's track-length estimator (pins E3, E8)."""
import numpy as np
import pytest

from oracle import Oracle
from workloads import configs as W


def _mesh_problem(nx=5, ny=4, nz=3, nt=6, G=2):
    """A bare problem whose only purpose is to carry a (x,y,z,t,g) mesh for score_segment()."""
    mats, ss = W._materials([dict(sigma_t=[1.0] * G, sigma_c=[1.0] * G, sigma_f=[0.0] * G, nu=[0.0] * G,
                                  chi=[0.0] * G, sigma_s=np.zeros((G, G)))], G)
    surfs = [W.plane_x(-100.0), W.plane_x(100.0)]
    cells = [([(0, +1), (1, -1)], 0)]
    pdf = np.zeros(G); pdf[0] = 1
    src = dict(lo=[0, 0, 0], hi=[0, 0, 0], t0=0.0, t1=0.0, pdf=pdf)
    mesh = dict(lo=[-1.0, 0.5, -2.0], hi=[4.0, 3.3, 1.0], n=[nx, ny, nz])
    T = np.array([0.0, 0.4, 1.0, 1.1, 2.5, 3.0, 4.0][: nt + 1])
    speed = [2.0, 0.5][:G]
    return W._assemble("mesh", mats, ss, speed, surfs, [1, 1], cells, src, mesh, T, T[1:].copy(), 1, 1, 1)


def _brute_score(p, r, o, t, g, w, d, n=200001):
    """Midpoint-rule binning of the segment: length w*d/n to the bin holding each sample point."""
    out = np.zeros(p.tally_shape())
    u = (np.arange(n) + 0.5) * (d / n)
    pts = r[None, :] + u[:, None] * o[None, :]
    tt = t + u / p.speed[g]
    ok = np.ones(n, dtype=bool)
    idx = []
    for a in range(3):
        lo, hi, na = p.mesh_lo[a], p.mesh_hi[a], int(p.mesh_n[a])
        ok &= (pts[:, a] >= lo) & (pts[:, a] < hi)
        i = np.floor((pts[:, a] - lo) / ((hi - lo) / na)).astype(int)
        idx.append(np.clip(i, 0, na - 1))
    it = np.searchsorted(p.time_edges, tt, side="right") - 1
    ok &= (it >= 0) & (it < p.n_time_bins)
    it = np.clip(it, 0, p.n_time_bins - 1)
    np.add.at(out, (it[ok], np.full(ok.sum(), g), idx[2][ok], idx[1][ok], idx[0][ok]), w * d / n)
    return out


def test_dda_matches_brute_force_binning():
    p = _mesh_problem()
    o = Oracle(p)
    rng = np.random.default_rng(7)
    for trial in range(25):
        r = rng.uniform([-2, 0, -3], [5, 4, 2])
        d_ = rng.normal(size=3); d_ /= np.linalg.norm(d_)
        if trial % 5 == 0:
            d_[trial % 3] = 0.0; d_ /= np.linalg.norm(d_)       # axis-parallel components
        g = int(rng.integers(0, 2)); t = rng.uniform(-0.5, 3.0); w = rng.uniform(0.2, 2.0)
        d = rng.uniform(0.1, 9.0)
        o.reset()
        o.score_segment(r, d_, t, g, w, d)
        o.close_batch(1)
        got, _ = o.tally_sums()
        ref = _brute_score(p, r, d_, t, g, w, d)
        assert np.abs(got - ref).max() < 3 * w * d / 200001 + 1e-12
        assert got.sum() == pytest.approx(ref.sum(), abs=3 * w * d / 200001)
        other = [k for k in range(2) if k != g]
        assert np.all(got[:, other] == 0.0)


def test_dda_total_length_is_the_clipped_length():
    p = _mesh_problem()
    o = Oracle(p)
    # fully inside the box and the time window: the bins must sum to w*d exactly (to rounding)
    r = np.array([-0.5, 1.0, -1.5]); d_ = np.array([0.6, 0.0, 0.8]); w, d = 1.7, 2.9
    o.score_segment(r, d_, 0.1, 0, w, d); o.close_batch(1)
    got, _ = o.tally_sums()
    assert got.sum() == pytest.approx(w * d, rel=1e-14)
    # starting before T[0]: only the part after T[0] counts: speed 2 -> enters at u = 2*0.25
    o.reset()
    o.score_segment(r, d_, -0.25, 0, w, d); o.close_batch(1)
    got, _ = o.tally_sums()
    assert got.sum() == pytest.approx(w * (d - 0.5), rel=1e-14)
    # zero-length segment scores nothing
    o.reset(); o.score_segment(r, d_, 0.1, 0, w, 0.0); o.close_batch(1)
    assert o.tally_sums()[0].sum() == 0.0


def test_time_index_on_an_edge_belongs_to_the_later_bin():
    # D16: time bin by comparison with the stored edge: a particle sitting exactly on T[2] scores in bin 2
    p = _mesh_problem()
    o = Oracle(p)
    o.score_segment([0.0, 1.0, 0.0], [1.0, 0.0, 0.0], p.time_edges[2], 0, 1.0, 0.1); o.close_batch(1)
    got, _ = o.tally_sums()
    assert got[2].sum() == pytest.approx(0.1, rel=1e-14) and got[1].sum() == 0.0


def test_unbounded_axes_accept_any_coordinate():
    p = W.config1_slab()
    o = Oracle(p)
    o.score_segment([1.0, 1e9, -1e12], [0.6, 0.8, 0.0], 0.0, 0, 1.0, 1.0); o.close_batch(1)
    got, _ = o.tally_sums()
    assert got.sum() == pytest.approx(1.0, rel=1e-14)
    # x from 1.0 to 1.6: bins 3 (0.9-1.2), 4 (1.2-1.5), 5 (1.5-1.8) hold 0.2, 0.3, 0.1 of x-extent => /0.6 of length
    assert got[:, 0, 0, 0, 3].sum() == pytest.approx(0.2 / 0.6, rel=1e-12)
    assert got[:, 0, 0, 0, 4].sum() == pytest.approx(0.3 / 0.6, rel=1e-12)
    assert got[:, 0, 0, 0, 5].sum() == pytest.approx(0.1 / 0.6, rel=1e-12)


def test_pure_absorber_beam_closed_form_E3_and_causality_E8():
    """Uncollided beam along +x from x=0 at t=0, v=1, Sigma_t=1 (x<10): the track length per history in
    bin (x in [a,b], t in [Tj,Tj+1]) is the integral of exp(-x) over [max(a,Tj), min(b,Tj+1)]."""
    N = 200_000
    p = W.config1a_pure_absorber_beam(n_histories=N, n_batches=100)
    o = Oracle(p)
    o.run(N, p.seed, n_batches=100)
    mean, sdev = o.tallies()
    mean = mean[:, 0, 0, 0, :]; sdev = sdev[:, 0, 0, 0, :]
    xe = np.linspace(0, 30, 101); T = p.time_edges

    def E(x):      # exp(-optical depth) integrated: F(x) = int_0^x exp(-tau(s)) ds, piecewise
        x = np.asarray(x, dtype=float)
        f1 = 1 - np.exp(-np.minimum(x, 10.0))
        f2 = np.exp(-10.0) * (1 - np.exp(-0.5 * np.clip(x - 10.0, 0, 10.0))) / 0.5
        f3 = np.exp(-15.0) * (1 - np.exp(-np.clip(x - 20.0, 0, 10.0)))
        return f1 + f2 + f3

    exact = np.zeros_like(mean)
    for j in range(50):
        for i in range(100):
            lo, hi = max(xe[i], T[j]), min(xe[i + 1], T[j + 1])
            if hi > lo + 1e-12:
                exact[j, i] = E(hi) - E(lo)
    # E8 causality: bins the beam has not reached yet or has already left hold nothing (a coincident x / t
    # edge may leak a piece of rounding length, A.7: "misassignments are bounded by rounding")
    assert mean[exact == 0.0].max() < 1e-14
    nz = exact > 0
    # north_star: uncollided transmission exp(-Sigma_t x); statistical agreement bin by bin
    z = (mean[nz] - exact[nz]) / np.maximum(sdev[nz], 1e-300)
    big = exact[nz] > 1e-4                      # bins with enough scores for a normal approximation
    assert np.abs(z[big]).max() < 4.5
    assert mean[nz][big].sum() == pytest.approx(exact[nz][big].sum(), rel=2e-3)
    # deterministic part: the first time bin [0, 0.2] is crossed uncollided with prob exp(-x); every history
    # contributes at most the bin width, and the total over all bins is the mean track length 1 - e^-10 + ...
    assert mean.sum() == pytest.approx(float(E(30.0)), rel=3 * 1.0 / np.sqrt(N))
    # the captures follow the same law: fraction absorbed before x=10 is 1-exp(-10)
    c = o.counters()
    assert c["capture"] / N == pytest.approx(1.0, abs=5e-4)
    assert c["source"] == c["capture"] + c["leak"] + c["census_final"]


def test_batch_statistics_definition():
    # A.9 with hand-made batches: S_b = 1, 2, 3, 6 with 2 histories each
    p = _mesh_problem()
    o = Oracle(p)
    for s in (1.0, 2.0, 3.0, 6.0):
        o.score_segment([0.0, 1.0, 0.0], [1.0, 0.0, 0.0], 0.0, 0, 1.0, s * 0.01); o.close_batch(2)
    mean, sdev = o.tallies()
    m_b = np.array([1.0, 2.0, 3.0, 6.0]) * 0.01 / 2
    assert mean.sum() == pytest.approx(m_b.mean(), rel=1e-13)
    assert sdev.max() == pytest.approx(m_b.std(ddof=0) / np.sqrt(3), rel=1e-10)   # sqrt(var_pop/(B-1))
