"""Pins for the oracle's history loop (pins E1, E2, E4, E5, E6, E7).

Closed forms named by BASELINE.json north_star: infinite-medium population N(t) = N0 exp(-(1-c) Sigma_t v t)
with c = (Sigma_s + nu Sigma_f)/Sigma_t, and the exact weight balance."""
import numpy as np
import pytest
import scipy.linalg as sl

from oracle import Oracle
from workloads import configs as W


def _balance(c):
    return c["source"] + c["production"] - (c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"] + c["lost"])


@pytest.fixture(scope="module")
def c0_run():
    p = W.config0_infinite_medium()
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=p.n_batches, record_history_events=True)
    return p, o


def test_E1_infinite_medium_flux_and_population(c0_run):
    p, o = c0_run
    N = p.n_histories
    lam = 0.1                                             # (1 - c) Sigma_t v, c = (0.5 + 2*0.2)/1 = 0.9
    k = np.arange(20)
    exact = (np.exp(-lam * k) - np.exp(-lam * (k + 1))) / lam
    assert exact[0] == pytest.approx(0.951626, abs=5e-7) and exact[19] == pytest.approx(0.142333, abs=5e-7)
    mean, sdev = o.tallies()
    mean, sdev = mean.ravel(), sdev.ravel()
    assert np.abs((mean - exact) / sdev).max() < 4.0
    # census populations: N(t_k)/N0 = exp(-0.1 k); binomial-ish noise, fission chains inflate the variance
    w, n = o.census()
    assert np.array_equal(w, n.astype(float))            # analog: all weights are 1
    popex = np.exp(-lam * np.arange(1, 21))
    # the per-bin sdev of the adjacent flux bins bounds the population noise (flux = integral of population)
    tol = 6.0 * np.maximum(sdev, 1e-3) + 1e-3
    assert np.all(np.abs(w / N - popex) < tol)


def test_E2_expected_event_counts_per_history(c0_run):
    p, o = c0_run
    ev = o.history_events().astype(np.float64)           # [N][coll, surf, children, census]
    N = ev.shape[0]
    exact = np.array([10 * (1 - np.exp(-2.0)),           # collisions: Sigma_t v int_0^20 e^{-0.1 t} dt
                      1.5 * 10 * (1 - np.exp(-2.0)),     # surface hits: Cauchy S/4V = 1.5 per cm of track
                      0.2 * 2.0 * 10 * (1 - np.exp(-2.0)),  # children: nu Sigma_f per cm of track
                      np.exp(-0.1 * np.arange(1, 21)).sum()])  # census events
    assert exact == pytest.approx([8.6466, 12.970, 3.4587, 8.2215], rel=2e-5)
    m = ev.mean(axis=0); se = ev.std(axis=0, ddof=1) / np.sqrt(N)
    assert np.all(np.abs(m - exact) / se < 4.0)
    c = o.counters()
    assert c["collisions"] == ev[:, 0].sum() and c["surf_hits"] == ev[:, 1].sum()
    assert c["children"] == ev[:, 2].sum() and c["census_events"] == ev[:, 3].sum()
    assert c["segments"] == c["collisions"] + c["surf_hits"] + c["census_events"]
    assert c["census_final"] / N == pytest.approx(np.exp(-2.0), abs=4 * np.sqrt(0.135 / N) * 3)
    # reaction branching: capture : fission = 0.3 : 0.2, scatter fraction 0.5
    absorbed = c["capture"] + c["fission_abs"]
    assert c["capture"] / absorbed == pytest.approx(0.6, abs=4 * np.sqrt(0.24 / absorbed))
    assert absorbed / c["collisions"] == pytest.approx(0.5, abs=4 * np.sqrt(0.25 / c["collisions"]))
    assert c["children"] / c["fission_abs"] == pytest.approx(2.0, abs=1e-12)   # nu = 2 exactly: floor(2 + xi) = 2


@pytest.mark.parametrize("name,N,B", [("config0", 20000, 20), ("config1", 20000, 10), ("config1a", 20000, 10),
                                      ("config2", 20000, 10), ("config3", 4000, 10)])
def test_E4_weight_balance_is_exact(name, N, B):
    p = W.get_config(name, n_histories=N, n_batches=B)
    o = Oracle(p)
    o.run(N, p.seed, n_batches=B)
    c = o.counters()
    assert c["source"] == N and c["lost"] == 0.0 and c["lost_n"] == 0
    assert _balance(c) == 0.0
    # every batch separately: run batch by batch on fresh handles
    o2 = Oracle(p)
    for b in range(3):
        o2.reset()
        o2.run(N // B, p.seed, n_batches=1, first_history_id=b * (N // B))
        assert _balance(o2.counters()) == 0.0
    # the census ledger agrees with the population arrays
    w, n = o.census()
    assert w[-1] == c["census_final"] and n.sum() == c["census_events"]


@pytest.mark.parametrize("name,N", [("config0", 5000), ("config1", 5000), ("config3", 1500)])
def test_E5_schedule_independence(name, N):
    p = W.get_config(name, n_histories=N, n_batches=5)
    base = Oracle(p); base.run(N, p.seed, n_batches=5, record_history_events=True)
    ev0 = base.history_events(); s0, _ = base.tally_sums(); c0 = base.counters()
    scale = np.abs(s0).max()
    for kw in (dict(bank_fifo=True), dict(reverse_histories=True), dict(bank_fifo=True, reverse_histories=True)):
        o = Oracle(p); o.run(N, p.seed, n_batches=5, record_history_events=True, **kw)
        assert np.array_equal(o.history_events(), ev0)
        s, _ = o.tally_sums()
        assert np.abs(s - s0).max() <= 1e-13 * scale
        assert o.counters() == c0
    # split ranges: two runs over disjoint history ranges accumulate to the same sums
    o = Oracle(p)
    h = N // 5
    o.run(2 * h, p.seed, n_batches=2, first_history_id=0, record_history_events=True)
    eva = o.history_events()
    o.run(3 * h, p.seed, n_batches=3, first_history_id=2 * h, record_history_events=True)
    evb = o.history_events()
    assert np.array_equal(np.vstack([eva, evb]), ev0)
    s, q = o.tally_sums(); s0, q0 = base.tally_sums()
    assert np.array_equal(s, s0) and np.array_equal(q, q0)
    assert o.counters() == c0
    # a different seed gives different trajectories
    o = Oracle(p); o.run(N, p.seed + 1, n_batches=5, record_history_events=True)
    assert not np.array_equal(o.history_events(), ev0)


@pytest.mark.parametrize("material", [0, 2])
def test_E6_multigroup_kinetics_matrix_exponential(material):
    """One config-3 material in a reflective box: n'(t) = A n, A[g][g'] = v_g'(Sigma_s[g'->g] + chi_g nu Sigma_f[g'])
    - delta v_g Sigma_t[g]; the group flux in a time bin is v_g times the time integral of n_g."""
    t_end = 2e-7 if material == 0 else 4e-7
    p = W.infinite_medium_multigroup(material=material, n_histories=60000, n_batches=20, t_end=t_end)
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=20)
    G = 7; v = p.speed; St = p.sigma_t[0]; Ss = p.sigma_s[0]; nuSf = p.nu[0] * p.sigma_f[0]; chi = p.chi[0]
    A = np.zeros((G, G))
    for g in range(G):
        for gp in range(G):
            A[g, gp] = v[gp] * (Ss[gp, g] + chi[g] * nuSf[gp])
        A[g, g] -= v[g] * St[g]
    n0 = p.src_group_pdf
    T = p.time_edges
    Ainv = np.linalg.inv(A)
    exact = np.array([v * (Ainv @ ((sl.expm(A * T[j + 1]) - sl.expm(A * T[j])) @ n0)) for j in range(20)])
    mean, sdev = o.tallies()
    mean, sdev = mean[:, :, 0, 0, 0], sdev[:, :, 0, 0, 0]
    big = exact > 1e-3 * exact.max()
    z = (mean - exact)[big] / sdev[big]
    assert np.abs(z).max() < 4.5
    assert mean[big].sum() == pytest.approx(exact[big].sum(), abs=4.0 * sdev[big].sum())   # fully-correlated bound
    assert _balance(o.counters()) == 0.0


def test_E7_slab_flux_is_symmetric_about_the_midplane():
    p = W.config1_slab(n_histories=40000, n_batches=40)
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=40)
    mean, sdev = o.tallies()
    m = mean[:, 0, 0, 0, :]; s = sdev[:, 0, 0, 0, :]
    diff = m - m[:, ::-1]
    err = np.sqrt(s ** 2 + s[:, ::-1] ** 2)
    ok = err > 0
    z = diff[ok] / err[ok]
    assert np.abs(z).max() < 5.0
    assert abs(z.mean()) < 0.2 and 0.7 < z.std() < 1.3


def test_E7_lattice_tally_has_the_symmetries_of_the_square():
    # centre source, 17 odd: the checkerboard maps to itself under the 8 symmetries of the square.
    p = W.config3_pin_lattice(n_histories=12000, n_batches=12)
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=12)
    mean, sdev = o.tallies()
    m = mean[:, :, 0].sum(axis=(0, 1))                    # [y][x] integrated over time and group
    # compare ring sums of each octant image: use the total of each quadrant-like wedge
    imgs = [m, m[::-1, :], m[:, ::-1], m[::-1, ::-1], m.T, m.T[::-1, :], m.T[:, ::-1], m.T[::-1, ::-1]]
    wedge = np.triu(np.ones((17, 17)), 1); wedge[:, :9] = 0   # one open octant
    sums = np.array([(im * wedge).sum() for im in imgs])
    assert sums.std() / sums.mean() < 0.06
    # x <-> y symmetry of the centre row / column
    assert m[8, :].sum() == pytest.approx(m[:, 8].sum(), rel=0.05)


def test_E8_causality_in_the_duct_box():
    # v = 1: a bin whose nearest point to the source cube [0,10]^3 is farther than T_{j+1} stays empty
    p = W.config2_lduct(n_histories=20000, n_batches=10)
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=10)
    mean, _ = o.tallies()
    m = mean[:, 0]                                        # [t][z][y][x]
    xc = np.arange(60.0); yc = np.arange(100.0); zc = np.arange(60.0)    # lower corners of the 1 cm bins
    dx = np.maximum(xc - 10.0, 0); dy = np.maximum(yc - 10.0, 0); dz = np.maximum(zc - 10.0, 0)
    dist = np.sqrt(dz[:, None, None] ** 2 + dy[None, :, None] ** 2 + dx[None, None, :] ** 2)
    for j in range(20):
        far = dist > p.time_edges[j + 1] + 1e-9
        assert m[j][far].max(initial=0.0) == 0.0
    assert m.sum() > 0


def test_source_sampling_moments():
    # A.3: uniform box, uniform time, isotropic direction (first flight through a void-like problem is
    # awkward to observe; use the duct box and the per-history leak of an all-vacuum... instead check the
    # integrated first-bin quantities): mean x of track in the first 1 cm mesh layer etc. is covered by E1-E3.
    # Here: isotropy via the slab beam-free problem: flux symmetric in +/-x (E7) and mean cosine zero:
    p = W.config1_slab(n_histories=20000, n_batches=10)
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=10)
    c = o.counters()
    # source times uniform in [0,1]: census k (T=0.2k, k<=5) has seen a fraction 0.2k of the sources, minus absorption
    w, _ = o.census()
    frac = w[:5] / p.n_histories
    assert np.all(np.diff(frac) > 0.15) and frac[0] == pytest.approx(0.2, abs=0.02)
    assert c["leak"] == 0 or c["leak"] / p.n_histories < 0.05


def test_stress_geometry_balance_lost_sources_and_mesh_independence():
    """General quadrics, reflective sphere, two-neighbour face: the ledger still closes exactly (E4); source points
    inside the mirror ball (no cell there) are lost at the rate of its volume fraction of the source box; the
    trajectories do not depend on the tally mesh, and a mesh that clips the geometry scores less track."""
    N = 120_000
    pa, pb = W.stress_geometry(n_histories=N, covering_mesh=False), W.stress_geometry(n_histories=N, covering_mesh=True)
    oa, ob = Oracle(pa), Oracle(pb)
    oa.run(N, pa.seed, n_batches=pa.n_batches, record_history_events=True)
    ob.run(N, pb.seed, n_batches=pb.n_batches, record_history_events=True)
    ca, cb = oa.counters(), ob.counters()
    assert _balance(ca) == 0.0 and ca == cb
    assert np.array_equal(oa.history_events(), ob.history_events())
    frac = (4.0 / 3.0) * np.pi * 0.4 ** 3 / (5.6 * 3.6 * 3.6)
    assert abs(ca["lost_n"] - N * frac) < 4.0 * np.sqrt(N * frac)
    assert ca["leak"] > 0 and ca["children"] > 0 and ca["census_final"] > 0
    ma, _ = oa.tallies(); mb, _ = ob.tallies()
    assert 0.0 < ma.sum() < mb.sum()
    # covering mesh, time grid [0, 6] = whole run: total track per history = sum over segments of their lengths;
    # per group g the time-integrated flux equals (time alive in g) * v_g, so sum_g flux_g / v_g = mean lifetime
    life = (mb.sum(axis=(0, 2, 3, 4)) / pb.speed).sum()
    assert 0.0 < life < 6.0 * (1.0 + cb["production"] / N)      # no particle lives longer than the run
