"""GPU parity for the NEXT-1 rows (implicit capture, weight roulette, population control at census; DESIGN.md
Appendix G) and the NEXT-3 row (accumulators exported, summed over ranks and imported back), against the oracle on
the same seeded inputs.  Weights are real numbers here, so ledger entries and census weights are compared to
rounding (1e-12) and integer event counts exactly."""
import numpy as np
import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(600)]

INT_COUNTS = ("histories", "segments", "collisions", "surf_hits", "census_events", "children", "lost_n", "batches",
              "pc_removed", "pc_added")
REAL_LEDGER = ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "vr_gain", "vr_loss")

TECHS = {
    "ic": dict(implicit_capture=True),
    "ic_wr": dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0),
    "wr_only": dict(wr_threshold=1.5, wr_survive=3.0),
    "pc": dict(population_control=True),
    "pc_target": dict(population_control=True, pc_target=700),
    "all": dict(implicit_capture=True, wr_threshold=0.3, wr_survive=0.6, population_control=True),
}


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2409_04668_b200 as M
    M.lib()
    return M


def _pair(M, p, tech, scheduler=0, **gkw):
    """scheduler 0 = the history kernel k_warp (weighted variant; one launch per census step when the population
    control is on); 1 = the census-stepped kernel k_transport."""
    from oracle import Oracle
    o = Oracle(p); o.set_technique(**tech)
    o.run(p.n_histories, p.seed, n_batches=p.n_batches, record_history_events=True)
    g = M.Problem(p, **gkw); g.set_technique(**tech)
    g.run(record_history_events=True, scheduler=scheduler)
    return o, g


def _compare(o, g, rtol_bins, frac=0.99999):
    co, cg = o.counters(), g.counters()
    for k in INT_COUNTS:
        assert cg[k] == co[k], (k, cg[k], co[k])
    for k in REAL_LEDGER:
        # sums of ~1e6 real terms taken in different orders: |difference| <= n 2^-53 relative, ~1e-10 here
        assert cg[k] == pytest.approx(co[k], rel=1e-10, abs=1e-9), (k, cg[k], co[k])
    gain = cg["source"] + cg["production"] + cg["vr_gain"]
    loss = cg["capture"] + cg["fission_abs"] + cg["leak"] + cg["census_final"] + cg["lost"] + cg["vr_loss"]
    assert abs(gain - loss) <= 1e-10 * gain
    eo, eg = o.history_events(), g.history_events()
    assert np.all(eo == eg, axis=1).mean() >= frac
    mo, so = o.tallies(); mg, sg = g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= rtol_bins * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)
    assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * scale)
    wo, no = o.census(); wg, ng = g.census()
    assert np.array_equal(no, ng) and np.allclose(wo, wg, rtol=1e-10)
    wo, no = o.census_after(); wg, ng = g.census_after()
    assert np.array_equal(no, ng) and np.allclose(wo, wg, rtol=1e-10)


@pytest.mark.parametrize("scheduler", [0, 1])
@pytest.mark.parametrize("tech", sorted(TECHS))
def test_config0_with_techniques_matches_the_oracle(M, tech, scheduler):
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=40000, n_batches=20)
    if tech == "ic":                                       # without roulette chains only end by fission: no fission here
        p.sigma_s = np.array([[[0.7]]]); p.sigma_c = np.array([[0.3]]); p.sigma_f = np.array([[0.0]]); p.nu = np.array([[0.0]])
    o, g = _pair(M, p, TECHS[tech], scheduler=scheduler)
    _compare(o, g, rtol_bins=1e-9)
    if tech != "ic":                                       # the closed form through the GPU path as well (pin G-b)
        mg, sg = g.tallies()
        k = np.arange(20)
        exact = (np.exp(-0.1 * k) - np.exp(-0.1 * (k + 1))) / 0.1
        assert np.abs((mg.ravel() - exact) / sg.ravel()).max() < 4.0
    else:                                                  # pin G-d: weight 0.7^collisions per history, exactly
        ev = g.history_events()
        assert g.counters()["census_final"] == pytest.approx((0.7 ** ev[:, 0].astype(np.float64)).sum(), rel=1e-12)
    g.close()


@pytest.mark.parametrize("name,N,B,tech,scheduler", [
    ("config1", 100_000, 20, "all", 0), ("config1a", 50_000, 10, "ic", 0), ("config1a", 50_000, 10, "ic", 1),
    ("config3", 40_000, 20, "all", 0), ("config3", 40_000, 20, "all", 1), ("config3", 100_000, 20, "pc", 0),
    ("config2", 60_000, 12, "all", 0), ("config3", 100_000, 20, "ic_wr", 0), ("config3", 40_000, 20, "ic_wr", 1),
    ("config2", 60_000, 12, "ic_wr", 0), ("config2", 60_000, 12, "ic_wr", 1), ("stress", 120_000, 12, "ic_wr", 0)])
def test_larger_configs_with_techniques(M, name, N, B, tech, scheduler):
    from workloads import configs as W
    p = W.stress_geometry(n_histories=N, n_batches=B) if name == "stress" else W.get_config(name, n_histories=N, n_batches=B)
    o, g = _pair(M, p, TECHS[tech], scheduler=scheduler)
    _compare(o, g, rtol_bins=1e-7)
    g.close()


def test_population_control_needs_whole_batches_per_slot(M):
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=4000, n_batches=1)
    g = M.Problem(p, max_histories_per_subbatch=1000, max_batches_in_flight=2)
    g.set_technique(population_control=True)
    with pytest.raises(M.McdcError) as e:
        g.run()
    assert e.value.code == -1
    g.set_technique()                                      # back to analog: the same handle runs again
    g.run()
    assert g.counters()["vr_gain"] == 0.0
    with pytest.raises(M.McdcError):
        g.set_technique(wr_threshold=1.0, wr_survive=0.5)
    g.close()


def test_state_export_sum_import_equals_the_single_run(M):
    """NEXT-3 on one device: two handles run the two halves of the history range (what two ranks would do), their
    exported accumulators are added (what the all-reduce does) and imported into a third handle."""
    import torch
    from workloads import configs as W
    from paper_2409_04668_b200.sharding import shard_range
    N, B = 60_000, 12
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    whole = M.Problem(p); whole.run()
    parts = []
    for r in range(2):
        first, n, nb = shard_range(N, 2, r, n_batches=B)
        h = M.Problem(p); h.run(n, p.seed, nb, first_history_id=first)
        parts.append(h)
    n = whole.state_size()
    assert n == 2 * p.n_bins + 2 * p.n_census + 20
    dev = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in parts]
    for h, b in zip(parts, dev):
        h.state_export(b)
    host = torch.empty(n, dtype=torch.float64)
    parts[0].state_export(host)
    assert torch.equal(host, dev[0].cpu())                 # host and device buffers carry the same vector
    with pytest.raises(M.McdcError):
        parts[0].state_export(torch.empty(n - 1, dtype=torch.float64))
    merged = M.Problem(p)
    merged.state_import(dev[0] + dev[1])
    mw, sw = whole.tallies(); mm, sm = merged.tallies()
    assert np.allclose(mm, mw, rtol=1e-13, atol=0) and np.allclose(sm, sw, rtol=1e-9, atol=1e-18)
    cw, cm = whole.counters(), merged.counters()
    for k in ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "histories", "segments",
              "collisions", "surf_hits", "census_events", "children", "batches"):
        assert cm[k] == cw[k], k
    assert np.array_equal(whole.census()[1], merged.census()[1])
    # all_reduce on a single rank (no process group) is the identity
    before = whole.tallies()[0].copy()
    whole.all_reduce()
    assert np.array_equal(whole.tallies()[0], before)
    for h in parts + [whole, merged]:
        h.close()


@pytest.mark.parametrize("scheduler", [0, 1])
def test_population_control_to_a_target_beyond_the_bank_reports_overflow(M, scheduler):
    """A control target far above what the census bank of a batch holds makes the control append more copies than fit:
    the run must answer MCDC_ERR_BANK_OVERFLOW (device flag, no host read inside the census loop), not write past the bank."""
    from workloads import configs as W
    p = W.config3_pin_lattice(n_histories=4000, n_batches=2)
    g = M.Problem(p)
    g.set_technique(population_control=True, pc_target=400 * 2000)
    with pytest.raises(M.McdcError) as e:
        g.run(scheduler=scheduler)
    assert e.value.code == -6
    g.set_technique(population_control=True)                # the handle is still usable
    g.reset(); g.run(scheduler=scheduler)
    c = g.counters()
    assert c["histories"] == 4000 and c["lost"] == 0.0
    g.close()


@pytest.mark.parametrize("scheduler", [0, 1])
def test_control_that_splits_every_particle_appends_copies_in_place(M, scheduler):
    """A target of three times the batch: every arrival becomes about three particles at every census, so the in-place
    control of the history kernel appends twice the arrivals behind them (and the next launch reads them there)."""
    from workloads import configs as W
    p = W.config3_pin_lattice(n_histories=20_000, n_batches=10)
    o, g = _pair(M, p, dict(population_control=True, pc_target=3 * 2000), scheduler=scheduler, max_histories_per_subbatch=6 * 20_000)   # (banks sized for the tripled population)
    c = g.counters()
    assert c["pc_added"] > 2 * c["pc_removed"] and c["pc_added"] > 20_000
    _compare(o, g, 1e-7)
    g.close()


@pytest.mark.timeout(900)
def test_all_techniques_at_a_million_histories(M):
    """Config 3 with implicit capture, roulette and population control at 1e6 histories in 100 batches: every warp of the
    launch refills from the banks (chunked reservations, holes of the in-place control) and parks into them; integer
    counts exact, ledger and census weights to rounding, tallies to 1e-7 (the oracle takes ~30 s on one core)."""
    from workloads import configs as W
    p = W.config3_pin_lattice(n_histories=1_000_000, n_batches=100)
    o, g = _pair(M, p, TECHS["all"], scheduler=0)
    assert g.kernel_info().startswith("k_warp<1,1,2,1,512>")
    _compare(o, g, 1e-7)
    g.close()
