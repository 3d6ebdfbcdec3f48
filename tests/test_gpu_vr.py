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


def _vanishing_weight_problem():
    """One-group absorber (Sigma_c / Sigma_t = 0.9, no fission) under implicit capture without roulette, first census at
    t = 60: a history has had Poisson(60) collisions by then and weighs 0.1^collisions, below 2^-40 from the 13th on
    (P(fewer) ~ 1e-14), so every arrival truncates to 0 in the control's 2^-40 fixed-point sum."""
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=4000, n_batches=4, n_time=2, t_end=120.0)
    p.sigma_s = np.array([[[0.1]]]); p.sigma_c = np.array([[0.9]]); p.sigma_f = np.array([[0.0]]); p.nu = np.array([[0.0]])
    return p


@pytest.mark.parametrize("scheduler", [0, 1])
def test_population_control_of_a_batch_whose_weight_sums_to_zero_empties_the_bank(M, scheduler):
    """Appendix G.3 with W = 0: the oracle's control returns an empty bank and touches no counter.  The out-of-place
    kernel does the same by construction; the in-place one (scheduler 0: k_warp in census-step mode) has to mark every
    arrival as a hole, else the next launch transports them on."""
    p = _vanishing_weight_problem()
    o, g = _pair(M, p, dict(implicit_capture=True, population_control=True), scheduler=scheduler)
    wo, no = o.census()
    assert no[0] == p.n_histories and no[1] == 0 and 0.0 < wo[0] < p.n_histories * 2.0 ** -40     # the case is the one meant
    assert o.counters()["pc_removed"] == 0 and o.census_after()[1][0] == 0
    _compare(o, g, rtol_bins=1e-9)
    g.close()


def test_census_step_mode_stops_queueing_once_the_population_has_died_out(M):
    """A pure absorber with census every 20 mean free paths: no history reaches the first census (e^-20 each), and 399
    more census steps follow.  The census-step loop looks at the live counts every 16 steps (one snapshot late) and stops:
    same results as the oracle's full loop, a small fraction of its 400 x 3 launches."""
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=4000, n_batches=4, n_time=400, t_end=8000.0)
    p.sigma_s = np.array([[[0.0]]]); p.sigma_c = np.array([[1.0]]); p.sigma_f = np.array([[0.0]]); p.nu = np.array([[0.0]])
    o, g = _pair(M, p, dict(population_control=True), scheduler=0)
    assert "k_warp<" in g.kernel_info() and o.census()[1].sum() == 0
    _compare(o, g, rtol_bins=1e-9)
    assert g.counters()["kernel_launches"] <= 3 * 40, g.counters()["kernel_launches"]
    g.close()


def test_census_step_mode_keeps_a_full_pool_with_thousands_of_census_times(M):
    """K = 4000 census times: the block's census-weight array is K doubles.  The census-step variant sums census weight in
    registers and uses one copy of it, not the four of the weighted history kernel (which would leave ~40 pool slots per
    warp and switch table staging off)."""
    from workloads import configs as W
    # (8 batches: with 2 the batch variance of a bin is the difference of two nearly equal numbers, and the sdev bar of
    # _compare then measures summation order, not the method)
    p = W.config0_infinite_medium(n_histories=4000, n_batches=8, n_time=4000, t_end=20.0)
    o, g = _pair(M, p, dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0, population_control=True), scheduler=0)
    info = g.kernel_info()
    slots = int(next(t for t in info.split() if t.startswith("pool_slots=")).split("=")[1])
    assert "k_warp<" in info and slots >= 80, info
    _compare(o, g, rtol_bins=1e-9)
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
    # ... and the far side of the reduction against the ORACLE's run of the whole range (not only against this library's
    # own single run): mean / sdev at the bars of tests/test_gpu_parity.py, ledger and populations exactly
    from oracle import Oracle
    o = Oracle(p); o.run(N, p.seed, n_batches=B)
    mo, so = o.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mm - mo) <= 1e-7 * np.maximum(np.abs(mo), np.abs(mm)) + 1e-13 * scale)
    assert np.allclose(sm, so, rtol=1e-6, atol=1e-12 * scale)
    err = np.sqrt(so ** 2 + sm ** 2) + 1e-12 * scale
    assert np.all(np.abs(mm - mo) <= 4.0 * err) and mm.sum() == pytest.approx(mo.sum(), rel=1e-3)
    co, cmg = o.counters(), merged.counters()
    for k in REAL_LEDGER + INT_COUNTS:
        assert cmg[k] == co[k], (k, cmg[k], co[k])
    wo, no = o.census(); wm, nm = merged.census()
    assert np.array_equal(no, nm) and np.array_equal(wo, wm)
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


def test_exported_state_vector_has_the_layout_the_header_documents(M):
    """include/mcdc.h: after the tallies and populations come ledger[9], counts[9], histories, batches.  Read segments,
    vr_gain and pc_added (and their neighbours) at the documented offsets of a run in which none of them is zero."""
    import torch
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=8000, n_batches=4)
    g = M.Problem(p); g.set_technique(**TECHS["all"]); g.run()
    v = torch.empty(g.state_size(), dtype=torch.float64)
    g.state_export(v)
    v = v.numpy()
    T = 2 * p.n_bins + 2 * p.n_census
    assert v.size == T + 20
    c = g.counters()
    s, q = g.tally_sums()
    assert np.array_equal(v[:p.n_bins], s.ravel()) and np.array_equal(v[p.n_bins:2 * p.n_bins], q.ravel())
    w, n = g.census()
    assert np.array_equal(v[2 * p.n_bins:2 * p.n_bins + p.n_census], w) and np.array_equal(v[T - p.n_census:T], n.astype(np.float64))
    for i, k in enumerate(REAL_LEDGER):
        assert v[T + i] == c[k], (k, i)
    for i, k in enumerate(("histories", "segments", "collisions", "surf_hits", "census_events", "children", "lost_n",
                           "pc_removed", "pc_added")):
        assert v[T + 9 + i] == c[k], (k, i)
    assert v[T + 7] == c["vr_gain"] > 0 and v[T + 10] == c["segments"] > 0 and v[T + 17] == c["pc_added"] > 0
    assert v[T + 18] == p.n_histories and v[T + 19] == p.n_batches
    g.close()


def test_one_rank_nccl_all_reduce_of_the_exported_state_is_the_identity_and_matches_the_oracle(M):
    """NCCL with one rank: the first time ncclAllReduce touches the device buffer that mcdc_state_export fills and
    mcdc_state_import reads back (multi-GPU boxes do not exist in this pool).  The state must come back unchanged and
    still be the oracle's."""
    import socket
    import torch
    import torch.distributed as dist
    from oracle import Oracle
    from workloads import configs as W
    p = W.config3_pin_lattice(n_histories=40_000, n_batches=8)
    g = M.Problem(p); g.run()
    before = torch.empty(g.state_size(), dtype=torch.float64, device="cuda"); g.state_export(before)
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0)); port = sk.getsockname()[1]
    dist.init_process_group("nccl", init_method=f"tcp://127.0.0.1:{port}", world_size=1, rank=0, device_id=torch.device("cuda:0"))
    try:
        assert dist.get_backend() == "nccl"
        g.all_reduce()
        torch.cuda.synchronize()
    finally:
        dist.destroy_process_group()
    after = torch.empty_like(before); g.state_export(after)
    assert torch.equal(before, after)
    o = Oracle(p); o.run(p.n_histories, p.seed, n_batches=p.n_batches)
    mo, so = o.tallies(); mg, sg = g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= 1e-7 * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)
    assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * scale)
    co, cg = o.counters(), g.counters()
    for k in REAL_LEDGER + INT_COUNTS:
        assert cg[k] == co[k], (k, cg[k], co[k])
    g.close()


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
