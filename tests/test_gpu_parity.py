"""GPU parity tests: libmcdc.so (through the C ABI binding) against the oracle, element by element on the
same seeded inputs.  Bars (BASELINE.json north_star): config 0 -- per-history integer event counts
bit-exact for >= 99.999 % of histories and every tally bin within 1e-9 relative; larger configs -- every
bin within |z| <= 4 combined standard errors and the integrated flux within 1e-3 (we also hold them to the
much tighter bound the shared trajectories allow)."""
import numpy as np
import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(300)]

LEDGER = ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost")
COUNTS = ("histories", "segments", "collisions", "surf_hits", "census_events", "children", "lost_n", "batches")


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2409_04668_b200 as M
    M.lib()                       # fails loudly if libmcdc.so is missing
    return M


def _pair(M, p, record=True, scheduler=0, **gkw):
    from oracle import Oracle
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=p.n_batches, record_history_events=record)
    g = M.Problem(p, **gkw)
    g.run(record_history_events=record, scheduler=scheduler)
    return o, g


def _check_counters(o, g, exact=True):
    co, cg = o.counters(), g.counters()
    for k in LEDGER + COUNTS:
        if exact:
            assert cg[k] == co[k], (k, cg[k], co[k])
    assert cg["source"] + cg["production"] == cg["capture"] + cg["fission_abs"] + cg["leak"] + cg["census_final"] + cg["lost"]
    assert cg["segments"] == cg["collisions"] + cg["surf_hits"] + cg["census_events"]
    return co, cg


def _check_tallies(o, g, rtol, official=True):
    mo, so = o.tallies(); mg, sg = g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= rtol * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)      # D26
    assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * scale)
    if official:
        err = np.sqrt(so ** 2 + sg ** 2) + 1e-12 * scale
        assert np.abs(mg - mo).max() <= 4.0 * err.max() and np.all(np.abs(mg - mo) <= 4.0 * err)
        assert mg.sum() == pytest.approx(mo.sum(), rel=1e-3)


@pytest.mark.parametrize("scheduler", [0, 1])
def test_config0_bit_exact_event_counts_and_1e9_tallies(M, scheduler):
    from workloads import configs as W
    p = W.config0_infinite_medium()                     # 1e5 histories, 20 batches: BASELINE config 0 as stated
    o, g = _pair(M, p, scheduler=scheduler)
    _check_counters(o, g)
    eo, eg = o.history_events(), g.history_events()
    same = np.all(eo == eg, axis=1).mean()
    assert same >= 0.99999
    _check_tallies(o, g, rtol=1e-9)
    wo, no = o.census(); wg, ng = g.census()
    assert np.array_equal(wo, wg) and np.array_equal(no, ng)
    # closed form through the GPU path as well (E1)
    mg, sg = g.tallies()
    k = np.arange(20)
    exact = (np.exp(-0.1 * k) - np.exp(-0.1 * (k + 1))) / 0.1
    assert np.abs((mg.ravel() - exact) / sg.ravel()).max() < 4.0
    g.close()


@pytest.mark.parametrize("scheduler", [0, 1])
@pytest.mark.parametrize("name,N,B", [("config1", 200_000, 20), ("config1a", 200_000, 20),
                                      ("config2", 300_000, 20), ("config3", 100_000, 20)])
def test_larger_configs_match_the_oracle(M, name, N, B, scheduler):
    from workloads import configs as W
    p = W.get_config(name, n_histories=N, n_batches=B)
    o, g = _pair(M, p, scheduler=scheduler)
    _check_counters(o, g)
    eo, eg = o.history_events(), g.history_events()
    assert np.all(eo == eg, axis=1).mean() >= 0.99999
    _check_tallies(o, g, rtol=1e-7)
    wo, no = o.census(); wg, ng = g.census()
    assert np.array_equal(no, ng) and np.allclose(wo, wg, rtol=1e-14)
    g.close()


@pytest.mark.parametrize("scheduler", [0, 1])
@pytest.mark.parametrize("N,B", [(1, 1), (31, 1), (33, 3), (257, 1), (1000, 8)])
def test_ragged_and_tiny_runs(M, N, B, scheduler):
    from workloads import configs as W
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    o, g = _pair(M, p, scheduler=scheduler)
    _check_counters(o, g)
    assert np.array_equal(o.history_events(), g.history_events())
    _check_tallies(o, g, rtol=1e-9, official=False)
    g.close()


@pytest.mark.parametrize("scheduler", [0, 1])
@pytest.mark.parametrize("covering", [False, True])
def test_stress_geometry_takes_the_slow_paths_and_still_matches(M, covering, scheduler):
    """General quadric cells, a reflective sphere, a face with two neighbours (no certified neighbour), lost source
    particles, a tally mesh that clips / is unaligned with the cells, census times off the tally time edges."""
    from workloads import configs as W
    p = W.stress_geometry(n_histories=240_000, n_batches=12, covering_mesh=covering)
    o, g = _pair(M, p, scheduler=scheduler)
    co, cg = _check_counters(o, g)
    assert cg["lost_n"] > 0 and cg["leak"] > 0 and cg["children"] > 0
    assert np.all(o.history_events() == g.history_events(), axis=1).mean() >= 0.99999
    _check_tallies(o, g, rtol=1e-9)
    wo, no = o.census(); wg, ng = g.census()
    assert np.array_equal(no, ng) and np.array_equal(wo, wg)
    g.close()


def test_sub_batching_and_split_batches_do_not_change_results(M):
    """A workspace too small for the whole run forces several sub-batches; a batch larger than a slot is split
    into pieces spread over the slots."""
    from workloads import configs as W
    p = W.config1_slab(n_histories=64_000, n_batches=16)
    o, g = _pair(M, p)
    ref_ev = g.history_events(); ref_s, ref_q = g.tally_sums(); ref_c = g.counters()
    g.close()
    for nh, nb in ((16_000, 4), (8_000, 16), (4_000, 1), (1_000, 4)):
        for scheduler in (0, 1):
            h = M.Problem(p, max_histories_per_subbatch=nh, max_batches_in_flight=nb)
            h.run(record_history_events=True, scheduler=scheduler)
            assert np.array_equal(h.history_events(), ref_ev)
            s, q = h.tally_sums()
            assert np.allclose(s, ref_s, rtol=1e-12, atol=1e-14 * np.abs(ref_s).max())
            assert np.allclose(q, ref_q, rtol=1e-11, atol=1e-14 * np.abs(ref_q).max())
            c = h.counters()
            for k in LEDGER + COUNTS:
                assert c[k] == ref_c[k], (nh, nb, scheduler, k)
            h.close()
    co = o.counters()
    for k in LEDGER + COUNTS:
        assert co[k] == ref_c[k]


def test_history_ranges_accumulate_like_one_run(M):
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=20_000, n_batches=10)
    o, g = _pair(M, p, record=False)
    s1, q1 = g.tally_sums(); c1 = g.counters()
    g.reset()
    assert g.counters()["histories"] == 0 and g.tally_sums()[0].sum() == 0.0
    g.run(8_000, p.seed, 4, first_history_id=0)
    g.run(12_000, p.seed, 6, first_history_id=8_000)
    s2, q2 = g.tally_sums(); c2 = g.counters()
    assert np.allclose(s2, s1, rtol=1e-13) and np.allclose(q2, q1, rtol=1e-12)
    for k in LEDGER + COUNTS:
        assert c1[k] == c2[k]
    # a different batch size on an accumulating handle is refused
    with pytest.raises(M.McdcError):
        g.run(1000, p.seed, 1)
    g.close()


def test_errors_are_reported_not_swallowed(M):
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=1000, n_batches=10)
    h = M.mcdc_problem_create(p)
    with pytest.raises(M.McdcError) as e:
        M.mcdc_run(h, 1000, 1)                          # no workspace bound
    assert e.value.code == -5
    with pytest.raises(M.McdcError) as e:
        M.mcdc_tallies_get(h, p.n_bins + 1)
    assert e.value.code == -4
    M.mcdc_problem_destroy(h)
    g = M.Problem(p)
    with pytest.raises(M.McdcError) as e:
        g.run(1001, p.seed, 10)                         # B does not divide N
    assert e.value.code == -1
    g.close()


def test_bank_overflow_is_detected(M):
    """A supercritical medium multiplies until a bank overflows: the run must say so."""
    from workloads import configs as W
    p = W.config0_infinite_medium(n_histories=2000, n_batches=1)
    p.sigma_f = p.sigma_f.copy(); p.sigma_c = p.sigma_c.copy(); p.nu = p.nu.copy()
    p.sigma_f[0, 0] = 0.45; p.sigma_c[0, 0] = 0.05; p.nu[0, 0] = 3.0       # c = 1.85: grows ~ e^{0.85 t}
    for scheduler in (0, 1):
        g = M.Problem(p)
        with pytest.raises(M.McdcError) as e:
            g.run(scheduler=scheduler)
        assert e.value.code == -6
        g.close()


def test_full_size_config3_sampled_against_the_oracle(M):
    """BASELINE config 3 at its full size (1e7 histories, 100 batches) in the launch configuration bench.py
    times; the oracle recomputes sampled histories one by one (trajectories depend only on seed and id)."""
    from oracle import Oracle
    from workloads import configs as W
    p = W.config3_pin_lattice()
    g = M.Problem(p)
    g.run(record_history_events=True)
    ev = g.history_events()
    c = g.counters()
    assert c["histories"] == p.n_histories and c["batches"] == p.n_batches and c["lost_n"] == 0
    assert c["source"] + c["production"] == c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"]
    assert ev[:, 0].sum() == c["collisions"] and ev[:, 1].sum() == c["surf_hits"]
    assert ev[:, 2].sum() == c["children"] and ev[:, 3].sum() == c["census_events"]
    o = Oracle(p)
    for first in (0, 4_999_700, 9_999_400):
        o.reset()
        o.run(600, p.seed, n_batches=1, first_history_id=first, record_history_events=True)
        assert np.array_equal(o.history_events(), ev[first:first + 600])
    mean, sdev = g.tallies()
    assert np.all(mean >= 0) and np.all(np.isfinite(sdev))
    # E7 on the GPU result: the 8 symmetries of the square
    m = mean[:, :, 0].sum(axis=(0, 1))
    assert np.allclose(m, m[::-1, :], rtol=0.05) and np.allclose(m, m.T, rtol=0.05)
    # (the per-bin comparison with the oracle at this size is tests/test_gpu_fullsize.py)
    g.close()


def test_certificates_one_bin_cells_and_async_only_workspace(M):
    """What problem creation derives from the geometry, and the small workspace that serves
    the asynchronous scheduler alone."""
    from workloads import configs as W
    p3 = W.config3_pin_lattice(n_histories=4000, n_batches=4)
    g = M.Problem(p3, async_only=True)
    i3 = g.info()
    # 289 moderator cells x (4 pitch planes + cylinder) + 289 fuel cylinders, minus the 68 reflective outer planes
    assert i3["transmission_halfspaces"] == 289 * 6 - 68 and i3["certified_halfspaces"] == i3["transmission_halfspaces"]
    assert i3["cells"] == 578 and i3["one_bin_cells"] == 578 and i3["warp_kernel_ok"] == 1 and i3["score_fast"] == 1
    assert i3["hot_table_bytes"] < 64 * 1024
    # every pin / moderator cell lies in one pin bin and census = time edges: the kernel without the DDA scorer;
    # the point source at the lattice centre sits strictly inside the centre pin (cell 288)
    assert i3["all_one_bin"] == 1 and i3["source_cell"] == 288
    # box sources inside one axis-aligned box cell are certified too (config 1a's beam starts ON the cell's face: the
    # cell is only a candidate there, every particle fails the strict check and takes the search)
    for cfg, one_bin, src_cell in (("config0", 1, 0), ("config1", 0, 1), ("config1a", 0, 0), ("config2", 0, None)):
        q = M.Problem(W.get_config(cfg, n_histories=1000, n_batches=1))
        iq = q.info()
        assert iq["all_one_bin"] == one_bin, (cfg, iq)
        assert iq["source_cell"] == src_cell if src_cell is not None else iq["source_cell"] >= 0, (cfg, iq)
        q.close()
    ps0 = W.stress_geometry(n_histories=1200, n_batches=12)        # source box spans several cells: nothing to certify
    q = M.Problem(ps0); assert q.info()["source_cell"] == -1; q.close()
    full = M.mcdc_workspace_size(g._h, 4000, 4)
    assert g.workspace_bytes < full
    g.run(record_history_events=True)
    ev = g.history_events()
    with pytest.raises(M.McdcError) as e:
        g.run(scheduler=1)                               # no particle banks in this workspace
    assert e.value.code == -5
    g.close()
    h = M.Problem(p3)
    h.run(record_history_events=True)
    assert np.array_equal(h.history_events(), ev)
    h.close()
    ps = W.stress_geometry(n_histories=1200, n_batches=12)
    g = M.Problem(ps)
    i_s = g.info()
    # certified: only the pin <-> its box (z-cylinder); nothing next to a sphere, nothing on the two-neighbour face
    assert 0 < i_s["certified_halfspaces"] < i_s["transmission_halfspaces"]
    assert i_s["one_bin_cells"] == 0 and i_s["score_fast"] == 0
    g.close()
    p2 = W.config2_lduct(n_histories=1000, n_batches=1)
    g = M.Problem(p2)
    i2 = g.info()
    assert i2["certified_halfspaces"] == i2["transmission_halfspaces"] > 0 and i2["one_bin_cells"] == 0
    g.close()


def test_problem_beyond_the_history_kernels_tables_falls_back_and_still_matches(M):
    """More census times than the compact particle word holds (4095): mcdc_problem_info says so, the asynchronous
    scheduler request is served by the census-stepped kernel, and the results are still the oracle's."""
    from oracle import Oracle
    from workloads import configs as W
    N, B = 6000, 6
    p = W.config0_infinite_medium(n_histories=N, n_batches=B)
    p.census_times = np.linspace(0.0, 20.0, 5001)[1:].copy()          # 5000 census steps over the same 20 s
    g = M.Problem(p)
    assert g.info()["warp_kernel_ok"] == 0
    g.run(record_history_events=True)
    assert g.kernel_info().startswith("k_transport")
    o = Oracle(p)
    o.run(N, p.seed, n_batches=B, record_history_events=True)
    co, cg = o.counters(), g.counters()
    for k in ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "collisions", "surf_hits",
              "census_events", "children"):
        assert cg[k] == co[k], (k, cg[k], co[k])
    assert np.array_equal(o.history_events(), g.history_events())
    (mo, _), (mg, _) = o.tallies(), g.tallies()
    assert np.allclose(mg, mo, rtol=1e-9, atol=1e-13 * np.abs(mo).max())
    wo, no = o.census(); wg, ng = g.census()
    assert np.array_equal(no, ng)
    g.close()


@pytest.mark.parametrize("scheduler", [0, 1])
def test_a_true_void_region_is_streamed_through(M, scheduler):
    """Sigma_t = 0 in the middle region of the slab (degenerate case of A.2: no collision distance): the history kernel
    reads 1 / Sigma_t = +inf there instead of testing Sigma_t; counts and tallies must still be the oracle's."""
    from oracle import Oracle
    from workloads import configs as W
    N, B = 60_000, 6
    p = W.config1_slab(n_histories=N, n_batches=B)
    for name in ("sigma_t", "sigma_c", "sigma_f", "nu", "chi"):
        a = getattr(p, name).copy(); a[1, :] = 0.0; setattr(p, name, a)
    s = p.sigma_s.copy(); s[1] = 0.0; p.sigma_s = s
    o = Oracle(p); g = M.Problem(p)
    o.run(N, p.seed, n_batches=B, record_history_events=True)
    g.run(record_history_events=True, scheduler=scheduler)
    co, cg = o.counters(), g.counters()
    for k in ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "collisions", "surf_hits",
              "census_events", "children"):
        assert cg[k] == co[k], (k, cg[k], co[k])
    assert co["collisions"] > 0 and co["lost"] == 0
    assert np.all(o.history_events() == g.history_events(), axis=1).mean() >= 0.99999
    (mo, _), (mg, _) = o.tallies(), g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= 1e-9 * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)
    g.close()


@pytest.mark.parametrize("scheduler", [0, 1])
def test_corner_hits_take_the_tie_break_and_the_cell_search(M, scheduler):
    """A beam along the lattice diagonal from a pin centre reaches every cell corner with two face distances that are
    equal to the last bit (D5: the earlier half-space of the cell's list wins) and a crossing point that lies on a second
    face (no certified neighbour applies: A.5's search decides).  Every history starts with such hits."""
    from oracle import Oracle
    from workloads import configs as W
    N, B = 40_000, 4
    p = W.config3_pin_lattice(n_histories=N, n_batches=B)
    p.src_dir_mode = W.DIR_FIXED
    p.src_dir = np.array([np.sqrt(0.5), np.sqrt(0.5), 0.0])
    o = Oracle(p); g = M.Problem(p)
    o.run(N, p.seed, n_batches=B, record_history_events=True)
    g.run(record_history_events=True, scheduler=scheduler)
    # Every history of this beam passes through points that lie on two planes at once, where the last bit of the moved
    # coordinate (fused multiply-add on the device, separate rounding in the oracle) can decide the
    # cell: the bar is the one of north_star for such flips -- a few histories in 1e5 may differ, nothing else.
    co, cg = o.counters(), g.counters()
    same = np.all(o.history_events() == g.history_events(), axis=1)
    assert same.mean() >= 0.9999, (~same).sum()
    for k in ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost", "collisions", "surf_hits",
              "census_events", "children"):
        assert abs(cg[k] - co[k]) <= 2e-4 * max(1.0, co[k]), (k, cg[k], co[k])
    # (a corner point whose rounded coordinates lie in no cell is lost, D13: a handful per run, on both sides)
    assert co["lost"] <= 1e-3 * N and abs(cg["lost"] - co["lost"]) <= 3
    assert cg["source"] + cg["production"] == cg["capture"] + cg["fission_abs"] + cg["leak"] + cg["census_final"] + cg["lost"]
    (mo, so), (mg, sg) = o.tallies(), g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= 4.0 * np.sqrt(so ** 2 + sg ** 2) + 1e-9 * scale)
    assert mg.sum() == pytest.approx(mo.sum(), rel=1e-3)
    # the beam really went through corners: the diagonal pins see flux that an x- or y-beam would not give them
    diag = mo.sum(axis=(0, 1))[0][np.arange(9, 17), np.arange(9, 17)]
    assert (diag > 0).all()
    g.close()
