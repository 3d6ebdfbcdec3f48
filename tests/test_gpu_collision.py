"""GPU parity for the collision-estimator tally of the paper's Fig. 3 (DESIGN.md Appendix I):
every bin against the oracle on the same seeded inputs, on both schedulers, with and without the techniques, and in
the k-eigenvalue mode.  The track-length tally must be unchanged by switching it on."""
import numpy as np
import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(600)]


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2409_04668_b200 as M
    M.lib()
    return M


def _close(a, b, rtol):
    scale = np.abs(a).max()
    return np.all(np.abs(a - b) <= rtol * np.maximum(np.abs(a), np.abs(b)) + 1e-13 * scale)


@pytest.mark.parametrize("scheduler", [0, 1])
@pytest.mark.parametrize("name,N,B,tech", [
    ("config0", 40_000, 20, None), ("config1", 100_000, 20, None), ("config1a", 100_000, 10, None),
    ("config2", 100_000, 10, None), ("config3", 60_000, 20, None), ("stress", 120_000, 12, None),
    ("config3", 40_000, 20, dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0)),
    ("config0", 40_000, 20, dict(implicit_capture=True, wr_threshold=0.3, wr_survive=0.6, population_control=True))])
def test_collision_tally_matches_the_oracle(M, name, N, B, tech, scheduler):
    from oracle import Oracle
    from workloads import configs as W
    p = W.stress_geometry(n_histories=N, n_batches=B) if name == "stress" else W.get_config(name, n_histories=N, n_batches=B)
    o = Oracle(p); o.enable_collision_tally()
    g = M.Problem(p); g.enable_collision_tally()
    if tech:
        o.set_technique(**tech); g.set_technique(**tech)
    o.run(N, p.seed, n_batches=B)
    g.run(scheduler=scheduler)
    mo, so = o.collision_tallies(); mg, sg = g.collision_tallies()
    assert mo.sum() > 0
    assert _close(mo, mg, 1e-9 if name == "config0" else 1e-7)
    assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * np.abs(mo).max())
    to, _ = o.tallies(); tg, _ = g.tallies()
    assert _close(to, tg, 1e-7)
    assert g.counters()["collisions"] == o.counters()["collisions"]
    if name == "config0" and tech is None:                 # pin I-a through the GPU path: Sigma_t = 1, unit weights
        assert mg.sum() * N == pytest.approx(g.counters()["collisions"], rel=1e-12)
    g.close()


def test_switching_it_on_leaves_the_track_length_tally_bitwise_alone_and_off_is_the_default(M):
    from workloads import configs as W
    p = W.config3_pin_lattice(n_histories=50_000, n_batches=10)
    a = M.Problem(p); a.run()
    with pytest.raises(M.McdcError):
        a.collision_tallies()                              # never enabled: nothing to report
    b = M.Problem(p); b.enable_collision_tally(); b.run()
    sa, qa = a.tally_sums(); sb, qb = b.tally_sums()
    assert np.allclose(sa, sb, rtol=1e-12, atol=0) and a.counters()["segments"] == b.counters()["segments"]
    b.reset(); b.enable_collision_tally(False); b.run()
    assert b.collision_tallies()[0].sum() == 0.0
    a.close(); b.close()


def test_collision_tally_in_the_eigenvalue_mode(M):
    from oracle import Oracle
    from workloads import configs as W
    N = 20_000
    p = W.as_eigenvalue(W.config3_pin_lattice(n_histories=N, n_batches=1))
    o = Oracle(p); o.enable_collision_tally()
    g = M.Problem(p, max_histories_per_subbatch=N, max_batches_in_flight=1, workspace_scale=2.0); g.enable_collision_tally()
    ko = o.run_eigenvalue(N, p.seed, 2, 4); kg = g.run_eigenvalue(N, p.seed, 2, 4)
    assert np.array_equal(ko, kg)
    mo, so = o.collision_tallies(); mg, sg = g.collision_tallies()
    assert _close(mo, mg, 1e-9) and np.allclose(sg, so, rtol=1e-6, atol=1e-12 * np.abs(mo).max())
    g.close()
