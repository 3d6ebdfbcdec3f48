"""GPU parity for the k-eigenvalue mode (DESIGN.md Appendix H): mcdc_run_eigenvalue against
the oracle's generation loop on the same seeded inputs.  Unit weights: k per generation, integer counts and census
counts are exact; tallies to 1e-9."""
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


def _both(M, p, N, n_in, n_act, tech=None):
    from oracle import Oracle
    o = Oracle(p); g = M.Problem(p, max_histories_per_subbatch=N, max_batches_in_flight=1, workspace_scale=2.0)
    if tech:
        o.set_technique(**tech); g.set_technique(**tech)
    ko = o.run_eigenvalue(N, p.seed, n_in, n_act)
    kg = g.run_eigenvalue(N, p.seed, n_in, n_act)
    return o, g, ko, kg


def _compare(o, g, ko, kg, exact=True):
    if exact:
        assert np.array_equal(ko, kg), (ko, kg)
    else:
        assert np.allclose(ko, kg, rtol=1e-10)
    co, cg = o.counters(), g.counters()
    # (counters()["histories"] counts generated source histories on the device: N here, not N x active generations)
    for k in ("batches", "collisions", "surf_hits", "census_events", "children", "pc_removed", "pc_added"):
        assert cg[k] == co[k], (k, cg[k], co[k])
    mo, so = o.tallies(); mg, sg = g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= 1e-9 * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)
    assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * scale)
    wo, no = o.census_after(); wg, ng = g.census_after()
    assert np.array_equal(no, ng) and np.allclose(wo, wg, rtol=1e-12)


def test_infinite_medium_k_matches_the_oracle_and_the_closed_form(M):
    from workloads import configs as W
    p = W.as_eigenvalue(W.config0_infinite_medium(n_histories=20000, n_batches=1))
    o, g, ko, kg = _both(M, p, 20000, 3, 17)
    _compare(o, g, ko, kg)
    assert abs(kg.mean() - 0.8) < 4.0 * np.sqrt(0.96 / 20000 / 20)      # pin H-a through the GPU path
    g.close()


def test_bare_slab_first_generation(M):
    from scipy.special import expn
    from workloads import configs as W
    N = 200_000
    p = W.bare_slab_absorber(thickness=2.0, n_histories=N)
    o, g, ko, kg = _both(M, p, N, 0, 2)
    _compare(o, g, ko, kg)
    p_esc = (0.5 - expn(3, 2.0)) / 2.0
    assert abs(kg[0] - 2.5 * 0.4 * (1 - p_esc)) < 4.0 * np.sqrt((6.5 * 0.4 * (1 - p_esc)) / N)   # pin H-b
    g.close()


@pytest.mark.parametrize("name,N,n_in,n_act", [("config3", 30_000, 3, 5), ("config1", 20_000, 2, 4), ("stress", 20_000, 1, 3)])
def test_lattice_slab_and_stress_geometry(M, name, N, n_in, n_act):
    from workloads import configs as W
    base = W.stress_geometry(n_histories=N, n_batches=1) if name == "stress" else W.get_config(name, n_histories=N, n_batches=1)
    p = W.as_eigenvalue(base)
    o, g, ko, kg = _both(M, p, N, n_in, n_act)
    _compare(o, g, ko, kg)
    g.close()


def test_eigenvalue_with_implicit_capture_and_roulette(M):
    from workloads import configs as W
    p = W.as_eigenvalue(W.config3_pin_lattice(n_histories=20_000, n_batches=1))
    o, g, ko, kg = _both(M, p, 20_000, 2, 4, tech=dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0))
    _compare(o, g, ko, kg, exact=False)
    g.close()


def test_argument_checks(M):
    from workloads import configs as W
    p = W.as_eigenvalue(W.config0_infinite_medium(n_histories=1000, n_batches=1))
    g = M.Problem(p, max_histories_per_subbatch=1000, max_batches_in_flight=1)
    with pytest.raises(M.McdcError):
        g.run_eigenvalue(1000, 1, 0, 0)
    g.set_technique(population_control=True)
    with pytest.raises(M.McdcError):
        g.run_eigenvalue(1000, 1, 1, 1)
    g.set_technique()
    with pytest.raises(M.McdcError):
        g.run_eigenvalue(5000, 1, 1, 1)                    # more particles than the workspace was bound for
    k = g.run_eigenvalue(1000, 1, 1, 2)
    assert k.shape == (3,) and np.all(k > 0)
    g.close()
