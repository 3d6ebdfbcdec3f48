"""GPU parity for universes / lattices (DESIGN.md Appendix K): mcdc_problem_create_lattice
against the oracle (which expands the same description with its own code) on the mixed lattice, and config 3 given
as a lattice against config 3 written out by hand."""
import numpy as np
import pytest

pytestmark = [pytest.mark.gpu, pytest.mark.timeout(600)]

LEDGER = ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost")
COUNTS = ("histories", "segments", "collisions", "surf_hits", "census_events", "children", "lost_n", "batches")


@pytest.fixture(scope="module")
def M():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2409_04668_b200 as M
    M.lib()
    return M


@pytest.mark.parametrize("scheduler", [0, 1])
@pytest.mark.parametrize("tech", [None, dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0, population_control=True)])
def test_mixed_lattice_matches_the_oracle(M, tech, scheduler):
    from oracle import Oracle
    from workloads import configs as W
    N, B = 120_000, 12
    p = W.lattice_mixed(n_histories=N, n_batches=B)
    o = Oracle(p); g = M.Problem(p)
    info = g.info()
    assert info["warp_kernel_ok"] == 1 and info["cells"] == o.prob.n_cells == 27
    if tech:
        o.set_technique(**tech); g.set_technique(**tech)
    o.run(N, p.seed, n_batches=B, record_history_events=True)
    g.run(record_history_events=True, scheduler=scheduler)
    co, cg = o.counters(), g.counters()
    for k in COUNTS:
        assert cg[k] == co[k], (k, cg[k], co[k])
    for k in LEDGER:
        assert cg[k] == pytest.approx(co[k], rel=1e-10), k
    assert cg["lost"] == 0.0
    assert np.all(o.history_events() == g.history_events(), axis=1).mean() >= 0.99999
    (mo, so), (mg, sg) = o.tallies(), g.tallies()
    scale = np.abs(mo).max()
    assert np.all(np.abs(mg - mo) <= 1e-7 * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)
    assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * scale)
    wo, no = o.census(); wg, ng = g.census()
    assert np.array_equal(no, ng)
    g.close()


def test_config3_as_a_lattice_is_config3(M):
    """The same tables (tests/test_lattice_host.py) give the same derived structure and the same run."""
    from workloads import configs as W
    N, B = 200_000, 20
    a = M.Problem(W.config3_pin_lattice(n_histories=N, n_batches=B))
    b = M.Problem(W.config3_lattice(n_histories=N, n_batches=B))
    assert a.info() == b.info() and b.info()["all_one_bin"] == 1 and b.info()["certified_halfspaces"] == 1666
    a.run(record_history_events=True); b.run(record_history_events=True)
    assert a.kernel_info().split(" queue_children")[0] == b.kernel_info().split(" queue_children")[0]   # (that count depends on timing)
    assert np.array_equal(a.history_events(), b.history_events())
    ca, cb = a.counters(), b.counters()
    for k in COUNTS + LEDGER:
        assert ca[k] == cb[k], k
    (ma, _), (mb, _) = a.tallies(), b.tallies()
    assert np.allclose(ma, mb, rtol=1e-12, atol=0.0)       # same trajectories; the REDs land in any order
    a.close(); b.close()
