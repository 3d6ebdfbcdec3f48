"""GPU parity for general CSG regions (DESIGN.md Appendix J): mcdc_problem_create_csg against
the oracle on the union / complement geometry -- integer event counts per history bit-exact, tallies to 1e-7, and
the closed form of pin J-b through the GPU path."""
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
@pytest.mark.parametrize("tech", [None, dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0),
                                  dict(implicit_capture=True, wr_threshold=0.25, wr_survive=1.0, population_control=True)])
def test_union_and_complement_cells_match_the_oracle(M, tech, scheduler):
    from oracle import Oracle
    from workloads import configs as W
    N, B = 120_000, 12
    p = W.csg_union_geometry(n_histories=N, n_batches=B)
    o = Oracle(p); g = M.Problem(p)
    assert g.info()["warp_kernel_ok"] == 1                 # regions run on the history kernel too (its RGN instantiations)
    o.enable_collision_tally(); g.enable_collision_tally()
    if tech:
        o.set_technique(**tech); g.set_technique(**tech)
    o.run(N, p.seed, n_batches=B, record_history_events=True)
    g.run(record_history_events=True, scheduler=scheduler)
    assert g.kernel_info().startswith("k_transport" if scheduler else "k_warp<1,1,%d,0,512,rgn>" %
                                      (2 if tech and tech.get("population_control") else 1))
    co, cg = o.counters(), g.counters()
    for k in COUNTS:
        assert cg[k] == co[k], (k, cg[k], co[k])
    for k in LEDGER:
        assert cg[k] == pytest.approx(co[k], rel=1e-10), k
    assert cg["lost"] == 0.0
    assert np.all(o.history_events() == g.history_events(), axis=1).mean() >= 0.99999
    for (mo, so), (mg, sg) in ((o.tallies(), g.tallies()), (o.collision_tallies(), g.collision_tallies())):
        scale = np.abs(mo).max()
        assert np.all(np.abs(mg - mo) <= 1e-7 * np.maximum(np.abs(mo), np.abs(mg)) + 1e-13 * scale)
        assert np.allclose(sg, so, rtol=1e-6, atol=1e-12 * scale)
    g.close()


def test_beam_through_the_union_closed_form_on_the_gpu(M):
    from workloads import configs as W
    N = 200_000
    p = W.csg_union_geometry(n_histories=N, n_batches=10, beam=True)
    g = M.Problem(p); g.run()
    assert g.kernel_info().startswith("k_warp<1,0,0,0,512,rgn>")
    c = g.counters()
    t_exact = np.exp(-6.5)                                 # union of the two spheres along the axis: x = 1 .. 7.5
    assert c["leak"] / N == pytest.approx(t_exact, abs=4.5 * np.sqrt(t_exact * (1 - t_exact) / N))
    assert c["capture"] + c["leak"] == N and c["lost"] == 0.0
    g.close()


def test_malformed_regions_are_refused(M):
    from workloads import configs as W
    p = W.csg_union_geometry(n_histories=100, n_batches=1)
    for off, tok in (([0, 2, 2, 2], [0, 1]), ([0, 2, 2, 2], [0, -2]), ([0, 3, 3, 3], [0, 5, -2]), ([0, 3, 3, 3], [0, 1, -7]),
                     ([1, 3, 3, 3], [0, 0, 1, -2])):
        with pytest.raises(M.McdcError) as e:
            M.mcdc_problem_create_csg(p, off, tok + [0])
        assert e.value.code == -3
    h = M.mcdc_problem_create_csg(p, [0, 0, 0, 0], [0])    # no expression anywhere: plain intersections
    M.mcdc_problem_destroy(h)
