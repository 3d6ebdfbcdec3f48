"""Pins of the oracle's universe / lattice expansion (DESIGN.md Appendix K; oracle/lattice.py).
K-a the config-3 lattice description expands to exactly the 578 hand-written cells of config 3 (two independently
    written generators), and its transport equals config 3's bit for bit;
K-b point location in a lattice that starts off the origin, with unequal pitches and three different universes, equals
    the membership written out directly here (i = floor((x - x0) / px), local circle / ball tests);
K-c the translated quadric evaluates to f(r - c);
K-d transport through the mixed lattice: exact balance, nothing lost, order independence;
K-e malformed descriptions are refused."""
import copy

import numpy as np
import pytest

from oracle import Oracle, expand_lattice, translate_quadric
from workloads import configs as W


def test_Ka_config3_lattice_expands_to_the_hand_written_cells():
    hand = W.config3_pin_lattice(n_histories=2000, n_batches=4)
    lat = W.config3_lattice(n_histories=2000, n_batches=4)
    e = expand_lattice(lat.meta["lattice"])
    for k in ("surf_coef", "surf_bc", "cell_offset", "hs_surface", "hs_sense", "cell_material"):
        a, b = np.asarray(getattr(hand, k)), e[k]
        assert a.shape == b.shape and a.dtype == b.dtype and a.tobytes() == b.tobytes(), k
    o1, o2 = Oracle(hand), Oracle(lat)
    o1.run(2000, hand.seed, n_batches=4, record_history_events=True)
    o2.run(2000, lat.seed, n_batches=4, record_history_events=True)
    assert np.array_equal(o1.history_events(), o2.history_events())
    assert o1.tallies()[0].tobytes() == o2.tallies()[0].tobytes()


def _direct_cell(r):
    """Cell id of a point in W.lattice_mixed, from the definition: element (i, j), then the universe's own cells."""
    L = W.LATTICE_MIXED
    fill = [[0, 1, 2, 0], [2, 0, 0, 1], [0, 2, 1, 0]]
    n_cells = {0: 3, 1: 1, 2: 2}
    if not (L["z_lo"] < r[2] < L["z_hi"]):
        return -1
    i = int(np.floor((r[0] - L["x0"]) / L["pitch_x"])); j = int(np.floor((r[1] - L["y0"]) / L["pitch_y"]))
    if not (0 <= i < L["nx"] and 0 <= j < L["ny"]):
        return -1
    base = sum(n_cells[fill[jj][ii]] for jj in range(L["ny"]) for ii in range(L["nx"]) if (jj, ii) < (j, i))
    lx = r[0] - (L["x0"] + (i + 0.5) * L["pitch_x"]); ly = r[1] - (L["y0"] + (j + 0.5) * L["pitch_y"])
    u = fill[j][i]
    if u == 0:
        rho2 = lx * lx + ly * ly
        return base + (0 if rho2 < L["r_fuel"] ** 2 else 1 if rho2 < L["r_clad"] ** 2 else 2)
    if u == 1:
        return base
    bx, by, bz, br = L["ball"]
    return base + (0 if (lx - bx) ** 2 + (ly - by) ** 2 + (r[2] - bz) ** 2 < br * br else 1)


def test_Kb_location_in_the_mixed_lattice_equals_the_direct_formula():
    p = W.lattice_mixed(n_histories=100, n_batches=1)
    o = Oracle(p)
    L = W.LATTICE_MIXED
    assert o.prob.n_cells == sum({0: 3, 1: 1, 2: 2}[u] for row in p.meta["lattice"]["fill"] for u in row)
    rng = np.random.default_rng(11)
    seen = set()
    for _ in range(6000):
        r = np.array([rng.uniform(L["x0"] - 0.3, L["x0"] + L["nx"] * L["pitch_x"] + 0.3),
                      rng.uniform(L["y0"] - 0.3, L["y0"] + L["ny"] * L["pitch_y"] + 0.3),
                      rng.uniform(L["z_lo"] - 0.2, L["z_hi"] + 0.2)])
        want = _direct_cell(r)
        assert o.locate(r, [0.3, 0.5, 0.81]) == want, r
        seen.add(want)
    assert seen == set(range(-1, o.prob.n_cells))              # every cell of every element was hit, and the outside
    # materials follow the universes
    mats = {0: [0, 1, 2], 1: [2], 2: [0, 2]}
    assert list(o.prob.cell_material) == [m for row in p.meta["lattice"]["fill"] for u in row for m in mats[u]]
    # boundary conditions sit on the outer planes only
    bc = o.prob.surf_bc
    nx, ny = L["nx"], L["ny"]
    assert list(bc[:nx + 1]) == [1, 0, 0, 0, 1] and list(bc[nx + 1:nx + ny + 2]) == [2, 0, 0, 2]
    assert list(bc[nx + ny + 2:nx + ny + 4]) == [2, 1] and not bc[nx + ny + 4:].any()


def test_Kc_translated_quadric_is_f_of_r_minus_c():
    rng = np.random.default_rng(3)
    for _ in range(50):
        coef = rng.normal(size=10); c = rng.normal(size=3) * 3
        t = translate_quadric(coef, c)

        def f(q, r):
            x, y, z = r
            return (q[0] * x * x + q[1] * y * y + q[2] * z * z + q[3] * x * y + q[4] * x * z + q[5] * y * z + q[6] * x +
                    q[7] * y + q[8] * z + q[9])
        for _ in range(5):
            r = rng.normal(size=3) * 4
            assert f(t, r) == pytest.approx(f(coef, r - c), rel=1e-12, abs=1e-10)
    # the pin of config 3: a local z-cylinder moved to (x0, y0) is W.cylinder_z(x0, y0, r) to the last bit
    assert translate_quadric(W.cylinder_z(0.0, 0.0, 0.54), (3.5 * 1.26, 7.5 * 1.26, 0.0)).tobytes() == \
        W.cylinder_z(3.5 * 1.26, 7.5 * 1.26, 0.54).tobytes()


def test_Kd_transport_through_the_mixed_lattice_balances_and_is_order_independent():
    p = W.lattice_mixed(n_histories=6000, n_batches=6)
    o = Oracle(p)
    o.run(6000, p.seed, n_batches=6, record_history_events=True)
    c = o.counters()
    assert c["lost"] == 0.0 and c["lost_n"] == 0
    assert c["source"] + c["production"] == c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"]
    assert c["leak"] > 0 and c["surf_hits"] > 3 * c["histories"]
    ev = o.history_events().copy()
    o2 = Oracle(p)
    o2.run(3000, p.seed, n_batches=3, first_history_id=3000, record_history_events=True)
    assert np.array_equal(o2.history_events(), ev[3000:])       # a later range alone = the same histories
    # flux appears in every material region that the source covers
    m, _ = o.tallies()
    assert (m.sum(axis=(0, 1)) > 0).all()


def test_Ke_malformed_lattices_are_refused():
    base = W.lattice_mixed(n_histories=10, n_batches=1).meta["lattice"]
    for edit in (lambda l: l.__setitem__("fill", [[0, 1, 2, 3], [2, 0, 0, 1], [0, 2, 1, 0]]),     # universe 3 does not exist
                 lambda l: l.__setitem__("fill", [[0, 1, 2, 0], [2, 0, 0, 1]]),                   # not [ny][nx]
                 lambda l: l.__setitem__("pitch_x", 0.0),
                 lambda l: l.__setitem__("z_hi", l["z_lo"]),
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([(0, +1)], 2)),             # local surface 0 of a universe without surfaces
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([(-7, +1)], 2)),            # unknown face code
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([(-1, 0)], 2)),             # sense 0
                 lambda l: l["universes"][1]["cells"].__setitem__(0, ([], 2))):                   # empty cell
        lat = copy.deepcopy(base)
        edit(lat)
        with pytest.raises(ValueError):
            expand_lattice(lat)
