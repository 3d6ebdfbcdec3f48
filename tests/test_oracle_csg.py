"""Pins for the oracle's general CSG regions (second half; DESIGN.md Appendix J): cells given
as postfix expressions (AND / OR / NOT) over half-spaces.  (J-a) point location agrees with membership written out by
hand for the test geometry (union of two spheres, a cylinder, the box minus both); (J-b) a beam through the union of
two overlapping absorbing spheres is attenuated over the length of the UNION along its axis, exp(-L), and the
collisions fall as exp(-x) inside it -- the intersection or either sphere alone gives another number; (J-c) streaming
visits cells in the order geometry dictates; (J-d) the weight balance stays exact and nothing is lost; (J-e) malformed
expressions are refused."""
import ctypes as C

import numpy as np
import pytest

from oracle import Oracle
from oracle import binding as B
from workloads import configs as W


def _member(r):
    """cell id of point r for workloads.csg_union_geometry, written out from the geometry's description"""
    x, y, z = r
    bx, by, bz = W.CSG_BOX
    if any(((x - a) ** 2 + (y - b) ** 2 + (z - c) ** 2) < rr * rr for a, b, c, rr in W.CSG_SPHERES):
        return 0
    cx, cy, cr = W.CSG_CYL
    if (x - cx) ** 2 + (y - cy) ** 2 < cr * cr and 0.0 < z < bz:
        return 1
    if 0.0 < x < bx and 0.0 < y < by and 0.0 < z < bz:
        return 2
    return -1


def test_Ja_point_location_against_hand_written_membership():
    p = W.csg_union_geometry(n_histories=100, n_batches=1)
    o = Oracle(p)
    rng = np.random.default_rng(3)
    pts = rng.uniform([-1, -1, -1], [13, 9, 9], size=(4000, 3))
    got = np.array([o.locate(r, [0.3, 0.5, 0.81]) for r in pts])
    want = np.array([_member(r) for r in pts])
    assert np.array_equal(got, want)
    assert set(want) == {-1, 0, 1, 2}
    # the lens where both spheres overlap and the far caps of either sphere all belong to the union
    for r in ([4.25, 4.0, 4.0], [1.5, 4.0, 4.0], [7.0, 4.0, 4.0]):
        assert o.locate(r, [1, 0, 0]) == 0


def test_Jb_beam_through_the_union_of_two_absorbing_spheres():
    N = 200_000
    p = W.csg_union_geometry(n_histories=N, n_batches=10, beam=True)
    o = Oracle(p); o.enable_collision_tally()
    o.run(N, p.seed, n_batches=10)
    c = o.counters()
    (x0, _, _, r0), (x1, _, _, r1) = W.CSG_SPHERES
    L = (x1 + r1) - (x0 - r0)                             # 1 .. 7.5 on the axis through both centres
    t_exact = np.exp(-1.0 * L)
    assert c["leak"] / N == pytest.approx(t_exact, abs=4.5 * np.sqrt(t_exact * (1 - t_exact) / N))
    assert c["capture"] + c["leak"] == N and c["lost"] == 0.0
    # neither sphere alone (exp(-4)) nor the overlap lens (exp(-1.5)) is within reach of that tolerance
    assert abs(np.exp(-4.0) - t_exact) > 0.01 and abs(np.exp(-1.5) - t_exact) > 0.01
    mc, _ = o.collision_tallies()                         # x profile of the collisions: bins of 1 cm from x = 0
    per_x = mc.sum(axis=(0, 1, 2, 3)) * N                 # Sigma_t = 1: collisions per x bin
    expect = np.zeros(12)
    for i in range(12):
        a, b = max(i, x0 - r0), min(i + 1.0, x1 + r1)
        if b > a:
            expect[i] = N * (np.exp(-(a - (x0 - r0))) - np.exp(-(b - (x0 - r0))))
    assert np.all(np.abs(per_x - expect) < 4.5 * np.sqrt(np.maximum(expect, 1.0)))
    assert per_x[0] == 0.0 and per_x[8:].sum() == 0.0


def test_Jc_streaming_visits_cells_in_geometric_order():
    p = W.csg_union_geometry(n_histories=100, n_batches=1)
    o = Oracle(p)
    # along the axis: box -> union (enter sphere 0, cross the two inner sphere surfaces without leaving) -> box -> out
    r, om, cell = [0.5, 4.0, 4.0], [1.0, 0.0, 0.0], 2
    seen = [cell]
    for _ in range(8):
        n, r, om, cell = o.stream(r, om, cell, 1)
        if n == 0 or cell < 0:
            break
        seen.append(cell)
    assert seen[0] == 2 and 0 in seen and 1 in seen       # the cylinder at x = 9 lies on the axis too
    assert [c for i, c in enumerate(seen) if i == 0 or c != seen[i - 1]] == [2, 0, 2, 1, 2]


def test_Jd_balance_and_no_lost_particles():
    p = W.csg_union_geometry(n_histories=20_000, n_batches=10)
    o = Oracle(p)
    o.run(p.n_histories, p.seed, n_batches=10)
    c = o.counters()
    assert c["lost"] == 0.0 and c["children"] > 0 and c["leak"] > 0
    assert c["source"] + c["production"] == c["capture"] + c["fission_abs"] + c["leak"] + c["census_final"]
    # order independence holds here as everywhere
    q = Oracle(p); q.run(p.n_histories, p.seed, n_batches=10, reverse_histories=True, bank_fifo=True)
    assert q.counters() == c


def test_Je_malformed_expressions_are_refused():
    p = W.csg_union_geometry(n_histories=100, n_batches=1)
    o = Oracle(p)
    L = B._load()
    ip = C.POINTER(C.c_int32)
    def rc(off, tok):
        a = np.array(off, dtype=np.int32); b = np.array(tok + [0], dtype=np.int32)
        return L.orc_regions_set(o._h, a.ctypes.data_as(ip), b.ctypes.data_as(ip))
    assert rc([0, 3, 3, 3], [0, 1, -2]) == 0
    assert rc([0, 2, 2, 2], [0, 1]) != 0                  # two values left
    assert rc([0, 2, 2, 2], [0, -2]) != 0                 # operator without operands
    assert rc([0, 3, 3, 3], [0, 5, -2]) != 0              # operand out of the cell's list
    assert rc([0, 3, 3, 3], [0, 1, -7]) != 0              # unknown token
    assert L.orc_regions_set(o._h, None, None) == 0       # back to plain intersections
