"""Pins for the oracle's geometry (pin E10): distances against brute force,
reflection invariants, cell location against a direct formula."""
import numpy as np
import pytest

import oracle
from oracle import Oracle
from workloads import configs as W


def f_eval(c, p):
    x, y, z = p
    return (c[0] * x * x + c[1] * y * y + c[2] * z * z + c[3] * x * y + c[4] * x * z + c[5] * y * z
            + c[6] * x + c[7] * y + c[8] * z + c[9])


def brute_distance(c, r, o, umax=40.0, n=400001):
    """First sign change of f along the ray, refined by bisection (independent of the quadratic formula)."""
    u = np.linspace(0.0, umax, n)[1:]
    pts = r[None, :] + u[:, None] * o[None, :]
    x, y, z = pts[:, 0], pts[:, 1], pts[:, 2]
    f = (c[0] * x * x + c[1] * y * y + c[2] * z * z + c[3] * x * y + c[4] * x * z + c[5] * y * z
         + c[6] * x + c[7] * y + c[8] * z + c[9])
    s = np.sign(f)
    idx = np.nonzero(s[1:] * s[:-1] < 0)[0]
    if len(idx) == 0:
        return np.inf
    lo, hi = u[idx[0]], u[idx[0] + 1]
    flo = f_eval(c, r + lo * o)
    for _ in range(80):
        mid = 0.5 * (lo + hi)
        fm = f_eval(c, r + mid * o)
        if fm * flo <= 0:
            hi = mid
        else:
            lo, flo = mid, fm
    return 0.5 * (lo + hi)


def _rand_dir(rng):
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


@pytest.mark.parametrize("kind", ["plane", "cyl", "sphere", "general"])
def test_distance_vs_brute_force(kind):
    rng = np.random.default_rng({"plane": 1, "cyl": 2, "sphere": 3, "general": 4}[kind])
    checked = 0
    for _ in range(60):
        if kind == "plane":
            n = _rand_dir(rng); c = np.zeros(10); c[6:9] = n * rng.uniform(0.5, 2); c[9] = rng.uniform(-3, 3)
        elif kind == "cyl":
            c = W.cylinder_z(rng.uniform(-2, 2), rng.uniform(-2, 2), rng.uniform(0.3, 2.0))
        elif kind == "sphere":
            c = W.sphere(*rng.uniform(-2, 2, 3), rng.uniform(0.3, 2.5))
        else:  # ellipsoid / hyperboloid with cross terms
            A = rng.normal(size=(3, 3)); Q = A + A.T
            c = np.array([Q[0, 0], Q[1, 1], Q[2, 2], 2 * Q[0, 1], 2 * Q[0, 2], 2 * Q[1, 2],
                          *rng.normal(size=3), rng.normal()])
        r = rng.uniform(-4, 4, 3)
        o = rng.uniform(-1.5, 1.5, 3) - r; o /= np.linalg.norm(o)      # aim at the region the surfaces live in
        d = oracle.surface_distance(c, r, o)
        b = brute_distance(c, r, o)
        if np.isinf(b):
            # the march can miss a tangential double root, or the root lies beyond umax
            assert np.isinf(d) or d > 40.0 or abs(f_eval(c, r + d * o)) < 1e-9
        else:
            assert d == pytest.approx(b, rel=1e-9, abs=1e-9)
            checked += 1
        if np.isfinite(d):
            assert abs(f_eval(c, r + d * o)) < 1e-8 * (1 + np.abs(c).max() * (1 + d * d + (np.abs(r) ** 2).sum()))
    assert checked > 15


def test_on_surface_rule_skips_the_current_surface():
    # plane: a particle flagged on the plane never re-hits it
    c = W.plane_x(1.0)
    assert np.isinf(oracle.surface_distance(c, [1.0 + 1e-17, 0, 0], [1, 0, 0], True))
    assert np.isinf(oracle.surface_distance(c, [1.0, 0, 0], [-1, 0, 0], True))
    # cylinder r=1: on the surface heading inward -> chord length -b/a = 2 cos(angle)
    c = W.cylinder_z(0, 0, 1.0)
    th = 0.3
    d = oracle.surface_distance(c, [1.0, 0.0, 0.0], [-np.cos(th), np.sin(th), 0.0], True)
    assert d == pytest.approx(2 * np.cos(th), rel=1e-14)
    # heading outward: no positive root
    assert np.isinf(oracle.surface_distance(c, [1.0, 0.0, 0.0], [np.cos(th), np.sin(th), 0.0], True))
    # with a polar component the chord stretches by 1/sin^2... (a = 1 - uz^2): u = 2 cos(th) s / s^2
    s = np.sqrt(1 - 0.36)
    d = oracle.surface_distance(c, [1.0, 0.0, 0.0], [-np.cos(th) * s, np.sin(th) * s, 0.6], True)
    assert d == pytest.approx(2 * np.cos(th) / s, rel=1e-14)


def test_textbook_distances():
    # sphere of radius R from the centre: R in every direction; from outside along the axis: gap and gap+2R
    c = W.sphere(0, 0, 0, 2.0)
    rng = np.random.default_rng(3)
    for _ in range(10):
        assert oracle.surface_distance(c, [0, 0, 0], _rand_dir(rng)) == pytest.approx(2.0, rel=1e-15)
    assert oracle.surface_distance(c, [-5, 0, 0], [1, 0, 0]) == pytest.approx(3.0, rel=1e-15)
    assert np.isinf(oracle.surface_distance(c, [-5, 0, 0], [-1, 0, 0]))
    assert np.isinf(oracle.surface_distance(c, [-5, 2.5, 0], [1, 0, 0]))       # misses
    assert oracle.surface_distance(W.plane_z(10.0), [0, 0, 4], [0, 0.6, 0.8]) == pytest.approx(7.5, rel=1e-15)


def test_reflective_cube_invariants():
    p = W.config0_infinite_medium()
    o = Oracle(p)
    rng = np.random.default_rng(11)
    for _ in range(5):
        r = rng.uniform(0.05, 0.95, 3); d = _rand_dir(rng)
        n, r2, d2, cell = o.stream(r, d, 0, 10000)
        assert n == 10000 and cell == 0
        assert abs(np.linalg.norm(d2) - 1.0) < 1e-12
        assert np.all(r2 > -1e-12) and np.all(r2 < 1 + 1e-12)
        # specular reflection off axis-aligned planes only flips signs
        assert np.allclose(np.abs(d2), np.abs(d), rtol=0, atol=1e-15)


def test_reflective_cube_path_is_the_unfolded_straight_line():
    # unfolding the reflections: after n events the particle has moved a straight line in the tiled
    # space; folding that point back into the cube must give the oracle's position.
    p = W.config0_infinite_medium()
    o = Oracle(p)
    r = np.array([0.3, 0.6, 0.2]); d = np.array([0.48, -0.6, 0.64])
    n, r2, d2, _ = o.stream(r, d, 0, 25)
    # total path length: 25th crossing of the unfolded lattice planes
    ts = []
    for a in range(3):
        k = np.arange(-40, 41)
        t = (k - r[a]) / d[a]
        ts.extend(t[t > 1e-15])
    L = np.sort(ts)[24]
    q = r + L * d
    fold = np.abs(((q + 1) % 2) - 1)
    assert np.allclose(fold, r2, atol=1e-12)


def test_locate_pin_lattice_against_direct_formula():
    p = W.config3_pin_lattice()
    o = Oracle(p)
    rng = np.random.default_rng(5)
    pitch, rad = 1.26, 0.54
    for _ in range(400):
        r = np.array([rng.uniform(0, 17 * pitch), rng.uniform(0, 17 * pitch), rng.uniform(0, 10)])
        i, j = int(r[0] // pitch), int(r[1] // pitch)
        inside = (r[0] - (i + 0.5) * pitch) ** 2 + (r[1] - (j + 0.5) * pitch) ** 2 < rad * rad
        expect = 2 * (j * 17 + i) + (0 if inside else 1)
        assert o.locate(r, [0, 0, 1]) == expect
    assert o.locate([5.0, 5.0, 10.5], [0, 0, 1]) == -1
    # a point exactly on a pitch plane is assigned by the direction of travel (A.3 tie rule)
    x = p.surf_coef[3][9] * -1.0          # plane x = 3 pitch
    assert o.locate([x, 0.1, 5.0], [1, 0, 0]) == 2 * (0 * 17 + 3) + 1
    assert o.locate([x, 0.1, 5.0], [-1, 0, 0]) == 2 * (0 * 17 + 2) + 1


def test_crossing_moves_to_the_neighbour_cell():
    p = W.config3_pin_lattice()
    o = Oracle(p)
    pitch = 1.26
    # start in the moderator corner of pin (2,3), head +x just above the pin's bottom edge: next cell is
    # the moderator of pin (3,3), then (4,3) ...
    r = [2 * pitch + 0.01, 3 * pitch + 0.01, 5.0]
    n, r2, d2, cell = o.stream(r, [1.0, 0.0, 0.0], 2 * (3 * 17 + 2) + 1, 3)
    assert n == 3 and cell == 2 * (3 * 17 + 5) + 1
    assert r2[0] == pytest.approx(5 * pitch, rel=1e-14)
    # through the middle of a pin: mod -> fuel -> mod -> next pin's mod
    r = [2 * pitch + 0.01, 3.5 * pitch, 5.0]
    cells = []
    rr, dd, c = np.array(r), np.array([1.0, 0, 0]), 2 * (3 * 17 + 2) + 1
    for _ in range(3):
        _, rr, dd, c = o.stream(rr, dd, c, 1)
        cells.append(c)
    # note: stream() restarts with last_surface = -1, harmless here because the hit surface is then
    # re-evaluated with c = f(r) ~ 1e-16 and the particle keeps moving away from it or through it
    assert cells[0] == 2 * (3 * 17 + 2) and cells[1] == 2 * (3 * 17 + 2) + 1
