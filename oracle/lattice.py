"""Universes and lattices for the ORACLE (test infrastructure; shares no code with the CUDA library).

The paper says "full three-dimensional constructive solid geometry" and nothing more; SURVEY.md 8(f)
NEXT-4 lists universes / lattices.  Reading (DESIGN.md Appendix K), written out step by step:

  A lattice is an nx x ny array of box elements of size pitch_x x pitch_y whose corner is (x0, y0), all spanning
  z_lo .. z_hi.  Element (i, j) is filled with universe fill[j][i].  A universe is a list of quadric surfaces given in
  coordinates LOCAL to an element (origin = the element's centre in x and y; z is not shifted) and a list of cells,
  each the intersection of half-spaces of the universe's own surfaces (index >= 0) or of the element's
  faces (-1 x-lo, -2 x-hi, -3 y-lo, -4 y-hi, -5 z-lo, -6 z-hi), with a material.

  K.1 surfaces of the flat geometry, in this order: the planes x = x0 + i pitch_x (i = 0..nx), the planes
      y = y0 + j pitch_y (j = 0..ny), z = z_lo, z = z_hi -- the outer ones with the lattice's boundary conditions, the
      inner ones transmission -- then, element by element (j outer, i inner), the universe's surfaces translated to
      the element's centre c = (x0 + (i + 1/2) pitch_x, y0 + (j + 1/2) pitch_y, 0), all transmission.
  K.2 translation of f(r) = A x^2 + B y^2 + C z^2 + D xy + E xz + F yz + G x + H y + I z + J to f(r - c):
      second-order coefficients unchanged;  G' = G - 2 A cx - D cy - E cz  (H', I' alike);
      J' = J + (A cx^2 + B cy^2 + C cz^2 + D cx cy + E cx cz + F cy cz) - (G cx + H cy + I cz).
  K.3 cells of the flat geometry: element by element in the same order, the universe's cells in their order, each
      half-space list in its order with local surfaces and face codes replaced by the flat surface ids.

expand_lattice returns the flat arrays of SURVEY A.1; everything after that is the ordinary oracle.
"""
from __future__ import annotations

import numpy as np

FACE_CODES = (-1, -2, -3, -4, -5, -6)


def translate_quadric(coef, c):
    """K.2: coefficients of f(r - c)."""
    A, B, C_, D, E, F, G, H, I, J = (float(v) for v in coef)
    cx, cy, cz = (float(v) for v in c)
    out = np.zeros(10)
    out[0:6] = (A, B, C_, D, E, F)
    out[6] = G - 2.0 * A * cx - D * cy - E * cz
    out[7] = H - 2.0 * B * cy - D * cx - F * cz
    out[8] = I - 2.0 * C_ * cz - E * cx - F * cy
    quad = A * cx * cx + B * cy * cy + C_ * cz * cz + D * cx * cy + E * cx * cz + F * cy * cz
    lin = G * cx + H * cy + I * cz
    out[9] = J + quad - lin
    return out


def _plane(axis, a):
    c = np.zeros(10)
    c[6 + axis] = 1.0
    c[9] = -a
    return c


def expand_lattice(lat):
    """lat: the dict of workloads.configs (universes, nx, ny, x0, y0, pitch_x, pitch_y, z_lo, z_hi, fill, bc).
    -> dict(surf_coef [S][10], surf_bc [S], cell_offset [C+1], hs_surface, hs_sense, cell_material [C])."""
    nx, ny = int(lat["nx"]), int(lat["ny"])
    U = lat["universes"]
    fill = np.asarray(lat["fill"], dtype=np.int64)
    if nx < 1 or ny < 1 or fill.shape != (ny, nx):
        raise ValueError("lattice: fill must be [ny][nx]")
    if fill.min() < 0 or fill.max() >= len(U):
        raise ValueError("lattice: universe id out of range")
    if not (lat["pitch_x"] > 0 and lat["pitch_y"] > 0 and lat["z_hi"] > lat["z_lo"]):
        raise ValueError("lattice: pitches must be positive and z_hi > z_lo")
    bc = [int(b) for b in lat["bc"]]
    surf, sbc = [], []
    for i in range(nx + 1):                                # K.1
        surf.append(_plane(0, lat["x0"] + i * lat["pitch_x"])); sbc.append(bc[0] if i == 0 else bc[1] if i == nx else 0)
    for j in range(ny + 1):
        surf.append(_plane(1, lat["y0"] + j * lat["pitch_y"])); sbc.append(bc[2] if j == 0 else bc[3] if j == ny else 0)
    oy, oz = nx + 1, nx + 1 + ny + 1
    surf.append(_plane(2, lat["z_lo"])); sbc.append(bc[4])
    surf.append(_plane(2, lat["z_hi"])); sbc.append(bc[5])
    first = {}                                             # (i, j) -> flat id of the element's first universe surface
    for j in range(ny):
        for i in range(nx):
            u = U[fill[j, i]]
            first[(i, j)] = len(surf)
            c = (lat["x0"] + (i + 0.5) * lat["pitch_x"], lat["y0"] + (j + 0.5) * lat["pitch_y"], 0.0)
            for coef in u["surf"]:
                surf.append(translate_quadric(coef, c)); sbc.append(0)
    off, hs_s, hs_n, mat = [0], [], [], []
    for j in range(ny):                                    # K.3
        for i in range(nx):
            u = U[fill[j, i]]
            face = {-1: i, -2: i + 1, -3: oy + j, -4: oy + j + 1, -5: oz, -6: oz + 1}
            for hs, m in u["cells"]:
                if not hs:
                    raise ValueError("lattice: empty universe cell")
                for s, sense in hs:
                    if s >= 0:
                        if s >= len(u["surf"]):
                            raise ValueError("lattice: local surface index out of range")
                        hs_s.append(first[(i, j)] + s)
                    elif s in face:
                        hs_s.append(face[s])
                    else:
                        raise ValueError("lattice: unknown face code")
                    if sense not in (1, -1):
                        raise ValueError("lattice: sense must be +1 or -1")
                    hs_n.append(sense)
                off.append(len(hs_s)); mat.append(int(m))
    return dict(surf_coef=np.ascontiguousarray(np.stack(surf), dtype=np.float64), surf_bc=np.asarray(sbc, dtype=np.int32),
                cell_offset=np.asarray(off, dtype=np.int32), hs_surface=np.asarray(hs_s, dtype=np.int32),
                hs_sense=np.asarray(hs_n, dtype=np.int32), cell_material=np.asarray(mat, dtype=np.int32))


def flat_problem(prob):
    """A copy of `prob` (workloads Problem with meta["lattice"]) whose flat geometry arrays hold the expansion."""
    import copy
    q = copy.copy(prob)
    q.meta = {k: v for k, v in prob.meta.items() if k != "lattice"}
    for k, v in expand_lattice(prob.meta["lattice"]).items():
        setattr(q, k, v)
    return q
