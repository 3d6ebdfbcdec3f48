"""Concrete synthetic inputs for the five BASELINE.json configs.

Every array is C-contiguous numpy with the dtype the C-ABI expects (float64 / int32).
Quadric coefficient order:
    f(x,y,z) = A x^2 + B y^2 + C z^2 + D xy + E xz + F yz + G x + H y + I z + J
Boundary conditions: 0 transmission, 1 vacuum, 2 reflective.
Half-space sense: +1 means f(r) > 0, -1 means f(r) < 0; a cell is the intersection of its
half-spaces (CSR: cell_offset / hs_surface / hs_sense).

Config 2 stands in for the paper's time-dependent Kobayashi dog-leg problem;
configs 3/4 stand in for a multigroup pin-lattice workload.  Nothing here reproduces a
published benchmark's own tables; the recipes are the ones written out in Appendix C.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

BC_TRANSMISSION, BC_VACUUM, BC_REFLECTIVE = 0, 1, 2
DIR_ISOTROPIC, DIR_FIXED = 0, 1

_BASE_SEED = 2409046680


def run_seed(k: int) -> int:
    """Run seed for config k (Appendix C: 2409046680 + k)."""
    return _BASE_SEED + k


@dataclass
class Problem:
    name: str
    # materials
    sigma_t: np.ndarray  # [M][G]
    sigma_c: np.ndarray  # [M][G]
    sigma_f: np.ndarray  # [M][G]
    nu: np.ndarray  # [M][G]
    chi: np.ndarray  # [M][G]
    sigma_s: np.ndarray  # [M][G][G]  g -> g'
    speed: np.ndarray  # [G]
    # geometry
    surf_coef: np.ndarray  # [S][10]
    surf_bc: np.ndarray  # [S]
    cell_offset: np.ndarray  # [C+1]
    hs_surface: np.ndarray
    hs_sense: np.ndarray
    cell_material: np.ndarray  # [C]
    # source
    src_lo: np.ndarray
    src_hi: np.ndarray
    src_t0: float
    src_t1: float
    src_group_pdf: np.ndarray  # [G]
    src_dir_mode: int
    src_dir: np.ndarray
    # tally mesh
    mesh_lo: np.ndarray
    mesh_hi: np.ndarray
    mesh_n: np.ndarray  # [3] int32 (nx, ny, nz)
    time_edges: np.ndarray  # [Nt+1]
    census_times: np.ndarray  # [K]
    # default run parameters of the config
    n_histories: int = 0
    n_batches: int = 1
    seed: int = _BASE_SEED
    meta: dict = field(default_factory=dict)

    @property
    def n_groups(self) -> int:
        return int(self.speed.shape[0])

    @property
    def n_materials(self) -> int:
        return int(self.sigma_t.shape[0])

    @property
    def n_surfaces(self) -> int:
        return int(self.surf_coef.shape[0])

    @property
    def n_cells(self) -> int:
        return int(self.cell_material.shape[0])

    @property
    def n_time_bins(self) -> int:
        return int(self.time_edges.shape[0]) - 1

    @property
    def n_census(self) -> int:
        return int(self.census_times.shape[0])

    @property
    def n_bins(self) -> int:
        nx, ny, nz = (int(v) for v in self.mesh_n)
        return self.n_time_bins * self.n_groups * nz * ny * nx

    def tally_shape(self):
        nx, ny, nz = (int(v) for v in self.mesh_n)
        return (self.n_time_bins, self.n_groups, nz, ny, nx)


# ----------------------------------------------------------------------------------------
# small builders
# ----------------------------------------------------------------------------------------
def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _i32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def plane_x(a):
    c = np.zeros(10)
    c[6] = 1.0
    c[9] = -a
    return c


def plane_y(a):
    c = np.zeros(10)
    c[7] = 1.0
    c[9] = -a
    return c


def plane_z(a):
    c = np.zeros(10)
    c[8] = 1.0
    c[9] = -a
    return c


def cylinder_z(x0, y0, r):
    c = np.zeros(10)
    c[0] = 1.0
    c[1] = 1.0
    c[6] = -2.0 * x0
    c[7] = -2.0 * y0
    c[9] = x0 * x0 + y0 * y0 - r * r
    return c


def sphere(x0, y0, z0, r):
    c = np.zeros(10)
    c[0] = c[1] = c[2] = 1.0
    c[6], c[7], c[8] = -2.0 * x0, -2.0 * y0, -2.0 * z0
    c[9] = x0 * x0 + y0 * y0 + z0 * z0 - r * r
    return c


def _cells_to_csr(cells):
    """cells: list of (list of (surface, sense), material)."""
    off = [0]
    hs_s, hs_n, mat = [], [], []
    for hs, m in cells:
        for s, sense in hs:
            hs_s.append(s)
            hs_n.append(sense)
        off.append(len(hs_s))
        mat.append(m)
    return _i32(off), _i32(hs_s), _i32(hs_n), _i32(mat)


def _materials(rows, G):
    """rows: list of dict(sigma_t, sigma_c, sigma_f, nu, chi, sigma_s)."""
    M = len(rows)
    out = {k: np.zeros((M, G)) for k in ("sigma_t", "sigma_c", "sigma_f", "nu", "chi")}
    ss = np.zeros((M, G, G))
    for m, r in enumerate(rows):
        for k in out:
            out[k][m, :] = np.asarray(r.get(k, np.zeros(G)), dtype=np.float64)
        ss[m] = np.asarray(r["sigma_s"], dtype=np.float64).reshape(G, G)
    return out, ss


def _assemble(name, mats, ss, speed, surfs, bcs, cells, src, mesh, time_edges, census,
              n_histories, n_batches, seed, meta=None):
    off, hs_s, hs_n, cmat = _cells_to_csr(cells)
    return Problem(
        name=name,
        sigma_t=_f64(mats["sigma_t"]), sigma_c=_f64(mats["sigma_c"]), sigma_f=_f64(mats["sigma_f"]),
        nu=_f64(mats["nu"]), chi=_f64(mats["chi"]), sigma_s=_f64(ss), speed=_f64(speed),
        surf_coef=_f64(np.stack(surfs)), surf_bc=_i32(bcs),
        cell_offset=off, hs_surface=hs_s, hs_sense=hs_n, cell_material=cmat,
        src_lo=_f64(src["lo"]), src_hi=_f64(src["hi"]), src_t0=float(src["t0"]), src_t1=float(src["t1"]),
        src_group_pdf=_f64(src["pdf"]), src_dir_mode=int(src.get("mode", DIR_ISOTROPIC)),
        src_dir=_f64(src.get("dir", [0.0, 0.0, 1.0])),
        mesh_lo=_f64(mesh["lo"]), mesh_hi=_f64(mesh["hi"]), mesh_n=_i32(mesh["n"]),
        time_edges=_f64(time_edges), census_times=_f64(census),
        n_histories=int(n_histories), n_batches=int(n_batches), seed=int(seed), meta=meta or {},
    )


# ----------------------------------------------------------------------------------------
# C0: one-group infinite homogeneous medium (reflective 1 cm cube)
# ----------------------------------------------------------------------------------------
def config0_infinite_medium(n_histories=100_000, n_batches=20, n_time=20, t_end=20.0):
    G = 1
    mats, ss = _materials([dict(sigma_t=[1.0], sigma_c=[0.3], sigma_f=[0.2], nu=[2.0], chi=[1.0],
                                sigma_s=[[0.5]])], G)
    surfs = [plane_x(0.0), plane_x(1.0), plane_y(0.0), plane_y(1.0), plane_z(0.0), plane_z(1.0)]
    bcs = [BC_REFLECTIVE] * 6
    cells = [([(0, +1), (1, -1), (2, +1), (3, -1), (4, +1), (5, -1)], 0)]
    src = dict(lo=[0, 0, 0], hi=[1, 1, 1], t0=0.0, t1=0.0, pdf=[1.0])
    mesh = dict(lo=[0, 0, 0], hi=[1, 1, 1], n=[1, 1, 1])
    T = np.array([k * (t_end / n_time) for k in range(n_time + 1)], dtype=np.float64)
    return _assemble("config0_infinite_medium", mats, ss, [1.0], surfs, bcs, cells, src, mesh, T, T[1:].copy(),
                     n_histories, n_batches, run_seed(0))


# ----------------------------------------------------------------------------------------
# C1: three-region slab; C1a: pure-absorber beam variant
# ----------------------------------------------------------------------------------------
def _slab_geometry():
    surfs = [plane_x(0.0), plane_x(10.0), plane_x(20.0), plane_x(30.0)]
    bcs = [BC_VACUUM, BC_TRANSMISSION, BC_TRANSMISSION, BC_VACUUM]
    cells = [([(0, +1), (1, -1)], 0), ([(1, +1), (2, -1)], 1), ([(2, +1), (3, -1)], 0)]
    return surfs, bcs, cells


def _slab_mesh_time():
    mesh = dict(lo=[0.0, -np.inf, -np.inf], hi=[30.0, np.inf, np.inf], n=[100, 1, 1])
    T = np.array([k * 0.2 for k in range(51)], dtype=np.float64)
    return mesh, T


def config1_slab(n_histories=1_000_000, n_batches=100):
    G = 1
    mats, ss = _materials([
        dict(sigma_t=[1.0], sigma_c=[0.2], sigma_f=[0.0], nu=[0.0], chi=[0.0], sigma_s=[[0.8]]),
        dict(sigma_t=[0.5], sigma_c=[0.2], sigma_f=[0.1], nu=[2.4], chi=[1.0], sigma_s=[[0.2]]),
    ], G)
    surfs, bcs, cells = _slab_geometry()
    src = dict(lo=[10.0, 0.0, 0.0], hi=[20.0, 0.0, 0.0], t0=0.0, t1=1.0, pdf=[1.0])
    mesh, T = _slab_mesh_time()
    return _assemble("config1_slab", mats, ss, [1.0], surfs, bcs, cells, src, mesh, T, T[1:].copy(),
                     n_histories, n_batches, run_seed(1))


def config1a_pure_absorber_beam(n_histories=1_000_000, n_batches=100):
    G = 1
    mats, ss = _materials([
        dict(sigma_t=[1.0], sigma_c=[1.0], sigma_f=[0.0], nu=[0.0], chi=[0.0], sigma_s=[[0.0]]),
        dict(sigma_t=[0.5], sigma_c=[0.5], sigma_f=[0.0], nu=[0.0], chi=[0.0], sigma_s=[[0.0]]),
    ], G)
    surfs, bcs, cells = _slab_geometry()
    src = dict(lo=[0.0, 0.0, 0.0], hi=[0.0, 0.0, 0.0], t0=0.0, t1=0.0, pdf=[1.0],
               mode=DIR_FIXED, dir=[1.0, 0.0, 0.0])
    mesh, T = _slab_mesh_time()
    return _assemble("config1a_pure_absorber_beam", mats, ss, [1.0], surfs, bcs, cells, src, mesh, T,
                     T[1:].copy(), n_histories, n_batches, run_seed(1))


# ----------------------------------------------------------------------------------------
# C2: L-duct shielding box (stand-in for the paper's dog-leg void-duct workload)
# ----------------------------------------------------------------------------------------
def config2_lduct(n_histories=10_000_000, n_batches=100):
    G = 1
    mats, ss = _materials([
        dict(sigma_t=[0.1], sigma_c=[0.05], sigma_f=[0.0], nu=[0.0], chi=[0.0], sigma_s=[[0.05]]),   # shield
        dict(sigma_t=[1e-4], sigma_c=[5e-5], sigma_f=[0.0], nu=[0.0], chi=[0.0], sigma_s=[[5e-5]]),  # void
    ], G)
    xs, ys, zs = [0.0, 10.0, 60.0], [0.0, 10.0, 50.0, 60.0, 100.0], [0.0, 10.0, 60.0]
    surfs, bcs = [], []
    for i, a in enumerate(xs):
        surfs.append(plane_x(a)); bcs.append(BC_VACUUM if i in (0, len(xs) - 1) else BC_TRANSMISSION)
    for j, a in enumerate(ys):
        surfs.append(plane_y(a)); bcs.append(BC_VACUUM if j in (0, len(ys) - 1) else BC_TRANSMISSION)
    for k, a in enumerate(zs):
        surfs.append(plane_z(a)); bcs.append(BC_VACUUM if k in (0, len(zs) - 1) else BC_TRANSMISSION)
    ox, oy, oz = 0, len(xs), len(xs) + len(ys)
    cells = []
    for kz in range(2):
        for jy in range(4):
            for ix in range(2):
                # void: {x in [0,10], z in [0,10], y in [10,60]} U {x in [10,60], y in [50,60], z in [0,10]}
                void = (kz == 0) and ((ix == 0 and jy in (1, 2)) or (ix == 1 and jy == 2))
                hs = [(ox + ix, +1), (ox + ix + 1, -1), (oy + jy, +1), (oy + jy + 1, -1),
                      (oz + kz, +1), (oz + kz + 1, -1)]
                cells.append((hs, 1 if void else 0))
    src = dict(lo=[0, 0, 0], hi=[10, 10, 10], t0=0.0, t1=50.0, pdf=[1.0])
    mesh = dict(lo=[0, 0, 0], hi=[60, 100, 60], n=[60, 100, 60])
    T = np.array([k * 10.0 for k in range(21)], dtype=np.float64)
    return _assemble("config2_lduct", mats, ss, [1.0], surfs, bcs, cells, src, mesh, T, T[1:].copy(),
                     n_histories, n_batches, run_seed(2))


# ----------------------------------------------------------------------------------------
# C3 / C4: 7-group 17x17 pin lattice with seed-drawn cross sections
# ----------------------------------------------------------------------------------------
_M64 = (1 << 64) - 1
_GAMMA = 0x9E3779B97F4A7C15


def _mix64(z):
    z &= _M64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & _M64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & _M64
    z ^= z >> 31
    return z


class _Stream:
    """Input-recipe stream of Appendix C: s += gamma; u = (M(s) >> 11) * 2^-53."""

    def __init__(self, s0):
        self.s = s0 & _M64

    def u(self):
        self.s = (self.s + _GAMMA) & _M64
        return (_mix64(self.s) >> 11) * (2.0 ** -53)


def config3_xs(pitch=1.26, radius=0.54, k_target=0.95):
    """Cross sections of config 3 (materials: 0 fuel A, 1 fuel B, 2 moderator), G = 7.

    Returns (mats dict, sigma_s[M][G][G], speed[G], k0) where k0 is the homogenised
    infinite-medium multiplication factor *before* nu was rescaled to k_target.
    """
    G, M = 7, 3
    st = _Stream(2409046683)
    sig_t = np.zeros((M, G)); sig_s = np.zeros((M, G, G)); sig_f = np.zeros((M, G))
    nu = np.zeros((M, G)); chi = np.zeros((M, G))
    for m in range(M):
        fuel = m < 2
        kappa = 1.0 if fuel else 0.5
        for g in range(G):
            sig_t[m, g] = 0.2 * 10.0 ** st.u()
            c_s = (0.55 + 0.25 * st.u()) if fuel else (0.985 + 0.01 * st.u())
            w = np.zeros(G)
            for gp in range(g, G):
                w[gp] = np.exp(-kappa * (gp - g)) * (0.5 + st.u())
            if g == G - 1:
                w[G - 2] = 0.2 * (0.5 + st.u())
            sig_s[m, g, :] = c_s * sig_t[m, g] * w / w.sum()
            sig_a = sig_t[m, g] - c_s * sig_t[m, g]
            if fuel:
                f = (0.3 + 0.4 * st.u()) if g >= 3 else (0.1 + 0.2 * st.u())
                sig_f[m, g] = f * sig_a
                nu[m, g] = 2.4 + 0.2 * st.u()
        if fuel:
            c = np.array([(0.5 + st.u()) * k for k in (6.0, 3.0, 1.0)])
            chi[m, :3] = c / c.sum()
    # volume-homogenised infinite medium: fuel fraction split 145:144 between A and B
    ff = np.pi * radius * radius / (pitch * pitch)
    frac = np.array([ff * 145.0 / 289.0, ff * 144.0 / 289.0, 1.0 - ff])
    St = (frac[:, None] * sig_t).sum(0)
    Ss = (frac[:, None, None] * sig_s).sum(0)              # [g][g']
    Fm = sum(frac[m] * np.outer(chi[m], nu[m] * sig_f[m]) for m in range(M))  # [g][g'] production into g
    A = np.diag(St) - Ss.T                                  # loss - inscatter (column = from-group)
    phi = np.ones(G)
    k0 = 1.0
    for _ in range(500):
        src = Fm @ phi
        phi_new = np.linalg.solve(A, src)
        k_new = (Fm @ phi_new).sum() / src.sum()
        phi = phi_new / np.abs(phi_new).sum()
        if abs(k_new - k0) < 1e-14 * abs(k_new):
            k0 = k_new
            break
        k0 = k_new
    nu *= k_target / k0
    sig_c = sig_t - sig_s.sum(axis=2) - sig_f               # validation identity to rounding
    sig_c = np.where(np.abs(sig_c) < 1e-15, 0.0, sig_c)
    speed = np.array([2e9 * (1e-4) ** (g / 6.0) for g in range(G)])
    mats = dict(sigma_t=sig_t, sigma_c=sig_c, sigma_f=sig_f, nu=nu, chi=chi)
    return mats, sig_s, speed, float(k0)


def config3_pin_lattice(n_histories=10_000_000, n_batches=100, n_pins=17):
    p, r, H = 1.26, 0.54, 10.0
    n = n_pins
    mats, ss, speed, k0 = config3_xs(p, r)
    surfs, bcs = [], []
    for i in range(n + 1):
        surfs.append(plane_x(i * p)); bcs.append(BC_REFLECTIVE if i in (0, n) else BC_TRANSMISSION)
    for j in range(n + 1):
        surfs.append(plane_y(j * p)); bcs.append(BC_REFLECTIVE if j in (0, n) else BC_TRANSMISSION)
    oy, oz = n + 1, 2 * (n + 1)
    surfs.append(plane_z(0.0)); bcs.append(BC_VACUUM)
    surfs.append(plane_z(H)); bcs.append(BC_VACUUM)
    oc = oz + 2
    for j in range(n):
        for i in range(n):
            surfs.append(cylinder_z((i + 0.5) * p, (j + 0.5) * p, r)); bcs.append(BC_TRANSMISSION)
    cells = []
    for j in range(n):
        for i in range(n):
            cyl = oc + j * n + i
            cells.append(([(cyl, -1), (oz, +1), (oz + 1, -1)], 0 if (i + j) % 2 == 0 else 1))
            cells.append(([(i, +1), (i + 1, -1), (oy + j, +1), (oy + j + 1, -1), (cyl, +1),
                           (oz, +1), (oz + 1, -1)], 2))
    c = 0.5 * n * p
    src = dict(lo=[c, c, 0.5 * H], hi=[c, c, 0.5 * H], t0=0.0, t1=0.0, pdf=mats["chi"][0].copy())
    mesh = dict(lo=[0.0, 0.0, 0.0], hi=[n * p, n * p, H], n=[n, n, 1])
    T = np.array([k * 5e-7 for k in range(21)], dtype=np.float64)
    return _assemble("config3_pin_lattice", mats, ss, speed, surfs, bcs, cells, src, mesh, T, T[1:].copy(),
                     n_histories, n_batches, run_seed(3), meta=dict(k0=k0, pitch=p, radius=r))


def infinite_medium_multigroup(material=0, n_histories=200_000, n_batches=20, n_time=20, t_end=2e-7):
    """One config-3 material in a reflective unit cube (pin E6: multigroup kinetics ODE)."""
    mats, ss, speed, _ = config3_xs()
    G = 7
    m1 = {k: v[material:material + 1].copy() for k, v in mats.items()}
    s1 = ss[material:material + 1].copy()
    if m1["chi"].sum() == 0.0:
        m1["chi"][0, 0] = 1.0
    surfs = [plane_x(0.0), plane_x(1.0), plane_y(0.0), plane_y(1.0), plane_z(0.0), plane_z(1.0)]
    bcs = [BC_REFLECTIVE] * 6
    cells = [([(0, +1), (1, -1), (2, +1), (3, -1), (4, +1), (5, -1)], 0)]
    pdf = np.zeros(G); pdf[0] = 1.0
    src = dict(lo=[0, 0, 0], hi=[1, 1, 1], t0=0.0, t1=0.0, pdf=pdf)
    mesh = dict(lo=[0, 0, 0], hi=[1, 1, 1], n=[1, 1, 1])
    T = np.array([k * (t_end / n_time) for k in range(n_time + 1)], dtype=np.float64)
    return _assemble("infinite_medium_multigroup", m1, s1, speed, surfs, bcs, cells, src, mesh, T, T[1:].copy(),
                     n_histories, n_batches, run_seed(3))


def as_eigenvalue(p, t_far=1e30):
    """The same problem for the k-eigenvalue mode (DESIGN.md Appendix H): time plays no part there, so the tally has
    one time bin [0, t_far] and the only census is at t_far (never reached); the source is born at t = 0."""
    import copy
    q = copy.deepcopy(p)
    q.name = p.name + "_eigenvalue"
    q.time_edges = _f64([0.0, t_far]); q.census_times = _f64([t_far])
    q.src_t0 = 0.0; q.src_t1 = 0.0
    return q


def bare_slab_absorber(thickness=2.0, sigma_t=1.0, sigma_f=0.4, nu=2.5, n_histories=100_000):
    """One-group slab with vacuum faces, no scattering (pin H-b: first-flight collision probability), uniform
    isotropic source over the slab, 10 x-bins."""
    mats, ss = _materials([dict(sigma_t=[sigma_t], sigma_c=[sigma_t - sigma_f], sigma_f=[sigma_f], nu=[nu], chi=[1.0],
                                sigma_s=[[0.0]])], 1)
    surfs = [plane_x(0.0), plane_x(thickness)]
    bcs = [BC_VACUUM, BC_VACUUM]
    cells = [([(0, +1), (1, -1)], 0)]
    src = dict(lo=[0.0, 0.0, 0.0], hi=[thickness, 0.0, 0.0], t0=0.0, t1=0.0, pdf=[1.0])
    mesh = dict(lo=[0.0, -np.inf, -np.inf], hi=[thickness, np.inf, np.inf], n=[10, 1, 1])
    T = _f64([0.0, 1e30])
    return _assemble("bare_slab_absorber", mats, ss, [1.0], surfs, bcs, cells, src, mesh, T, T[1:].copy(),
                     n_histories, 1, run_seed(5))


CONFIGS = {
    "config0": config0_infinite_medium,
    "config1": config1_slab,
    "config1a": config1a_pure_absorber_beam,
    "config2": config2_lduct,
    "config3": config3_pin_lattice,
}


# ----------------------------------------------------------------------------------------
# Stress geometry (parity tests only): what the five configs do not reach -- a general quadric (sphere) cell,
# a reflective sphere with nothing inside (sources drawn there are lost), a face shared with two neighbours
# (no certified neighbour), a z-cylinder inside one of them, a tally mesh smaller than the geometry or
# unaligned with the cells, census times that do not coincide with the tally time edges, two groups.
# ----------------------------------------------------------------------------------------
def stress_geometry(n_histories=60_000, n_batches=12, covering_mesh=False):
    G = 2
    mats, ss = _materials([
        dict(sigma_t=[0.6, 0.9], sigma_c=[0.1, 0.2], sigma_f=[0.0, 0.0], nu=[0.0, 0.0], chi=[0.0, 0.0],
             sigma_s=[[0.3, 0.2], [0.1, 0.6]]),
        dict(sigma_t=[0.8, 1.2], sigma_c=[0.15, 0.4], sigma_f=[0.05, 0.1], nu=[2.2, 2.5], chi=[0.7, 0.3],
             sigma_s=[[0.4, 0.2], [0.0, 0.7]]),
    ], G)
    surfs = [plane_x(0.0), plane_x(2.0), plane_x(6.0), plane_y(0.0), plane_y(2.0), plane_y(4.0), plane_z(0.0),
             plane_z(4.0), sphere(1.0, 2.0, 2.0, 0.7), sphere(5.0, 1.0, 2.0, 0.4), cylinder_z(4.0, 3.0, 0.5)]
    bcs = [BC_REFLECTIVE, BC_TRANSMISSION, BC_VACUUM, BC_VACUUM, BC_TRANSMISSION, BC_VACUUM, BC_VACUUM,
           BC_REFLECTIVE, BC_TRANSMISSION, BC_REFLECTIVE, BC_TRANSMISSION]
    cells = [
        ([(8, -1)], 1),                                                              # fuel sphere
        ([(0, +1), (1, -1), (3, +1), (5, -1), (6, +1), (7, -1), (8, +1)], 0),        # x in [0,2], outside it
        ([(1, +1), (2, -1), (3, +1), (4, -1), (6, +1), (7, -1), (9, +1)], 1),        # y in [0,2], outside the mirror ball
        ([(1, +1), (2, -1), (4, +1), (5, -1), (6, +1), (7, -1), (10, +1)], 0),       # y in [2,4], outside the pin
        ([(10, -1), (6, +1), (7, -1)], 1),                                           # the pin
    ]
    src = dict(lo=[0.2, 0.2, 0.2], hi=[5.8, 3.8, 3.8], t0=0.0, t1=1.5, pdf=[0.6, 0.4])
    if covering_mesh:
        mesh = dict(lo=[0.0, 0.0, 0.0], hi=[6.0, 4.0, 4.0], n=[7, 5, 3])
        T = np.array([0.0, 0.5, 2.0, 3.5, 6.0])
    else:
        mesh = dict(lo=[0.5, 0.5, 0.0], hi=[5.5, 3.5, 4.0], n=[5, 3, 2])
        T = np.array([0.25, 0.5, 2.0, 3.5, 5.0])
    census = np.array([1.3, 2.9, 6.0])
    return _assemble("stress_geometry" + ("_covering" if covering_mesh else ""), mats, ss, [1.0, 0.4], surfs, bcs,
                     cells, src, mesh, T, census, n_histories, n_batches, run_seed(9))


CONFIGS["stress"] = stress_geometry


# ----------------------------------------------------------------------------------------
# General CSG regions (DESIGN.md Appendix J; parity tests only): a vacuum box that holds the UNION of two overlapping
# spheres (cell 0) and a z-cylinder that does not touch them (cell 1); cell 2 is the box MINUS those: the
# complement of a union.  Regions are postfix expressions over a cell's half-space list: t >= 0 operand, -1 AND,
# -2 OR, -3 NOT; they travel in meta["regions"] = (region_offset, region_rpn).
# ----------------------------------------------------------------------------------------
RGN_AND, RGN_OR, RGN_NOT = -1, -2, -3
CSG_SPHERES = ((3.0, 4.0, 4.0, 2.0), (5.5, 4.0, 4.0, 2.0))      # (x0, y0, z0, r): centres 2.5 apart on the x axis
CSG_CYL = (9.0, 4.0, 1.0)                                        # (x0, y0, r), parallel to z
CSG_BOX = (12.0, 8.0, 8.0)


def csg_union_geometry(n_histories=60_000, n_batches=12, beam=False):
    G = 2
    if beam:                                              # pin J-b: absorber in the union, nothing anywhere else
        mats, ss = _materials([
            dict(sigma_t=[1.0, 1.0], sigma_c=[1.0, 1.0], sigma_f=[0.0, 0.0], nu=[0.0, 0.0], chi=[0.0, 0.0],
                 sigma_s=[[0.0, 0.0], [0.0, 0.0]]),
            dict(sigma_t=[0.0, 0.0], sigma_c=[0.0, 0.0], sigma_f=[0.0, 0.0], nu=[0.0, 0.0], chi=[0.0, 0.0],
                 sigma_s=[[0.0, 0.0], [0.0, 0.0]])], G)
        cell_mats = [0, 1, 1]
    else:
        mats, ss = _materials([
            dict(sigma_t=[0.8, 1.2], sigma_c=[0.15, 0.4], sigma_f=[0.05, 0.1], nu=[2.2, 2.5], chi=[0.7, 0.3],
                 sigma_s=[[0.4, 0.2], [0.0, 0.7]]),
            dict(sigma_t=[0.3, 0.5], sigma_c=[0.05, 0.1], sigma_f=[0.0, 0.0], nu=[0.0, 0.0], chi=[0.0, 0.0],
                 sigma_s=[[0.2, 0.05], [0.02, 0.38]])], G)
        cell_mats = [0, 0, 1]
    bx, by, bz = CSG_BOX
    surfs = [plane_x(0.0), plane_x(bx), plane_y(0.0), plane_y(by), plane_z(0.0), plane_z(bz),
             sphere(*CSG_SPHERES[0]), sphere(*CSG_SPHERES[1]), cylinder_z(*CSG_CYL)]
    bcs = [BC_VACUUM] * 6 + [BC_TRANSMISSION] * 3
    cells = [
        ([(6, -1), (7, -1)], cell_mats[0]),                                           # inside sphere 0 OR sphere 1
        ([(8, -1), (4, +1), (5, -1)], cell_mats[1]),                                  # the cylinder (plain intersection)
        ([(0, +1), (1, -1), (2, +1), (3, -1), (4, +1), (5, -1), (6, -1), (7, -1), (8, -1)], cell_mats[2]),
    ]
    A, O, N = RGN_AND, RGN_OR, RGN_NOT
    rpn = [[0, 1, O],
           [],
           [0, 1, A, 2, A, 3, A, 4, A, 5, A, 6, 7, O, 8, O, N, A]]                     # box AND NOT (s0 OR s1 OR cyl)
    off = np.cumsum([0] + [len(r) for r in rpn]).astype(np.int32)
    tok = np.array([t for r in rpn for t in r], dtype=np.int32)
    if beam:
        src = dict(lo=[0.0, 4.0, 4.0], hi=[0.0, 4.0, 4.0], t0=0.0, t1=0.0, pdf=[1.0, 0.0], mode=DIR_FIXED,
                   dir=[1.0, 0.0, 0.0])
    else:
        src = dict(lo=[0.5, 0.5, 0.5], hi=[11.5, 7.5, 7.5], t0=0.0, t1=1.0, pdf=[0.6, 0.4])
    mesh = dict(lo=[0.0, 0.0, 0.0], hi=[bx, by, bz], n=[12, 4, 2])
    T = np.array([0.0, 2.0, 5.0, 9.0, 20.0])
    p = _assemble("csg_union" + ("_beam" if beam else ""), mats, ss, [1.0, 0.4], surfs, bcs, cells, src, mesh, T,
                  T[1:].copy(), n_histories, n_batches, run_seed(11))
    p.meta["regions"] = (off, tok)
    return p


# ----------------------------------------------------------------------------------------
# Universes and lattices (DESIGN.md Appendix K): geometry given as a rectangular array of elements, each filled with
# a universe -- surfaces and cells in coordinates local to the element (origin at its centre in x and y, z unshifted).
# A universe cell lists half-spaces of the universe's own surfaces (index >= 0) or of the element's six faces
# (LAT_XLO .. LAT_ZHI).  The description travels in meta["lattice"]; the flat arrays of the Problem stay empty and
# the library / the oracle each expand it themselves.  Input tables only: no arithmetic of the method.
# ----------------------------------------------------------------------------------------
LAT_XLO, LAT_XHI, LAT_YLO, LAT_YHI, LAT_ZLO, LAT_ZHI = -1, -2, -3, -4, -5, -6


def _lattice_problem(name, mats, ss, speed, lattice, src, mesh, time_edges, census, n_histories, n_batches, seed, meta=None):
    p = _assemble(name, mats, ss, speed, [np.zeros(10)], [0], [], src, mesh, time_edges, census, n_histories, n_batches,
                  seed, meta=dict(meta or {}, lattice=lattice))
    p.surf_coef = np.zeros((0, 10)); p.surf_bc = _i32([])                   # no flat geometry: see meta["lattice"]
    return p


def config3_lattice(n_histories=10_000_000, n_batches=100, n_pins=17):
    """Config 3 written as a 17 x 17 lattice of two pin-cell universes (fuel A / fuel B in a checkerboard) instead of
    578 hand-written cells; the expansion must give config3_pin_lattice's tables exactly."""
    p, r, H = 1.26, 0.54, 10.0
    n = n_pins
    mats, ss, speed, k0 = config3_xs(p, r)

    def pin_universe(fuel):
        return dict(surf=[cylinder_z(0.0, 0.0, r)],
                    cells=[([(0, -1), (LAT_ZLO, +1), (LAT_ZHI, -1)], fuel),
                           ([(LAT_XLO, +1), (LAT_XHI, -1), (LAT_YLO, +1), (LAT_YHI, -1), (0, +1), (LAT_ZLO, +1),
                             (LAT_ZHI, -1)], 2)])
    lattice = dict(universes=[pin_universe(0), pin_universe(1)], nx=n, ny=n, x0=0.0, y0=0.0, pitch_x=p, pitch_y=p,
                   z_lo=0.0, z_hi=H, fill=[[(i + j) % 2 for i in range(n)] for j in range(n)],
                   bc=[BC_REFLECTIVE, BC_REFLECTIVE, BC_REFLECTIVE, BC_REFLECTIVE, BC_VACUUM, BC_VACUUM])
    c = 0.5 * n * p
    src = dict(lo=[c, c, 0.5 * H], hi=[c, c, 0.5 * H], t0=0.0, t1=0.0, pdf=mats["chi"][0].copy())
    mesh = dict(lo=[0.0, 0.0, 0.0], hi=[n * p, n * p, H], n=[n, n, 1])
    T = np.array([k * 5e-7 for k in range(21)], dtype=np.float64)
    return _lattice_problem("config3_lattice", mats, ss, speed, lattice, src, mesh, T, T[1:].copy(), n_histories,
                            n_batches, run_seed(3), meta=dict(k0=k0, pitch=p, radius=r))


LATTICE_MIXED = dict(nx=4, ny=3, x0=-2.5, y0=1.0, pitch_x=1.5, pitch_y=2.0, z_lo=-1.0, z_hi=3.0,
                     r_fuel=0.4, r_clad=0.55, ball=(0.1, -0.2, 1.0, 0.45))   # ball: local centre and radius


def lattice_mixed(n_histories=60_000, n_batches=12):
    """Parity / pin workload: a 4 x 3 lattice that does not start at the origin, with unequal pitches and three
    universes -- a clad pin (two concentric z-cylinders, three cells), a bare moderator box (one cell, no surface) and
    a box holding an off-centre ball (a translated general quadric); vacuum in x, reflective in y and at the bottom,
    vacuum on top; two groups; a source box over the whole lattice; a mesh that does not follow the elements."""
    G = 2
    L = LATTICE_MIXED
    mats, ss = _materials([
        dict(sigma_t=[0.8, 1.2], sigma_c=[0.15, 0.4], sigma_f=[0.05, 0.1], nu=[2.2, 2.5], chi=[0.7, 0.3],
             sigma_s=[[0.4, 0.2], [0.0, 0.7]]),                                  # fuel
        dict(sigma_t=[0.3, 0.5], sigma_c=[0.05, 0.1], sigma_f=[0.0, 0.0], nu=[0.0, 0.0], chi=[0.0, 0.0],
             sigma_s=[[0.2, 0.05], [0.02, 0.38]]),                               # clad
        dict(sigma_t=[0.6, 0.9], sigma_c=[0.1, 0.2], sigma_f=[0.0, 0.0], nu=[0.0, 0.0], chi=[0.0, 0.0],
             sigma_s=[[0.3, 0.2], [0.1, 0.6]]),                                  # moderator
    ], G)
    box = [(LAT_XLO, +1), (LAT_XHI, -1), (LAT_YLO, +1), (LAT_YHI, -1), (LAT_ZLO, +1), (LAT_ZHI, -1)]
    u_pin = dict(surf=[cylinder_z(0.0, 0.0, L["r_fuel"]), cylinder_z(0.0, 0.0, L["r_clad"])],
                 cells=[([(0, -1), (LAT_ZLO, +1), (LAT_ZHI, -1)], 0),
                        ([(0, +1), (1, -1), (LAT_ZLO, +1), (LAT_ZHI, -1)], 1),
                        (box + [(1, +1)], 2)])
    u_box = dict(surf=[], cells=[(box, 2)])
    u_ball = dict(surf=[sphere(*L["ball"])], cells=[([(0, -1)], 0), (box + [(0, +1)], 2)])
    fill = [[0, 1, 2, 0],
            [2, 0, 0, 1],
            [0, 2, 1, 0]]
    lattice = dict(universes=[u_pin, u_box, u_ball], nx=L["nx"], ny=L["ny"], x0=L["x0"], y0=L["y0"],
                   pitch_x=L["pitch_x"], pitch_y=L["pitch_y"], z_lo=L["z_lo"], z_hi=L["z_hi"], fill=fill,
                   bc=[BC_VACUUM, BC_VACUUM, BC_REFLECTIVE, BC_REFLECTIVE, BC_REFLECTIVE, BC_VACUUM])
    x1 = L["x0"] + L["nx"] * L["pitch_x"]; y1 = L["y0"] + L["ny"] * L["pitch_y"]
    src = dict(lo=[L["x0"], L["y0"], L["z_lo"]], hi=[x1, y1, L["z_hi"]], t0=0.0, t1=1.0, pdf=[0.6, 0.4])
    mesh = dict(lo=[L["x0"], L["y0"], L["z_lo"]], hi=[x1, y1, L["z_hi"]], n=[5, 4, 2])
    T = np.array([0.0, 1.0, 2.5, 5.0, 9.0])
    return _lattice_problem("lattice_mixed", mats, ss, [1.0, 0.4], lattice, src, mesh, T, np.array([2.0, 4.5, 9.0]),
                            n_histories, n_batches, run_seed(13))


CONFIGS["csg_union"] = csg_union_geometry
CONFIGS["config3_lattice"] = config3_lattice
CONFIGS["lattice_mixed"] = lattice_mixed


def get_config(name: str, **kw) -> Problem:
    return CONFIGS[name](**kw)
