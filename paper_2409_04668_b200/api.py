"""Thin ctypes binding of libmcdc.so: same names as include/mcdc.h, argument marshalling only.

PyTorch is used for exactly two things: the device workspace (a uint8 CUDA tensor whose data_ptr is
handed to mcdc_workspace_bind) and the CUDA stream handle.  If libmcdc.so is missing this module
raises at import of the first call -- there is no fallback path.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("MCDC_LIB_PATH") or os.path.join(_HERE, "libmcdc.so")

EXPORTED_SYMBOLS = [
    "mcdc_problem_create", "mcdc_problem_destroy", "mcdc_problem_reset", "mcdc_workspace_size", "mcdc_workspace_size_async", "mcdc_problem_info_get",
    "mcdc_workspace_bind", "mcdc_run", "mcdc_run_ex", "mcdc_tallies_get", "mcdc_tally_sums_get",
    "mcdc_counters_get", "mcdc_census_get", "mcdc_history_events_get", "mcdc_strerror",
    "mcdc_last_cuda_error", "mcdc_version", "mcdc_technique_set", "mcdc_census_after_get",
    "mcdc_state_size", "mcdc_state_export", "mcdc_state_import", "mcdc_run_eigenvalue",
    "mcdc_collision_tally_enable", "mcdc_collision_tallies_get", "mcdc_problem_create_csg", "mcdc_kernel_info_get",
    "mcdc_lattice_expand_size", "mcdc_lattice_expand", "mcdc_problem_create_lattice", "mcdc_tallies_get_noalloc",
]

NOALLOC_MAX_BINS = 1 << 20   # MCDC_NOALLOC_MAX_BINS of include/mcdc.h

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class McdcError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        msg = f"{where}: {mcdc_strerror(code)} ({code})"
        if detail:
            msg += f" [{detail}]"
        super().__init__(msg)


class ProblemDesc(C.Structure):
    _fields_ = [
        ("n_groups", C.c_int32), ("n_materials", C.c_int32), ("n_surfaces", C.c_int32), ("n_cells", C.c_int32),
        ("sigma_t", _dp), ("sigma_c", _dp), ("sigma_f", _dp), ("nu", _dp), ("chi", _dp),
        ("sigma_s", _dp), ("speed", _dp),
        ("surf_coef", _dp), ("surf_bc", _ip),
        ("cell_offset", _ip), ("hs_surface", _ip), ("hs_sense", _ip), ("cell_material", _ip),
        ("src_lo", C.c_double * 3), ("src_hi", C.c_double * 3), ("src_t0", C.c_double), ("src_t1", C.c_double),
        ("src_group_pdf", _dp), ("src_dir_mode", C.c_int32), ("src_dir", C.c_double * 3),
        ("mesh_lo", C.c_double * 3), ("mesh_hi", C.c_double * 3), ("mesh_n", C.c_int32 * 3),
        ("n_time_bins", C.c_int32), ("time_edges", _dp), ("n_census", C.c_int32), ("census_times", _dp),
    ]


class LatticeDesc(C.Structure):
    _fields_ = [("n_universes", C.c_int32), ("usurf_offset", _ip), ("usurf_coef", _dp), ("ucell_offset", _ip),
                ("uhs_offset", _ip), ("uhs_surface", _ip), ("uhs_sense", _ip), ("ucell_material", _ip),
                ("nx", C.c_int32), ("ny", C.c_int32), ("x0", C.c_double), ("y0", C.c_double), ("pitch_x", C.c_double),
                ("pitch_y", C.c_double), ("z_lo", C.c_double), ("z_hi", C.c_double), ("fill", _ip), ("bc", C.c_int32 * 6)]


class RunOpts(C.Structure):
    _fields_ = [("n_batches", C.c_uint32), ("first_history_id", C.c_uint64), ("record_history_events", C.c_int32),
                ("scheduler", C.c_int32), ("debug_pool_slots", C.c_uint32), ("debug_stage_tables", C.c_int32)]


class Counters(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost")] + \
               [(n, C.c_uint64) for n in ("histories", "segments", "collisions", "surf_hits", "census_events",
                                          "children", "lost_n", "batches", "kernel_launches")] + \
               [("ms_run", C.c_double), ("ms_transport", C.c_double), ("vr_gain", C.c_double), ("vr_loss", C.c_double),
                ("pc_removed", C.c_uint64), ("pc_added", C.c_uint64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class Technique(C.Structure):
    _fields_ = [("implicit_capture", C.c_int32), ("wr_threshold", C.c_double), ("wr_survive", C.c_double),
                ("population_control", C.c_int32), ("pc_target", C.c_uint64)]


_lib = None


class ProblemInfo(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("transmission_halfspaces", "certified_halfspaces", "cells", "one_bin_cells",
                                          "hot_table_bytes")] + [("warp_kernel_ok", C.c_int32), ("score_fast", C.c_int32),
                                                                     ("all_one_bin", C.c_int32), ("source_cell", C.c_int32)]


def lib_path() -> str:
    return _LIB_PATH


def lib():
    """Load libmcdc.so (once).  Raises if the CUDA extension has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} not found: build it with `python -m paper_2409_04668_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(_LIB_PATH)
    vp = C.c_void_p
    L.mcdc_problem_create.argtypes = [C.POINTER(ProblemDesc), C.POINTER(vp)]; L.mcdc_problem_create.restype = C.c_int
    L.mcdc_problem_create_csg.argtypes = [C.POINTER(ProblemDesc), _ip, _ip, C.POINTER(vp)]
    L.mcdc_problem_create_csg.restype = C.c_int
    i32p = C.POINTER(C.c_int32)
    L.mcdc_lattice_expand_size.argtypes = [C.POINTER(LatticeDesc), i32p, i32p, i32p]; L.mcdc_lattice_expand_size.restype = C.c_int
    L.mcdc_lattice_expand.argtypes = [C.POINTER(LatticeDesc), _dp, _ip, _ip, _ip, _ip, _ip]; L.mcdc_lattice_expand.restype = C.c_int
    L.mcdc_problem_create_lattice.argtypes = [C.POINTER(ProblemDesc), C.POINTER(LatticeDesc), C.POINTER(vp)]
    L.mcdc_problem_create_lattice.restype = C.c_int
    L.mcdc_problem_destroy.argtypes = [vp]; L.mcdc_problem_destroy.restype = None
    L.mcdc_problem_reset.argtypes = [vp]; L.mcdc_problem_reset.restype = C.c_int
    L.mcdc_workspace_size.argtypes = [vp, C.c_uint64, C.c_uint32, C.POINTER(C.c_size_t)]
    L.mcdc_workspace_size.restype = C.c_int
    L.mcdc_workspace_size_async.argtypes = [vp, C.c_uint64, C.c_uint32, C.POINTER(C.c_size_t)]
    L.mcdc_workspace_size_async.restype = C.c_int
    L.mcdc_problem_info_get.argtypes = [vp, C.POINTER(ProblemInfo)]; L.mcdc_problem_info_get.restype = C.c_int
    L.mcdc_workspace_bind.argtypes = [vp, vp, C.c_size_t, C.c_uint64, C.c_uint32, vp]
    L.mcdc_workspace_bind.restype = C.c_int
    L.mcdc_run.argtypes = [vp, C.c_uint64, C.c_uint64]; L.mcdc_run.restype = C.c_int
    L.mcdc_run_ex.argtypes = [vp, C.c_uint64, C.c_uint64, C.POINTER(RunOpts)]; L.mcdc_run_ex.restype = C.c_int
    L.mcdc_tallies_get.argtypes = [vp, _dp, _dp, C.c_size_t]; L.mcdc_tallies_get.restype = C.c_int
    L.mcdc_tallies_get_noalloc.argtypes = [vp, _dp, _dp, C.c_size_t]; L.mcdc_tallies_get_noalloc.restype = C.c_int
    L.mcdc_tally_sums_get.argtypes = [vp, _dp, _dp, C.c_size_t]; L.mcdc_tally_sums_get.restype = C.c_int
    L.mcdc_counters_get.argtypes = [vp, C.POINTER(Counters)]; L.mcdc_counters_get.restype = C.c_int
    L.mcdc_census_get.argtypes = [vp, _dp, C.POINTER(C.c_uint64), C.c_size_t]; L.mcdc_census_get.restype = C.c_int
    L.mcdc_history_events_get.argtypes = [vp, C.POINTER(C.c_uint32), C.c_size_t]
    L.mcdc_history_events_get.restype = C.c_int
    L.mcdc_run_eigenvalue.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, _dp]
    L.mcdc_run_eigenvalue.restype = C.c_int
    L.mcdc_collision_tally_enable.argtypes = [vp, C.c_int]; L.mcdc_collision_tally_enable.restype = C.c_int
    L.mcdc_collision_tallies_get.argtypes = [vp, _dp, _dp, C.c_size_t]; L.mcdc_collision_tallies_get.restype = C.c_int
    L.mcdc_technique_set.argtypes = [vp, C.POINTER(Technique)]; L.mcdc_technique_set.restype = C.c_int
    L.mcdc_census_after_get.argtypes = [vp, _dp, C.POINTER(C.c_uint64), C.c_size_t]
    L.mcdc_census_after_get.restype = C.c_int
    L.mcdc_state_size.argtypes = [vp, C.POINTER(C.c_size_t)]; L.mcdc_state_size.restype = C.c_int
    L.mcdc_state_export.argtypes = [vp, vp, C.c_size_t, C.c_int]; L.mcdc_state_export.restype = C.c_int
    L.mcdc_state_import.argtypes = [vp, vp, C.c_size_t, C.c_int]; L.mcdc_state_import.restype = C.c_int
    L.mcdc_kernel_info_get.argtypes = [vp, C.c_char_p, C.c_size_t]; L.mcdc_kernel_info_get.restype = C.c_int
    L.mcdc_strerror.argtypes = [C.c_int]; L.mcdc_strerror.restype = C.c_char_p
    L.mcdc_last_cuda_error.argtypes = [vp]; L.mcdc_last_cuda_error.restype = C.c_char_p
    L.mcdc_version.argtypes = []; L.mcdc_version.restype = C.c_char_p
    _lib = L
    return L


def mcdc_strerror(code: int) -> str:
    return lib().mcdc_strerror(int(code)).decode()


def mcdc_version() -> str:
    return lib().mcdc_version().decode()


def _check(rc, where, handle=None):
    if rc != 0:
        detail = ""
        if handle is not None and rc == -7:
            detail = lib().mcdc_last_cuda_error(handle).decode()
        raise McdcError(rc, where, detail)


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _vec3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


def _make_desc(prob):
    """workloads.Problem (or any object with the same attributes) -> (ProblemDesc, keep-alive list)."""
    d = ProblemDesc()
    keep = []
    d.n_groups, d.n_materials = int(prob.n_groups), int(prob.n_materials)
    d.n_surfaces, d.n_cells = int(prob.n_surfaces), int(prob.n_cells)
    for name in ("sigma_t", "sigma_c", "sigma_f", "nu", "chi", "sigma_s", "speed", "surf_coef"):
        a = np.ascontiguousarray(getattr(prob, name), dtype=np.float64); keep.append(a)
        setattr(d, name, _d(a))
    for name in ("surf_bc", "cell_offset", "hs_surface", "hs_sense", "cell_material"):
        a = np.ascontiguousarray(getattr(prob, name), dtype=np.int32); keep.append(a)
        setattr(d, name, _i(a))
    d.src_lo, d.src_hi = _vec3(prob.src_lo), _vec3(prob.src_hi)
    d.src_t0, d.src_t1 = float(prob.src_t0), float(prob.src_t1)
    pdf = np.ascontiguousarray(prob.src_group_pdf, dtype=np.float64); keep.append(pdf)
    d.src_group_pdf = _d(pdf)
    d.src_dir_mode = int(prob.src_dir_mode); d.src_dir = _vec3(prob.src_dir)
    d.mesh_lo, d.mesh_hi = _vec3(prob.mesh_lo), _vec3(prob.mesh_hi)
    d.mesh_n = (C.c_int32 * 3)(*[int(v) for v in prob.mesh_n])
    te = np.ascontiguousarray(prob.time_edges, dtype=np.float64); keep.append(te)
    ce = np.ascontiguousarray(prob.census_times, dtype=np.float64); keep.append(ce)
    d.n_time_bins, d.time_edges = len(te) - 1, _d(te)
    d.n_census, d.census_times = len(ce), _d(ce)
    return d, keep


def _make_lattice(lat):
    """The lattice dict of workloads.configs (universes = [{surf: [coef10, ...], cells: [([(surface, sense), ...],
    material), ...]}, ...], nx, ny, x0, y0, pitch_x, pitch_y, z_lo, z_hi, fill [ny][nx], bc [6]) -> (LatticeDesc, keep-alive)."""
    us_off, uc_off, uh_off, coef, hs_s, hs_n, mat = [0], [0], [0], [], [], [], []
    for u in lat["universes"]:
        coef += [np.asarray(c, dtype=np.float64).reshape(10) for c in u["surf"]]
        us_off.append(len(coef))
        for hs, m in u["cells"]:
            for s, sense in hs:
                hs_s.append(int(s)); hs_n.append(int(sense))
            uh_off.append(len(hs_s)); mat.append(int(m))
        uc_off.append(len(mat))
    arr = dict(us_off=np.asarray(us_off, dtype=np.int32), uc_off=np.asarray(uc_off, dtype=np.int32),
               uh_off=np.asarray(uh_off, dtype=np.int32), hs_s=np.asarray(hs_s, dtype=np.int32),
               hs_n=np.asarray(hs_n, dtype=np.int32), mat=np.asarray(mat, dtype=np.int32),
               coef=np.ascontiguousarray(np.stack(coef) if coef else np.zeros((1, 10)), dtype=np.float64),
               fill=np.ascontiguousarray(np.asarray(lat["fill"], dtype=np.int32).reshape(-1)))
    d = LatticeDesc()
    d.n_universes = len(lat["universes"])
    d.usurf_offset, d.usurf_coef, d.ucell_offset, d.uhs_offset = _i(arr["us_off"]), _d(arr["coef"]), _i(arr["uc_off"]), _i(arr["uh_off"])
    d.uhs_surface, d.uhs_sense, d.ucell_material = _i(arr["hs_s"]), _i(arr["hs_n"]), _i(arr["mat"])
    d.nx, d.ny = int(lat["nx"]), int(lat["ny"])
    if arr["fill"].size != d.nx * d.ny:
        raise McdcError(-3, "mcdc_lattice", "fill must be [ny][nx]")
    d.x0, d.y0, d.pitch_x, d.pitch_y = float(lat["x0"]), float(lat["y0"]), float(lat["pitch_x"]), float(lat["pitch_y"])
    d.z_lo, d.z_hi = float(lat["z_lo"]), float(lat["z_hi"])
    d.fill = _i(arr["fill"])
    d.bc = (C.c_int32 * 6)(*[int(b) for b in lat["bc"]])
    return d, arr


def mcdc_lattice_expand(lat) -> dict:
    """The flat geometry of a lattice description (mcdc_lattice_expand_size + mcdc_lattice_expand; no device needed)."""
    d, keep = _make_lattice(lat)
    nS, nC, nH = C.c_int32(), C.c_int32(), C.c_int32()
    _check(lib().mcdc_lattice_expand_size(C.byref(d), C.byref(nS), C.byref(nC), C.byref(nH)), "mcdc_lattice_expand_size")
    out = dict(surf_coef=np.empty((nS.value, 10)), surf_bc=np.empty(nS.value, dtype=np.int32),
               cell_offset=np.empty(nC.value + 1, dtype=np.int32), hs_surface=np.empty(nH.value, dtype=np.int32),
               hs_sense=np.empty(nH.value, dtype=np.int32), cell_material=np.empty(nC.value, dtype=np.int32))
    _check(lib().mcdc_lattice_expand(C.byref(d), _d(out["surf_coef"]), _i(out["surf_bc"]), _i(out["cell_offset"]),
                                     _i(out["hs_surface"]), _i(out["hs_sense"]), _i(out["cell_material"])), "mcdc_lattice_expand")
    return out


def mcdc_lattice_expand_size(lat):
    d, keep = _make_lattice(lat)
    nS, nC, nH = C.c_int32(), C.c_int32(), C.c_int32()
    _check(lib().mcdc_lattice_expand_size(C.byref(d), C.byref(nS), C.byref(nC), C.byref(nH)), "mcdc_lattice_expand_size")
    return nS.value, nC.value, nH.value


def mcdc_problem_create_lattice(prob, lat):
    d, keep = _make_desc(prob)
    ld, keep2 = _make_lattice(lat)
    h = C.c_void_p()
    _check(lib().mcdc_problem_create_lattice(C.byref(d), C.byref(ld), C.byref(h)), "mcdc_problem_create_lattice")
    return h


# ---- functions with the names of include/mcdc.h ------------------------------------------------
def mcdc_problem_create(prob):
    """prob.meta["regions"] = (region_offset, region_rpn), when present, makes this mcdc_problem_create_csg;
    prob.meta["lattice"] makes it mcdc_problem_create_lattice."""
    lat = (getattr(prob, "meta", None) or {}).get("lattice")
    if lat is not None:
        return mcdc_problem_create_lattice(prob, lat)
    rgn = (getattr(prob, "meta", None) or {}).get("regions")
    if rgn is not None:
        return mcdc_problem_create_csg(prob, rgn[0], rgn[1])
    d, keep = _make_desc(prob)
    h = C.c_void_p()
    _check(lib().mcdc_problem_create(C.byref(d), C.byref(h)), "mcdc_problem_create")
    return h


def mcdc_problem_create_csg(prob, region_offset, region_rpn):
    d, keep = _make_desc(prob)
    ro = np.ascontiguousarray(region_offset, dtype=np.int32); rt = np.ascontiguousarray(region_rpn, dtype=np.int32)
    h = C.c_void_p()
    _check(lib().mcdc_problem_create_csg(C.byref(d), _i(ro), _i(rt), C.byref(h)), "mcdc_problem_create_csg")
    return h


def mcdc_problem_destroy(h):
    lib().mcdc_problem_destroy(h)


def mcdc_problem_reset(h):
    _check(lib().mcdc_problem_reset(h), "mcdc_problem_reset", h)


def mcdc_workspace_size(h, max_histories_per_subbatch, max_batches_in_flight) -> int:
    n = C.c_size_t()
    _check(lib().mcdc_workspace_size(h, int(max_histories_per_subbatch), int(max_batches_in_flight), C.byref(n)),
           "mcdc_workspace_size", h)
    return int(n.value)


def mcdc_problem_info_get(h) -> dict:
    info = ProblemInfo()
    _check(lib().mcdc_problem_info_get(h, C.byref(info)), "mcdc_problem_info_get", h)
    return {n: int(getattr(info, n)) for n, _ in ProblemInfo._fields_}


def mcdc_kernel_info_get(h) -> str:
    buf = C.create_string_buffer(256)
    _check(lib().mcdc_kernel_info_get(h, buf, 256), "mcdc_kernel_info_get", h)
    return buf.value.decode()


def mcdc_workspace_size_async(h, max_histories_per_subbatch, max_batches_in_flight) -> int:
    n = C.c_size_t(0)
    _check(lib().mcdc_workspace_size_async(h, int(max_histories_per_subbatch), int(max_batches_in_flight), C.byref(n)),
           "mcdc_workspace_size_async", h)
    return int(n.value)


def mcdc_workspace_bind(h, dev_ptr, nbytes, max_histories_per_subbatch, max_batches_in_flight, cuda_stream=0):
    _check(lib().mcdc_workspace_bind(h, C.c_void_p(int(dev_ptr)), int(nbytes), int(max_histories_per_subbatch),
                                     int(max_batches_in_flight), C.c_void_p(int(cuda_stream))),
           "mcdc_workspace_bind", h)


def mcdc_run(h, n_histories, seed):
    _check(lib().mcdc_run(h, int(n_histories), int(seed)), "mcdc_run", h)


SCHED_ASYNC, SCHED_CENSUS_STEPPED = 0, 1


def mcdc_run_ex(h, n_histories, seed, n_batches=1, first_history_id=0, record_history_events=False, scheduler=0,
                debug_pool_slots=0, debug_stage_tables=0):
    o = RunOpts(int(n_batches), int(first_history_id), int(bool(record_history_events)), int(scheduler),
                int(debug_pool_slots), int(debug_stage_tables))
    _check(lib().mcdc_run_ex(h, int(n_histories), int(seed), C.byref(o)), "mcdc_run_ex", h)


def mcdc_run_eigenvalue(h, n_particles, seed, n_inactive, n_active):
    k = np.zeros(int(n_inactive) + int(n_active))
    _check(lib().mcdc_run_eigenvalue(h, int(n_particles), int(seed), int(n_inactive), int(n_active), _d(k)),
           "mcdc_run_eigenvalue", h)
    return k


def mcdc_tallies_get(h, n_bins, out=None):
    """out = (mean, sdev): caller-owned contiguous float64 arrays of n_bins elements to fill (e.g. views of pinned
    host memory, which the device-to-host copy then reaches at full PCIe rate); default: fresh arrays."""
    if out is None:
        mean = np.empty(n_bins); sdev = np.empty(n_bins)
    else:
        mean, sdev = out
        if mean.size != n_bins or sdev.size != n_bins or mean.dtype != np.float64 or sdev.dtype != np.float64 or \
                not mean.flags.c_contiguous or not sdev.flags.c_contiguous:
            raise McdcError(-4, "mcdc_tallies_get", "out arrays must be contiguous float64 of n_bins elements")
    _check(lib().mcdc_tallies_get(h, _d(mean), _d(sdev), n_bins), "mcdc_tallies_get", h)
    return mean, sdev


def mcdc_tallies_get_noalloc(h, n_bins, out=None):
    """mcdc_tallies_get for a caller that must not allocate on the GPU (all device memory belongs to a pool, or the
    read-out sits in a timing-critical loop): same numbers, but the device scratch is a fixed 16 MiB array inside
    libmcdc.so, so no cudaMalloc / cudaFree happens.  Limits (include/mcdc.h): at most NOALLOC_MAX_BINS bins, else
    McdcError(-4) whose text names the limit; one array per GPU shared by all handles, so do not run two of these
    calls concurrently on one GPU; make the first call per GPU before any stream capture starts.  out as in
    mcdc_tallies_get (pass pinned arrays to keep the host side allocation-free as well)."""
    if out is None:
        mean = np.empty(n_bins); sdev = np.empty(n_bins)
    else:
        mean, sdev = out
        if mean.size != n_bins or sdev.size != n_bins or mean.dtype != np.float64 or sdev.dtype != np.float64 or \
                not mean.flags.c_contiguous or not sdev.flags.c_contiguous:
            raise McdcError(-4, "mcdc_tallies_get_noalloc", "out arrays must be contiguous float64 of n_bins elements")
    rc = lib().mcdc_tallies_get_noalloc(h, _d(mean), _d(sdev), n_bins)
    if rc in (-1, -4):   # the library leaves the reason (over the limit / wrong current device) in its error text
        raise McdcError(rc, "mcdc_tallies_get_noalloc", lib().mcdc_last_cuda_error(h).decode())
    _check(rc, "mcdc_tallies_get_noalloc", h)
    return mean, sdev


def mcdc_collision_tally_enable(h, on=True):
    _check(lib().mcdc_collision_tally_enable(h, int(bool(on))), "mcdc_collision_tally_enable", h)


def mcdc_collision_tallies_get(h, n_bins):
    mean = np.empty(n_bins); sdev = np.empty(n_bins)
    _check(lib().mcdc_collision_tallies_get(h, _d(mean), _d(sdev), n_bins), "mcdc_collision_tallies_get", h)
    return mean, sdev


def mcdc_tally_sums_get(h, n_bins):
    s = np.empty(n_bins); q = np.empty(n_bins)
    _check(lib().mcdc_tally_sums_get(h, _d(s), _d(q), n_bins), "mcdc_tally_sums_get", h)
    return s, q


def mcdc_counters_get(h) -> dict:
    c = Counters()
    _check(lib().mcdc_counters_get(h, C.byref(c)), "mcdc_counters_get", h)
    return c.as_dict()


def mcdc_census_get(h, n_census):
    w = np.empty(n_census); n = np.empty(n_census, dtype=np.uint64)
    _check(lib().mcdc_census_get(h, _d(w), n.ctypes.data_as(C.POINTER(C.c_uint64)), n_census), "mcdc_census_get", h)
    return w, n


def mcdc_history_events_get(h, n_histories):
    ev = np.empty((n_histories, 4), dtype=np.uint32)
    _check(lib().mcdc_history_events_get(h, ev.ctypes.data_as(C.POINTER(C.c_uint32)), n_histories),
           "mcdc_history_events_get", h)
    return ev


def mcdc_technique_set(h, implicit_capture=False, wr_threshold=0.0, wr_survive=0.0, population_control=False,
                       pc_target=0):
    t = Technique(int(bool(implicit_capture)), float(wr_threshold), float(wr_survive), int(bool(population_control)),
                  int(pc_target))
    _check(lib().mcdc_technique_set(h, C.byref(t)), "mcdc_technique_set", h)


def mcdc_census_after_get(h, n_census):
    w = np.empty(n_census); n = np.empty(n_census, dtype=np.uint64)
    _check(lib().mcdc_census_after_get(h, _d(w), n.ctypes.data_as(C.POINTER(C.c_uint64)), n_census),
           "mcdc_census_after_get", h)
    return w, n


def mcdc_state_size(h) -> int:
    n = C.c_size_t(0)
    _check(lib().mcdc_state_size(h, C.byref(n)), "mcdc_state_size", h)
    return int(n.value)


def mcdc_state_export(h, ptr, n_doubles, on_device):
    _check(lib().mcdc_state_export(h, C.c_void_p(int(ptr)), int(n_doubles), int(bool(on_device))), "mcdc_state_export", h)


def mcdc_state_import(h, ptr, n_doubles, on_device):
    _check(lib().mcdc_state_import(h, C.c_void_p(int(ptr)), int(n_doubles), int(bool(on_device))), "mcdc_state_import", h)


# ---- convenience wrapper: owns the handle and the torch workspace ------------------------------
class Problem:
    """Handle + PyTorch-owned workspace.  Marshalling only; all work happens in libmcdc.so."""

    def __init__(self, prob, max_histories_per_subbatch=None, max_batches_in_flight=None, device="cuda:0",
                 workspace_scale=1.0, async_only=False):
        import torch  # device memory and stream only

        if not torch.cuda.is_available():
            raise RuntimeError("paper_2409_04668_b200 needs a CUDA device (no CPU fallback)")
        self.prob = prob
        self.n_bins = int(prob.n_bins)
        self.shape = prob.tally_shape()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self._h = mcdc_problem_create(prob)
        nb = int(max_batches_in_flight or max(1, getattr(prob, "n_batches", 1)))
        nh = int(max_histories_per_subbatch or max(1, getattr(prob, "n_histories", 1)))
        self._async_only = bool(async_only)
        self._bind(nh, nb, workspace_scale)

    def _bind(self, nh, nb, scale=1.0):
        import torch

        size = mcdc_workspace_size_async if self._async_only else mcdc_workspace_size
        nbytes = int(size(self._h, nh, nb) * scale)
        self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self._ws.data_ptr() + 255) // 256 * 256
        self._stream = torch.cuda.current_stream(self.device)
        mcdc_workspace_bind(self._h, ptr, nbytes, nh, nb, self._stream.cuda_stream)
        self.workspace_bytes = nbytes
        self.max_hist, self.max_slots = nh, nb

    def close(self):
        if getattr(self, "_h", None):
            mcdc_problem_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self):
        mcdc_problem_reset(self._h)

    def info(self):
        return mcdc_problem_info_get(self._h)

    def kernel_info(self):
        return mcdc_kernel_info_get(self._h)

    def run(self, n_histories=None, seed=None, n_batches=None, first_history_id=0, record_history_events=False,
            scheduler=0, debug_pool_slots=0, debug_stage_tables=0):
        n = int(n_histories if n_histories is not None else self.prob.n_histories)
        s = int(seed if seed is not None else self.prob.seed)
        b = int(n_batches if n_batches is not None else self.prob.n_batches)
        mcdc_run_ex(self._h, n, s, b, first_history_id, record_history_events, scheduler, debug_pool_slots,
                    debug_stage_tables)
        self._last_n = n

    def run_eigenvalue(self, n_particles=None, seed=None, n_inactive=0, n_active=1):
        n = int(n_particles if n_particles is not None else self.prob.n_histories)
        s = int(seed if seed is not None else self.prob.seed)
        return mcdc_run_eigenvalue(self._h, n, s, n_inactive, n_active)

    def tallies(self):
        m, s = mcdc_tallies_get(self._h, self.n_bins)
        return m.reshape(self.shape), s.reshape(self.shape)

    def tallies_noalloc(self):
        """tallies() through mcdc_tallies_get_noalloc: no device allocation, at most NOALLOC_MAX_BINS bins."""
        m, s = mcdc_tallies_get_noalloc(self._h, self.n_bins)
        return m.reshape(self.shape), s.reshape(self.shape)

    def enable_collision_tally(self, on=True):
        mcdc_collision_tally_enable(self._h, on)

    def collision_tallies(self):
        m, s = mcdc_collision_tallies_get(self._h, self.n_bins)
        return m.reshape(self.shape), s.reshape(self.shape)

    def tally_sums(self):
        a, b = mcdc_tally_sums_get(self._h, self.n_bins)
        return a.reshape(self.shape), b.reshape(self.shape)

    def counters(self):
        return mcdc_counters_get(self._h)

    def census(self):
        return mcdc_census_get(self._h, int(self.prob.n_census))

    def history_events(self):
        return mcdc_history_events_get(self._h, self._last_n)

    def set_technique(self, **kw):
        mcdc_technique_set(self._h, **kw)

    def census_after(self):
        return mcdc_census_after_get(self._h, int(self.prob.n_census))

    # ---- multi-rank: the accumulators as one fp64 vector (include/mcdc.h) ----
    def state_size(self):
        return mcdc_state_size(self._h)

    def state_export(self, tensor):
        """tensor: contiguous float64 torch tensor of state_size() elements, on this device or on the host."""
        mcdc_state_export(self._h, tensor.data_ptr(), tensor.numel(), tensor.is_cuda)

    def state_import(self, tensor):
        mcdc_state_import(self._h, tensor.data_ptr(), tensor.numel(), tensor.is_cuda)

    def all_reduce(self, group=None):
        """Sum the accumulators of all ranks into every rank's handle (NCCL on the device buffer)."""
        from .sharding import all_reduce_state
        all_reduce_state(self, group=group, device=self.device)
