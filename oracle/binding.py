"""ctypes binding of the oracle library (oracle/mcdc_oracle.cpp).  Test infrastructure only."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mcdc_oracle.cpp")
# ORACLE_SANITIZE=1: a second build with AddressSanitizer + UBSan (-O1 -g, same -ffp-contract=off), loaded instead of
# the plain one; run the suite with LD_PRELOAD=$(gcc -print-file-name=libasan.so) (profiles/r02_sanitizers.md)
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")
_LIB = os.path.join(_HERE, "libmcdc_oracle_asan.so" if _SANITIZE else "libmcdc_oracle.so")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class _Desc(C.Structure):
    _fields_ = [
        ("G", C.c_int32), ("M", C.c_int32), ("S", C.c_int32), ("C", C.c_int32),
        ("sigma_t", _dp), ("sigma_c", _dp), ("sigma_f", _dp), ("nu", _dp), ("chi", _dp),
        ("sigma_s", _dp), ("speed", _dp),
        ("surf_coef", _dp), ("surf_bc", _ip),
        ("cell_offset", _ip), ("hs_surface", _ip), ("hs_sense", _ip), ("cell_material", _ip),
        ("src_lo", C.c_double * 3), ("src_hi", C.c_double * 3), ("src_t0", C.c_double), ("src_t1", C.c_double),
        ("src_group_pdf", _dp), ("src_dir_mode", C.c_int32), ("src_dir", C.c_double * 3),
        ("mesh_lo", C.c_double * 3), ("mesh_hi", C.c_double * 3), ("mesh_n", C.c_int32 * 3),
        ("Nt", C.c_int32), ("time_edges", _dp), ("K", C.c_int32), ("census", _dp),
    ]


class Counters(C.Structure):
    _fields_ = [(n, C.c_double) for n in
                ("source", "production", "capture", "fission_abs", "leak", "census_final", "lost")] + \
               [(n, C.c_uint64) for n in
                ("histories", "segments", "collisions", "surf_hits", "census_events", "children", "lost_n", "batches")] + \
               [("vr_gain", C.c_double), ("vr_loss", C.c_double), ("pc_removed", C.c_uint64), ("pc_added", C.c_uint64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class _Technique(C.Structure):
    _fields_ = [("implicit_capture", C.c_int32), ("wr_threshold", C.c_double), ("wr_survive", C.c_double),
                ("population_control", C.c_int32), ("pc_target", C.c_uint64)]


class _RunOpts(C.Structure):
    _fields_ = [("n_batches", C.c_uint32), ("first_history_id", C.c_uint64), ("record_history_events", C.c_int32),
                ("bank_fifo", C.c_int32), ("reverse_histories", C.c_int32)]


def lib_path() -> str:
    return _LIB


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -ffp-contract=off).  Building the checker is not using it."""
    hdr = os.path.join(_HERE, "mcdc_oracle.h")
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(_SRC), os.path.getmtime(hdr))):
        return _LIB
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] \
        if _SANITIZE else ["-O2"]
    cmd = ["g++"] + opt + ["-ffp-contract=off", "-std=c++17", "-fPIC", "-shared", "-Wall", "-o", _LIB, _SRC]
    subprocess.check_call(cmd)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = C.CDLL(_LIB)
    vp = C.c_void_p
    L.orc_create.argtypes = [C.POINTER(_Desc), C.POINTER(vp)]; L.orc_create.restype = C.c_int
    L.orc_destroy.argtypes = [vp]; L.orc_destroy.restype = None
    L.orc_reset.argtypes = [vp]; L.orc_reset.restype = None
    L.orc_run.argtypes = [vp, C.c_uint64, C.c_uint64, C.POINTER(_RunOpts)]; L.orc_run.restype = C.c_int
    L.orc_tallies_get.argtypes = [vp, _dp, _dp, C.c_size_t]; L.orc_tallies_get.restype = C.c_int
    L.orc_tally_sums_get.argtypes = [vp, _dp, _dp, C.c_size_t]; L.orc_tally_sums_get.restype = C.c_int
    L.orc_counters_get.argtypes = [vp, C.POINTER(Counters)]; L.orc_counters_get.restype = C.c_int
    L.orc_census_get.argtypes = [vp, _dp, C.POINTER(C.c_uint64), C.c_size_t]; L.orc_census_get.restype = C.c_int
    L.orc_history_events_get.argtypes = [vp, C.POINTER(C.c_uint32), C.c_size_t]; L.orc_history_events_get.restype = C.c_int
    L.orc_mix64.argtypes = [C.c_uint64]; L.orc_mix64.restype = C.c_uint64
    L.orc_source_key.argtypes = [C.c_uint64, C.c_uint64]; L.orc_source_key.restype = C.c_uint64
    L.orc_child_key.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32]; L.orc_child_key.restype = C.c_uint64
    L.orc_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
    L.orc_philox4x32_10.restype = None
    L.orc_draws.argtypes = [C.c_uint64, C.c_uint32, C.c_size_t, _dp]; L.orc_draws.restype = None
    L.orc_surface_distance.argtypes = [_dp, _dp, _dp, C.c_int]; L.orc_surface_distance.restype = C.c_double
    L.orc_locate.argtypes = [vp, _dp, _dp]; L.orc_locate.restype = C.c_int
    L.orc_stream.argtypes = [vp, _dp, _dp, _ip, C.c_int]; L.orc_stream.restype = C.c_int
    L.orc_score_segment.argtypes = [vp, _dp, _dp, C.c_double, C.c_int, C.c_double, C.c_double]
    L.orc_score_segment.restype = C.c_int
    L.orc_close_batch.argtypes = [vp, C.c_uint64]; L.orc_close_batch.restype = C.c_int
    L.orc_run_eigenvalue.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_int32, _dp]
    L.orc_run_eigenvalue.restype = C.c_int
    L.orc_collision_tally_enable.argtypes = [vp, C.c_int]; L.orc_collision_tally_enable.restype = C.c_int
    L.orc_collision_tallies_get.argtypes = [vp, _dp, _dp, C.c_size_t]; L.orc_collision_tallies_get.restype = C.c_int
    L.orc_regions_set.argtypes = [vp, _ip, _ip]; L.orc_regions_set.restype = C.c_int
    L.orc_technique_set.argtypes = [vp, C.POINTER(_Technique)]; L.orc_technique_set.restype = C.c_int
    L.orc_census_after_get.argtypes = [vp, _dp, C.POINTER(C.c_uint64), C.c_size_t]; L.orc_census_after_get.restype = C.c_int
    L.orc_population_control.argtypes = [vp, C.c_size_t, _dp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint32), C.c_uint64,
                                         _ip, _dp]
    L.orc_population_control.restype = C.c_int
    _lib = L
    return L


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _vec3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


# ---- unit-level helpers -------------------------------------------------------------------
def mix64(z: int) -> int:
    return int(_load().orc_mix64(C.c_uint64(z & (2 ** 64 - 1))))


def source_key(seed: int, h: int) -> int:
    return int(_load().orc_source_key(seed, h))


def child_key(parent_key: int, c0: int, j: int) -> int:
    return int(_load().orc_child_key(parent_key, c0, j))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) for x in ctr]); k = (C.c_uint32 * 2)(*[int(x) for x in key])
    o = (C.c_uint32 * 4)()
    _load().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def draws(key: int, first_ctr: int, n: int) -> np.ndarray:
    out = np.empty(n, dtype=np.float64)
    _load().orc_draws(key, first_ctr, n, _d(out))
    return out


def surface_distance(coef, r, omega, on_surface=False) -> float:
    c = np.ascontiguousarray(coef, dtype=np.float64)
    rr = np.ascontiguousarray(r, dtype=np.float64); oo = np.ascontiguousarray(omega, dtype=np.float64)
    return float(_load().orc_surface_distance(_d(c), _d(rr), _d(oo), int(bool(on_surface))))


# ---- problem handle -------------------------------------------------------------------------
class Oracle:
    """Oracle problem handle built from a workloads.Problem."""

    def __init__(self, prob):
        L = _load()
        self._L = L
        if getattr(prob, "meta", {}).get("lattice") is not None:   # universes / lattices: expanded here (oracle/lattice.py)
            from .lattice import flat_problem
            prob = flat_problem(prob)
        self.prob = prob
        d = _Desc()
        d.G, d.M, d.S, d.C = prob.n_groups, prob.n_materials, prob.n_surfaces, prob.n_cells
        self._keep = []
        for name in ("sigma_t", "sigma_c", "sigma_f", "nu", "chi", "sigma_s", "speed", "surf_coef"):
            a = np.ascontiguousarray(getattr(prob, name), dtype=np.float64); self._keep.append(a)
            setattr(d, name, _d(a))
        for name in ("surf_bc", "cell_offset", "hs_surface", "hs_sense", "cell_material"):
            a = np.ascontiguousarray(getattr(prob, name), dtype=np.int32); self._keep.append(a)
            setattr(d, name, _i(a))
        d.src_lo = _vec3(prob.src_lo); d.src_hi = _vec3(prob.src_hi)
        d.src_t0, d.src_t1 = prob.src_t0, prob.src_t1
        pdf = np.ascontiguousarray(prob.src_group_pdf, dtype=np.float64); self._keep.append(pdf)
        d.src_group_pdf = _d(pdf)
        d.src_dir_mode = prob.src_dir_mode; d.src_dir = _vec3(prob.src_dir)
        d.mesh_lo = _vec3(prob.mesh_lo); d.mesh_hi = _vec3(prob.mesh_hi)
        d.mesh_n = (C.c_int32 * 3)(*[int(v) for v in prob.mesh_n])
        te = np.ascontiguousarray(prob.time_edges, dtype=np.float64); self._keep.append(te)
        ce = np.ascontiguousarray(prob.census_times, dtype=np.float64); self._keep.append(ce)
        d.Nt, d.time_edges, d.K, d.census = prob.n_time_bins, _d(te), prob.n_census, _d(ce)
        h = C.c_void_p()
        rc = L.orc_create(C.byref(d), C.byref(h))
        if rc != 0:
            raise RuntimeError(f"orc_create failed: {rc}")
        self._h = h
        self.n_bins = prob.n_bins
        self._last_n = 0
        rgn = getattr(prob, "meta", {}).get("regions")     # (region_offset, region_rpn) of a general-CSG workload
        if rgn is not None:
            ro = np.ascontiguousarray(rgn[0], dtype=np.int32); rt = np.ascontiguousarray(rgn[1], dtype=np.int32)
            self._keep += [ro, rt]
            if L.orc_regions_set(h, _i(ro), _i(rt)) != 0:
                raise RuntimeError("orc_regions_set failed")

    def close(self):
        if getattr(self, "_h", None):
            self._L.orc_destroy(self._h); self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def reset(self):
        self._L.orc_reset(self._h)

    def set_technique(self, implicit_capture=False, wr_threshold=0.0, wr_survive=0.0, population_control=False,
                      pc_target=0):
        t = _Technique(int(implicit_capture), float(wr_threshold), float(wr_survive), int(population_control),
                       int(pc_target))
        if self._L.orc_technique_set(self._h, C.byref(t)) != 0:
            raise RuntimeError("orc_technique_set failed")

    def census_after(self):
        K = self.prob.n_census
        w = np.empty(K); n = np.empty(K, dtype=np.uint64)
        self._L.orc_census_after_get(self._h, _d(w), n.ctypes.data_as(C.POINTER(C.c_uint64)), K)
        return w, n

    def population_control(self, w, key, ctr, target):
        w = np.ascontiguousarray(w, dtype=np.float64); key = np.ascontiguousarray(key, dtype=np.uint64)
        ctr = np.ascontiguousarray(ctr, dtype=np.uint32)
        n_out = np.zeros(len(w), dtype=np.int32); w_t = C.c_double(0.0)
        self._L.orc_population_control(self._h, len(w), _d(w), key.ctypes.data_as(C.POINTER(C.c_uint64)),
                                       ctr.ctypes.data_as(C.POINTER(C.c_uint32)), int(target), _i(n_out), C.byref(w_t))
        return n_out, w_t.value

    def run(self, n_histories, seed, n_batches=1, first_history_id=0, record_history_events=False,
            bank_fifo=False, reverse_histories=False):
        o = _RunOpts(int(n_batches), int(first_history_id), int(record_history_events), int(bank_fifo),
                     int(reverse_histories))
        rc = self._L.orc_run(self._h, int(n_histories), int(seed), C.byref(o))
        if rc != 0:
            raise RuntimeError(f"orc_run failed: {rc}")
        self._last_n = int(n_histories)

    def run_eigenvalue(self, n_particles, seed, n_inactive, n_active, reverse_order=False):
        k = np.zeros(int(n_inactive) + int(n_active))
        rc = self._L.orc_run_eigenvalue(self._h, int(n_particles), int(seed), int(n_inactive), int(n_active),
                                        int(reverse_order), _d(k))
        if rc != 0:
            raise RuntimeError(f"orc_run_eigenvalue failed: {rc}")
        return k

    def tallies(self):
        mean = np.empty(self.n_bins); sdev = np.empty(self.n_bins)
        rc = self._L.orc_tallies_get(self._h, _d(mean), _d(sdev), self.n_bins)
        if rc != 0:
            raise RuntimeError(f"orc_tallies_get failed: {rc}")
        shp = self.prob.tally_shape()
        return mean.reshape(shp), sdev.reshape(shp)

    def enable_collision_tally(self, on=True):
        self._L.orc_collision_tally_enable(self._h, int(bool(on)))

    def collision_tallies(self):
        mean = np.empty(self.n_bins); sdev = np.empty(self.n_bins)
        rc = self._L.orc_collision_tallies_get(self._h, _d(mean), _d(sdev), self.n_bins)
        if rc != 0:
            raise RuntimeError(f"orc_collision_tallies_get failed: {rc}")
        shp = self.prob.tally_shape()
        return mean.reshape(shp), sdev.reshape(shp)

    def tally_sums(self):
        s = np.empty(self.n_bins); q = np.empty(self.n_bins)
        rc = self._L.orc_tally_sums_get(self._h, _d(s), _d(q), self.n_bins)
        if rc != 0:
            raise RuntimeError(f"orc_tally_sums_get failed: {rc}")
        shp = self.prob.tally_shape()
        return s.reshape(shp), q.reshape(shp)

    def counters(self) -> dict:
        c = Counters()
        self._L.orc_counters_get(self._h, C.byref(c))
        return c.as_dict()

    def census(self):
        K = self.prob.n_census
        w = np.empty(K); n = np.empty(K, dtype=np.uint64)
        self._L.orc_census_get(self._h, _d(w), n.ctypes.data_as(C.POINTER(C.c_uint64)), K)
        return w, n

    def history_events(self):
        ev = np.empty((self._last_n, 4), dtype=np.uint32)
        rc = self._L.orc_history_events_get(self._h, ev.ctypes.data_as(C.POINTER(C.c_uint32)), self._last_n)
        if rc != 0:
            raise RuntimeError(f"orc_history_events_get failed: {rc}")
        return ev

    def locate(self, r, omega):
        rr = np.ascontiguousarray(r, dtype=np.float64); oo = np.ascontiguousarray(omega, dtype=np.float64)
        return int(self._L.orc_locate(self._h, _d(rr), _d(oo)))

    def stream(self, r, omega, cell, max_events):
        rr = np.array(r, dtype=np.float64); oo = np.array(omega, dtype=np.float64)
        c = np.array([cell], dtype=np.int32)
        n = self._L.orc_stream(self._h, _d(rr), _d(oo), _i(c), int(max_events))
        return n, rr, oo, int(c[0])

    def score_segment(self, r, omega, t, g, w, d):
        rr = np.ascontiguousarray(r, dtype=np.float64); oo = np.ascontiguousarray(omega, dtype=np.float64)
        rc = self._L.orc_score_segment(self._h, _d(rr), _d(oo), float(t), int(g), float(w), float(d))
        if rc != 0:
            raise RuntimeError("orc_score_segment failed")

    def close_batch(self, histories_in_batch=1):
        rc = self._L.orc_close_batch(self._h, int(histories_in_batch))
        if rc != 0:
            raise RuntimeError("orc_close_batch failed")
