"""ctypes front end of the CPU oracle (oracle/oracle.c).  TEST INFRASTRUCTURE ONLY.

May be imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs -- never by the product package.  Shares no code with the
CUDA path; the only thing both receive is the input data of
``paper_1101_1245_b200.inputs`` (plain arrays).
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import build as _build

_lib = None


class _Tables(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_energy", C.c_int32),
                ("e_min", C.c_double), ("e_max", C.c_double),
                ("photon", C.c_void_p), ("electron", C.c_void_p),
                ("n_K", C.c_int32), ("lnK_min", C.c_double), ("lnK_max", C.c_double),
                ("ms_a", C.c_void_p), ("e_cut", C.c_double), ("p_cut", C.c_double)]


class _Options(C.Structure):
    _fields_ = [("es_max_cm", C.c_double), ("f_eloss_max", C.c_double),
                ("boundary_nudge", C.c_double), ("pair_mode", C.c_int32),
                ("photon_only", C.c_int32), ("majorant_scale", C.c_double), ("hom_tol", C.c_double)]


class _Source(C.Structure):
    _fields_ = [("particle", C.c_int32), ("shape", C.c_int32),
                ("cx", C.c_double), ("cy", C.c_double), ("wx", C.c_double), ("wy", C.c_double),
                ("energy", C.c_double), ("n_spec", C.c_int32),
                ("spec_E", C.c_void_p), ("spec_w", C.c_void_p),
                ("n_phsp", C.c_int64), ("phsp", C.c_void_p)]


class Counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in (
        "n_histories", "photon_flights", "photon_compton", "photon_photo", "photon_pair",
        "photon_fict", "ch_steps", "hard_moller", "hard_brems", "hard_fict", "pushes_e",
        "pushes_g", "stack_high_water")] + [(n, C.c_double) for n in (
            "e_incident", "e_dep_continuous", "e_dep_cutoff", "e_escaped", "e_pair_rest")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.orc_uniform.restype = C.c_double
        _lib.orc_uniform.argtypes = [C.c_uint32]
        _lib.orc_lookup.restype = C.c_double
        _lib.orc_lookup.argtypes = [C.c_void_p, C.c_int32, C.c_double, C.c_double, C.c_double]
        _lib.orc_run.restype = C.c_int
        _lib.orc_run_pathlen.restype = C.c_int
        _lib.orc_run_moments.restype = C.c_int
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


@dataclass
class Options:
    es_max_cm: float = 0.5
    f_eloss_max: float = 0.25
    boundary_nudge: float = 1e-4
    pair_mode: int = 1
    photon_only: int = 0
    majorant_scale: float = 1.0
    hom_tol: float = 0.0

    def c(self):
        f32 = lambda v: float(np.float32(v))
        return _Options(f32(self.es_max_cm), f32(self.f_eloss_max), f32(self.boundary_nudge), self.pair_mode,
                        self.photon_only, f32(self.majorant_scale), f32(self.hom_tol))


def _tables_c(tb):
    keep = (np.ascontiguousarray(tb.photon, np.float32), np.ascontiguousarray(tb.electron, np.float32),
            np.ascontiguousarray(tb.ms_a, np.float32))
    f32 = lambda v: float(np.float32(v))   # the boundary (include/gpumcd.h) carries these as float32
    t = _Tables(tb.n_materials, tb.n_energy, f32(tb.e_min), f32(tb.e_max), _p(keep[0]), _p(keep[1]),
                tb.n_K, f32(tb.lnK_min), f32(tb.lnK_max), _p(keep[2]), f32(tb.e_cut), f32(tb.p_cut))
    return t, keep


def _source_c(src):
    keep = ()
    n_spec = 0
    pe = pw = None
    if src.spec_edges is not None:
        e = np.ascontiguousarray(src.spec_edges, np.float32)
        w = np.ascontiguousarray(src.spec_weights, np.float32)
        keep = (e, w)
        n_spec = int(w.size)
        pe, pw = _p(e), _p(w)
    n_phsp, pp = 0, None
    if getattr(src, "phsp", None) is not None:
        ps = np.ascontiguousarray(src.phsp, np.float32).reshape(-1, 8)
        keep = keep + (ps,)
        n_phsp, pp = int(ps.shape[0]), _p(ps)
    f32 = lambda v: float(np.float32(v))   # the boundary (include/gpumcd.h) carries these as float32
    s = _Source(src.particle, src.shape, f32(src.cx), f32(src.cy), f32(src.wx), f32(src.wy), f32(src.energy),
                n_spec, pe, pw, n_phsp, pp)
    return s, keep


# ---------------------------------------------------------------------------
def philox(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def philox_batch(ctr_key: np.ndarray) -> np.ndarray:
    """ctr_key: uint32 [n, 6] = counter (4 words) and key (2 words) per row; returns the blocks, uint32 [n, 4]."""
    a = np.ascontiguousarray(ctr_key, np.uint32)
    out = np.zeros((a.shape[0], 4), np.uint32)
    lib().orc_philox_batch(_p(a), _p(out), C.c_int64(a.shape[0]))
    return out


def uniform(w: int) -> float:
    return lib().orc_uniform(int(w) & 0xFFFFFFFF)


def lookup(col: np.ndarray, x_min: float, x_max: float, x: float) -> float:
    col = np.ascontiguousarray(col, np.float32)
    return lib().orc_lookup(_p(col), col.size, x_min, x_max, x)


def majorants(tb, rho_max):
    t, keep = _tables_c(tb)
    rm = np.ascontiguousarray(rho_max, np.float64)
    mu = np.zeros(tb.n_energy)
    me = np.zeros(tb.n_energy)
    lib().orc_majorants(C.byref(t), _p(rm), _p(mu), _p(me))
    return mu, me


def batch_compton(E, seed, n):
    eps, cost, phi = np.zeros(n), np.zeros(n), np.zeros(n)
    lib().orc_batch_compton(C.c_double(E), C.c_uint64(seed), C.c_int64(n), _p(eps), _p(cost), _p(phi))
    return eps, cost, phi


def batch_sauter(E, seed, n):
    nu = np.zeros(n)
    lib().orc_batch_sauter(C.c_double(E), C.c_uint64(seed), C.c_int64(n), _p(nu))
    return nu


def batch_pair(E, seed, n):
    T1, c1, c2 = np.zeros(n), np.zeros(n), np.zeros(n)
    lib().orc_batch_pair(C.c_double(E), C.c_uint64(seed), C.c_int64(n), _p(T1), _p(c1), _p(c2))
    return T1, c1, c2


def batch_moller(T, k_cut, seed, n):
    eps, cp, cd = np.zeros(n), np.zeros(n), np.zeros(n)
    lib().orc_batch_moller(C.c_double(T), C.c_double(k_cut), C.c_uint64(seed), C.c_int64(n),
                           _p(eps), _p(cp), _p(cd))
    return eps, cp, cd


def batch_brems(T, k_c, seed, n):
    k = np.zeros(n)
    lib().orc_batch_brems(C.c_double(T), C.c_double(k_c), C.c_uint64(seed), C.c_int64(n), _p(k))
    return k


def batch_ms(a, seed, n):
    c = np.zeros(n)
    lib().orc_batch_ms(C.c_double(a), C.c_uint64(seed), C.c_int64(n), _p(c))
    return c


def rotate(d, cost, phi):
    dd = (C.c_double * 3)(*d)
    o = (C.c_double * 3)()
    lib().orc_rotate(dd, C.c_double(cost), C.c_double(phi), o)
    return np.array(list(o))


@dataclass
class Result:
    edep: np.ndarray            # float64 [nz, ny, nx], MeV
    dose: np.ndarray            # float32 [nz, ny, nx], MeV/g per history
    counters: dict
    trace: Optional[np.ndarray]


def run(density, material, voxel_cm, tables, source, n_histories, seed, options: Options = None,
        hist_begin: int = 0, want_trace: bool = False, n_threads: int = 0) -> Result:
    options = options or Options()
    density = np.ascontiguousarray(density, np.float32)
    material = np.ascontiguousarray(material, np.uint8)
    nz, ny, nx = density.shape
    t, keep_t = _tables_c(tables)
    s, keep_s = _source_c(source)
    o = options.c()
    edep = np.zeros((nz, ny, nx), np.float64)
    dose = np.zeros((nz, ny, nx), np.float32)
    trace = np.zeros(int(n_histories), np.uint64) if want_trace else None
    cnt = Counters()
    rc = lib().orc_run(_p(density), _p(material), C.c_int32(nx), C.c_int32(ny), C.c_int32(nz),
                       C.c_double(float(np.float32(voxel_cm))), C.byref(t), C.byref(o), C.byref(s),
                       C.c_uint64(hist_begin), C.c_uint64(int(n_histories)), C.c_uint64(seed),
                       _p(edep), _p(dose), _p(trace), C.byref(cnt), C.c_int32(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_run failed with code {rc}")
    del keep_t, keep_s
    return Result(edep, dose, cnt.as_dict(), trace)


def run_moments(density, material, voxel_cm, tables, source, n_histories, seed, options: Options = None,
                hist_begin: int = 0, n_threads: int = 0):
    """History-by-history first and second moments (Eq. 13).  Returns (edep, edep_sq, counters):
    per voxel the sum over histories of the energy a history deposits, and of its square."""
    options = options or Options()
    density = np.ascontiguousarray(density, np.float32)
    material = np.ascontiguousarray(material, np.uint8)
    nz, ny, nx = density.shape
    t, keep_t = _tables_c(tables)
    s, keep_s = _source_c(source)
    o = options.c()
    edep = np.zeros((nz, ny, nx), np.float64)
    esq = np.zeros((nz, ny, nx), np.float64)
    cnt = Counters()
    rc = lib().orc_run_moments(_p(density), _p(material), C.c_int32(nx), C.c_int32(ny), C.c_int32(nz),
                               C.c_double(float(np.float32(voxel_cm))), C.byref(t), C.byref(o), C.byref(s),
                               C.c_uint64(hist_begin), C.c_uint64(int(n_histories)), C.c_uint64(seed),
                               _p(edep), _p(esq), C.byref(cnt), C.c_int32(n_threads))
    if rc != 0:
        raise RuntimeError(f"orc_run_moments failed with code {rc}")
    del keep_t, keep_s
    return edep, esq, cnt.as_dict()


def uncertainty_from_moments(edep, edep_sq, n_histories):
    """PAPER.md Eq. 13 in energy units per history: sqrt((<e^2> - <e>^2)/(N - 1))."""
    n = float(n_histories)
    var = (edep_sq / n - (edep / n) ** 2) / (n - 1.0)
    return np.sqrt(np.maximum(var, 0.0))


def run_workload(w, n_histories=None, options: Options = None, want_trace=False, n_threads=0, hist_begin=0):
    n = w.n_histories if n_histories is None else n_histories
    return run(w.density, w.material, w.voxel_cm, w.tables, w.source, n, w.seed, options,
               hist_begin=hist_begin, want_trace=want_trace, n_threads=n_threads)


def run_pathlen(density, material, voxel_cm, tables, source, n_histories, seed, options: Options = None):
    options = options or Options()
    density = np.ascontiguousarray(density, np.float32)
    material = np.ascontiguousarray(material, np.uint8)
    nz, ny, nx = density.shape
    t, keep_t = _tables_c(tables)
    s, keep_s = _source_c(source)
    o = options.c()
    out = np.zeros(int(n_histories))
    rc = lib().orc_run_pathlen(_p(density), _p(material), C.c_int32(nx), C.c_int32(ny), C.c_int32(nz),
                               C.c_double(voxel_cm), C.byref(t), C.byref(o), C.byref(s),
                               C.c_uint64(int(n_histories)), C.c_uint64(seed), _p(out))
    if rc != 0:
        raise RuntimeError(f"orc_run_pathlen failed with code {rc}")
    del keep_t, keep_s
    return out


VLOG_COLS = 24
VLOG = {"hist": 0, "kind": 1, "parent_track": 2, "parent_ctr": 3, "E0": 4, "d0": slice(5, 8), "E1": 8,
        "d1": slice(9, 12), "child_type": 12, "child_track": 13, "child_E": 14, "child_d": slice(15, 18),
        "x": slice(18, 21)}
COMPTON, PHOTO, PAIR, MOLLER, BREMS = 1, 2, 3, 4, 5


def run_endstate(density, material, voxel_cm, tables, source, n_histories, seed, options: Options = None,
                 max_steps: int = 0):
    """End state of every history's primary track: (end[n, 8] = x, y, z, u, v, w, E, steps taken;
    pathmat[n, n_materials] = the primary electron's path length per material)."""
    options = options or Options()
    density = np.ascontiguousarray(density, np.float32)
    material = np.ascontiguousarray(material, np.uint8)
    nz, ny, nx = density.shape
    t, keep_t = _tables_c(tables)
    s, keep_s = _source_c(source)
    o = options.c()
    end = np.zeros((int(n_histories), 8))
    pathmat = np.zeros((int(n_histories), tables.n_materials))
    f = lib().orc_run_endstate
    f.restype = C.c_int
    rc = f(_p(density), _p(material), C.c_int32(nx), C.c_int32(ny), C.c_int32(nz),
           C.c_double(float(np.float32(voxel_cm))), C.byref(t), C.byref(o), C.byref(s),
           C.c_uint64(int(n_histories)), C.c_uint64(seed), C.c_int64(int(max_steps)), _p(end), _p(pathmat))
    if rc != 0:
        raise RuntimeError(f"orc_run_endstate failed with code {rc}")
    del keep_t, keep_s
    return end, pathmat


def run_vertices(density, material, voxel_cm, tables, source, n_histories, seed, options: Options = None,
                 cap: int = 4_000_000):
    """Log of every pushed secondary with its vertex: (rows[n_pushed, VLOG_COLS], counters); columns in VLOG."""
    options = options or Options()
    density = np.ascontiguousarray(density, np.float32)
    material = np.ascontiguousarray(material, np.uint8)
    nz, ny, nx = density.shape
    t, keep_t = _tables_c(tables)
    s, keep_s = _source_c(source)
    o = options.c()
    rows = np.zeros((int(cap), VLOG_COLS))
    n_out = C.c_int64(0)
    cnt = Counters()
    f = lib().orc_run_vertices
    f.restype = C.c_int
    rc = f(_p(density), _p(material), C.c_int32(nx), C.c_int32(ny), C.c_int32(nz),
           C.c_double(float(np.float32(voxel_cm))), C.byref(t), C.byref(o), C.byref(s),
           C.c_uint64(int(n_histories)), C.c_uint64(seed), _p(rows), C.c_int64(int(cap)), C.byref(n_out),
           C.byref(cnt))
    if rc != 0:
        raise RuntimeError(f"orc_run_vertices failed with code {rc}")
    if n_out.value > cap:
        raise RuntimeError(f"vertex log too small: {n_out.value} secondaries, capacity {cap}")
    del keep_t, keep_s
    return rows[:n_out.value].copy(), cnt.as_dict()
