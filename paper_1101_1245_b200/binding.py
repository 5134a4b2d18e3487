"""Thin ctypes binding of libgpumcd.so: same names as include/gpumcd.h, argument marshalling only.

Every step of the hot path runs inside the CUDA library; PyTorch appears here only as the owner
of device memory and streams.  There is no CPU fallback: if the library cannot be loaded, or no
CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgpumcd.so")

GPUMCD_OK = 0
GPUMCD_ERR_INVALID_ARG = -1
GPUMCD_ERR_CUDA = -2
GPUMCD_ERR_OOM = -3
GPUMCD_ERR_BANK_OVERFLOW = -4
GPUMCD_ERR_NO_SOURCE = -5
GPUMCD_ERR_TABLE_RANGE = -6
GPUMCD_STATIC_MAX_VOXELS = 64 * 64 * 64   # include/gpumcd.h: largest phantom of gpumcd_run_uncertainty_static

EXPORTS = ("gpumcd_default_options", "gpumcd_create", "gpumcd_create_host", "gpumcd_set_phantom",
           "gpumcd_set_phantom_host", "gpumcd_set_source", "gpumcd_run",
           "gpumcd_run_host", "gpumcd_run_uncertainty", "gpumcd_run_uncertainty_static", "gpumcd_run_trace", "gpumcd_get_counters", "gpumcd_get_energy_tally",
           "gpumcd_set_history_offset", "gpumcd_set_profiling", "gpumcd_get_profile", "gpumcd_probe_tally",
           "gpumcd_selftest_philox", "gpumcd_release_l2",
           "gpumcd_last_error", "gpumcd_destroy")


class gpumcd_tables(C.Structure):
    _fields_ = [("n_materials", C.c_int32), ("n_energy", C.c_int32), ("e_min", C.c_float), ("e_max", C.c_float),
                ("photon", C.c_void_p), ("electron", C.c_void_p), ("n_K", C.c_int32), ("lnK_min", C.c_float),
                ("lnK_max", C.c_float), ("ms_a", C.c_void_p), ("e_cut", C.c_float), ("p_cut", C.c_float)]


class gpumcd_options(C.Structure):
    _fields_ = [("es_max_cm", C.c_float), ("f_eloss_max", C.c_float), ("boundary_nudge", C.c_float),
                ("pair_mode", C.c_int32), ("photon_only", C.c_int32), ("majorant_scale", C.c_float),
                ("wave_size", C.c_uint32), ("bank_factor", C.c_uint32), ("scheduler", C.c_int32),
                ("warp_stack", C.c_uint32), ("cta_threads", C.c_uint32), ("hom_tol", C.c_float),
                ("tally_mode", C.c_int32), ("table_memory", C.c_int32), ("bank_high_g", C.c_uint32),
                ("bank_high_e", C.c_uint32), ("bank_low", C.c_uint32), ("steps_per_refill", C.c_uint32),
                ("l2_persist", C.c_int32)]


class gpumcd_source(C.Structure):
    _fields_ = [("particle", C.c_int32), ("shape", C.c_int32), ("cx", C.c_float), ("cy", C.c_float),
                ("wx", C.c_float), ("wy", C.c_float), ("energy", C.c_float), ("n_spec", C.c_int32),
                ("spec_E", C.c_void_p), ("spec_w", C.c_void_p),
                ("n_phsp", C.c_uint64), ("phsp", C.c_void_p), ("phsp_on_host", C.c_int32)]


class gpumcd_counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in (
        "n_histories", "photon_flights", "photon_compton", "photon_photo", "photon_pair", "photon_fict",
        "ch_steps", "hard_moller", "hard_brems", "hard_fict", "pushes_e", "pushes_g", "bank_high_water",
        "overflow_count")] + [(n, C.c_double) for n in (
            "e_incident", "e_dep_continuous", "e_dep_cutoff", "e_escaped", "e_pair_rest")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class gpumcd_profile(C.Structure):
    _fields_ = [("launches", C.c_uint64), ("n_source", C.c_uint32), ("n_photon", C.c_uint32),
                ("n_electron", C.c_uint32), ("n_finalize", C.c_uint32), ("ms_source", C.c_float),
                ("ms_photon", C.c_float), ("ms_electron", C.c_float), ("ms_finalize", C.c_float)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class GpumcdError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"gpumcd status {status}: {message}")
        self.status = status


_lib = None


def load_library():
    """Load the in-tree CUDA library; raises if it has not been built (no fallback exists)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1101_1245_b200.build` "
                               "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        lib.gpumcd_default_options.argtypes = [C.POINTER(gpumcd_options)]
        lib.gpumcd_create.argtypes = [C.POINTER(vp), vp, vp, C.c_int, C.c_int, C.c_int, C.c_float,
                                      C.POINTER(gpumcd_tables), C.POINTER(gpumcd_options)]
        lib.gpumcd_create_host.argtypes = lib.gpumcd_create.argtypes
        lib.gpumcd_set_phantom.argtypes = [vp, vp, vp]
        lib.gpumcd_set_phantom_host.argtypes = [vp, vp, vp]
        lib.gpumcd_set_source.argtypes = [vp, C.POINTER(gpumcd_source)]
        lib.gpumcd_run.argtypes = [vp, C.c_uint64, C.c_uint64, vp, vp]
        lib.gpumcd_run_host.argtypes = [vp, C.c_uint64, C.c_uint64, vp, vp]
        lib.gpumcd_run_trace.argtypes = [vp, C.c_uint64, C.c_uint64, vp, vp]
        lib.gpumcd_run_uncertainty.argtypes = [vp, C.c_uint64, C.c_uint32, C.c_uint64, vp, vp, vp]
        lib.gpumcd_run_uncertainty_static.argtypes = lib.gpumcd_run_uncertainty.argtypes
        lib.gpumcd_get_counters.argtypes = [vp, C.POINTER(gpumcd_counters)]
        lib.gpumcd_get_energy_tally.argtypes = [vp, vp]
        lib.gpumcd_set_history_offset.argtypes = [vp, C.c_uint64]
        lib.gpumcd_set_profiling.argtypes = [vp, C.c_int]
        lib.gpumcd_get_profile.argtypes = [vp, C.POINTER(gpumcd_profile)]
        lib.gpumcd_probe_tally.argtypes = [vp, C.c_uint64, C.POINTER(C.c_double), vp]
        lib.gpumcd_selftest_philox.argtypes = [vp, vp, vp, C.c_uint64, vp]
        lib.gpumcd_release_l2.argtypes = [vp]
        lib.gpumcd_last_error.argtypes = [vp]
        lib.gpumcd_last_error.restype = C.c_char_p
        lib.gpumcd_destroy.argtypes = [vp]
        lib.gpumcd_destroy.restype = None
        for name in EXPORTS:
            if name not in ("gpumcd_last_error", "gpumcd_destroy"):
                getattr(lib, name).restype = C.c_int
        _lib = lib
    return _lib


def gpumcd_default_options(**overrides) -> gpumcd_options:
    opt = gpumcd_options()
    load_library().gpumcd_default_options(C.byref(opt))
    for k, v in overrides.items():
        if not hasattr(opt, k):
            raise AttributeError(k)
        setattr(opt, k, v)
    return opt


def _hptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _tables_struct(tb):
    keep = (np.ascontiguousarray(tb.photon, np.float32), np.ascontiguousarray(tb.electron, np.float32),
            np.ascontiguousarray(tb.ms_a, np.float32))
    t = gpumcd_tables(tb.n_materials, tb.n_energy, tb.e_min, tb.e_max, _hptr(keep[0]), _hptr(keep[1]), tb.n_K,
                      tb.lnK_min, tb.lnK_max, _hptr(keep[2]), tb.e_cut, tb.p_cut)
    return t, keep


class Context:
    """Owner of one gpumcd_ctx.  Methods mirror the C calls one to one."""

    def __init__(self, handle, shape_zyx):
        self._h = C.c_void_p(handle)
        self.shape = tuple(shape_zyx)

    def _check(self, rc):
        if rc != GPUMCD_OK:
            raise GpumcdError(rc, gpumcd_last_error(self))
        return rc

    def close(self):
        if self._h:
            load_library().gpumcd_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def _create(fn, density_ptr, material_ptr, shape_zyx, voxel_cm, tables, options):
    nz, ny, nx = shape_zyx
    t, keep = _tables_struct(tables)
    h = C.c_void_p()
    rc = fn(C.byref(h), density_ptr, material_ptr, nx, ny, nz, C.c_float(voxel_cm), C.byref(t),
            C.byref(options) if options is not None else None)
    del keep
    if rc != GPUMCD_OK:
        raise GpumcdError(rc, load_library().gpumcd_last_error(None).decode())
    return Context(h.value, shape_zyx)


def gpumcd_create(density_dev, material_dev, voxel_cm, tables, options: Optional[gpumcd_options] = None) -> Context:
    """density_dev: torch float32 CUDA tensor [nz,ny,nx]; material_dev: torch uint8 CUDA tensor [nz,ny,nx]."""
    import torch
    assert density_dev.is_cuda and material_dev.is_cuda, "gpumcd_create takes CUDA tensors (no CPU path)"
    assert density_dev.dtype == torch.float32 and material_dev.dtype == torch.uint8
    assert density_dev.is_contiguous() and material_dev.is_contiguous() and density_dev.shape == material_dev.shape
    return _create(load_library().gpumcd_create, C.c_void_p(density_dev.data_ptr()),
                   C.c_void_p(material_dev.data_ptr()), tuple(density_dev.shape), voxel_cm, tables, options)


def gpumcd_create_host(density: np.ndarray, material: np.ndarray, voxel_cm, tables,
                       options: Optional[gpumcd_options] = None) -> Context:
    density = np.ascontiguousarray(density, np.float32)
    material = np.ascontiguousarray(material, np.uint8)
    assert density.shape == material.shape and density.ndim == 3
    return _create(load_library().gpumcd_create_host, _hptr(density), _hptr(material), density.shape, voxel_cm,
                   tables, options)


def gpumcd_set_phantom(ctx: Context, density_dev, material_dev) -> None:
    """New phantom of the same shape from CUDA tensors (float32 / uint8, [nz,ny,nx])."""
    assert density_dev.is_cuda and material_dev.is_cuda and density_dev.is_contiguous() and material_dev.is_contiguous()
    assert tuple(density_dev.shape) == ctx.shape == tuple(material_dev.shape)
    assert density_dev.element_size() == 4 and material_dev.element_size() == 1
    ctx._check(load_library().gpumcd_set_phantom(ctx._h, C.c_void_p(density_dev.data_ptr()),
                                                 C.c_void_p(material_dev.data_ptr())))


def gpumcd_set_phantom_host(ctx: Context, density: np.ndarray, material: np.ndarray) -> None:
    """New phantom of the same shape from host arrays (float32 / uint8, [nz,ny,nx]; pinned memory copies fastest)."""
    assert density.dtype == np.float32 and material.dtype == np.uint8
    assert density.flags.c_contiguous and material.flags.c_contiguous
    assert density.shape == ctx.shape == material.shape
    ctx._check(load_library().gpumcd_set_phantom_host(ctx._h, _hptr(density), _hptr(material)))


def gpumcd_set_source(ctx: Context, source) -> None:
    """``source``: an inputs.Source (particle, shape, cx, cy, wx, wy, energy, spec_edges, spec_weights, phsp)."""
    n_spec, pe, pw, keep = 0, None, None, ()
    if getattr(source, "spec_edges", None) is not None:
        e = np.ascontiguousarray(source.spec_edges, np.float32)
        w = np.ascontiguousarray(source.spec_weights, np.float32)
        keep = (e, w)
        n_spec, pe, pw = int(w.size), _hptr(e), _hptr(w)
    n_phsp, pp, on_host = 0, None, 0
    ps = getattr(source, "phsp", None)
    if ps is not None:  # a torch CUDA tensor (device records) or a numpy array (host records), float32 [n, 8]
        if isinstance(ps, np.ndarray):
            ps = np.ascontiguousarray(ps, np.float32).reshape(-1, 8)
            n_phsp, pp, on_host = int(ps.shape[0]), _hptr(ps), 1
        else:
            assert ps.is_cuda and ps.is_contiguous() and str(ps.dtype) == "torch.float32" and ps.shape[-1] == 8
            n_phsp, pp = int(ps.numel() // 8), ps.data_ptr()
        keep = keep + (ps,)
    s = gpumcd_source(source.particle, source.shape, source.cx, source.cy, source.wx, source.wy, source.energy,
                      n_spec, pe, pw, n_phsp, pp, on_host)
    ctx._check(load_library().gpumcd_set_source(ctx._h, C.byref(s)))
    del keep


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(getattr(stream, "cuda_stream", stream))


def gpumcd_run(ctx: Context, n_histories: int, seed: int, dose_out_dev, stream=None) -> None:
    """dose_out_dev: torch float32 CUDA tensor with nx*ny*nz elements, overwritten."""
    assert dose_out_dev.is_cuda and dose_out_dev.is_contiguous() and dose_out_dev.numel() == int(np.prod(ctx.shape))
    ctx._check(load_library().gpumcd_run(ctx._h, int(n_histories), int(seed), C.c_void_p(dose_out_dev.data_ptr()),
                                         _stream_ptr(stream)))


def gpumcd_run_host(ctx: Context, n_histories: int, seed: int, dose_out: np.ndarray, stream=None) -> None:
    assert dose_out.dtype == np.float32 and dose_out.flags.c_contiguous and dose_out.size == int(np.prod(ctx.shape))
    ctx._check(load_library().gpumcd_run_host(ctx._h, int(n_histories), int(seed), _hptr(dose_out),
                                              _stream_ptr(stream)))


def gpumcd_run_uncertainty(ctx: Context, n_histories: int, n_batches: int, seed: int, dose_out_dev, sigma_out_dev,
                           stream=None) -> None:
    """dose_out_dev, sigma_out_dev: torch float32 CUDA tensors of the phantom's shape (include/gpumcd.h)."""
    for t in (dose_out_dev, sigma_out_dev):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 4 and t.numel() == int(np.prod(ctx.shape))
    ctx._check(load_library().gpumcd_run_uncertainty(ctx._h, int(n_histories), int(n_batches), int(seed),
                                                     C.c_void_p(dose_out_dev.data_ptr()),
                                                     C.c_void_p(sigma_out_dev.data_ptr()), _stream_ptr(stream)))


def gpumcd_run_uncertainty_static(ctx: Context, n_histories: int, n_batches: int, seed: int, dose_out_dev,
                                  sigma_out_dev, stream=None) -> None:
    """gpumcd_run_uncertainty with its scratch in the library's static device array: no device allocation
    (include/gpumcd.h; at most GPUMCD_STATIC_MAX_VOXELS voxels)."""
    for t in (dose_out_dev, sigma_out_dev):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 4 and t.numel() == int(np.prod(ctx.shape))
    ctx._check(load_library().gpumcd_run_uncertainty_static(ctx._h, int(n_histories), int(n_batches), int(seed),
                                                            C.c_void_p(dose_out_dev.data_ptr()),
                                                            C.c_void_p(sigma_out_dev.data_ptr()), _stream_ptr(stream)))


def gpumcd_run_trace(ctx: Context, n_histories: int, seed: int, trace_out_dev, stream=None) -> None:
    """trace_out_dev: torch int64 CUDA tensor with n_histories elements (bit pattern of the uint64 codes)."""
    assert trace_out_dev.is_cuda and trace_out_dev.is_contiguous() and trace_out_dev.numel() == int(n_histories)
    assert trace_out_dev.element_size() == 8
    ctx._check(load_library().gpumcd_run_trace(ctx._h, int(n_histories), int(seed),
                                               C.c_void_p(trace_out_dev.data_ptr()), _stream_ptr(stream)))


def gpumcd_get_counters(ctx: Context) -> dict:
    c = gpumcd_counters()
    ctx._check(load_library().gpumcd_get_counters(ctx._h, C.byref(c)))
    return c.as_dict()


def gpumcd_get_energy_tally(ctx: Context, edep_out_dev) -> None:
    """edep_out_dev: torch float64 CUDA tensor with nx*ny*nz elements."""
    assert edep_out_dev.is_cuda and edep_out_dev.is_contiguous() and edep_out_dev.element_size() == 8
    assert edep_out_dev.numel() == int(np.prod(ctx.shape))
    ctx._check(load_library().gpumcd_get_energy_tally(ctx._h, C.c_void_p(edep_out_dev.data_ptr())))


def gpumcd_set_history_offset(ctx: Context, first_history: int) -> None:
    ctx._check(load_library().gpumcd_set_history_offset(ctx._h, int(first_history)))


def gpumcd_release_l2(ctx: Context) -> None:
    ctx._check(load_library().gpumcd_release_l2(ctx._h))


def gpumcd_set_profiling(ctx: Context, enable: bool) -> None:
    ctx._check(load_library().gpumcd_set_profiling(ctx._h, int(bool(enable))))


def gpumcd_get_profile(ctx: Context) -> dict:
    p = gpumcd_profile()
    ctx._check(load_library().gpumcd_get_profile(ctx._h, C.byref(p)))
    return p.as_dict()


def gpumcd_probe_tally(ctx: Context, n_updates: int, stream=None) -> float:
    """fp64 atomic adds per second into the context's energy grid under the source's field (include/gpumcd.h)."""
    r = C.c_double(0.0)
    ctx._check(load_library().gpumcd_probe_tally(ctx._h, int(n_updates), C.byref(r), _stream_ptr(stream)))
    return r.value


def gpumcd_selftest_philox(ctr_key_dev, out_dev, uniform_dev=None, stream=None) -> None:
    """ctr_key_dev: torch int32 CUDA tensor [n, 6] (bit patterns of the uint32 counter and key words); out_dev: int32
    [n, 4]; uniform_dev: float32 [n, 4] or None (include/gpumcd.h)."""
    n = ctr_key_dev.shape[0]
    for t, cols in ((ctr_key_dev, 6), (out_dev, 4)) + (((uniform_dev, 4),) if uniform_dev is not None else ()):
        assert t.is_cuda and t.is_contiguous() and t.element_size() == 4 and tuple(t.shape) == (n, cols)
    rc = load_library().gpumcd_selftest_philox(C.c_void_p(ctr_key_dev.data_ptr()), C.c_void_p(out_dev.data_ptr()),
                                               C.c_void_p(uniform_dev.data_ptr()) if uniform_dev is not None else None,
                                               int(n), _stream_ptr(stream))
    if rc != GPUMCD_OK:
        raise GpumcdError(rc, "gpumcd_selftest_philox failed")


def gpumcd_last_error(ctx: Optional[Context]) -> str:
    s = load_library().gpumcd_last_error(ctx._h if ctx is not None else None)
    return s.decode() if s else ""


def gpumcd_destroy(ctx: Context) -> None:
    ctx.close()
