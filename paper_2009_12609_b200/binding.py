"""ctypes binding of the C-ABI library declared in include/loc.h (argument marshalling only).

Every function below has the name of the C entry point it forwards to; all arithmetic runs in the CUDA
kernels of libloc_b200.so.  PyTorch is used for device memory and streams only.  There is no CPU fallback:
importing works without a GPU (the library loads and its symbols can be inspected), but every compute call
needs a CUDA device and raises LocError otherwise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

LOC_OK, LOC_EINVAL, LOC_ESTATE, LOC_ENOMEM, LOC_ECUDA, LOC_ENONFINITE = 0, -1, -2, -3, -4, -5
LOC_OPT_WINDOW_XMIN, LOC_OPT_WINDOW_EPS_TAU, LOC_OPT_SPAN_XCLIP, LOC_OPT_SIM3D_PARTS, LOC_OPT_SOLVER = 1, 2, 3, 4, 5
LOC_OPT_SOLVER_LOCAL = LOC_OPT_SOLVER
LOC_OPT_SIM3D_WARPS = 6
LOC_OPT_SPAN_XFULL = 7
LOC_GRID_SHELL, LOC_GRID_OCTREE = 1, 2
LOC_MAX_HFS = 8

SYMBOLS = ("loc_workspace_bytes", "loc_create_model", "loc_set_species", "loc_refresh_cells", "loc_set_directions", "loc_set_populations",
           "loc_init_lte", "loc_simulate", "loc_get_counters", "loc_solve", "loc_iterate", "loc_set_ali",
           "loc_set_option", "loc_iterate_until", "loc_spectra", "loc_spectra_map", "loc_line_area", "loc_tex",
           "loc_get_stats", "loc_destroy_model", "loc_last_error", "loc_set_hyperfine", "loc_spectra_shells_static")
LOC_STATIC_MAX_SHELLS = 4096


class LocError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"loc error {code}: {msg}")
        self.code = code


class loc_grid(C.Structure):
    _fields_ = [("kind", C.c_int), ("nshell", C.c_int), ("r_out", C.c_void_p), ("nray", C.c_int), ("ray_p", C.c_void_p),
                ("ray_w", C.c_void_p), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("root_cell_cm", C.c_double),
                ("nlevel", C.c_int), ("level_offset", C.c_void_p), ("child", C.c_void_p)]


class loc_cells(C.Structure):
    _fields_ = [("density", C.c_void_p), ("tkin", C.c_void_p), ("sigma", C.c_void_p), ("vx", C.c_void_p),
                ("vy", C.c_void_p), ("vz", C.c_void_p), ("abundance", C.c_void_p)]


class loc_stats(C.Structure):
    _fields_ = [("ncell", C.c_int64), ("steps", C.c_int64), ("ntrans_sim", C.c_int), ("nchannel", C.c_int),
                ("kernel_launches", C.c_int64), ("counter_stride", C.c_int), ("active_channels", C.c_int64), ("setup_steps", C.c_int64),
                ("setup_ms", C.c_double), ("active_updates", C.c_int64)]


_lib = None


def lib_path() -> str:
    return _build.SO


def lib():
    """Loads libloc_b200.so (building it with nvcc if the sources are newer).  Fails loudly if it cannot."""
    global _lib
    if _lib is None:
        if _build.needs_build():
            _build.build()
        if not os.path.exists(_build.SO):
            raise LocError(LOC_ESTATE, "libloc_b200.so is missing: run python -m paper_2009_12609_b200.build")
        L = C.CDLL(_build.SO)
        L.loc_workspace_bytes.restype = C.c_int64
        L.loc_workspace_bytes.argtypes = [C.POINTER(loc_grid), C.c_int, C.c_int, C.c_int, C.c_int]
        L.loc_create_model.argtypes = [C.POINTER(loc_grid), C.POINTER(loc_cells), C.c_int, C.c_double, C.c_double, C.c_int,
                                       C.c_int, C.c_int, C.c_void_p, C.c_int64, C.c_void_p, C.POINTER(C.c_void_p)]
        L.loc_set_species.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                      C.c_void_p]
        L.loc_refresh_cells.argtypes = [C.c_void_p]
        L.loc_set_directions.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.loc_set_populations.argtypes = [C.c_void_p, C.c_void_p]
        L.loc_init_lte.argtypes = [C.c_void_p]
        L.loc_simulate.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int]
        L.loc_get_counters.argtypes = [C.c_void_p, C.POINTER(C.c_void_p), C.POINTER(C.c_int), C.POINTER(C.c_void_p),
                                       C.POINTER(C.c_void_p)]
        L.loc_solve.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.loc_iterate.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double)]
        L.loc_set_ali.argtypes = [C.c_void_p, C.c_int]
        L.loc_set_hyperfine.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.loc_iterate_until.argtypes = [C.c_void_p, C.c_int, C.c_double, C.POINTER(C.c_int), C.POINTER(C.c_double)]
        L.loc_spectra.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        L.loc_set_option.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.loc_spectra_map.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_void_p, C.c_void_p]
        L.loc_tex.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.loc_line_area.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        L.loc_get_stats.argtypes = [C.c_void_p, C.POINTER(loc_stats)]
        L.loc_spectra_shells_static.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p,
                                                C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_double,
                                                C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_char_p, C.c_int]
        L.loc_destroy_model.argtypes = [C.c_void_p]
        L.loc_destroy_model.restype = None
        L.loc_last_error.argtypes = [C.c_void_p]
        L.loc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc, handle=None):
    if rc != LOC_OK:
        msg = lib().loc_last_error(handle)
        raise LocError(rc, msg.decode() if msg else "")


def _np(a, dt):
    return np.ascontiguousarray(a, dtype=dt)


def _hp(a):
    return a.ctypes.data_as(C.c_void_p)


def _dp(t):
    """device pointer of a torch CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise LocError(LOC_EINVAL, "expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr())


def make_shell_grid(r_out, ray_p, ray_w):
    """returns (loc_grid, keepalive)"""
    r, p, w = _np(r_out, np.float64), _np(ray_p, np.float64), _np(ray_w, np.float64)
    g = loc_grid(kind=LOC_GRID_SHELL, nshell=len(r), r_out=_hp(r), nray=len(p), ray_p=_hp(p), ray_w=_hp(w))
    return g, (r, p, w)


def make_octree_grid(nx, ny, nz, root_cell_cm, level_offset, child_dev):
    off = _np(level_offset, np.int64)
    g = loc_grid(kind=LOC_GRID_OCTREE, nx=nx, ny=ny, nz=nz, root_cell_cm=float(root_cell_cm), nlevel=len(off) - 1,
                 level_offset=_hp(off), child=_dp(child_dev))
    return g, (off, child_dev)


def loc_workspace_bytes(grid: loc_grid, nchannel: int, nlevel_species: int, ntrans: int, ndir_max: int) -> int:
    n = lib().loc_workspace_bytes(C.byref(grid), nchannel, nlevel_species, ntrans, ndir_max)
    if n < 0:
        raise LocError(int(n), "loc_workspace_bytes: invalid arguments")
    return int(n)


def loc_create_model(grid: loc_grid, cells: loc_cells, nchannel, band_halfwidth_cm_s, t_background_K, nlevel_species,
                     ntrans, ndir_max, workspace, stream_ptr=0):
    h = C.c_void_p()
    rc = lib().loc_create_model(C.byref(grid), C.byref(cells), nchannel, float(band_halfwidth_cm_s), float(t_background_K),
                                nlevel_species, ntrans, ndir_max, _dp(workspace), workspace.numel() * workspace.element_size(),
                                C.c_void_p(stream_ptr), C.byref(h))
    _check(rc, None)
    return h


def loc_set_species(h, sp):
    """sp: object with energy_K, g, upper, lower, einstein_A, mass_amu, cu, cl, temps_K, rate_down"""
    e, g = _np(sp.energy_K, np.float64), _np(sp.g, np.float64)
    up, lo, A = _np(sp.upper, np.int32), _np(sp.lower, np.int32), _np(sp.einstein_A, np.float64)
    cu, cl = _np(sp.cu, np.int32), _np(sp.cl, np.int32)
    tk, rd = _np(sp.temps_K, np.float64), _np(sp.rate_down, np.float64)
    _check(lib().loc_set_species(h, len(e), _hp(e), _hp(g), len(up), _hp(up), _hp(lo), _hp(A), float(sp.mass_amu), len(cu),
                                 _hp(cu), _hp(cl), len(tk), _hp(tk), _hp(rd)), h)


def loc_refresh_cells(h):
    _check(lib().loc_refresh_cells(h), h)


def loc_set_directions(h, dirs):
    d = _np(dirs, np.float64).reshape(-1, 3)
    _check(lib().loc_set_directions(h, len(d), _hp(d)), h)


def loc_set_populations(h, dev_pops):
    _check(lib().loc_set_populations(h, _dp(dev_pops)), h)


def loc_init_lte(h):
    _check(lib().loc_init_lte(h), h)


def loc_simulate(h, trans_idx=None, geometry_counters=False):
    if trans_idx is None or len(trans_idx) == 0:
        _check(lib().loc_simulate(h, 0, None, int(geometry_counters)), h)
    else:
        t = _np(trans_idx, np.int32)
        _check(lib().loc_simulate(h, len(t), _hp(t), int(geometry_counters)), h)


def loc_get_counters(h):
    """returns (counters_ptr, ntrans_padded, visits_ptr, pathz_ptr) as integers (borrowed device pointers)"""
    c, v, p, n = C.c_void_p(), C.c_void_p(), C.c_void_p(), C.c_int()
    _check(lib().loc_get_counters(h, C.byref(c), C.byref(n), C.byref(v), C.byref(p)), h)
    return c.value, n.value, v.value, p.value


def loc_solve(h) -> float:
    r = C.c_double(0.0)
    _check(lib().loc_solve(h, C.byref(r)), h)
    return r.value


def loc_iterate(h, niter: int) -> float:
    r = C.c_double(0.0)
    _check(lib().loc_iterate(h, int(niter), C.byref(r)), h)
    return r.value


def loc_tex(h, trans: int, dev_tex) -> None:
    _check(lib().loc_tex(h, int(trans), _dp(dev_tex)), h)


def loc_line_area(h, dev_cube, npix: int, dev_w) -> None:
    _check(lib().loc_line_area(h, _dp(dev_cube), int(npix), _dp(dev_w)), h)


def loc_set_hyperfine(h, trans: int, dv_cm_s, weight) -> None:
    dv = np.ascontiguousarray(dv_cm_s, np.float64)
    w = np.ascontiguousarray(weight, np.float64)
    assert dv.shape == w.shape and dv.ndim == 1
    _check(lib().loc_set_hyperfine(h, int(trans), len(dv), dv.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p)), h)


def loc_set_ali(h, ali: bool) -> None:
    _check(lib().loc_set_ali(h, int(bool(ali))), h)


def loc_iterate_until(h, max_iter: int, tol: float):
    """returns (iterations run, max relative change of the last one)"""
    r, n = C.c_double(0.0), C.c_int(0)
    _check(lib().loc_iterate_until(h, int(max_iter), float(tol), C.byref(n), C.byref(r)), h)
    return n.value, r.value


def loc_spectra(h, trans, dev_out, nx, ny=1, dir=None, aff=None, offsets_cm=None):
    d = _np(dir, np.float64) if dir is not None else None
    a = _np(aff, np.int64) if aff is not None else None
    o = _np(offsets_cm, np.float64) if offsets_cm is not None else None
    _check(lib().loc_spectra(h, int(trans), _hp(d) if d is not None else None, int(nx), int(ny),
                             _hp(a) if a is not None else None, _hp(o) if o is not None else None, _dp(dev_out)), h)


def loc_set_option(h, key: int, value: float) -> None:
    _check(lib().loc_set_option(h, int(key), float(value)), h)


def loc_spectra_map(h, trans, dev_out, nx, ny, dir, pixel_cm, centre_cm):
    d, c = _np(dir, np.float64), _np(centre_cm, np.float64)
    _check(lib().loc_spectra_map(h, int(trans), _hp(d), int(nx), int(ny), float(pixel_cm), _hp(c), _dp(dev_out)), h)


def loc_spectra_shells_static(r_out, dev_vrad, dev_sigma, dev_tkin, mass_amu, dev_pop_u, dev_pop_l, freq_hz, einstein_A,
                              g_upper, g_lower, nchannel, band_halfwidth_cm_s, t_background_K, offsets_cm, dev_out,
                              stream_ptr=0) -> None:
    """Shell-model spectra for callers that cannot allocate device memory (include/loc.h): no model, no workspace; the
    kernel's scratch is a fixed array inside the library (at most LOC_STATIC_MAX_SHELLS shells).  This wrapper only
    marshals: it creates no tensor -- inputs and dev_out are the caller's CUDA tensors, r_out and offsets_cm host arrays.
    All calls on a device share the scratch array: keep them on one stream (or otherwise serialised), and make the first
    call on each device during start-up."""
    r, o = _np(r_out, np.float64), _np(offsets_cm, np.float64)
    err = C.create_string_buffer(512)
    rc = lib().loc_spectra_shells_static(len(r), _hp(r), _dp(dev_vrad), _dp(dev_sigma), _dp(dev_tkin), float(mass_amu),
                                         _dp(dev_pop_u), _dp(dev_pop_l), float(freq_hz), float(einstein_A), float(g_upper),
                                         float(g_lower), int(nchannel), float(band_halfwidth_cm_s), float(t_background_K),
                                         len(o), _hp(o), _dp(dev_out), C.c_void_p(stream_ptr), err, len(err))
    if rc != LOC_OK:
        raise LocError(rc, err.value.decode())


def loc_get_stats(h) -> dict:
    s = loc_stats()
    _check(lib().loc_get_stats(h, C.byref(s)), h)
    return {k: getattr(s, k) for k, _ in loc_stats._fields_}


def loc_destroy_model(h):
    lib().loc_destroy_model(h)
