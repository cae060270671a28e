"""Thin Python binding of libgammanav.so (include/gammanav.h) -- argument marshalling only.

Every step of the path runs in the CUDA kernels; torch is used for device memory and streams.  There is
no CPU fallback: if the library is missing or no CUDA device is present, calls raise GammaNavError.
Names mirror the C ABI: Geometry(...) = gn_geometry_create, nav_locate, nav_compute_step, transport_run.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.environ.get("GN_LIBRARY") or os.path.join(_HERE, "libgammanav.so")      # GN_LIBRARY: load another build of the same library (diagnostics)
_lib = None

EXPORTS = ("gn_geometry_create", "gn_geometry_destroy", "gn_geometry_num_places", "gn_geometry_tolerance",
           "gn_geometry_voxel_info", "gn_nav_locate", "gn_nav_compute_step", "gn_nav_compute_step_noalloc", "gn_nav_compute_step_normal", "gn_nav_compute_safety", "gn_transport_run", "gn_nav_query_host",
           "gn_transport_run_host", "gn_free_path_run", "gn_free_path_run_host", "gn_selftest_arith", "gn_selftest_pipe_peak",
           "gn_host_source_frame", "gn_host_compose_transforms", "gn_host_voxel_tables", "gn_last_error", "gn_version")


class GammaNavError(RuntimeError):
    pass


class Opts(C.Structure):
    _fields_ = [("tol64", C.c_double), ("tol32", C.c_double), ("sigma_pe0", C.c_double), ("e_cut", C.c_double),
                ("voxel_min_daughters", C.c_int32), ("stuck_limit", C.c_int32), ("steps_per_pass", C.c_int32), ("first_pass_steps", C.c_int32),
                ("tail_photons", C.c_int32), ("regroup_percent", C.c_int32), ("secondaries", C.c_int32), ("refill", C.c_int32),
                ("no_voxel_pass", C.c_int32), ("rayleigh", C.c_int32), ("sigma_r0", C.c_double), ("pe_table_per_decade", C.c_int32), ("pe_k_edge", C.c_int32)]


class CSource(C.Structure):
    _fields_ = [("kind", C.c_int32), ("energy_kind", C.c_int32), ("origin", C.c_double * 3), ("axis", C.c_double * 3),
                ("sigma", C.c_double), ("half_angle", C.c_double), ("e0", C.c_double), ("e1", C.c_double)]


class RunStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck", "n_photons")] + \
               [(n, C.c_double) for n in ("e_escaped", "e_stuck", "e_source", "e_deposited")] + \
               [("n_passes", C.c_uint64), ("n_kernel_launches", C.c_uint64), ("kernel_ms", C.c_double), ("step_pass_ms", C.c_double),
                ("n_steps_step_pass", C.c_uint64), ("n_rayleigh", C.c_uint64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


def library_path() -> str:
    return _LIB_PATH


def lib():
    """Load libgammanav.so (built in-tree by paper_1209_5235_b200.build).  Fails loudly when absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise GammaNavError(f"{_LIB_PATH} not built: run `python -m paper_1209_5235_b200.build` (there is no CPU fallback)")
        L = C.CDLL(_LIB_PATH)
        L.gn_last_error.restype = C.c_char_p
        L.gn_version.restype = C.c_char_p
        L.gn_geometry_tolerance.restype = C.c_double
        L.gn_geometry_tolerance.argtypes = [C.c_void_p, C.c_int]
        L.gn_geometry_num_places.restype = C.c_int32
        L.gn_geometry_num_places.argtypes = [C.c_void_p]
        L.gn_geometry_destroy.argtypes = [C.c_void_p]
        L.gn_geometry_voxel_info.argtypes = [C.c_void_p, C.c_void_p]
        L.gn_nav_locate.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.gn_nav_compute_step.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.gn_nav_compute_step_noalloc.argtypes = L.gn_nav_compute_step.argtypes
        L.gn_nav_compute_safety.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
        L.gn_nav_compute_step_normal.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.gn_transport_run.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_uint64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                       C.c_void_p, C.c_void_p, C.c_void_p]
        L.gn_nav_query_host.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]
        L.gn_selftest_arith.argtypes = [C.c_int64, C.c_void_p]
        L.gn_selftest_pipe_peak.argtypes = [C.c_int, C.c_void_p]
        L.gn_host_source_frame.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.gn_host_compose_transforms.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        L.gn_host_voxel_tables.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_void_p,
                                           C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.gn_free_path_run_host.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_void_p, C.c_void_p]
        L.gn_free_path_run.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p]
        L.gn_transport_run_host.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_uint64, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        _lib = L
    return _lib


def _check(rc, what):
    if rc != 0:
        raise GammaNavError(f"{what} failed ({rc}): {lib().gn_last_error().decode()}")


def _np(a, dtype):
    return np.ascontiguousarray(a, dtype)


def _csource(src) -> CSource:
    s = CSource()
    s.kind, s.energy_kind = int(src.kind), int(src.energy_kind)
    s.origin[:] = [float(v) for v in src.origin]
    s.axis[:] = [float(v) for v in src.axis]
    s.sigma, s.half_angle, s.e0, s.e1 = float(src.sigma), float(src.half_angle), float(src.e0), float(src.e1)
    return s


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise GammaNavError("no CUDA device: this library has no CPU fallback")
    return torch


def _real_dtype(torch, precision):
    if precision == 32:
        return torch.float32
    if precision == 64:
        return torch.float64
    raise GammaNavError("precision must be 32 or 64")


def _stream_ptr(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class Geometry:
    """gn_geometry_create: materials, solids, placements, transforms -> device-resident geometry store."""

    def __init__(self, geom, **opts):
        L = lib()
        self._h = C.c_void_p()
        mats = _np(geom.materials, np.float64); st = _np(geom.solid_type, np.int32); sp = _np(geom.solid_params, np.float64)
        pl = _np(geom.placements, np.int32); tr = _np(geom.transforms, np.float64)
        o = Opts(**opts) if opts else None
        rc = L.gn_geometry_create(mats.ctypes.data_as(C.c_void_p), C.c_int32(mats.shape[0]), st.ctypes.data_as(C.c_void_p),
                                  sp.ctypes.data_as(C.c_void_p), C.c_int32(st.shape[0]), pl.ctypes.data_as(C.c_void_p),
                                  C.c_int32(pl.shape[0]), tr.ctypes.data_as(C.c_void_p), C.c_int32(tr.shape[0]),
                                  C.byref(o) if o else None, C.byref(self._h))
        _check(rc, "gn_geometry_create")
        self.n_places = int(L.gn_geometry_num_places(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().gn_geometry_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def tolerance(self, precision):
        return lib().gn_geometry_tolerance(self._h, precision)

    def voxel_info(self):
        info = (C.c_int64 * 4)()
        _check(lib().gn_geometry_voxel_info(self._h, info), "gn_geometry_voxel_info")
        return {"grids": info[0], "cells": info[1], "candidates": info[2], "device_bytes": info[3]}


def nav_locate(geo: Geometry, pos, dirs=None, precision=None, out=None):
    """gn_nav_locate on device tensors: pos (n,3), dirs (n,3) or None -> int32 volume indices (n,)."""
    torch = _torch()
    precision = precision or (32 if pos.dtype == torch.float32 else 64)
    dt = _real_dtype(torch, precision)
    if pos.dtype != dt or not pos.is_cuda or (dirs is not None and (dirs.dtype != dt or not dirs.is_cuda)):
        raise GammaNavError("nav_locate: pos/dirs must be CUDA tensors of the selected precision")
    pos = pos.contiguous(); n = pos.shape[0]
    dirs = None if dirs is None else dirs.contiguous()
    if out is None:
        out = torch.empty(n, dtype=torch.int32, device=pos.device)
    _check(lib().gn_nav_locate(geo._h, precision, C.c_void_p(pos.data_ptr()), C.c_void_p(dirs.data_ptr()) if dirs is not None else None,
                               C.c_int64(n), C.c_void_p(out.data_ptr()), _stream_ptr(torch)), "gn_nav_locate")
    return out


def nav_compute_step(geo: Geometry, pos, dirs, vol, max_step=None, precision=None, out=None):
    """gn_nav_compute_step on device tensors -> (step (n,) Real, next_vol (n,) int32)."""
    torch = _torch()
    precision = precision or (32 if pos.dtype == torch.float32 else 64)
    dt = _real_dtype(torch, precision)
    if pos.dtype != dt or dirs.dtype != dt or vol.dtype != torch.int32 or not (pos.is_cuda and dirs.is_cuda and vol.is_cuda):
        raise GammaNavError("nav_compute_step: tensors must be CUDA, Real / int32")
    pos = pos.contiguous(); dirs = dirs.contiguous(); vol = vol.contiguous(); n = pos.shape[0]
    if max_step is not None:
        max_step = max_step.to(dt).contiguous()
    if out is None:
        out = (torch.empty(n, dtype=dt, device=pos.device), torch.empty(n, dtype=torch.int32, device=pos.device))
    _check(lib().gn_nav_compute_step(geo._h, precision, C.c_void_p(pos.data_ptr()), C.c_void_p(dirs.data_ptr()), C.c_void_p(vol.data_ptr()),
                                     C.c_void_p(max_step.data_ptr()) if max_step is not None else None, C.c_int64(n),
                                     C.c_void_p(out[0].data_ptr()), C.c_void_p(out[1].data_ptr()), _stream_ptr(torch)), "gn_nav_compute_step")
    return out


def nav_compute_step_noalloc(geo: Geometry, pos, dirs, vol, out, max_step=None, precision=None):
    """gn_nav_compute_step_noalloc: gn_nav_compute_step without any allocation inside the library (scratch in a fixed device
    array; n <= NOALLOC_MAX_QUERIES).  The caller passes every buffer, outputs included: out = (step (n,) Real, next_vol (n,)
    int32), contiguous CUDA tensors; nothing is converted or copied here."""
    torch = _torch()
    precision = precision or (32 if pos.dtype == torch.float32 else 64)
    dt = _real_dtype(torch, precision)
    tensors = [pos, dirs, vol, out[0], out[1]] + ([max_step] if max_step is not None else [])
    if pos.dtype != dt or dirs.dtype != dt or vol.dtype != torch.int32 or out[0].dtype != dt or out[1].dtype != torch.int32 or \
            (max_step is not None and max_step.dtype != dt) or not all(t.is_cuda and t.is_contiguous() for t in tensors):
        raise GammaNavError("nav_compute_step_noalloc: tensors must be contiguous CUDA tensors, Real / int32")
    n = pos.shape[0]
    if out[0].numel() < n or out[1].numel() < n or vol.numel() < n or dirs.shape[0] < n:
        raise GammaNavError("nav_compute_step_noalloc: buffers shorter than n")
    _check(lib().gn_nav_compute_step_noalloc(geo._h, precision, C.c_void_p(pos.data_ptr()), C.c_void_p(dirs.data_ptr()), C.c_void_p(vol.data_ptr()),
                                             C.c_void_p(max_step.data_ptr()) if max_step is not None else None, C.c_int64(n),
                                             C.c_void_p(out[0].data_ptr()), C.c_void_p(out[1].data_ptr()), _stream_ptr(torch)), "gn_nav_compute_step_noalloc")
    return out


NOALLOC_MAX_QUERIES = 1 << 20      # GN_NOALLOC_MAX_QUERIES of include/gammanav.h


def nav_compute_step_normal(geo: Geometry, pos, dirs, vol, max_step=None, precision=None):
    """gn_nav_compute_step_normal on device tensors -> (step (n,), next_vol (n,) int32, normal (n, 3))."""
    torch = _torch()
    precision = precision or (32 if pos.dtype == torch.float32 else 64)
    dt = _real_dtype(torch, precision)
    if pos.dtype != dt or dirs.dtype != dt or vol.dtype != torch.int32 or not (pos.is_cuda and dirs.is_cuda and vol.is_cuda):
        raise GammaNavError("nav_compute_step_normal: tensors must be CUDA, Real / int32")
    pos = pos.contiguous(); dirs = dirs.contiguous(); vol = vol.contiguous(); n = pos.shape[0]
    if max_step is not None:
        max_step = max_step.to(dt).contiguous()
    step = torch.empty(n, dtype=dt, device=pos.device); nxt = torch.empty(n, dtype=torch.int32, device=pos.device)
    nrm = torch.empty((n, 3), dtype=dt, device=pos.device)
    _check(lib().gn_nav_compute_step_normal(geo._h, precision, C.c_void_p(pos.data_ptr()), C.c_void_p(dirs.data_ptr()), C.c_void_p(vol.data_ptr()),
                                            C.c_void_p(max_step.data_ptr()) if max_step is not None else None, C.c_int64(n),
                                            C.c_void_p(step.data_ptr()), C.c_void_p(nxt.data_ptr()), C.c_void_p(nrm.data_ptr()), _stream_ptr(torch)),
           "gn_nav_compute_step_normal")
    return step, nxt, nrm


def nav_compute_safety(geo: Geometry, pos, vol, precision=None):
    """gn_nav_compute_safety on device tensors -> safety (n,) Real."""
    torch = _torch()
    precision = precision or (32 if pos.dtype == torch.float32 else 64)
    dt = _real_dtype(torch, precision)
    if pos.dtype != dt or vol.dtype != torch.int32 or not (pos.is_cuda and vol.is_cuda):
        raise GammaNavError("nav_compute_safety: tensors must be CUDA, Real / int32")
    pos = pos.contiguous(); vol = vol.contiguous(); n = pos.shape[0]
    out = torch.empty(n, dtype=dt, device=pos.device)
    _check(lib().gn_nav_compute_safety(geo._h, precision, C.c_void_p(pos.data_ptr()), C.c_void_p(vol.data_ptr()), C.c_int64(n),
                                       C.c_void_p(out.data_ptr()), _stream_ptr(torch)), "gn_nav_compute_safety")
    return out


def transport_run(geo: Geometry, source, seed, n_photons, precision=32, first_photon_id=0, per_photon=False, edep=None):
    """gn_transport_run -> dict(edep: cuda float64 tensor (n_places,), stats: dict[, hash, nsteps, efinal])."""
    torch = _torch()
    _real_dtype(torch, precision)
    dev = torch.device("cuda", torch.cuda.current_device())
    if edep is None:
        edep = torch.empty(geo.n_places, dtype=torch.float64, device=dev)
    st = RunStats(); cs = _csource(source)
    h = ns = ef = None
    if per_photon:
        h = torch.empty(n_photons, dtype=torch.int64, device=dev)     # uint64 bit pattern
        ns = torch.empty(n_photons, dtype=torch.int32, device=dev)
        ef = torch.empty(n_photons, dtype=torch.float64, device=dev)
    _check(lib().gn_transport_run(geo._h, precision, C.byref(cs), C.c_uint64(seed), C.c_int64(first_photon_id), C.c_int64(n_photons),
                                  C.c_void_p(edep.data_ptr()), C.byref(st),
                                  C.c_void_p(h.data_ptr()) if per_photon else None, C.c_void_p(ns.data_ptr()) if per_photon else None,
                                  C.c_void_p(ef.data_ptr()) if per_photon else None, _stream_ptr(torch)), "gn_transport_run")
    out = {"edep": edep, "stats": st.as_dict()}
    if per_photon:
        out.update(hash=h, nsteps=ns, efinal=ef)
    return out


def free_path_run(geo: Geometry, pos, dirs, Y, mu_mass, precision=None, out=None, nsteps=True):
    """gn_free_path_run on device tensors -> (T (n,) Real, nsteps (n,) int32 bit pattern of uint32 or None)."""
    torch = _torch()
    precision = precision or (32 if pos.dtype == torch.float32 else 64)
    dt = _real_dtype(torch, precision)
    if pos.dtype != dt or dirs.dtype != dt or Y.dtype != dt or not (pos.is_cuda and dirs.is_cuda and Y.is_cuda):
        raise GammaNavError("free_path_run: tensors must be CUDA and Real")
    pos = pos.contiguous(); dirs = dirs.contiguous(); Y = Y.contiguous(); n = pos.shape[0]
    T = out if out is not None else torch.empty(n, dtype=dt, device=pos.device)
    ns = torch.empty(n, dtype=torch.int32, device=pos.device) if nsteps else None
    _check(lib().gn_free_path_run(geo._h, precision, C.c_void_p(pos.data_ptr()), C.c_void_p(dirs.data_ptr()), C.c_void_p(Y.data_ptr()), C.c_int64(n),
                                  C.c_double(float(mu_mass)), C.c_void_p(T.data_ptr()), C.c_void_p(ns.data_ptr()) if nsteps else None,
                                  _stream_ptr(torch)), "gn_free_path_run")
    return T, ns


def free_path_run_host(geo: Geometry, pos: np.ndarray, dirs: np.ndarray, Y: np.ndarray, mu_mass, precision=64):
    """gn_free_path_run_host: host numpy buffers in, T (and steps) out; the copies happen inside (Algorithm 2 phases 4-6)."""
    R = np.float32 if precision == 32 else np.float64
    pos = _np(pos, R); dirs = _np(dirs, R); Y = _np(Y, R); n = pos.shape[0]
    T = np.empty(n, R); ns = np.empty(n, np.uint32)
    _check(lib().gn_free_path_run_host(geo._h, precision, pos.ctypes.data_as(C.c_void_p), dirs.ctypes.data_as(C.c_void_p), Y.ctypes.data_as(C.c_void_p),
                                       C.c_int64(n), C.c_double(float(mu_mass)), T.ctypes.data_as(C.c_void_p), ns.ctypes.data_as(C.c_void_p)), "gn_free_path_run_host")
    return T, ns


def nav_query_host(geo: Geometry, pos: np.ndarray, dirs: np.ndarray, precision=64, out=None):
    """gn_nav_query_host: host numpy buffers in, host numpy out (locate + compute_step, copies inside).
    out = (vol int32 (n,), step Real (n,), next int32 (n,)) numpy arrays to fill (page-locked ones let the copies overlap)."""
    R = np.float32 if precision == 32 else np.float64
    pos = _np(pos, R); dirs = _np(dirs, R); n = pos.shape[0]
    if out is not None:
        vol, step, nxt = out
        if vol.dtype != np.int32 or nxt.dtype != np.int32 or step.dtype != R or min(vol.size, step.size, nxt.size) < n or \
                not (vol.flags.c_contiguous and step.flags.c_contiguous and nxt.flags.c_contiguous):
            raise GammaNavError("nav_query_host: out must be contiguous (int32, Real, int32) arrays of at least n elements")
    else:
        vol = np.empty(n, np.int32); step = np.empty(n, R); nxt = np.empty(n, np.int32)
    _check(lib().gn_nav_query_host(geo._h, precision, pos.ctypes.data_as(C.c_void_p), dirs.ctypes.data_as(C.c_void_p), C.c_int64(n),
                                   vol.ctypes.data_as(C.c_void_p), step.ctypes.data_as(C.c_void_p), nxt.ctypes.data_as(C.c_void_p)), "gn_nav_query_host")
    return vol, step, nxt


def transport_run_host(geo: Geometry, source, seed, n_photons, precision=32, first_photon_id=0):
    """gn_transport_run_host: per-volume edep returned in a host numpy array."""
    edep = np.empty(geo.n_places, np.float64); st = RunStats(); cs = _csource(source)
    _check(lib().gn_transport_run_host(geo._h, precision, C.byref(cs), C.c_uint64(seed), C.c_int64(first_photon_id), C.c_int64(n_photons),
                                       edep.ctypes.data_as(C.c_void_p), C.byref(st)), "gn_transport_run_host")
    return {"edep": edep, "stats": st.as_dict()}


def selftest_arith(n_div_pairs=1 << 30):
    """gn_selftest_arith: in-line fp32 division / square root of the kernels vs. the IEEE intrinsics, bit for bit."""
    _torch()
    out = (C.c_uint64 * 4)()
    _check(lib().gn_selftest_arith(C.c_int64(n_div_pairs), out), "gn_selftest_arith")
    return {"sqrt_mismatches": out[0], "div_mismatches": out[1], "first_bad_sqrt": out[2], "first_bad_div": out[3]}


def selftest_pipe_peak(precision=32):
    """gn_selftest_pipe_peak: FFMA / DFMA pipe peak of the current device (the flops leg of the roofline)."""
    _torch()
    out = (C.c_double * 4)()
    _check(lib().gn_selftest_pipe_peak(int(precision), out), "gn_selftest_pipe_peak")
    return {"tflops": out[0], "sm_mhz": out[1], "ms": out[2], "sms": int(out[3])}


def host_source_frame(source, precision=64):
    """gn_host_source_frame (host-only hook): rows a, e1, e2 of the source frame as rounded to `precision`."""
    out = np.empty(9, np.float64); cs = _csource(source)
    _check(lib().gn_host_source_frame(C.byref(cs), int(precision), out.ctypes.data_as(C.c_void_p)), "gn_host_source_frame")
    return out.reshape(3, 3)


def host_compose_transforms(geom):
    """gn_host_compose_transforms (host-only hook): composed global->local (M (n, 9), T (n, 3)) of every placement, fp64."""
    pl = _np(geom.placements, np.int32); tr = _np(geom.transforms, np.float64)
    M = np.empty((pl.shape[0], 9), np.float64); T = np.empty((pl.shape[0], 3), np.float64)
    _check(lib().gn_host_compose_transforms(pl.ctypes.data_as(C.c_void_p), C.c_int32(pl.shape[0]), tr.ctypes.data_as(C.c_void_p), C.c_int32(tr.shape[0]),
                                            M.ctypes.data_as(C.c_void_p), T.ctypes.data_as(C.c_void_p)), "gn_host_compose_transforms")
    return M, T


def host_voxel_tables(geom, **opts):
    """gn_host_voxel_tables: the voxel grids, candidate lists, node flags and sibling hints gn_geometry_create builds for `geom`,
    as numpy arrays (host only, no device needed)."""
    L = lib()
    mats = _np(geom.materials, np.float64); st = _np(geom.solid_type, np.int32); sp = _np(geom.solid_params, np.float64)
    pl = _np(geom.placements, np.int32); tr = _np(geom.transforms, np.float64)
    o = Opts(**opts) if opts else None
    counts = (C.c_int64 * 3)()

    def call(info, link, hint, grids, cell_start, cand):
        p = lambda a: a.ctypes.data_as(C.c_void_p) if a is not None else None
        _check(L.gn_host_voxel_tables(p(mats), C.c_int32(mats.shape[0]), p(st), p(sp), C.c_int32(st.shape[0]), p(pl), C.c_int32(pl.shape[0]),
                                      p(tr), C.c_int32(tr.shape[0]), C.byref(o) if o else None, counts, p(info), p(link), p(hint), p(grids),
                                      p(cell_start), p(cand)), "gn_host_voxel_tables")
    call(None, None, None, None, None, None)
    V, ng, nc, nk = pl.shape[0], counts[0], counts[1], counts[2]
    info = np.empty(V, np.int32); link = np.empty(V, np.int32); hint = np.empty((V, 4), np.int32)
    grids = np.empty((max(ng, 1), 11), np.float64); cell_start = np.empty(nc + 1, np.int32); cand = np.empty(max(nk, 1), np.int32)
    call(info, link, hint, grids, cell_start, cand)
    return {"info": info, "link": link, "hint": hint, "grids": grids[:ng], "cell_start": cell_start, "cand": cand[:nk]}
