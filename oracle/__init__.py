"""ctypes binding of the CPU oracle (oracle/oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  It imports nothing from the product package; geometries and sources are
passed as objects with the plain-array attributes described in oracle.h.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None


class Opts(C.Structure):
    _fields_ = [("tol64", C.c_double), ("tol32", C.c_double), ("sigma_pe0", C.c_double), ("e_cut", C.c_double),
                ("grid_min_daughters", C.c_int32), ("stuck_limit", C.c_int32), ("secondaries", C.c_int32), ("rayleigh", C.c_int32),
                ("sigma_r0", C.c_double), ("pe_table_per_decade", C.c_int32), ("pe_k_edge", C.c_int32)]


class CSource(C.Structure):
    _fields_ = [("kind", C.c_int32), ("energy_kind", C.c_int32), ("origin", C.c_double * 3), ("axis", C.c_double * 3),
                ("sigma", C.c_double), ("half_angle", C.c_double), ("e0", C.c_double), ("e1", C.c_double)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("n_steps", "n_compton", "n_pe", "n_pair", "n_cut", "n_escaped", "n_stuck", "n_photons")] + \
               [(n, C.c_double) for n in ("e_escaped", "e_stuck", "e_source", "e_deposited")] + [("n_rayleigh", C.c_uint64)]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


def lib():
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.oracle_geometry_tolerance.restype = C.c_double
        L.oracle_sigma_kn.restype = C.c_double; L.oracle_sigma_kn.argtypes = [C.c_double]
        L.oracle_sigma_pair.restype = C.c_double; L.oracle_sigma_pair.argtypes = [C.c_double, C.c_double]
        L.oracle_sigma_pe.restype = C.c_double; L.oracle_sigma_pe.argtypes = [C.c_double, C.c_double, C.c_double]
        L.oracle_uniform_from_lane.restype = C.c_double; L.oracle_uniform_from_lane.argtypes = [C.c_uint64, C.c_int]
        L.oracle_draw.restype = C.c_double; L.oracle_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_int]
        L.oracle_mu_rayleigh.restype = C.c_double; L.oracle_mu_rayleigh.argtypes = [C.c_void_p, C.c_int, C.c_int32, C.c_double]
        L.oracle_fnv1a_bytes.restype = C.c_uint64; L.oracle_fnv1a_bytes.argtypes = [C.c_void_p, C.c_int64]
        L.oracle_history_hash.restype = C.c_uint64; L.oracle_history_hash.argtypes = [C.c_void_p, C.c_int64]
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _real(precision):
    return np.float32 if precision == 32 else np.float64


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def _csource(src):
    s = CSource()
    s.kind, s.energy_kind = int(src.kind), int(src.energy_kind)
    s.origin[:] = [float(v) for v in src.origin]; s.axis[:] = [float(v) for v in src.axis]
    s.sigma, s.half_angle, s.e0, s.e1 = float(src.sigma), float(src.half_angle), float(src.e0), float(src.e1)
    return s


class OracleGeometry:
    def __init__(self, geom, **opts):
        o = Opts(**opts) if opts else None
        self._h = C.c_void_p()
        self.n_places = int(geom.placements.shape[0])
        arrs = [np.ascontiguousarray(geom.materials, np.float64), np.ascontiguousarray(geom.solid_type, np.int32),
                np.ascontiguousarray(geom.solid_params, np.float64), np.ascontiguousarray(geom.placements, np.int32),
                np.ascontiguousarray(geom.transforms, np.float64)]
        rc = lib().oracle_geometry_create(_p(arrs[0]), C.c_int32(arrs[0].shape[0]), _p(arrs[1]), _p(arrs[2]), C.c_int32(arrs[1].shape[0]),
                                          _p(arrs[3]), C.c_int32(arrs[3].shape[0]), _p(arrs[4]), C.c_int32(arrs[4].shape[0]),
                                          C.byref(o) if o else None, C.byref(self._h))
        self.rc = rc
        _check(rc, "geometry_create")

    def __del__(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().oracle_geometry_destroy(self._h); self._h = C.c_void_p()

    def tolerance(self, precision):
        return lib().oracle_geometry_tolerance(self._h, C.c_int(precision))

    def locate(self, pos, dirs=None, precision=64, use_grid=True):
        R = _real(precision)
        pos = np.ascontiguousarray(pos, R); n = pos.shape[0]
        dirs = None if dirs is None else np.ascontiguousarray(dirs, R)
        out = np.empty(n, np.int32)
        _check(lib().oracle_nav_locate(self._h, C.c_int(precision), _p(pos), _p(dirs), C.c_int64(n), _p(out), C.c_int(int(use_grid))), "nav_locate")
        return out

    def locate_bruteforce(self, pos):
        pos = np.ascontiguousarray(pos, np.float64); out = np.empty(pos.shape[0], np.int32)
        _check(lib().oracle_nav_locate_bruteforce(self._h, _p(pos), C.c_int64(pos.shape[0]), _p(out)), "locate_bruteforce")
        return out

    def compute_step(self, pos, dirs, vol, max_step=None, precision=64, use_grid=True):
        R = _real(precision)
        pos = np.ascontiguousarray(pos, R); dirs = np.ascontiguousarray(dirs, R); vol = np.ascontiguousarray(vol, np.int32)
        ms = None if max_step is None else np.ascontiguousarray(max_step, R)
        n = pos.shape[0]
        step = np.empty(n, R); nxt = np.empty(n, np.int32)
        _check(lib().oracle_nav_compute_step(self._h, C.c_int(precision), _p(pos), _p(dirs), _p(vol), _p(ms), C.c_int64(n), _p(step), _p(nxt),
                                             C.c_int(int(use_grid))), "nav_compute_step")
        return step, nxt

    def compute_step_normal(self, pos, dirs, vol, max_step=None, precision=64, use_grid=True):
        R = _real(precision)
        pos = np.ascontiguousarray(pos, R); dirs = np.ascontiguousarray(dirs, R); vol = np.ascontiguousarray(vol, np.int32)
        ms = None if max_step is None else np.ascontiguousarray(max_step, R)
        n = pos.shape[0]
        step = np.empty(n, R); nxt = np.empty(n, np.int32); nrm = np.empty((n, 3), R)
        _check(lib().oracle_nav_compute_step_normal(self._h, C.c_int(precision), _p(pos), _p(dirs), _p(vol), _p(ms), C.c_int64(n), _p(step), _p(nxt),
                                                    _p(nrm), C.c_int(int(use_grid))), "nav_compute_step_normal")
        return step, nxt, nrm

    def compute_safety(self, pos, vol, precision=64):
        R = _real(precision)
        pos = np.ascontiguousarray(pos, R); vol = np.ascontiguousarray(vol, np.int32)
        out = np.empty(pos.shape[0], R)
        _check(lib().oracle_nav_compute_safety(self._h, C.c_int(precision), _p(pos), _p(vol), C.c_int64(pos.shape[0]), _p(out)), "nav_compute_safety")
        return out

    def transport(self, src, seed, n, precision=64, first_id=0, per_photon=False, use_grid=True, tally=False):
        """tally=True adds per volume the sum of the squared deposits and the number of deposits (edep_sq, n_dep)."""
        edep = np.zeros(self.n_places, np.float64); st = Stats()
        h = np.empty(n, np.uint64) if per_photon else None
        ns = np.empty(n, np.uint32) if per_photon else None
        ef = np.empty(n, np.float64) if per_photon else None
        sq = np.zeros(self.n_places, np.float64) if tally else None
        nd = np.zeros(self.n_places, np.uint32) if tally else None
        cs = _csource(src)
        _check(lib().oracle_transport_run_tally(self._h, C.c_int(precision), C.byref(cs), C.c_uint64(seed), C.c_int64(first_id), C.c_int64(n),
                                                _p(edep), _p(sq), _p(nd), C.byref(st), _p(h), _p(ns), _p(ef), C.c_int(int(use_grid))), "transport_run")
        out = {"edep": edep, "stats": st.as_dict()}
        if per_photon:
            out.update(hash=h, nsteps=ns, efinal=ef)
        if tally:
            out.update(edep_sq=sq, n_dep=nd)
        return out

    OP_NAMES = ("add", "mul", "div", "sqrt", "cmp", "fma", "trans", "flops")

    def transport_count_ops(self, src, seed, n, first_id=0):
        """Operation counts of n histories (S:8(d) instrumented oracle) -> (dict of counts, stats)."""
        c = np.zeros(8, np.uint64); st = Stats(); cs = _csource(src)
        _check(lib().oracle_transport_count_ops(self._h, C.byref(cs), C.c_uint64(seed), C.c_int64(first_id), C.c_int64(n), _p(c), C.byref(st)), "transport_count_ops")
        return dict(zip(self.OP_NAMES, (int(v) for v in c))), st.as_dict()

    def nav_count_ops(self, pos, dirs):
        """Operation counts of len(pos) navigation queries (locate, then ComputeStep)."""
        pos = np.ascontiguousarray(pos, np.float64); dirs = np.ascontiguousarray(dirs, np.float64)
        c = np.zeros(8, np.uint64)
        _check(lib().oracle_nav_count_ops(self._h, _p(pos), _p(dirs), C.c_int64(pos.shape[0]), _p(c)), "nav_count_ops")
        return dict(zip(self.OP_NAMES, (int(v) for v in c)))

    def composed_transforms(self, precision=64):
        """Global->local (M row-major, T) of every node as stored for `precision` (test hook, S:C0)."""
        M = np.empty((self.n_places, 9)); T = np.empty((self.n_places, 3))
        _check(lib().oracle_composed_transforms(self._h, C.c_int(precision), _p(M), _p(T)), "composed_transforms")
        return M, T

    def free_path(self, pos, dirs, Y, mu_mass, precision=64, use_grid=True):
        """The paper's benchmark (Algorithm 2 phase 5): T_i from (x0, w, Y)_i, attenuation only.  -> (T, nsteps)."""
        R = _real(precision)
        pos = np.ascontiguousarray(pos, R); dirs = np.ascontiguousarray(dirs, R); Y = np.ascontiguousarray(Y, R)
        n = pos.shape[0]
        T = np.empty(n, R); ns = np.empty(n, np.uint32)
        _check(lib().oracle_free_path_run(self._h, C.c_int(precision), _p(pos), _p(dirs), _p(Y), C.c_int64(n), C.c_double(mu_mass), _p(T), _p(ns),
                                          C.c_int(int(use_grid))), "free_path_run")
        return T, ns

    def mu_rayleigh(self, material, E, precision=64):
        return lib().oracle_mu_rayleigh(self._h, precision, int(material), float(E))

    def mu(self, material, E, precision=64):
        m = np.empty(3, np.float64)
        _check(lib().oracle_mu(self._h, C.c_int(precision), C.c_int32(material), C.c_double(E), _p(m)), "mu")
        return m


def solid_eval(stype, params, tol, what, pos, dirs=None, precision=64):
    """what: 'inside' | 'dist_in' | 'dist_out' for one solid on many points."""
    R = _real(precision)
    code = {"inside": 0, "dist_in": 1, "dist_out": 2, "normal": 3, "safety_in": 4, "safety_out": 5}[what]
    pos = np.ascontiguousarray(pos, R)
    dirs = np.ascontiguousarray(dirs if dirs is not None else np.zeros_like(pos), R)
    p5 = np.zeros(5, np.float64); p5[:len(params)] = params
    out = np.empty((pos.shape[0], 3) if what == "normal" else pos.shape[0], R)
    _check(lib().oracle_solid_eval(C.c_int32(stype), _p(p5), C.c_double(tol), C.c_int(precision), C.c_int(code), _p(pos), _p(dirs),
                                   C.c_int64(pos.shape[0]), _p(out)), "solid_eval")
    return out.astype(np.int32) if what == "inside" else out


def sigma_kn(k):
    return lib().oracle_sigma_kn(float(k))


def sigma_pair(k, Z):
    return lib().oracle_sigma_pair(float(k), float(Z))


def sigma_pe(E, Z, s0=1750.0):
    return lib().oracle_sigma_pe(float(E), float(Z), float(s0))


def pair_directions(seed, first_id, n, precision=64):
    """Directions of the two annihilation photons of photons first_id .. first_id + n - 1 (test hook)."""
    w1 = np.empty((n, 3), np.float64); w2 = np.empty((n, 3), np.float64)
    _check(lib().oracle_pair_directions(C.c_int(precision), C.c_uint64(seed), C.c_int64(first_id), C.c_int64(n), _p(w1), _p(w2)), "pair_directions")
    return w1, w2


def fnv1a_bytes(data: bytes) -> int:
    """FNV-1a-64 of a byte string through the oracle's own byte step (test hook for the history hash, S:C9)."""
    buf = np.frombuffer(bytes(data), np.uint8) if len(data) else np.zeros(0, np.uint8)
    return int(lib().oracle_fnv1a_bytes(_p(np.ascontiguousarray(buf)) if len(buf) else None, C.c_int64(len(buf))))


def history_hash(words) -> int:
    """History hash of a list of 32-bit words (vol_before, event, vol_before, event, ...)."""
    w = np.ascontiguousarray(np.asarray(words, dtype=np.int64) & 0xffffffff, np.uint32)
    return int(lib().oracle_history_hash(_p(w) if len(w) else None, C.c_int64(len(w))))


def source_frame(src, precision=64):
    """(a, e1, e2) of a source as rounded to `precision` (D:reading 4)."""
    out = np.empty(9); cs = _csource(src)
    _check(lib().oracle_source_frame(C.byref(cs), C.c_int(precision), _p(out)), "source_frame")
    return out.reshape(3, 3)


def philox(counter, key):
    out = (C.c_uint32 * 4)()
    lib().oracle_philox4x32_10(*[C.c_uint32(int(c)) for c in counter], C.c_uint32(int(key[0])), C.c_uint32(int(key[1])), out)
    return [int(v) for v in out]


def uniform_from_lane(lane, precision=64):
    return lib().oracle_uniform_from_lane(int(lane), precision)


def draw(seed, pid, j, precision=64):
    return lib().oracle_draw(int(seed), int(pid), int(j), precision)


def kn_sample(E, seed, n, precision=64, first_id=0):
    eps = np.empty(n); cost = np.empty(n); nt = np.empty(n, np.int32)
    _check(lib().oracle_kn_sample(C.c_int(precision), C.c_double(E), C.c_uint64(seed), C.c_int64(first_id), C.c_int64(n), _p(eps), _p(cost), _p(nt)), "kn_sample")
    return eps, cost, nt


def rayleigh_sample(seed, n, precision=64, first_id=0):
    """n cosines of the Rayleigh scattering angle (rejection from 1 + c^2) and the trials each took."""
    c = np.empty(n); nt = np.empty(n, np.int32)
    _check(lib().oracle_rayleigh_sample(C.c_int(precision), C.c_uint64(seed), C.c_int64(first_id), C.c_int64(n), _p(c), _p(nt)), "rayleigh_sample")
    return c, nt


def rotate(w, cost, phi, precision=64):
    w = np.ascontiguousarray(w, np.float64); cost = np.ascontiguousarray(cost, np.float64); phi = np.ascontiguousarray(phi, np.float64)
    out = np.empty_like(w)
    _check(lib().oracle_rotate(C.c_int(precision), _p(w), _p(cost), _p(phi), C.c_int64(w.shape[0]), _p(out)), "rotate")
    return out


def move(pos, dirs, step, precision=64):
    R = _real(precision)
    pos = np.ascontiguousarray(pos, R); dirs = np.ascontiguousarray(dirs, R); step = np.ascontiguousarray(step, R)
    out = np.empty_like(pos)
    _check(lib().oracle_move(C.c_int(precision), _p(pos), _p(dirs), _p(step), C.c_int64(pos.shape[0]), _p(out)), "move")
    return out


def source_sample(src, seed, n, precision=64, first_id=0):
    pos = np.empty((n, 3)); d = np.empty((n, 3)); e = np.empty(n); nd = np.empty(n, np.int32)
    cs = _csource(src)
    _check(lib().oracle_source_sample(C.c_int(precision), C.byref(cs), C.c_uint64(seed), C.c_int64(first_id), C.c_int64(n), _p(pos), _p(d), _p(e), _p(nd)), "source_sample")
    return pos, d, e, nd
