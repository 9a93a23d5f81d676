"""ctypes loader for the fp64 CPU oracle (TEST INFRASTRUCTURE -- see oracle/chisao_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from the CUDA path; it accepts any object with the attributes of
`paper_2606_26164_b200.inputs.Workload` (plain arrays and numbers).
"""
from __future__ import annotations

import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import build as _build  # noqa: E402  (oracle/build.py)

X, F, G, V, STUCK, REMOVED, HIST_S, HIST_Y, HIST_LEN, STALLED, CTRL = range(11)
P, LS_B, LS_MARGIN, ASC_MARGIN, CURV_MARGIN, GHAT, HLC_F, RS_SRC, RS_CAND, RS_MARGIN, HLC_U = range(20, 31)
SIGMA = 33
RS_SCORE = 34
PH_RELEASE_EVAL, PH_STICK, PH_DEDUP, PH_RESEED, PH_HLC_STEP, PH_ANTI_STEP, PH_LBFGS_ITER = 1, 2, 3, 4, 5, 6, 11

_fp = C.POINTER(C.c_float)


class _Objective(C.Structure):
    _fields_ = [("id", C.c_int32), ("d", C.c_int32), ("K", C.c_int32),
                ("means", _fp), ("mats", _fp), ("vec_a", _fp), ("vec_b", _fp),
                ("scalar0", C.c_float), ("sigma_noise", C.c_float)]


class _Config(C.Structure):
    _fields_ = [("d", C.c_int32), ("N", C.c_int32), ("lo", _fp), ("hi", _fp)] + \
               [(n, C.c_int32) for n in ("n_osc", "n_conv", "n_anti", "n_cloud", "hlc_M", "lbfgs_m",
                                         "ls_max", "reseed_cands")] + \
               [(n, C.c_float) for n in ("fd_h", "eps_grad", "eps_dup", "log_delta", "mu", "alpha_anti",
                                         "eta_hlc", "sigma_s", "ls_c1", "ls_shrink")] + \
               [("hlc_baseline", C.c_int32), ("phase_mask", C.c_uint32), ("seed", C.c_uint64)]


class Stats(C.Structure):
    _fields_ = [("cycle", C.c_int32), ("n_stuck", C.c_int32), ("k_lost", C.c_int32),
                ("n_active", C.c_int32), ("reseed_strategy", C.c_int32), ("gr_enabled", C.c_int32),
                ("evals", C.c_uint64 * 8), ("f_max", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_create.restype = C.c_void_p
        L.orc_create.argtypes = [C.POINTER(_Config), C.POINTER(_Objective), _fp]
        L.orc_destroy.argtypes = [C.c_void_p]
        L.orc_set_threads.argtypes = [C.c_void_p, C.c_int]
        L.orc_step.argtypes = [C.c_void_p, C.POINTER(Stats)]
        L.orc_phase.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.orc_modes.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.POINTER(C.c_int32)]
        L.orc_get.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_uint64]
        L.orc_set.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_uint64]
        L.orc_stats_now.argtypes = [C.c_void_p, C.POINTER(Stats)]
        L.orc_objective_values.argtypes = [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]
        L.orc_fd_gradient.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_two_loop.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_philox4x32_10.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        for fn in (L.orc_uniform, L.orc_normal):
            fn.restype = C.c_double
            fn.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint64]
        L.orc_gr_basis.argtypes = [C.c_void_p, C.c_int, C.c_void_p]
        L.orc_noise.restype = C.c_double
        L.orc_noise.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_fp) if a is not None else C.cast(None, _fp)


_FIELD_DTYPE = {STUCK: np.uint8, REMOVED: np.uint8, STALLED: np.uint8, HIST_LEN: np.int32, CTRL: np.int32,
                LS_B: np.int32, RS_SRC: np.int32, RS_CAND: np.int32}


class Oracle:
    """One CHISAO run on the CPU in fp64.  `wl` is an inputs.Workload-like object."""

    def __init__(self, wl, threads: int = 1):
        o, h = wl.obj, wl.hp
        self.d, self.N, self.m, self.M = h.d, h.N, h.lbfgs_m, h.hlc_M
        self._keep = [np.ascontiguousarray(a, np.float32) if a is not None else None
                      for a in (o.means, o.mats, o.vec_a, o.vec_b, h.lo, h.hi, wl.x0)]
        me, ma, va, vb, lo, hi, x0 = self._keep
        self._obj = _Objective(o.id, o.d, o.K, _p(me), _p(ma), _p(va), _p(vb), o.scalar0, o.sigma_noise)
        self._cfg = _Config(h.d, h.N, _p(lo), _p(hi), h.n_osc, h.n_conv, h.n_anti, h.n_cloud, h.hlc_M,
                            h.lbfgs_m, h.ls_max, h.reseed_cands, h.fd_h, h.eps_grad, h.eps_dup,
                            h.log_delta, h.mu, h.alpha_anti, h.eta_hlc, h.sigma_s, h.ls_c1, h.ls_shrink,
                            h.hlc_baseline, h.phase_mask & 0xFFFFFFFF, h.seed)
        self._h = lib().orc_create(C.byref(self._cfg), C.byref(self._obj), _p(x0))
        if not self._h:
            raise ValueError("orc_create rejected the configuration")
        lib().orc_set_threads(self._h, threads)

    def close(self):
        if self._h:
            lib().orc_destroy(self._h)
            self._h = None

    __del__ = close

    def _shape(self, field):
        N, d, m, M = self.N, self.d, self.m, self.M
        return {X: (N, d), G: (N, d), V: (N, d), P: (N, d), GHAT: (N, d), HIST_S: (m, N, d), HIST_Y: (m, N, d),
                HLC_F: (N, M), HLC_U: (N, M, d), CTRL: (8,), SIGMA: (1,), RS_SCORE: (N, 16)}.get(field, (N,))

    def get(self, field):
        a = np.empty(self._shape(field), _FIELD_DTYPE.get(field, np.float64))
        rc = lib().orc_get(self._h, field, a.ctypes.data, a.nbytes)
        if rc:
            raise RuntimeError(f"orc_get({field}) -> {rc}")
        return a

    def set(self, field, value):
        a = np.ascontiguousarray(value, _FIELD_DTYPE.get(field, np.float64)).reshape(self._shape(field))
        rc = lib().orc_set(self._h, field, a.ctypes.data, a.nbytes)
        if rc:
            raise RuntimeError(f"orc_set({field}) -> {rc}")

    def step(self) -> Stats:
        st = Stats()
        rc = lib().orc_step(self._h, C.byref(st))
        if rc:
            raise RuntimeError(f"orc_step -> {rc}")
        return st

    def stats(self) -> Stats:
        st = Stats()
        lib().orc_stats_now(self._h, C.byref(st))
        return st

    def phase(self, phase_id, it=0):
        rc = lib().orc_phase(self._h, phase_id, it)
        if rc:
            raise RuntimeError(f"orc_phase({phase_id}) -> {rc}")

    def modes(self):
        n = C.c_int32(0)
        x = np.empty((max(self.N, 1), self.d)); f = np.empty(max(self.N, 1)); idx = np.empty(max(self.N, 1), np.int32)
        lib().orc_modes(self._h, x.ctypes.data, f.ctypes.data, idx.ctypes.data, self.N, C.byref(n))
        return x[:n.value].copy(), f[:n.value].copy(), idx[:n.value].copy()

    def values(self, pts):
        pts = np.ascontiguousarray(pts, np.float64).reshape(-1, self.d)
        out = np.empty(pts.shape[0])
        lib().orc_objective_values(self._h, pts.ctypes.data, pts.shape[0], out.ctypes.data)
        return out

    def fd_gradient(self, x):
        x = np.ascontiguousarray(x, np.float64)
        f = np.empty(1); g = np.empty(self.d)
        lib().orc_fd_gradient(self._h, x.ctypes.data, f.ctypes.data, g.ctypes.data)
        return float(f[0]), g

    def gr_basis(self, cycle):
        q = np.empty((self.d, self.d))
        lib().orc_gr_basis(self._h, cycle, q.ctypes.data)
        return q

    def noise(self, cycle, sample, phase, it, slot):
        return lib().orc_noise(self._h, cycle, sample, phase, it, slot)


def two_loop(S, Y, gamma):
    S = np.ascontiguousarray(S, np.float64); Y = np.ascontiguousarray(Y, np.float64)
    gamma = np.ascontiguousarray(gamma, np.float64)
    r = np.empty_like(gamma)
    lib().orc_two_loop(gamma.shape[0], S.shape[0], S.ctypes.data, Y.ctypes.data, gamma.ctypes.data, r.ctypes.data)
    return r


def philox(ctr, key):
    c = np.asarray(ctr, np.uint32); k = np.asarray(key, np.uint32); o = np.empty(4, np.uint32)
    lib().orc_philox4x32_10(c.ctypes.data, k.ctypes.data, o.ctypes.data)
    return o


def tag(phase, it, purpose):
    return (phase << 24) | ((it & 0xFFFF) << 8) | purpose


def uniform(seed, c1, c2, c3, n):
    return lib().orc_uniform(seed, c1, c2, c3, n)


def normal(seed, c1, c2, c3, n):
    return lib().orc_normal(seed, c1, c2, c3, n)
