"""Thin ctypes binding of libchisao.so (include/chisao.h): argument marshalling only.

Every step of the CHISAO cycle runs in the CUDA kernels behind the C ABI; PyTorch is used here for device
memory (the population and the workspace are torch tensors owned by the `Chisao` object) and for the
stream.  There is no CPU fallback: a missing library or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libchisao.so")

OK, E_INVALID, E_WORKSPACE, E_CAPACITY, E_CUDA, E_STATE = 0, -1, -2, -3, -4, -5
X, F, G, V, STUCK, REMOVED, HIST_S, HIST_Y, HIST_LEN, STALLED, CTRL = range(11)
P, LS_B, GHAT, HLC_F, RS_SRC, RS_CAND, XT, GR_Q, SIGMA = 20, 21, 25, 26, 27, 28, 31, 32, 33
PH_RELEASE_EVAL, PH_STICK, PH_DEDUP, PH_RESEED, PH_HLC_STEP, PH_ANTI_STEP, PH_LBFGS_ITER = 1, 2, 3, 4, 5, 6, 11
PH_LBFGS_DIRECTION = 12
OPT_STENCIL_AWARE = 1
OPT_CUDA_GRAPH = 2
OPT_LS_TILE_LOCAL = 3
OPT_LBFGS_RESIDENT = 4
INFO_EVALUATOR = 1
INFO_GRAPH_LAUNCHES = 2
INFO_LS_TILE_LOCAL = 3
INFO_LBFGS_RESIDENT = 4
EVALUATOR_NAMES = ("fp32-fma", "tcgen05 3xTF32 (x - c)", "tcgen05 x-stationary tf32 hi/lo", "tcgen05 x-stationary fp16 hi/lo",
                   "tcgen05 exact fixed-point fp16 pieces (random-Fourier phases)", "tcgen05 scaled fp16 hi/lo (x - c)")
TIMING_CLASSES = ("eval_fd", "eval_points", "hlc", "lbfgs_direction", "lbfgs_update", "select", "reseed")

EXPORTS = ("chisao_workspace_bytes", "chisao_init", "chisao_seed_population", "chisao_step", "chisao_step_host",
           "chisao_modes", "chisao_get_state", "chisao_set_state", "chisao_phase", "chisao_get_stats",
           "chisao_set_option", "chisao_get_info", "chisao_launch_count", "chisao_timing_enable", "chisao_timing_reset", "chisao_timing_get",
           "chisao_measure_peak", "chisao_stick_test_static", "chisao_last_error", "chisao_destroy")
STATIC_MAX_N = 262144                       # CHISAO_STATIC_MAX_N
STATIC_SCRATCH_BYTES = 256 + 4 * STATIC_MAX_N

_fp = C.POINTER(C.c_float)


class Objective(C.Structure):
    _fields_ = [("id", C.c_int32), ("d", C.c_int32), ("K", C.c_int32),
                ("means", _fp), ("mats", _fp), ("vec_a", _fp), ("vec_b", _fp),
                ("scalar0", C.c_float), ("sigma_noise", C.c_float)]


class Config(C.Structure):
    _fields_ = [("d", C.c_int32), ("N", C.c_int32), ("lo", _fp), ("hi", _fp)] + \
               [(n, C.c_int32) for n in ("n_osc", "n_conv", "n_anti", "n_cloud", "hlc_M", "lbfgs_m", "ls_max",
                                         "reseed_cands")] + \
               [(n, C.c_float) for n in ("fd_h", "eps_grad", "eps_dup", "log_delta", "mu", "alpha_anti",
                                         "eta_hlc", "sigma_s", "ls_c1", "ls_shrink")] + \
               [("hlc_baseline", C.c_int32), ("phase_mask", C.c_uint32), ("seed", C.c_uint64)]


class Stats(C.Structure):
    _fields_ = [("cycle", C.c_int32), ("n_stuck", C.c_int32), ("k_lost", C.c_int32), ("n_active", C.c_int32),
                ("reseed_strategy", C.c_int32), ("gr_enabled", C.c_int32), ("evals", C.c_uint64 * 8),
                ("f_max", C.c_float)]

    def total_evals(self) -> int:
        return int(sum(self.evals[k] for k in (0, 1, 2, 5, 6)))


class ChisaoError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"libchisao error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: Optional[str] = None):
    """Load libchisao.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise FileNotFoundError(f"{p} not found: build it with `python -m paper_2606_26164_b200.build` "
                                "(there is no CPU fallback)")
    L = C.CDLL(p)
    vp = C.c_void_p
    L.chisao_workspace_bytes.argtypes = [C.POINTER(Config), C.POINTER(Objective), C.POINTER(C.c_size_t)]
    L.chisao_init.argtypes = [C.POINTER(vp), C.POINTER(Config), C.POINTER(Objective), vp, vp, C.c_size_t, vp]
    L.chisao_seed_population.argtypes = [vp]
    L.chisao_step.argtypes = [vp, C.POINTER(Stats)]
    L.chisao_step_host.argtypes = [vp, vp, vp, vp, vp, C.POINTER(Stats)]
    L.chisao_modes.argtypes = [vp, vp, vp, vp, C.c_int32, C.POINTER(C.c_int32)]
    L.chisao_get_state.argtypes = [vp, C.c_int32, vp, C.c_size_t]
    L.chisao_set_state.argtypes = [vp, C.c_int32, vp, C.c_size_t]
    L.chisao_phase.argtypes = [vp, C.c_int32, C.c_int32]
    L.chisao_get_stats.argtypes = [vp, C.POINTER(Stats)]
    L.chisao_set_option.argtypes = [vp, C.c_int32, C.c_int32]
    L.chisao_get_info.argtypes = [vp, C.c_int32, C.POINTER(C.c_int32)]
    L.chisao_launch_count.argtypes = [vp]
    L.chisao_launch_count.restype = C.c_uint64
    L.chisao_timing_enable.argtypes = [vp, C.c_int32]
    L.chisao_timing_reset.argtypes = [vp]
    L.chisao_timing_get.argtypes = [vp, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]
    L.chisao_measure_peak.argtypes = [C.c_int32, vp, vp, C.POINTER(C.c_double)]
    L.chisao_stick_test_static.argtypes = [vp, vp, C.c_int32, C.c_int32, C.c_float, C.c_float, vp, vp, vp, vp]
    L.chisao_last_error.argtypes = [vp]
    L.chisao_last_error.restype = C.c_char_p
    L.chisao_destroy.argtypes = [vp]
    L.chisao_destroy.restype = None
    if path is None:
        _lib = L
    return L


def _p(a):
    return a.ctypes.data_as(_fp) if a is not None else C.cast(None, _fp)


def marshal(wl):
    """(Config, Objective, keepalive) ctypes records for an `inputs.Workload`-like object."""
    o, h = wl.obj, wl.hp
    keep = [np.ascontiguousarray(a, np.float32) if a is not None else None
            for a in (o.means, o.mats, o.vec_a, o.vec_b, h.lo, h.hi)]
    me, ma, va, vb, lo, hi = keep
    obj = Objective(o.id, o.d, o.K, _p(me), _p(ma), _p(va), _p(vb), o.scalar0, o.sigma_noise)
    cfg = Config(h.d, h.N, _p(lo), _p(hi), h.n_osc, h.n_conv, h.n_anti, h.n_cloud, h.hlc_M, h.lbfgs_m, h.ls_max,
                 h.reseed_cands, h.fd_h, h.eps_grad, h.eps_dup, h.log_delta, h.mu, h.alpha_anti, h.eta_hlc,
                 h.sigma_s, h.ls_c1, h.ls_shrink, h.hlc_baseline, h.phase_mask & 0xFFFFFFFF, h.seed)
    return cfg, obj, keep


def workspace_bytes(wl) -> int:
    cfg, obj, _keep = marshal(wl)
    n = C.c_size_t(0)
    rc = load_library().chisao_workspace_bytes(C.byref(cfg), C.byref(obj), C.byref(n))
    if rc:
        raise ChisaoError(rc, load_library().chisao_last_error(None).decode())
    return n.value


PEAK_FP32_FMA, PEAK_SFU = 0, 1


def measure_peak(which: int, device="cuda:0") -> float:
    """chisao_measure_peak: FP32 FMA rate (TFLOP/s) or MUFU rate (T op/s) of `device`, by the library's own probe kernels"""
    import torch
    L = load_library()
    dev = torch.device(device)
    with torch.cuda.device(dev):
        scratch = torch.zeros(64, dtype=torch.float32, device=dev)
        v = C.c_double(0.0)
        rc = L.chisao_measure_peak(int(which), C.c_void_p(scratch.data_ptr()),
                                   C.c_void_p(torch.cuda.current_stream(dev).cuda_stream), C.byref(v))
    if rc:
        raise ChisaoError(rc, "chisao_measure_peak failed")
    return float(v.value)


def stick_test_static(g, f, eps_grad: float, log_delta: float, stuck, n_stuck=None, f_max=None, stream=None) -> None:
    """chisao_stick_test_static: Eq. 3 on the caller's DEVICE tensors with no device allocation (the scratch is a static
    array inside the library, STATIC_SCRATCH_BYTES per GPU; N <= STATIC_MAX_N).  g [N][d] fp32, f [N] fp32 are read;
    stuck [N] uint8 and, if given, n_stuck [1] int32 and f_max [1] fp32 are written.  Asynchronous on `stream` (default:
    torch's current stream of g's device).  Calls that overlap on the GPU race on the shared scratch."""
    import torch
    L = load_library()
    N, d = (int(g.shape[0]), int(g.shape[1]))
    for t, dt, n in ((g, torch.float32, N * d), (f, torch.float32, N), (stuck, torch.uint8, N)):
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() == n and t.device == g.device):
            raise ValueError("stick_test_static: g [N][d] f32, f [N] f32, stuck [N] u8: contiguous CUDA tensors on one device")
    for t, dt in ((n_stuck, torch.int32), (f_max, torch.float32)):
        if t is not None and not (t.is_cuda and t.dtype == dt and t.numel() >= 1 and t.device == g.device):
            raise ValueError("stick_test_static: n_stuck int32 [1] / f_max f32 [1] on g's device")
    with torch.cuda.device(g.device):
        st = stream if stream is not None else torch.cuda.current_stream(g.device)
        rc = L.chisao_stick_test_static(C.c_void_p(g.data_ptr()), C.c_void_p(f.data_ptr()), N, d, float(eps_grad),
                                        float(log_delta), C.c_void_p(stuck.data_ptr()),
                                        C.c_void_p(n_stuck.data_ptr() if n_stuck is not None else None),
                                        C.c_void_p(f_max.data_ptr() if f_max is not None else None),
                                        C.c_void_p(st.cuda_stream))
    if rc:
        raise ChisaoError(rc, (L.chisao_last_error(None) or b"").decode())


_FIELD_DTYPE = {STUCK: np.uint8, REMOVED: np.uint8, STALLED: np.uint8, HIST_LEN: np.int32, CTRL: np.int32,
                LS_B: np.int32, RS_SRC: np.int32, RS_CAND: np.int32}


class Chisao:
    """One CHISAO run on `device` (a CUDA device).  `wl` is an `inputs.Workload`-like object; its x0 is the
    initial population unless `seed_population=True` (then x is drawn on the device from Philox)."""

    def __init__(self, wl, device="cuda:0", seed_population: bool = False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_26164_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self._L = load_library()
        self.device = torch.device(device)
        h = wl.hp
        self.d, self.N, self.m, self.M = h.d, h.N, h.lbfgs_m, h.hlc_M
        self._cfg, self._obj, self._keep = marshal(wl)
        n = C.c_size_t(0)
        self._ck(self._L.chisao_workspace_bytes(C.byref(self._cfg), C.byref(self._obj), C.byref(n)), None)
        with torch.cuda.device(self.device):
            self.stream = torch.cuda.current_stream(self.device)
            x0 = np.ascontiguousarray(wl.x0, np.float32).reshape(self.N, self.d)
            self.x = torch.from_numpy(x0.copy()).to(self.device) if self.N else \
                torch.empty((0, self.d), dtype=torch.float32, device=self.device)
            self.workspace = torch.empty(max(n.value, 256), dtype=torch.uint8, device=self.device)
            assert self.workspace.data_ptr() % 256 == 0
            h_ = C.c_void_p(None)
            rc = self._L.chisao_init(C.byref(h_), C.byref(self._cfg), C.byref(self._obj), C.c_void_p(self.x.data_ptr()),
                                     C.c_void_p(self.workspace.data_ptr()), n.value, C.c_void_p(self.stream.cuda_stream))
            self._ck(rc, None)
            self._h = h_
            if seed_population:
                self._ck(self._L.chisao_seed_population(self._h))
        self.workspace_bytes = n.value

    def _ck(self, rc, h="self"):
        if rc:
            hh = self._h if h == "self" else None
            raise ChisaoError(rc, self._L.chisao_last_error(hh).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._torch.cuda.synchronize(self.device)
            self._L.chisao_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the cycle -------------------------------------------------------------------------------------
    def step(self, stats: bool = True) -> Optional[Stats]:
        st = Stats()
        self._ck(self._L.chisao_step(self._h, C.byref(st) if stats else None))
        return st if stats else None

    def step_host(self, x_in=None, x_out=None, f_out=None, stuck_out=None, stats: bool = False):
        st = Stats()
        ptr = lambda a: C.c_void_p(a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr()) if a is not None else None
        self._ck(self._L.chisao_step_host(self._h, ptr(x_in), ptr(x_out), ptr(f_out), ptr(stuck_out),
                                          C.byref(st) if stats else None))
        return st if stats else None

    def phase(self, phase_id: int, it: int = 0):
        self._ck(self._L.chisao_phase(self._h, phase_id, it))

    def set_option(self, option: int, value: int):
        """chisao_set_option (OPT_STENCIL_AWARE: opt-in stencil-aware FD evaluator, reported separately;
        OPT_CUDA_GRAPH: submit each cycle as one CUDA graph launch, default on; OPT_LS_TILE_LOCAL: form of the line
        search, see include/chisao.h)."""
        self._ck(self._L.chisao_set_option(self._h, int(option), int(value)))

    def evaluator(self) -> int:
        """chisao_get_info(INFO_EVALUATOR): index into EVALUATOR_NAMES"""
        v = C.c_int32(0)
        self._ck(self._L.chisao_get_info(self._h, INFO_EVALUATOR, C.byref(v)))
        return int(v.value)

    def ls_tile_local(self) -> bool:
        """chisao_get_info(INFO_LS_TILE_LOCAL): the line search runs every trial of a tile in one launch"""
        v = C.c_int32(0)
        self._ck(self._L.chisao_get_info(self._h, INFO_LS_TILE_LOCAL, C.byref(v)))
        return bool(v.value)

    def lbfgs_resident(self) -> bool:
        """chisao_get_info(INFO_LBFGS_RESIDENT): Phase 1 runs as one launch with the (s, y) history in registers"""
        v = C.c_int32(0)
        self._ck(self._L.chisao_get_info(self._h, INFO_LBFGS_RESIDENT, C.byref(v)))
        return bool(v.value)

    def graph_launches(self) -> int:
        """chisao_get_info(INFO_GRAPH_LAUNCHES): cycles submitted as one CUDA graph launch so far"""
        v = C.c_int32(0)
        self._ck(self._L.chisao_get_info(self._h, INFO_GRAPH_LAUNCHES, C.byref(v)))
        return int(v.value)

    def stats(self) -> Stats:
        st = Stats()
        self._ck(self._L.chisao_get_stats(self._h, C.byref(st)))
        return st

    def modes(self, cap: Optional[int] = None):
        cap = self.N if cap is None else cap
        x = np.empty((max(cap, 1), self.d), np.float32)
        f = np.empty(max(cap, 1), np.float32)
        idx = np.empty(max(cap, 1), np.int32)
        n = C.c_int32(0)
        rc = self._L.chisao_modes(self._h, x.ctypes.data, f.ctypes.data, idx.ctypes.data, cap, C.byref(n))
        if rc and rc != E_CAPACITY:
            self._ck(rc)
        k = min(n.value, cap)
        return x[:k].copy(), f[:k].copy(), idx[:k].copy(), n.value

    # ---- state exchange ----------------------------------------------------------------------------------
    def _shape(self, field):
        N, d, m, M = self.N, self.d, self.m, self.M
        return {X: (N, d), G: (N, d), V: (N, d), P: (N, d), GHAT: (N, d), XT: (N, d), HIST_S: (m, N, d),
                HIST_Y: (m, N, d), HLC_F: (N, M), CTRL: (8,), GR_Q: (d, d), SIGMA: (1,)}.get(field, (N,))

    def get(self, field):
        a = np.empty(self._shape(field), _FIELD_DTYPE.get(field, np.float32))
        self._ck(self._L.chisao_get_state(self._h, field, a.ctypes.data, a.nbytes))
        return a

    def set(self, field, value):
        a = np.ascontiguousarray(value, _FIELD_DTYPE.get(field, np.float32)).reshape(self._shape(field))
        self._ck(self._L.chisao_set_state(self._h, field, a.ctypes.data, a.nbytes))

    # ---- instrumentation -----------------------------------------------------------------------------------
    def launch_count(self) -> int:
        return int(self._L.chisao_launch_count(self._h))

    def timing_enable(self, on=True):
        """on: False / True (every kernel class) or an iterable of class names from TIMING_CLASSES"""
        if isinstance(on, (bool, int)):
            v = 1 if on else 0
        else:
            v = sum(1 << (TIMING_CLASSES.index(name) + 1) for name in on)
        self._ck(self._L.chisao_timing_enable(self._h, v))

    def timing_reset(self):
        self._ck(self._L.chisao_timing_reset(self._h))

    def timing(self):
        out = {}
        for k, name in enumerate(TIMING_CLASSES):
            ms = C.c_double(0.0)
            n = C.c_uint64(0)
            self._ck(self._L.chisao_timing_get(self._h, k, C.byref(ms), C.byref(n)))
            out[name] = (ms.value, int(n.value))
        return out
