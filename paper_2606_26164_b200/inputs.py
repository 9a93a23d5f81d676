"""Seeded synthetic inputs for the CHISAO oscillation cycle (shared by the CUDA path and the oracle).

This module holds NO arithmetic of the method itself: it only writes down the *inputs* of a run --
objective parameter arrays, box bounds, the initial population and the hyper-parameter record -- as
fp32 numpy arrays.  Both `paper_2606_26164_b200.binding` (CUDA) and `oracle/` (fp64 CPU) consume
exactly these arrays; neither imports the other.

Workloads follow BASELINE.json `configs` C1..C5 (they stand in for the paper's workloads: the
isotropic Gaussian mixture of PAPER.md:629 App. D, the noisy mixture of PAPER.md:525 sec. 5.7, the
Group-A multimodal and Group-B ill-conditioned bowls of PAPER.md:272-287).  Values that BASELINE.json
leaves open follow SURVEY.md sec. 8(d) and are restated in DESIGN.md ("Input recipe").

Objective parameterisation (all arrays fp32, row-major):
  id 0 GMM_ISO : means[K][d], mats[0]=sigma,          vec_a[K] = log w_k - d/2 log(2 pi sigma^2)
  id 1 GMM_DIAG: means[K][d], mats[K][d]=1/sigma_kj,   vec_a[K] = log w_k - sum_j log sigma_kj - d/2 log 2pi
  id 2 GMM_FULL: means[K][d], mats[K][d][d]=W_k with Sigma_k^-1 = W_k^T W_k,
                 vec_a[K] = log w_k + log|det W_k| - d/2 log 2pi
  id 3 RFF     : mats[K][d]=w_j, vec_a[K]=a_j, vec_b[K]=b_j, scalar0 = 1/50
  id 4 QUAD    : means[1][d]=c,  mats[d][d]=W=diag(sqrt(lambda)) Q
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import numpy as np

OBJ_GMM_ISO, OBJ_GMM_DIAG, OBJ_GMM_FULL, OBJ_RFF, OBJ_QUAD = 0, 1, 2, 3, 4
# Appendix D of the paper: parameter-free benchmark functions, negated for maximisation
OBJ_RASTRIGIN, OBJ_ACKLEY, OBJ_SCHWEFEL, OBJ_STYBLINSKI_TANG, OBJ_MICHALEWICZ, OBJ_TRID, OBJ_BUKIN6 = 5, 6, 7, 8, 9, 10, 11
APPENDIX_D = {"rastrigin": 5, "ackley": 6, "schwefel": 7, "styblinski_tang": 8, "michalewicz": 9, "trid": 10, "bukin6": 11}


@dataclass
class Objective:
    id: int
    d: int
    K: int
    means: np.ndarray           # fp32
    mats: np.ndarray            # fp32
    vec_a: np.ndarray           # fp32
    vec_b: Optional[np.ndarray] = None
    scalar0: float = 0.0
    sigma_noise: float = 0.0
    # float64 ground truth the arrays were derived from (used by oracle *pins* only)
    truth: dict = field(default_factory=dict)


@dataclass
class Hyper:
    d: int
    N: int
    lo: np.ndarray
    hi: np.ndarray
    n_osc: int = 3
    n_conv: int = 10
    n_anti: int = 5
    n_cloud: int = 3
    hlc_M: int = 10
    lbfgs_m: int = 10
    ls_max: int = 10
    reseed_cands: int = 4
    fd_h: float = 1e-3
    eps_grad: float = 1e-6
    eps_dup: float = 1e-3
    log_delta: float = math.log(0.1)
    mu: float = 0.9
    alpha_anti: float = 1e-2
    eta_hlc: float = 1e-2
    sigma_s: float = 0.5
    ls_c1: float = 1e-4
    ls_shrink: float = 0.5
    hlc_baseline: int = 0
    phase_mask: int = 0xFFFFFFFF
    seed: int = 0


@dataclass
class Workload:
    name: str
    obj: Objective
    hp: Hyper
    x0: np.ndarray              # [N][d] fp32 initial population


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.Philox(seed))


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def _rotation(rng: np.random.Generator, d: int) -> np.ndarray:
    """Random orthogonal matrix: QR of a Gaussian matrix, signs fixed so that R_ii > 0."""
    g = rng.standard_normal((d, d))
    q, r = np.linalg.qr(g)
    return q * np.sign(np.diag(r))[None, :]


def gmm_iso(d: int, K: int, sigma: float, box: float, seed: int, means=None, sigma_noise=0.0) -> Objective:
    rng = _rng(seed)
    mu = rng.uniform(-box, box, size=(K, d)) if means is None else np.asarray(means, dtype=np.float64)
    K = mu.shape[0]
    logw = np.full(K, -math.log(K))
    # parameters are rounded to fp32 first; the constants are then derived from the rounded values
    mu32 = _f32(mu)
    sig32 = np.float32(sigma)
    a = logw - 0.5 * d * math.log(2.0 * math.pi * float(sig32) ** 2)
    return Objective(OBJ_GMM_ISO, d, K, mu32, _f32([sig32]), _f32(a), None, 0.0, sigma_noise,
                     truth=dict(mu=mu32.astype(np.float64), sigma=float(sig32), logw=logw))


def gmm_diag(d: int, K: int, box: float, seed: int, sigma_noise=0.0) -> Objective:
    rng = _rng(seed)
    mu = rng.uniform(-box, box, size=(K, d))
    sig = rng.uniform(0.1, 0.5, size=(K, d))
    e = -np.log(rng.uniform(size=K))          # Dirichlet(1) = normalised exponentials
    logw = np.log(e / e.sum())
    mu32 = _f32(mu)
    inv32 = _f32(1.0 / sig)
    sig_eff = 1.0 / inv32.astype(np.float64)
    a = logw - np.log(sig_eff).sum(axis=1) - 0.5 * d * math.log(2.0 * math.pi)
    return Objective(OBJ_GMM_DIAG, d, K, mu32, inv32, _f32(a), None, 0.0, sigma_noise,
                     truth=dict(mu=mu32.astype(np.float64), sig=sig_eff, logw=logw))


def gmm_full(d: int, K: int, box: float, seed: int, sigma_noise=0.0, eig=(0.05, 0.5)) -> Objective:
    rng = _rng(seed)
    mu = rng.uniform(-box, box, size=(K, d))
    W = np.empty((K, d, d))
    for k in range(K):
        R = _rotation(rng, d)
        lam = rng.uniform(eig[0], eig[1], size=d)      # eigenvalues of the COVARIANCE
        W[k] = (1.0 / np.sqrt(lam))[:, None] * R.T     # Sigma^-1 = W^T W
    logw = np.full(K, -math.log(K))
    mu32, W32 = _f32(mu), _f32(W)
    W64 = W32.astype(np.float64)
    logdet = np.array([np.linalg.slogdet(W64[k])[1] for k in range(K)])
    a = logw + logdet - 0.5 * d * math.log(2.0 * math.pi)
    prec = np.einsum("krc,krd->kcd", W64, W64)
    return Objective(OBJ_GMM_FULL, d, K, mu32, W32, _f32(a), None, 0.0, sigma_noise,
                     truth=dict(mu=mu32.astype(np.float64), prec=prec, logw=logw))


def rff(d: int, K: int, seed: int, sigma_noise=0.0) -> Objective:
    rng = _rng(seed)
    w = rng.standard_normal((K, d))
    a = rng.uniform(0.0, 0.5, size=K)
    b = rng.uniform(0.0, 2.0 * math.pi, size=K)
    return Objective(OBJ_RFF, d, K, np.zeros((1, d), np.float32), _f32(w), _f32(a), _f32(b),
                     float(np.float32(1.0 / 50.0)), sigma_noise,
                     truth=dict(w=_f32(w).astype(np.float64), a=_f32(a).astype(np.float64),
                                b=_f32(b).astype(np.float64), q=float(np.float32(1.0 / 50.0))))


def quad(d: int, seed: int, lam_max: float = 1e4, sigma_noise=0.0) -> Objective:
    rng = _rng(seed)
    Q = _rotation(rng, d)
    lam = np.logspace(0.0, math.log10(lam_max), d) if d > 1 else np.ones(1)
    c = rng.uniform(-2.0, 2.0, size=d)
    W32 = _f32(np.sqrt(lam)[:, None] * Q)
    c32 = _f32(c[None, :])
    W64 = W32.astype(np.float64)
    return Objective(OBJ_QUAD, d, 1, c32, W32, np.zeros(1, np.float32), None, 0.0, sigma_noise,
                     truth=dict(c=c32[0].astype(np.float64), A=W64.T @ W64))


def uniform_population(N: int, lo: np.ndarray, hi: np.ndarray, seed: int) -> np.ndarray:
    rng = _rng(seed)
    u = rng.uniform(size=(N, lo.shape[0]))
    return _f32(lo[None, :] + u * (hi - lo)[None, :])


def _box(d: int, b: float):
    return np.full(d, -b, np.float32), np.full(d, b, np.float32)


def n_conv_default(d: int) -> int:
    """PAPER.md:82  n_conv = max(10, 3 log2 d)."""
    return max(10, int(round(3 * math.log2(d))))


def config(c: int, N: Optional[int] = None, n_osc: Optional[int] = None, noise: Optional[float] = None,
           **over) -> Workload:
    """BASELINE.json configs[c-1]; `N`, `n_osc`, `noise` and any Hyper field may be overridden for
    reduced parity cases (same d, K and parameter seeds)."""
    if c == 1:
        d, N0 = 2, 256
        obj = gmm_iso(d, 4, 0.3, 3.0, 1001)
        lo, hi = _box(d, 3.0)
        hp = Hyper(d, N0, lo, hi, n_osc=10, n_conv=20, hlc_M=8, lbfgs_m=5, fd_h=1e-3, eps_grad=2e-3,
                   eps_dup=1e-3, sigma_s=0.5, alpha_anti=1e-2, eta_hlc=1e-2, hlc_baseline=1)
    elif c == 2:
        d, N0 = 8, 4096
        obj = gmm_diag(d, 16, 5.0, 1002, sigma_noise=0.1)
        lo, hi = _box(d, 5.0)
        hp = Hyper(d, N0, lo, hi, n_osc=20, n_conv=10, hlc_M=16, lbfgs_m=8, fd_h=0.1, eps_grad=2.8,
                   eps_dup=0.5, sigma_s=0.5, alpha_anti=5e-3, eta_hlc=5e-3, hlc_baseline=1)
    elif c == 3:
        d, N0 = 32, 16384
        obj = rff(d, 256, 1003)
        lo, hi = _box(d, 5.0)
        hp = Hyper(d, N0, lo, hi, n_osc=30, n_conv=15, hlc_M=32, lbfgs_m=10, fd_h=5e-3, eps_grad=5e-3,
                   eps_dup=2e-2, sigma_s=1.0, alpha_anti=2e-2, eta_hlc=2e-2, hlc_baseline=1)
    elif c == 4:
        d, N0 = 64, 16384
        obj = quad(d, 1004)
        lo, hi = _box(d, 4.0)
        hp = Hyper(d, N0, lo, hi, n_osc=30, n_conv=18, hlc_M=32, lbfgs_m=10, fd_h=1e-2, eps_grad=1e-1,
                   eps_dup=1e-2, sigma_s=1.0, alpha_anti=2e-5, eta_hlc=2e-5, hlc_baseline=1)
    elif c == 5:
        d, N0 = 64, 65536
        obj = gmm_full(d, 64, 10.0, 1005, sigma_noise=1.0)
        lo, hi = _box(d, 10.0)
        hp = Hyper(d, N0, lo, hi, n_osc=50, n_conv=18, hlc_M=32, lbfgs_m=10, fd_h=0.25, eps_grad=11.3,
                   eps_dup=3.0, log_delta=-8.0, sigma_s=1.0, alpha_anti=5e-3, eta_hlc=5e-3,
                   hlc_baseline=1)
    else:
        raise ValueError("config id must be 1..5")
    if noise is not None:
        obj.sigma_noise = float(noise)
    if N is not None:
        hp.N = int(N)
    if n_osc is not None:
        hp.n_osc = int(n_osc)
    hp.seed = 3000 + c
    for k, v in over.items():
        if not hasattr(hp, k):
            raise KeyError(k)
        setattr(hp, k, v)
    x0 = uniform_population(hp.N, hp.lo, hp.hi, 2000 + c)
    return Workload(f"C{c}", obj, hp, x0)


def noise_robustness(sigma_noise: float, trial: int = 0, N: int = 200) -> Workload:
    """The noise-robustness workload of PAPER.md:523-541 (sec. 5.7, Table 8): 2-mode isotropic Gaussian mixture in
    d = 6, peaks at +-2 e_1, sigma = 1 (mode separation 4 sigma), Theta = [-10, 10]^6, N = 200 and the
    defaults of Table 1 (n_osc = 3, n_conv = 10, n_anti = 5, n_cloud = 3, K = 10, m = 10).  The paper does not state
    the FD step or the thresholds it used under noise; they follow the FD noise floor sigma_noise / (sqrt(2) h) with
    h = sigma = 1."""
    d = 6
    means = np.zeros((2, d))
    means[0, 0], means[1, 0] = 2.0, -2.0
    obj = gmm_iso(d, 2, 1.0, 10.0, 1, means=means, sigma_noise=sigma_noise)
    h = 1.0
    lo, hi = _box(d, 10.0)
    hp = Hyper(d, N, lo, hi, n_osc=3, n_conv=10, n_anti=5, n_cloud=3, hlc_M=10, lbfgs_m=10, fd_h=h,
               eps_grad=max(4.0 * sigma_noise / (math.sqrt(2.0) * h), 1e-2), eps_dup=min(3.0, 0.2 + 6.0 * sigma_noise),
               log_delta=math.log(0.1) - 4.0 * sigma_noise, alpha_anti=0.05, eta_hlc=0.05, sigma_s=1.0, hlc_baseline=1)
    hp.seed = 500 + trial
    return Workload(f"noise{sigma_noise:g}", obj, hp, uniform_population(N, lo, hi, 501 + trial))


def appendix_d(name: str, d: int, N: int, seed: int = 11, **over) -> Workload:
    """One of the benchmark functions printed in the paper's Appendix D on its printed domain.
    Only the seven functions whose definitions are in the paper are available."""
    oid = APPENDIX_D[name]
    if name == "bukin6":
        d = 2
        lo, hi = np.array([-15.0, -3.0], np.float32), np.array([-5.0, 3.0], np.float32)
    elif name == "michalewicz":
        lo, hi = np.zeros(d, np.float32), np.full(d, np.float32(math.pi), np.float32)
    else:
        b = {"rastrigin": 5.12, "ackley": 32.768, "schwefel": 500.0, "styblinski_tang": 5.0, "trid": float(d * d)}[name]
        lo, hi = _box(d, b)
    obj = Objective(oid, d, 1, np.zeros((1, d), np.float32), np.zeros(1, np.float32), np.zeros(1, np.float32))
    hp = Hyper(d, N, lo, hi, n_conv=n_conv_default(d))
    hp.seed = seed
    for k, v in over.items():
        if not hasattr(hp, k):
            raise KeyError(k)
        setattr(hp, k, v)
    return Workload(name, obj, hp, uniform_population(N, lo.astype(np.float64), hi.astype(np.float64), seed + 1))


def custom(obj: Objective, box: float, N: int, seed: int = 7, **over) -> Workload:
    """A free-form workload on [-box, box]^d (used by pins and edge-case tests)."""
    lo, hi = _box(obj.d, box)
    hp = Hyper(obj.d, N, lo, hi, n_conv=n_conv_default(obj.d))
    hp.seed = seed
    for k, v in over.items():
        if not hasattr(hp, k):
            raise KeyError(k)
        setattr(hp, k, v)
    return Workload("custom", obj, hp, uniform_population(N, lo, hi, seed + 1))


def synthetic_converged_state(wl: Workload, frac_clustered: float = 0.6, n_clusters: int = 300, seed: int = 17):
    """A seeded post-convergence state (x, f, g) for cross-sample phase tests at any N -- inputs only, no arithmetic of
    the method: `frac_clustered` of the samples sit in `n_clusters` tight clusters (centres uniform in Theta, jitter
    well inside eps_dup, so the deduplication has many removals and exact / near ties), the rest stay at their
    seeded uniform positions; f is a seeded per-cluster level minus a jitter term (with exact ties), g is seeded
    noise whose magnitude straddles eps_grad; a few f / g entries are non-finite (R-12)."""
    hp = wl.hp
    N, d = hp.N, hp.d
    rng = _rng(seed)
    x = np.array(wl.x0, dtype=np.float64, copy=True)
    clustered = rng.uniform(size=N) < frac_clustered
    centres = rng.uniform(hp.lo.astype(np.float64) * 0.9, hp.hi.astype(np.float64) * 0.9, size=(n_clusters, d))
    which = rng.integers(0, n_clusters, size=N)
    jit = rng.uniform(-0.3, 0.3, size=(N, d)) * float(hp.eps_dup)
    x[clustered] = centres[which[clustered]] + jit[clustered]
    level = rng.uniform(-2.0, 0.0, size=n_clusters)          # most clusters inside the quality gate of the best one
    f = np.where(clustered, level[which] - np.round(np.abs(jit).max(axis=1) / float(hp.eps_dup), 2),
                 rng.uniform(-40.0, -1.0, size=N))           # two decimals: many exact ties inside a cluster
    gmag = float(hp.eps_grad) * np.where(clustered, rng.uniform(0.0, 1.25, size=N), rng.uniform(0.5, 50.0, size=N))
    g = rng.uniform(-1.0, 1.0, size=(N, d))
    g *= (gmag / np.abs(g).max(axis=1))[:, None]
    if N >= 64:
        f[5] = np.nan; f[17] = np.inf; f[33] = -np.inf; g[41, d - 1] = np.nan
    return _f32(x), _f32(f), _f32(g)
