"""Helpers of the GPU<->oracle parity tests.

Teacher forcing: the oracle runs free; before every compared unit its state is rounded to fp32 (so both
sides start from bit-identical inputs) and loaded into the CUDA context; exactly one unit runs on both
sides; outputs are compared with the tolerances of BASELINE.json north_star (f 1e-5 relative, FD / HLC
gradients 1e-3 relative with the fp32 finite-difference floor, updated positions 1e-4 relative to the
domain, discrete decisions exact away from thresholds).
"""
from __future__ import annotations

import numpy as np

EPS32 = float(np.finfo(np.float32).eps)

# tolerances (north_star + DESIGN.md "Tolerances")
F_REL = 1e-5
G_REL = 1e-3
X_REL = 1e-4
LS_MARGIN_MIN = 2e-5       # Armijo decisions closer than this (relative) are not required to agree
REL_MARGIN_MIN = 1e-3      # ascent / curvature tests
MAX_EXCLUDED_FRACTION = 0.005


def f32(a):
    return np.asarray(a, np.float64).astype(np.float32).astype(np.float64)


def sync_oracle_to_gpu(o, g, O, B, with_history=True):
    """Round the oracle's floating state to fp32 in place and load the same state into the CUDA context."""
    for fo, fg in ((O.X, B.X), (O.F, B.F), (O.G, B.G), (O.V, B.V)):
        a = f32(o.get(fo))
        o.set(fo, a)
        g.set(fg, a)
    for fo, fg in ((O.STUCK, B.STUCK), (O.REMOVED, B.REMOVED), (O.STALLED, B.STALLED), (O.HIST_LEN, B.HIST_LEN),
                   (O.CTRL, B.CTRL)):
        g.set(fg, o.get(fo))
    if with_history:
        for fo, fg in ((O.HIST_S, B.HIST_S), (O.HIST_Y, B.HIST_Y)):
            a = f32(o.get(fo))
            o.set(fo, a)
            g.set(fg, a)


def f_tol(f_orc):
    return F_REL * np.maximum(np.abs(f_orc), 1.0)


def fd_floor(f_orc, h, sigma_noise=0.0):
    """fp32 floor of a central difference: 8 eps32 max|f| / (2h) (+ the rounding of the noise draws)."""
    return 8.0 * EPS32 * (np.abs(f_orc) + 6.0 * sigma_noise + 1.0) / (2.0 * h)


def grad_ok(g_gpu, g_orc, f_orc, h, sigma_noise=0.0):
    """per-sample: ||dg||_inf <= 1e-3 ||g||_inf + floor"""
    err = np.max(np.abs(g_gpu - g_orc), axis=1)
    tol = G_REL * np.max(np.abs(g_orc), axis=1) + fd_floor(f_orc, h, sigma_noise)
    return err <= tol, err, tol


def x_tol(x_orc, lo, hi, step_inf=None, grad_inside=False):
    """rule 4: 1e-4 max(||x||_inf, half-width) (+ 1e-3 of the step when the unit computes its own gradient)"""
    half = float(np.max(np.asarray(hi, np.float64) - np.asarray(lo, np.float64)) / 2.0)
    tol = X_REL * np.maximum(np.max(np.abs(x_orc), axis=1), half)
    if grad_inside and step_inf is not None:
        tol = tol + G_REL * step_inf
    return tol


def match_modes(xa, xb, tol):
    """greedy one-to-one matching of two mode sets within L2 distance tol; returns #matched"""
    xa = np.asarray(xa, np.float64); xb = np.asarray(xb, np.float64)
    if len(xa) == 0 or len(xb) == 0:
        return 0
    used = np.zeros(len(xb), bool)
    n = 0
    for a in xa:
        dist = np.linalg.norm(xb - a[None, :], axis=1)
        dist[used] = np.inf
        j = int(np.argmin(dist))
        if dist[j] <= tol:
            used[j] = True
            n += 1
    return n


# ---- end-to-end mode-set comparison (R-14) ---------------------------------
def subset_workload(wl, x0, **over):
    """the same problem and hyper-parameters on another population (used by the oracle polish)"""
    import copy
    hp = copy.copy(wl.hp)
    hp.N = len(x0)
    for k, v in over.items():
        setattr(hp, k, v)
    obj = copy.copy(wl.obj)
    out = copy.copy(wl)
    out.obj, out.hp, out.x0 = obj, hp, np.ascontiguousarray(x0, np.float32)
    return out


def oracle_polish(O, wl, x_pts, f_max_ref, threads=8):
    """S-14's acceptance rule for a mode reported by the CUDA path that has no partner in the oracle's set: run the
    oracle's own Phase 1 (release + n_conv L-BFGS iterations, noise off) from the point; returns the L2 movement, and
    whether the polished point is stationary by the oracle's gradient test and passes the oracle's Eq. 1 / Eq. 3 quality
    gate f >= f_max_ref + log delta."""
    x_pts = np.asarray(x_pts, np.float64).reshape(-1, wl.hp.d)
    if len(x_pts) == 0:
        return np.zeros(0), np.zeros(0, bool), np.zeros(0)
    sub = subset_workload(wl, x_pts)
    sub.obj.sigma_noise = 0.0
    o = O.Oracle(sub, threads=threads)
    o.set(O.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(O.PH_RELEASE_EVAL)
    for it in range(1, sub.hp.n_conv + 1):
        o.phase(O.PH_LBFGS_ITER, it)
    x1, f1, g1 = o.get(O.X), o.get(O.F), o.get(O.G)
    o.close()
    move = np.linalg.norm(x1 - f32(x_pts), axis=1)
    ok = (np.max(np.abs(g1), axis=1) < wl.hp.eps_grad) & (f1 >= f_max_ref + wl.hp.log_delta)
    return move, ok, f1


def nearest(xa, xb):
    """for every row of xa: (L2 distance to, index of) the nearest row of xb"""
    xa = np.asarray(xa, np.float64); xb = np.asarray(xb, np.float64)
    if len(xa) == 0:
        return np.zeros(0), np.zeros(0, int)
    if len(xb) == 0:
        return np.full(len(xa), np.inf), np.full(len(xa), -1)
    D = np.linalg.norm(xa[:, None, :] - xb[None, :, :], axis=2)
    return D.min(axis=1), D.argmin(axis=1)


def mode_set_report(xg, fg, xo, fo, tol):
    """one-to-one matching within tol plus what is left over on either side"""
    xg = np.asarray(xg, np.float64); xo = np.asarray(xo, np.float64)
    used = np.zeros(len(xo), bool)
    pair = np.full(len(xg), -1)
    for q, a in enumerate(xg):
        if len(xo) == 0:
            break
        dist = np.linalg.norm(xo - a[None, :], axis=1)
        dist[used] = np.inf
        j = int(np.argmin(dist))
        if dist[j] <= tol:
            used[j] = True
            pair[q] = j
    only_g = np.flatnonzero(pair < 0)
    only_o = np.flatnonzero(~used)
    dg, _ = nearest(xg[only_g], xo)
    do, _ = nearest(xo[only_o], xg)
    text = (f"gpu {len(xg)} modes, oracle {len(xo)}, matched {int((pair >= 0).sum())} within {tol:g}; "
            f"gpu-only {len(only_g)} (nearest oracle mode at {np.round(dg, 4).tolist()}, f {np.round(np.asarray(fg)[only_g], 4).tolist()}); "
            f"oracle-only {len(only_o)} (nearest gpu mode at {np.round(do, 4).tolist()}, f {np.round(np.asarray(fo)[only_o], 4).tolist()})")
    return pair, only_g, only_o, text


RM_MARGIN_MIN = 1e-5


def rm_candidates_ok(O, o, cand_gpu, removed):
    """Repulse-Monkey candidate choice (R-8), protocol rule 3, checked decision by decision: the candidate the CUDA path
    kept must score (min squared distance to the frozen modes, by the ORACLE's fp64 scores) within 1e-5 relative of the
    oracle's best -- it IS the oracle's best wherever the runner-up is farther away than that; inside the band fp32
    rounding of the d-term squared distances may order near-equal candidates differently (short rays: t_max small against
    the distance to the modes).  Returns (mask of slots that kept the oracle's candidate, number of slots that did not)."""
    score = o.get(O.RS_SCORE)
    best = o.get(O.RS_CAND)
    rows = np.flatnonzero(removed)
    sb = score[rows, best[rows]]
    sg = score[rows, cand_gpu[rows]]
    assert np.all((cand_gpu[rows] >= 0) & (cand_gpu[rows] < 16))
    ok = sg >= sb * (1.0 - RM_MARGIN_MIN)
    assert np.all(ok), (int(np.sum(~ok)), float(np.min(sg / np.maximum(sb, 1e-300))))
    same = removed & (cand_gpu == best)
    return same, int(len(rows) - same.sum())
