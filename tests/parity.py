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
