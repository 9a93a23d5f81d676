"""Pins for the oracle's phases (Algorithm 1) against definitions, closed forms,
invariants and brute force -- none of them re-call the oracle's own routine for the expected value."""
import math

import numpy as np
import pytest
from scipy.optimize import minimize

from paper_2606_26164_b200 import inputs


# ----------------------------------------------------------------------------- L-BFGS (Phase 1)
def _dense_bfgs_H(S, Y):
    """Explicit BFGS inverse-Hessian recursion H <- (I - rho s y^T) H (I - rho y s^T) + rho s s^T
    from H0 = (s.y/y.y) I of the newest pair (Nocedal & Wright Eq. 6.17 / 7.16)."""
    d = S.shape[1]
    H = np.eye(d) * (S[-1] @ Y[-1]) / (Y[-1] @ Y[-1])
    for s, y in zip(S, Y):
        rho = 1.0 / (s @ y)
        V = np.eye(d) - rho * np.outer(y, s)
        H = V.T @ H @ V + rho * np.outer(s, s)
    return H


@pytest.mark.parametrize("d,m", [(2, 1), (5, 3), (8, 8), (8, 10)])
def test_two_loop_equals_dense_bfgs(orc, d, m):
    rng = np.random.default_rng(d * 100 + m)
    A = rng.standard_normal((d, d)); A = A @ A.T + d * np.eye(d)
    S = rng.standard_normal((m, d)); Y = S @ A                     # guarantees s.y > 0
    gamma = rng.standard_normal(d)
    r = orc.two_loop(S, Y, gamma)
    assert np.allclose(r, _dense_bfgs_H(S, Y) @ gamma, rtol=1e-10, atol=1e-12)
    # secant identity: H y_newest = s_newest
    assert np.allclose(orc.two_loop(S, Y, Y[-1]), S[-1], rtol=1e-10, atol=1e-12)
    # a transposed operand (swapping the roles of s and y) must not pass
    assert not np.allclose(orc.two_loop(Y, S, gamma), _dense_bfgs_H(S, Y) @ gamma, rtol=1e-3)


def test_two_loop_empty_history_is_identity(orc):
    g = np.array([1.0, -2.0, 3.0])
    assert np.array_equal(orc.two_loop(np.zeros((0, 3)), np.zeros((0, 3)), g), g)


def _run_phase1(o, orc, n_conv, cycle=1):
    o.set(orc.CTRL, [cycle, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    fs = [o.get(orc.F).copy()]
    for it in range(1, n_conv + 1):
        o.phase(orc.PH_LBFGS_ITER, it)
        fs.append(o.get(orc.F).copy())
    return np.array(fs)


def test_lbfgs_converges_to_exact_maximiser_of_quadratic(orc):
    """north_star: 'the exact maximiser of a quadratic, L-BFGS convergence on it'."""
    obj = inputs.quad(8, 11, lam_max=100.0)
    wl = inputs.custom(obj, 4.0, 16, fd_h=1e-2, eps_grad=1e-9, lbfgs_m=10)
    o = orc.Oracle(wl)
    fs = _run_phase1(o, orc, 60)
    x = o.get(orc.X)
    assert np.abs(x - obj.truth["c"][None]).max() < 1e-6     # positions are fp32-rounded
    assert np.all(np.diff(fs, axis=0) >= -1e-15)               # Armijo, noise-free: f never decreases
    assert np.all(fs[-1] > -1e-10)


def test_lbfgs_same_optimum_as_scipy_on_mixture(orc):
    wl = inputs.config(1, N=64, eps_grad=1e-7, n_conv=60)
    wl.hp.fd_h = 1e-4
    o = orc.Oracle(wl)
    _run_phase1(o, orc, 60)
    x, f = o.get(orc.X), o.get(orc.F)
    t = wl.obj.truth
    neg = lambda z: -float(o.values(z[None])[0])
    for i in range(0, 64, 7):
        res = minimize(neg, x[i], method="L-BFGS-B", options=dict(gtol=1e-10, ftol=1e-15))
        assert np.abs(res.x - x[i]).max() < 5e-5
        assert abs(-res.fun - f[i]) < 1e-7
        assert np.min(np.abs(x[i][None] - t["mu"]).max(axis=1)) < 1e-3   # at one of the means (separated)


def test_lbfgs_respects_bounds_and_counts_evaluations(orc):
    # maximiser outside the box: iterates must stop on the boundary
    obj = inputs.gmm_iso(2, 1, 1.0, 3.0, 5, means=[[5.0, 0.5]])
    wl = inputs.custom(obj, 3.0, 8, fd_h=1e-3, eps_grad=1e-8)
    o = orc.Oracle(wl)
    _run_phase1(o, orc, 25)
    x = o.get(orc.X)
    assert np.all(x <= 3.0) and np.all(x >= -3.0)
    assert np.allclose(x[:, 0], 3.0) and np.allclose(x[:, 1], 0.5, atol=1e-4)
    ev = o.stats().evals
    lsb = o.get(orc.LS_B)
    assert ev[0] == 8 * 5 and ev[2] % 4 == 0 and ev[1] >= ev[2] // 4
    assert set(np.unique(lsb)).issubset(set(range(-2, 11)))


def test_stationary_samples_are_skipped(orc):
    obj = inputs.gmm_iso(2, 1, 1.0, 3.0, 5, means=[[0.25, 0.5]])
    wl = inputs.custom(obj, 3.0, 4, eps_grad=1e-3)
    wl.x0[:] = np.float32([0.25, 0.5])
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    e0 = list(o.stats().evals)
    o.phase(orc.PH_LBFGS_ITER, 1)
    assert list(o.stats().evals) == e0 and np.all(o.get(orc.LS_B) == -2)


def test_first_step_length_is_min_1_inverse_gradient_norm(orc):
    """R-4 (iii): with an empty history the first trial step is t0 = min(1, 1/||gamma||_2) along p = -gamma.  On
    f = -1/2 ||x - c||^2 (central differences are exact, g = -(x - c), and every t <= 1 passes Armijo) the first trial
    is accepted, so a sample farther than 1 from c moves by exactly 1 towards c and a sample closer than 1 lands on c.
    t0 = 1 for everybody, or t0 = 1/||gamma||^2, fails."""
    obj = inputs.quad(3, 11, lam_max=1.0)                       # lambda = (1, 1, 1): W orthogonal, A = I
    c = obj.truth["c"]
    wl = inputs.custom(obj, 8.0, 6, fd_h=1e-2, eps_grad=1e-9)
    rng = np.random.default_rng(4)
    dirs = rng.standard_normal((6, 3)); dirs /= np.linalg.norm(dirs, axis=1)[:, None]
    radii = np.array([3.0, 2.0, 1.5, 0.75, 0.5, 0.1])
    wl.x0[:] = np.float32(c[None, :] + radii[:, None] * dirs)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    x0 = o.get(orc.X).copy()
    assert np.allclose(o.get(orc.G), -(x0 - c[None, :]), atol=1e-9)
    o.phase(orc.PH_LBFGS_ITER, 1)
    assert np.all(o.get(orc.LS_B) == 0)                          # first trial accepted
    x1 = o.get(orc.X)
    r0 = np.linalg.norm(x0 - c[None, :], axis=1)
    step = np.linalg.norm(x1 - x0, axis=1)
    far = r0 > 1.0
    assert far.sum() == 3
    assert np.allclose(step[far], 1.0, atol=2e-6)                # min(1, 1/||gamma||) ||gamma|| = 1 (positions are fp32)
    assert np.allclose(np.linalg.norm(x1[far] - c[None, :], axis=1), r0[far] - 1.0, atol=2e-6)   # towards c
    assert np.allclose(x1[~far], c[None, :], atol=2e-6)          # t0 = 1: the Newton step of A = I
    assert np.allclose(step[~far], r0[~far], atol=2e-6)
    assert np.all(o.get(orc.HIST_LEN) == 1)                      # s.y = ||s||^2 > 0: the pair is stored


def _cosine_1d(w, a, x0, **over):
    """f(x) = a cos(w x) on [-1, 1] (the random-Fourier objective with one feature, b = 0 and no quadratic term)"""
    obj = inputs.Objective(inputs.OBJ_RFF, 1, 1, np.zeros((1, 1), np.float32), np.float32([[w]]), np.float32([a]),
                           np.float32([0.0]), 0.0, 0.0)
    wl = inputs.custom(obj, 1.0, len(x0), **over)
    wl.x0[:] = np.float32(x0)[:, None]
    return wl


def test_curvature_pair_is_stored_only_for_positive_curvature(orc):
    """R-4 (vi): the pair (s, y) is stored iff s.y > 1e-10 |s||y|.  With s = x+ - x and y = gamma+ - gamma = -(g+ - g),
    s.y = -s^2 f''(xi): positive where f is concave, negative where f is convex.  f = 0.05 cos(2x): concave on
    |2x| < pi/2, convex on pi/2 < 2x < 3pi/2 (the small amplitude keeps the first step inside the region it starts in).  An accepted step inside the convex region must leave the history empty; inside the
    concave region it must store the pair."""
    wl = _cosine_1d(2.0, 0.05, [0.3, 1.0], fd_h=1e-4, eps_grad=1e-9, lbfgs_m=3)
    wl.hp.lo[:] = -2.0; wl.hp.hi[:] = 2.0                      # 2x up to 4: the convex region is inside the box
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    x0 = o.get(orc.X)[:, 0].copy(); g0 = o.get(orc.G)[:, 0].copy()
    o.phase(orc.PH_LBFGS_ITER, 1)
    x1 = o.get(orc.X)[:, 0]; g1 = o.get(orc.G)[:, 0]
    assert np.all(o.get(orc.LS_B) >= 0) and np.all(x1 != x0)     # both samples took an accepted step
    sy = (x1 - x0) * (-(g1 - g0))
    assert sy[0] > 0 and sy[1] < 0
    assert 1.0 < 2 * min(x0[1], x1[1]) * 2 / math.pi and 2 * max(x0[1], x1[1]) * 2 / math.pi < 3.0   # inside the convex region
    assert list(o.get(orc.HIST_LEN)) == [1, 0]
    S, Y = o.get(orc.HIST_S), o.get(orc.HIST_Y)
    assert S[0, 0, 0] == x1[0] - x0[0] and Y[0, 0, 0] == -(g1[0] - g0[0])
    assert not S[:, 1].any() and not Y[:, 1].any()


def test_failed_line_search_stalls_or_clears_history(orc):
    """R-4 (v): no trial accepted -> the sample is stalled (no further work) if its history was empty, else only the
    history is cleared.  f = 1/2 cos(40 x) just right of its maximum at 0 with an FD step h = 3 pi / 80 (w h = 3 pi / 2:
    the central difference has the wrong sign), so p points downhill for every trial t0 2^-b, b = 0..10: all ls_max + 1
    trials fail."""
    h = 3.0 * math.pi / 80.0
    wl = _cosine_1d(40.0, 0.5, [0.001, 0.001], fd_h=h, eps_grad=1e-3, lbfgs_m=2, ls_max=10)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    g0 = o.get(orc.G)[:, 0]
    assert np.all(g0 > 0.1) and np.all(g0 < 1.0)                 # wrong sign (true slope is negative), t0 = 1
    # sample 1 starts with one stored pair (s = y = 1: H = 1, the same direction p = g, t0 = 1)
    S = np.zeros((2, 2, 1)); S[0, 1, 0] = 1.0
    o.set(orc.HIST_S, S); o.set(orc.HIST_Y, S); o.set(orc.HIST_LEN, [0, 1])
    e0 = list(o.stats().evals)
    x0 = o.get(orc.X).copy(); f0 = o.get(orc.F).copy()
    o.phase(orc.PH_LBFGS_ITER, 1)
    e1 = list(o.stats().evals)
    assert list(o.get(orc.LS_B)) == [-1, -1]                     # nobody accepted
    assert e1[1] - e0[1] == 2 * 11 and e1[2] == e0[2]            # ls_max + 1 trials each, no FD gradient
    assert np.array_equal(o.get(orc.X), x0) and np.array_equal(o.get(orc.F), f0)   # no move
    assert list(o.get(orc.STALLED)) == [1, 0] and list(o.get(orc.HIST_LEN)) == [0, 0]
    # next iteration: the stalled sample does nothing; the other one searches again (now with an empty history) and stalls
    o.phase(orc.PH_LBFGS_ITER, 2)
    e2 = list(o.stats().evals)
    assert list(o.get(orc.LS_B)) == [-2, -1] and e2[1] - e1[1] == 11
    assert list(o.get(orc.STALLED)) == [1, 1]
    o.phase(orc.PH_LBFGS_ITER, 3)
    assert list(o.stats().evals) == e2 and list(o.get(orc.LS_B)) == [-2, -2]
    # release at the start of the next Phase 1 clears the flag (R-5)
    o.phase(orc.PH_RELEASE_EVAL)
    assert not o.get(orc.STALLED).any()


# ----------------------------------------------------------------------------- Phase 2: Eq. 3
def test_stick_is_eq3(orc):
    wl = inputs.config(1, N=200)
    o = orc.Oracle(wl)
    rng = np.random.default_rng(0)
    f = rng.normal(-2, 1.5, 200); g = rng.normal(0, 2e-3, (200, 2))
    f[5] = np.nan; f[6] = np.inf; g[7, 1] = np.nan
    o.set(orc.F, f); o.set(orc.G, g)
    o.phase(orc.PH_STICK)
    fmax = np.max(f[np.isfinite(f)])
    expect = (np.abs(g).max(axis=1) < np.float32(wl.hp.eps_grad)) & (f >= fmax + np.float32(wl.hp.log_delta))
    expect &= np.isfinite(f)
    expect[7] = False
    got = o.get(orc.STUCK).astype(bool)
    assert np.array_equal(got, expect) and 0 < got.sum() < 200
    assert o.stats().f_max == fmax and o.stats().n_stuck == got.sum()


def test_stick_thresholds_are_strict_and_nonstrict_as_printed(orc):
    wl = inputs.config(1, N=4)
    o = orc.Oracle(wl)
    eg, ld = float(np.float32(wl.hp.eps_grad)), float(np.float32(wl.hp.log_delta))
    o.set(orc.F, [0.0, ld, np.nextafter(ld, -np.inf), 0.0])
    o.set(orc.G, [[0, 0], [0, 0], [0, 0], [eg, 0]])
    o.phase(orc.PH_STICK)
    assert list(o.get(orc.STUCK)) == [1, 1, 0, 0]      # f >= f_max + log delta ; ||g||inf < eps_grad


# ----------------------------------------------------------------------------- Phase 3: Eq. 4
def _dedup_brute(x, f, stuck, eps):
    N = len(f)
    rem = np.zeros(N, bool)
    for i in range(N):
        if not stuck[i]:
            continue
        for j in range(N):
            if j != i and stuck[j] and np.abs(x[i] - x[j]).max() < eps and (f[j] > f[i] or (f[j] == f[i] and j < i)):
                rem[i] = True
    return rem


def test_dedup_definition_and_invariants(orc):
    wl = inputs.config(1, N=300, eps_dup=0.05)
    o = orc.Oracle(wl)
    rng = np.random.default_rng(1)
    centres = rng.uniform(-3, 3, (12, 2))
    x = np.float32(centres[rng.integers(0, 12, 300)] + rng.normal(0, 0.012, (300, 2))).astype(np.float64)
    f = rng.normal(0, 1, 300); f[10] = f[11] = 100.0; x[11] = x[10];            # exact tie -> lower index survives
    stuck = rng.uniform(size=300) < 0.8; stuck[10] = stuck[11] = True
    o.set(orc.X, x); o.set(orc.F, f); o.set(orc.STUCK, stuck)
    o.set(orc.REMOVED, np.zeros(300))
    eps = float(np.float32(0.05))
    o.phase(orc.PH_DEDUP)
    rem = o.get(orc.REMOVED).astype(bool); st = o.get(orc.STUCK).astype(bool)
    assert np.array_equal(rem, _dedup_brute(x, f, stuck, eps))
    assert rem.sum() > 50 and (stuck[10] and stuck[11]) <= (rem[11] and not rem[10])
    assert np.array_equal(st, stuck & ~rem)
    assert o.stats().k_lost == rem.sum() and o.stats().n_stuck == st.sum()
    assert o.stats().n_active == (~stuck).sum()
    # not a chain-removal: a survivor's cluster representative is the local f-maximum
    P = np.flatnonzero(st)
    for i in np.flatnonzero(rem):
        near = [j for j in np.flatnonzero(stuck) if np.abs(x[i] - x[j]).max() < eps]
        assert max(f[j] for j in near) > f[i] or min(j for j in near if f[j] == f[i]) < i
    # idempotent: survivors of a second pass = survivors of the first whenever clusters are cliques
    o.set(orc.REMOVED, np.zeros(300))
    o.phase(orc.PH_DEDUP)
    rem2 = o.get(orc.REMOVED).astype(bool)
    assert np.array_equal(rem2, _dedup_brute(x, f, st, eps))


def test_dedup_mask_off_removes_nothing(orc):
    wl = inputs.config(1, N=16, phase_mask=0xFFFFFFFF & ~(1 << 3))
    o = orc.Oracle(wl)
    o.set(orc.X, np.zeros((16, 2))); o.set(orc.STUCK, np.ones(16)); o.set(orc.F, np.arange(16.0))
    o.phase(orc.PH_DEDUP)
    assert o.get(orc.REMOVED).sum() == 0 and o.stats().k_lost == 0


# ----------------------------------------------------------------------------- Phase 4: reseeding
def _setup_reseed(orc, wl, stuck, removed, cycle=2, ctrl=None):
    o = orc.Oracle(wl)
    o.set(orc.STUCK, stuck); o.set(orc.REMOVED, removed)
    c = [cycle, 1, 0, 0, 0, int(removed.sum()), int(stuck.sum()), int((~stuck & ~removed).sum())]
    if ctrl:
        c[1:5] = ctrl
    o.set(orc.CTRL, c)
    return o


def test_repulse_monkey(orc):
    wl = inputs.config(2, N=64)
    x0 = wl.x0.astype(np.float64)
    stuck = np.zeros(64, bool); stuck[[3, 9, 20]] = True
    removed = np.zeros(64, bool); removed[[4, 5, 30, 63]] = True
    o = _setup_reseed(orc, wl, stuck, removed)
    o.phase(orc.PH_RESEED)
    x = o.get(orc.X); src = o.get(orc.RS_SRC); cand = o.get(orc.RS_CAND)
    assert o.stats().reseed_strategy == 1
    keep = ~removed
    assert np.array_equal(x[keep], x0[keep])                        # only removed slots are rewritten
    assert np.all(x >= -5) and np.all(x <= 5) and len(x) == 64      # population maintained at N, inside Theta
    assert o.get(orc.REMOVED).sum() == 0 and o.get(orc.STUCK)[removed].sum() == 0
    A = np.flatnonzero(~stuck & ~removed); P = np.flatnonzero(stuck)
    for r in np.flatnonzero(removed):
        assert src[r] in A
        w = orc.philox([0, r, 2, orc.tag(4, 0, 3)], [wl.hp.seed, 0])
        assert src[r] == A[(int(w[0]) * len(A)) >> 32]
        u = np.array([orc.normal(wl.hp.seed, r, 2, orc.tag(4, 0, 5), j) for j in range(8)])
        u /= np.linalg.norm(u)
        dvec = x[r] - x0[src[r]]
        t = np.linalg.norm(dvec)
        assert np.allclose(dvec / t, u, atol=1e-5)                  # on the ray, positive side
        # exit distance and the C candidates; the kept one maximises the distance to the frozen modes
        tmax = min(((5 if u[j] > 0 else -5) - x0[src[r], j]) / u[j] for j in range(8))
        U = [orc.uniform(wl.hp.seed, r, 2, orc.tag(4, 0, 4), c) for c in range(4)]
        assert 0 < t <= tmax * (1 + 1e-6)
        cands = [x0[src[r]] + tmax * Uc * u for Uc in U]
        score = [min(np.linalg.norm(cx - x0[p]) for p in P) for cx in cands]
        assert cand[r] == int(np.argmax(score))
        assert np.allclose(x[r], cands[cand[r]], atol=1e-5)


def test_golden_rooster_and_uniform_fallback(orc):
    wl = inputs.config(2, N=40)
    x0 = wl.x0.astype(np.float64)
    stuck = np.zeros(40, bool); stuck[[1, 2, 7]] = True
    removed = ~stuck; removed[[0, 39]] = False                      # 2 unfrozen < 5
    o = _setup_reseed(orc, wl, stuck, removed, cycle=3)
    Q = o.gr_basis(3)
    assert np.allclose(Q.T @ Q, np.eye(8), atol=1e-12)
    G = np.array([[orc.normal(wl.hp.seed, 0, 3, orc.tag(4, 0, 6), a * 8 + b) for b in range(8)] for a in range(8)])
    R = Q.T @ G
    assert np.allclose(np.tril(R, -1), 0, atol=1e-10) and np.all(np.diag(R) > 0)    # G = QR, R_ii > 0
    o.phase(orc.PH_RESEED)
    assert o.stats().reseed_strategy == 2
    x = o.get(orc.X); P = np.flatnonzero(stuck)
    for q, r in enumerate(np.flatnonzero(removed)):
        peak = P[q % 3]; col = (q // 3) % 8; sign = -1 if (q // 24) % 2 else 1
        dvec = x[r] - x0[peak]
        assert np.allclose(dvec / np.linalg.norm(dvec), sign * Q[:, col], atol=1e-5)
    assert np.array_equal(x[~removed], x0[~removed])
    assert np.all(np.abs(x) <= 5) and o.get(orc.STUCK).sum() == 3 and o.get(orc.REMOVED).sum() == 0
    ctrl = o.get(orc.CTRL)
    assert ctrl[4] == 1 and ctrl[3] == 3                            # gr_used_last, gr_prev_modes
    # disabled -> uniform refill of Theta
    o2 = _setup_reseed(orc, wl, stuck, removed, cycle=3, ctrl=[0, 2, 3, 0])
    o2.phase(orc.PH_RESEED)
    assert o2.stats().reseed_strategy == 3
    x2 = o2.get(orc.X)
    for r in np.flatnonzero(removed)[:5]:
        U = np.array([orc.uniform(wl.hp.seed, r, 3, orc.tag(4, 0, 7), j) for j in range(8)])
        assert np.allclose(x2[r], -5 + 10 * U, atol=1e-6)


def test_golden_rooster_self_disables_after_two_unproductive_generations(orc):
    wl = inputs.config(1)                                           # 4 modes; everything converges in cycle 1
    o = orc.Oracle(wl)
    strat, en = [], []
    for _ in range(5):
        st = o.step(); strat.append(st.reseed_strategy); en.append(st.gr_enabled)
    assert strat == [2, 2, 3, 3, 3] and en == [1, 1, 0, 0, 0]


def test_no_reseed_without_losses_or_when_masked(orc):
    wl = inputs.config(2, N=16)
    o = _setup_reseed(orc, wl, np.zeros(16, bool), np.zeros(16, bool))
    o.phase(orc.PH_RESEED)
    assert o.stats().reseed_strategy == 0 and np.array_equal(o.get(orc.X), wl.x0.astype(np.float64))


# ----------------------------------------------------------------------------- Phase 5: HLC (Eq. 5 / Eq. 9)
def test_hlc_estimator_is_unbiased_for_the_smoothed_gradient(orc):
    """Eq. 9: for a quadratic, grad f_sigma = grad f; the Monte-Carlo mean must agree
    within 4 standard errors, with and without the mean-value baseline."""
    obj = inputs.quad(3, 21, lam_max=10.0)
    t = obj.truth
    for baseline in (0, 1):
        wl = inputs.custom(obj, 4.0, 1, hlc_M=400_000, sigma_s=0.3, eta_hlc=0.0, hlc_baseline=baseline)
        o = orc.Oracle(wl)
        o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 1])
        x = o.get(orc.X)[0]
        o.phase(orc.PH_HLC_STEP, 1)
        gh = o.get(orc.GHAT)[0]; fk = o.get(orc.HLC_F)[0]; u = o.get(orc.HLC_U)[0]
        truth = -t["A"] @ (x - t["c"])
        b = fk.mean() if baseline else 0.0
        per_draw = (fk - b)[:, None] * u / float(np.float32(0.3))
        se = per_draw.std(axis=0) / math.sqrt(len(fk))
        assert np.all(np.abs(gh - truth) < 4.5 * se)
        if baseline:
            assert np.all(se < 0.05 * np.abs(truth).max())
        assert np.array_equal(o.get(orc.X)[0], x)                    # eta = 0 -> no move
        # draws are the documented Philox normals and every evaluation is at x + sigma u (unclipped)
        for k in (0, 1, 399_999):
            for j in range(3):
                assert u[k, j] == orc.normal(wl.hp.seed, 0, 1, orc.tag(5, 1, 2), k * 3 + j)
            assert math.isclose(fk[k], o.values((x + float(np.float32(0.3)) * u[k])[None])[0], rel_tol=1e-13)


def test_hlc_baseline_identity_and_step(orc):
    wl = inputs.config(2, N=6, noise=0.0, hlc_baseline=0)
    wl1 = inputs.config(2, N=6, noise=0.0, hlc_baseline=1)
    o0, o1 = orc.Oracle(wl), orc.Oracle(wl1)
    for o in (o0, o1):
        o.set(orc.CTRL, [2, 1, 0, 0, 0, 0, 1, 5])
        o.set(orc.STUCK, [0, 0, 1, 0, 0, 0])
        o.phase(orc.PH_HLC_STEP, 2)
    M, sig = 16, 0.5
    g0, g1, fk, u = o0.get(orc.GHAT), o1.get(orc.GHAT), o0.get(orc.HLC_F), o0.get(orc.HLC_U)
    for i in (0, 1, 3, 4, 5):
        assert np.allclose(g0[i] - g1[i], fk[i].mean() * u[i].sum(axis=0) / (M * sig), rtol=1e-10)
        assert np.allclose(g0[i], (fk[i][:, None] * u[i]).sum(axis=0) / (M * sig), rtol=1e-12)
    x0 = wl.x0.astype(np.float64); x = o0.get(orc.X)
    assert np.array_equal(x[2], x0[2])                                # frozen sample never moves
    expect = np.clip(x0 + float(np.float32(wl.hp.eta_hlc)) * g0, -5, 5)
    assert np.allclose(x, expect, atol=1e-6)


# ----------------------------------------------------------------------------- Phase 6: Eq. 6
def test_anti_convergence_is_the_eq6_linear_recurrence(orc):
    """On a quadratic, grad f = -A (x - c) and central FD is exact, so Eq. 6 is the linear map
    [e; v] <- [[I + alpha A, mu I], [alpha A, mu I]] [e; v] with e = x - c; compare with its matrix power."""
    obj = inputs.quad(4, 31, lam_max=50.0)
    t = obj.truth
    wl = inputs.custom(obj, 50.0, 3, alpha_anti=1e-3, mu=0.9, n_anti=5, fd_h=1e-2)
    wl.x0[:] = np.float32(np.random.default_rng(2).uniform(-1, 1, (3, 4)))   # stays inside the box for 5 steps
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 1, 2])
    o.set(orc.STUCK, [0, 1, 0])
    x0 = o.get(orc.X)
    o.set(orc.V, np.ones((3, 4)))                                      # must be reset: v_0 = 0 (R-12)
    for s in range(1, 6):
        o.phase(orc.PH_ANTI_STEP, s)
    al, mu = float(np.float32(1e-3)), float(np.float32(0.9))
    A = t["A"]; I = np.eye(4)
    T = np.block([[I + al * A, mu * I], [al * A, mu * I]])
    T5 = np.linalg.matrix_power(T, 5)
    x, v = o.get(orc.X), o.get(orc.V)
    for i in (0, 2):
        ev = T5 @ np.concatenate([x0[i] - t["c"], np.zeros(4)])
        assert np.allclose(x[i] - t["c"], ev[:4], rtol=2e-6, atol=1e-6)
        assert np.allclose(v[i], ev[4:], rtol=2e-6, atol=1e-6)
        assert o.values(x[i][None])[0] < o.values(x0[i][None])[0]      # descent: moves away from the peak
    assert np.array_equal(x[1], x0[1]) and np.array_equal(v[1], np.ones(4))
    assert o.stats().evals[6] == 2 * 5 * 2 * 4


# ----------------------------------------------------------------------------- Algorithm 1
def test_remark1_unimodal_everything_sticks_and_cycle_collapses(orc):
    """PAPER.md:218 (Remark 1) / Prop. 1: one mode -> every sample sticks, one mode survives."""
    obj = inputs.gmm_iso(3, 1, 0.8, 3.0, 5)
    wl = inputs.custom(obj, 3.0, 50, n_osc=2, n_conv=40, eps_grad=1e-4, eps_dup=1e-3, fd_h=1e-3)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    for it in range(1, 41):
        o.phase(orc.PH_LBFGS_ITER, it)
    o.phase(orc.PH_STICK)
    assert o.get(orc.STUCK).sum() == 50
    o.phase(orc.PH_DEDUP)
    st = o.stats()
    assert st.n_stuck == 1 and st.k_lost == 49
    xm, fm, _ = o.modes()
    assert np.abs(xm[0] - obj.truth["mu"][0]).max() < 1e-4


def test_last_cycle_skips_phases_4_to_6_and_counts_follow_eq8(orc):
    """PAPER.md:131 and the structure of Eq. 8."""
    wl = inputs.config(2, N=32, n_osc=2)
    o = orc.Oracle(wl)
    s1 = o.step(); x_after_1 = o.get(orc.X).copy()
    e1 = list(s1.evals)
    act1 = s1.n_active
    assert e1[0] == 32 * 17
    assert e1[5] == act1 * 3 * 16 and e1[6] == act1 * 5 * 16           # n_cloud*M and n_anti*2d per unfrozen
    assert e1[2] % 16 == 0 and e1[2] // 16 <= e1[1] <= 11 * 32 * 10
    s2 = o.step()
    e2 = list(s2.evals)
    assert e2[5] == e1[5] and e2[6] == e1[6] and s2.reseed_strategy == 0   # no exploration on k = n_osc
    stuck = o.get(orc.STUCK).astype(bool)
    xm, fm, idx = o.modes()
    assert np.array_equal(np.sort(idx), np.flatnonzero(stuck))
    assert np.all(np.diff(fm) <= 0)
    with pytest.raises(RuntimeError):
        o.step()


def test_frozen_samples_never_move_in_exploration_phases(orc):
    wl = inputs.config(1, N=128, n_osc=3)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    for it in range(1, 6):                       # few iterations: only part of the population converges
        o.phase(orc.PH_LBFGS_ITER, it)
    o.phase(orc.PH_STICK); o.phase(orc.PH_DEDUP)
    stuck = o.get(orc.STUCK).astype(bool)
    assert 0 < stuck.sum() < 128
    x0 = o.get(orc.X).copy()
    o.phase(orc.PH_RESEED)
    removed_before = np.flatnonzero(np.any(o.get(orc.X) != x0, axis=1))
    x1 = o.get(orc.X).copy()
    for t in range(1, 4):
        o.phase(orc.PH_HLC_STEP, t)
    for t in range(1, 6):
        o.phase(orc.PH_ANTI_STEP, t)
    x2 = o.get(orc.X)
    assert np.array_equal(x2[stuck], x0[stuck])
    moved = np.any(x2 != x1, axis=1)
    assert moved[~stuck].all() and np.all(np.abs(x2) <= 3)
    assert len(x2) == 128 and set(removed_before).isdisjoint(np.flatnonzero(stuck))


def test_modes_equal_brute_force_grid_enumeration_d2(orc):
    """north_star: 'a brute-force grid mode enumeration at d=2'.  Grid maxima -> Newton polish with
    the analytic gradient/Hessian -> Eq. 1 filter must equal the oracle's mode set."""
    wl = inputs.config(1)
    t = wl.obj.truth
    mu, sig = t["mu"], t["sigma"]
    n = 1201
    ax = np.linspace(-3, 3, n)
    XX, YY = np.meshgrid(ax, ax, indexing="ij")
    pts = np.stack([XX.ravel(), YY.ravel()], axis=1)
    o = orc.Oracle(wl)
    F = o.values(pts).reshape(n, n)
    c = F[1:-1, 1:-1]
    ismax = np.ones_like(c, bool)
    for dx in (-1, 0, 1):
        for dy in (-1, 0, 1):
            if dx or dy:
                ismax &= c > F[1 + dx:n - 1 + dx, 1 + dy:n - 1 + dy]
    seeds = np.stack([ax[1:-1][np.nonzero(ismax)[0]], ax[1:-1][np.nonzero(ismax)[1]]], axis=1)

    def grad_hess(x):
        dx = mu - x
        lw = -((dx ** 2).sum(axis=1)) / (2 * sig ** 2)
        r = np.exp(lw - lw.max()); r /= r.sum()
        g = (r[:, None] * dx).sum(axis=0) / sig ** 2
        m1 = (r[:, None] * dx).sum(axis=0) / sig ** 2
        H = -np.eye(2) / sig ** 2 + (r[:, None, None] * dx[:, :, None] * dx[:, None, :]).sum(axis=0) / sig ** 4 - np.outer(m1, m1)
        return g, H

    polished = []
    for s in seeds:
        x = s.copy()
        for _ in range(30):
            g, H = grad_hess(x)
            x = x - np.linalg.solve(H, g)
        g, H = grad_hess(x)
        assert np.abs(g).max() < 1e-10 and np.all(np.linalg.eigvalsh(H) < 0)
        polished.append(x)
    polished = np.array(polished)
    fpol = o.values(polished)
    keep = fpol >= fpol.max() + math.log(0.1)                          # Eq. 1 quality filter
    truth_modes = polished[keep]
    for _ in range(wl.hp.n_osc):
        o.step()
    xm, fm, _ = o.modes()
    assert len(xm) == len(truth_modes) == 4
    for m in truth_modes:
        assert np.min(np.linalg.norm(xm - m[None], axis=1)) < 1e-3


def test_hlc_eq5_form_on_a_quadratic_is_the_gradient_at_the_mean_perturbed_point(orc):
    """Paper form of Hands Like Clouds, Eq. 5: (1/K) sum_k grad f(x + sigma z_k).  On a quadratic the
    gradient is affine and central differences are exact, so the average equals the analytic gradient at the mean
    perturbed point -A (mean_k(x + sigma z_k) - c); the step and the evaluation count K 2d follow (Eq. 8)."""
    obj = inputs.quad(5, 21, lam_max=30.0)
    wl = inputs.custom(obj, 4.0, 12, hlc_M=7, sigma_s=0.3, eta_hlc=1e-3, fd_h=1e-2, hlc_baseline=2, seed=99)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [2, 1, 0, 0, 0, 0, 0, 0])
    x0 = o.get(orc.X).copy()
    stuck = np.zeros(12, np.uint8); stuck[3] = 1
    o.set(orc.STUCK, stuck)
    o.phase(orc.PH_HLC_STEP, 1)
    A, c = obj.truth["A"], obj.truth["c"]
    tag = orc.tag(5, 1, 2)
    for i in (0, 5, 11):
        z = np.array([[orc.normal(99, i, 2, tag, k * 5 + j) for j in range(5)] for k in range(7)])
        pts = (x0[i][None, :] + float(np.float32(0.3)) * z).astype(np.float32).astype(np.float64)
        expect = -(A @ (pts.mean(axis=0) - c))
        gh = o.get(orc.GHAT)[i]
        assert np.allclose(gh, expect, rtol=1e-7, atol=1e-7)
        assert np.allclose(o.get(orc.X)[i], np.clip(x0[i] + float(np.float32(1e-3)) * gh, -4, 4).astype(np.float32), atol=1e-7)
    assert np.array_equal(o.get(orc.X)[3], x0[3]) and not o.get(orc.GHAT)[3].any()
    assert o.stats().evals[5] == 11 * 7 * 2 * 5


def test_hlc_sigma_auto_is_c_times_the_pooled_std_of_the_unfrozen_samples(orc):
    """sigma = c std({x_i : not stuck_i}), c = 0.1 by default (R-18: pooled population std over all
    coordinates of the unfrozen samples); sigma_s > 0 is used as given."""
    obj = inputs.gmm_iso(3, 2, 0.5, 2.0, 5)
    wl = inputs.custom(obj, 3.0, 50, sigma_s=-0.1, hlc_M=4, eta_hlc=1e-3, seed=31)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    stuck = np.zeros(50, np.uint8); stuck[::3] = 1
    o.set(orc.STUCK, stuck)
    x0 = o.get(orc.X).copy()
    o.phase(orc.PH_HLC_STEP, 1)
    assert abs(o.get(orc.SIGMA)[0] - float(np.float32(0.1)) * np.std(x0[stuck == 0])) < 1e-12
    assert np.array_equal(o.get(orc.X)[stuck == 1], x0[stuck == 1]) and not np.array_equal(o.get(orc.X), x0)
    wl2 = inputs.custom(obj, 3.0, 50, sigma_s=0.25, hlc_M=4, seed=31)
    o2 = orc.Oracle(wl2); o2.phase(orc.PH_HLC_STEP, 1)
    assert o2.get(orc.SIGMA)[0] == 0.25
    # nobody unfrozen: sigma = 0 and nothing moves
    o.set(orc.STUCK, np.ones(50, np.uint8)); x1 = o.get(orc.X).copy()
    o.phase(orc.PH_HLC_STEP, 2)
    assert o.get(orc.SIGMA)[0] == 0.0 and np.array_equal(o.get(orc.X), x1)
