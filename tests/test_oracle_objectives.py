"""Pins for the oracle's objective values and finite-difference gradients.

Values are checked against library routines that are not the oracle's own code path
(scipy.stats.multivariate_normal / scipy.special.logsumexp, numpy matrix algebra on the float64
"truth" the fp32 parameter arrays were derived from, mpmath at 50 digits) and against closed forms;
FD gradients against analytic gradients ("or supplied analytically when available").
"""
import math

import mpmath
import numpy as np
import pytest
from scipy.special import logsumexp
from scipy.stats import multivariate_normal

from paper_2606_26164_b200 import inputs


def _pts(wl, n, seed=0):
    rng = np.random.default_rng(seed)
    return rng.uniform(wl.hp.lo.astype(np.float64), wl.hp.hi.astype(np.float64), size=(n, wl.hp.d))


def _gmm_ref(obj, X):
    t = obj.truth
    K, d = obj.K, obj.d
    cols = []
    for k in range(K):
        if obj.id == inputs.OBJ_GMM_ISO:
            cov = np.eye(d) * t["sigma"] ** 2
        elif obj.id == inputs.OBJ_GMM_DIAG:
            cov = np.diag(t["sig"][k] ** 2)
        else:
            cov = np.linalg.inv(t["prec"][k])
        cols.append(t["logw"][k] + multivariate_normal(t["mu"][k], cov, allow_singular=False).logpdf(X))
    return logsumexp(np.stack(cols, axis=1), axis=1)


def _gmm_grad(obj, x):
    """sum_k r_k(x) P_k (mu_k - x), r = responsibilities."""
    t = obj.truth
    K, d = obj.K, obj.d
    logp, grads = [], []
    for k in range(K):
        if obj.id == inputs.OBJ_GMM_ISO:
            P = np.eye(d) / t["sigma"] ** 2
        elif obj.id == inputs.OBJ_GMM_DIAG:
            P = np.diag(1.0 / t["sig"][k] ** 2)
        else:
            P = t["prec"][k]
        dx = t["mu"][k] - x
        logp.append(t["logw"][k] + 0.5 * np.linalg.slogdet(P)[1] - 0.5 * dx @ P @ dx)
        grads.append(P @ dx)
    r = np.exp(np.array(logp) - logsumexp(logp))
    return (r[:, None] * np.array(grads)).sum(axis=0)


CASES = {
    "iso": lambda: inputs.config(1, N=4),
    "diag": lambda: inputs.config(2, N=4, noise=0.0),
    "full8": lambda: inputs.custom(inputs.gmm_full(8, 5, 4.0, 77), 4.0, 4),
    "full64": lambda: inputs.config(5, N=4, noise=0.0),
}


@pytest.mark.parametrize("name", list(CASES))
def test_gmm_values_match_scipy(orc, name):
    wl = CASES[name]()
    o = orc.Oracle(wl)
    X = _pts(wl, 40)
    # also points near the component means, where the value is O(1) and cancellation matters
    X = np.concatenate([X, wl.obj.truth["mu"][: min(8, wl.obj.K)] + 0.05])
    ref = _gmm_ref(wl.obj, X)
    got = o.values(X)
    # vec_a is stored in fp32 -> absolute 1e-6-level differences are inherent to the inputs
    assert np.allclose(got, ref, rtol=2e-7, atol=5e-6)


def test_isolated_component_closed_form(orc):
    """f(mu_k) = log w_k + log-normaliser when the other components are far away."""
    obj = inputs.gmm_iso(3, 2, 0.3, 3.0, 5, means=[[-2.0, 0, 0], [2.0, 0, 0]])
    wl = inputs.custom(obj, 3.0, 2)
    o = orc.Oracle(wl)
    f = o.values(obj.truth["mu"])
    expect = math.log(0.5) - 1.5 * math.log(2 * math.pi * obj.truth["sigma"] ** 2)
    assert np.allclose(f, expect, atol=5e-7)      # other component contributes exp(-16/0.18) ~ 1e-39


def test_one_component_gmm_is_a_quadratic(orc):
    obj = inputs.gmm_iso(4, 1, 0.7, 3.0, 6)
    wl = inputs.custom(obj, 3.0, 2)
    o = orc.Oracle(wl)
    X = _pts(wl, 10)
    mu, sig = obj.truth["mu"][0], obj.truth["sigma"]
    expect = float(obj.vec_a[0]) - ((X - mu) ** 2).sum(axis=1) / (2 * sig ** 2)
    assert np.allclose(o.values(X), expect, rtol=1e-14, atol=1e-12)


def test_rff_values(orc):
    wl = inputs.config(3, N=4)
    o = orc.Oracle(wl)
    X = _pts(wl, 30)
    t = wl.obj.truth
    ref = -t["q"] * (X ** 2).sum(axis=1) + (t["a"][None, :] * np.cos(X @ t["w"].T + t["b"][None, :])).sum(axis=1)
    assert np.allclose(o.values(X), ref, rtol=1e-12, atol=1e-12)
    assert math.isclose(o.values(np.zeros((1, 32)))[0], float((t["a"] * np.cos(t["b"])).sum()), rel_tol=1e-13)
    # one point at 50 digits
    mpmath.mp.dps = 50
    x = X[0]
    acc = -mpmath.mpf(t["q"]) * sum(mpmath.mpf(float(v)) ** 2 for v in x)
    for j in range(wl.obj.K):
        arg = sum(mpmath.mpf(float(t["w"][j, c])) * mpmath.mpf(float(x[c])) for c in range(32)) + mpmath.mpf(float(t["b"][j]))
        acc += mpmath.mpf(float(t["a"][j])) * mpmath.cos(arg)
    assert abs(o.values(x[None])[0] - float(acc)) < 1e-12


def test_quadratic_closed_forms(orc):
    wl = inputs.config(4, N=4)
    o = orc.Oracle(wl)
    t = wl.obj.truth
    assert o.values(t["c"][None])[0] == 0.0
    X = _pts(wl, 20)
    ref = -0.5 * np.einsum("ni,ij,nj->n", X - t["c"], t["A"], X - t["c"])
    assert np.allclose(o.values(X), ref, rtol=1e-12)
    # along an eigen-direction Q^T e_i:  f(c + t q_i) = -1/2 lambda_i t^2
    lam, Q = np.linalg.eigh(t["A"])
    for i in (0, 31, 63):
        assert math.isclose(o.values((t["c"] + 0.3 * Q[:, i])[None])[0], -0.5 * lam[i] * 0.09, rel_tol=1e-9)
    assert lam.min() == pytest.approx(1.0, rel=1e-4) and lam.max() == pytest.approx(1e4, rel=1e-4)


@pytest.mark.parametrize("name", list(CASES))
def test_fd_gradient_vs_analytic_gmm(orc, name):
    wl = CASES[name]()
    wl.hp.fd_h = 1e-4
    o = orc.Oracle(wl)
    mu = wl.obj.truth["mu"]
    rng = np.random.default_rng(3)
    for k in range(min(6, wl.obj.K)):
        x = mu[k] + 0.3 * rng.standard_normal(wl.hp.d)
        f, g = o.fd_gradient(x)
        ga = _gmm_grad(wl.obj, x)
        assert f == o.values(x[None])[0]
        assert np.allclose(g, ga, rtol=1e-5, atol=1e-5 * np.abs(ga).max())


def test_fd_gradient_vs_analytic_rff_and_truncation_order(orc):
    wl = inputs.config(3, N=4)
    t = wl.obj.truth
    x = _pts(wl, 1, seed=5)[0]
    ga = -2 * t["q"] * x - (t["a"][:, None] * np.sin(t["w"] @ x + t["b"])[:, None] * t["w"]).sum(axis=0)
    errs = []
    for h in (2e-2, 1e-2):
        wl.hp.fd_h = h
        _, g = orc.Oracle(wl).fd_gradient(x)
        errs.append(np.abs(g - ga).max())
    assert errs[1] < 1e-3 * np.abs(ga).max()
    assert 3.5 < errs[0] / errs[1] < 4.5            # central differences: error ~ h^2


def test_fd_exact_on_quadratic_any_h(orc):
    wl = inputs.config(4, N=4)
    t = wl.obj.truth
    x = _pts(wl, 1, seed=8)[0]
    ga = -t["A"] @ (x - t["c"])
    for h in (1e-2, 0.5):
        wl.hp.fd_h = h
        _, g = orc.Oracle(wl).fd_gradient(x)
        assert np.allclose(g, ga, rtol=1e-9)


def test_fd_uses_2d_plus_1_evaluations_and_slots(orc):
    """Noise slots: 0 centre, 1+2j plus, 2+2j minus (R-2) -- reconstruct f, g from the noise-free parts."""
    wl = inputs.config(2, N=3)
    o = orc.Oracle(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    assert o.stats().evals[0] == 3 * (2 * 8 + 1)
    f, g, x = o.get(orc.F), o.get(orc.G), o.get(orc.X)
    h = float(np.float32(wl.hp.fd_h))
    for i in range(3):
        assert math.isclose(f[i], o.values(x[i][None])[0] + o.noise(1, i, 1, 0, 0), rel_tol=1e-14)
        for j in range(8):
            e = np.zeros(8); e[j] = h
            fp = o.values((x[i] + e)[None])[0] + o.noise(1, i, 1, 0, 1 + 2 * j)
            fm = o.values((x[i] - e)[None])[0] + o.noise(1, i, 1, 0, 2 + 2 * j)
            assert math.isclose(g[i, j], (fp - fm) / (2 * h), rel_tol=1e-12, abs_tol=1e-12)
