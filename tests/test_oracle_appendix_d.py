"""Pins for the oracle's Appendix-D objectives against the optima the paper prints and against
closed-form special points (none of them re-evaluates the oracle's own formula)."""
import math

import numpy as np
import pytest

from paper_2606_26164_b200 import inputs


def _o(orc, name, d):
    return orc.Oracle(inputs.appendix_d(name, d, 4))


@pytest.mark.parametrize("d", [1, 2, 7, 64])
def test_rastrigin_printed_optimum_and_integer_lattice(orc, d):
    o = _o(orc, "rastrigin", d)
    assert abs(o.values(np.zeros(d))[0]) < 1e-12                        # PAPER.md:614 "f(0) = 0"
    k = np.arange(d) % 5 - 2.0                                           # integers: cos(2 pi k) = 1 -> f = -sum k^2
    assert abs(o.values(k)[0] + np.sum(k * k)) < 1e-9
    assert abs(o.values(np.full(d, 0.5))[0] + d * (0.25 + 20.0)) < 1e-9  # half-integers: cos = -1


@pytest.mark.parametrize("d", [1, 3, 32])
def test_ackley_closed_forms(orc, d):
    o = _o(orc, "ackley", d)
    assert abs(o.values(np.zeros(d))[0]) < 1e-12                        # -[-a - e + a + e] = 0
    t = np.full(d, 3.0)                                                  # integer point: cos(2 pi 3) = 1, rms = 3
    assert abs(o.values(t)[0] + (-20.0 * math.exp(-0.6) - math.e + 20.0 + math.e)) < 1e-9


@pytest.mark.parametrize("d", [1, 4, 64])
def test_schwefel_printed_optimum(orc, d):
    o = _o(orc, "schwefel", d)
    x = np.full(d, 420.97)                                               # PAPER.md:619 "near theta_i = 420.97"
    f = o.values(x)[0]
    assert abs(f) < 2e-4 * d + 1e-6                                      # 418.9829 d - d * 418.98288...
    for dx in (-0.5, 0.5):
        assert o.values(x + dx)[0] < f                                   # a maximum along the diagonal
    assert abs(o.values(np.zeros(d))[0] + 418.9829 * d) < 1e-9


@pytest.mark.parametrize("d", [1, 5])
def test_styblinski_tang_stationary_points(orc, d):
    o = _o(orc, "styblinski_tang", d)
    roots = np.roots([4.0, 0.0, -32.0, 5.0]).real                       # d/dt (t^4 - 16 t^2 + 5 t) = 0
    tbest = roots[np.argmin(roots)]                                      # global maximiser of f, approx -2.9035
    fbest = o.values(np.full(d, tbest))[0]
    assert abs(fbest - d * 39.16616570377142) < 1e-6 * d                 # -(1/2)(t^4 - 16 t^2 + 5 t) at that root
    g = np.array([o.fd_gradient(np.full(d, r))[1] for r in roots])
    assert np.max(np.abs(g)) < 1e-3                                      # FD gradient vanishes at all three roots
    assert abs(o.values(np.zeros(d))[0]) < 1e-15


@pytest.mark.parametrize("d", [1, 2, 10])
def test_michalewicz_special_points(orc, d):
    o = _o(orc, "michalewicz", d)
    i = np.arange(1, d + 1)
    x = math.pi / np.sqrt(2.0 * i)                                       # i x^2 / pi = pi/2 -> sin^{20} = 1
    assert abs(o.values(x)[0] - np.sum(np.sin(x))) < 1e-12
    assert abs(o.values(np.zeros(d))[0]) < 1e-15 and abs(o.values(np.full(d, math.pi))[0]) < 1e-10
    x2 = math.pi / np.sqrt(i)                                            # i x^2 / pi = pi -> sin = 0
    assert abs(o.values(x2)[0]) < 1e-10


@pytest.mark.parametrize("d", [2, 6, 10])
def test_trid_printed_optimum(orc, d):
    o = _o(orc, "trid", d)
    i = np.arange(1, d + 1, dtype=np.float64)
    xs = i * (d + 1 - i)                                                 # PAPER.md:625 theta*_i = i (d + 1 - i)
    fs = o.values(xs)[0]
    assert abs(fs - d * (d + 4) * (d - 1) / 6.0) < 1e-9                  # f* = d (d + 4)(d - 1) / 6
    _, g = o.fd_gradient(xs)
    assert np.max(np.abs(g)) < 1e-6                                      # stationary (quadratic: FD exact)
    assert o.values(xs + 0.3)[0] < fs and o.values(xs - 0.3)[0] < fs


def test_bukin6_printed_optimum_and_ridge(orc):
    o = _o(orc, "bukin6", 2)
    assert abs(o.values(np.array([-10.0, 1.0]))[0]) < 1e-12             # PAPER.md:627 maximum at (-10, 1), f* = 0
    x = np.array([-8.0, 0.64])                                           # on the ridge y = 0.01 x^2: f = -0.01 |x + 10|
    assert abs(o.values(x)[0] + 0.02) < 1e-12
    assert abs(o.values(np.array([-10.0, 2.0]))[0] + 100.0) < 1e-12     # off the ridge by 1: -100 sqrt(1)
    with pytest.raises(ValueError):
        orc.Oracle(type(inputs.appendix_d("bukin6", 2, 4))("b", inputs.Objective(11, 3, 1, np.zeros((1, 3), np.float32), np.zeros(1, np.float32), np.zeros(1, np.float32)), inputs.Hyper(3, 4, np.zeros(3, np.float32), np.ones(3, np.float32)), np.zeros((4, 3), np.float32)))


# ---- whole-cycle pins: the mode sets of these functions are known in closed form ---------------------------------
RUNS = {
    "rastrigin": dict(d=2, N=512, n_osc=4, n_conv=25, fd_h=1e-3, eps_grad=5e-3, eps_dup=0.1, log_delta=-200.0, sigma_s=0.5),
    "trid": dict(d=6, N=256, n_osc=2, n_conv=60, fd_h=1e-2, eps_grad=1e-2, eps_dup=0.2, log_delta=-1e9, sigma_s=3.0),
    "styblinski_tang": dict(d=4, N=512, n_osc=3, n_conv=30, fd_h=1e-3, eps_grad=5e-3, eps_dup=0.1, log_delta=-1e9, sigma_s=0.5),
    "schwefel": dict(d=2, N=512, n_osc=3, n_conv=30, fd_h=1e-2, eps_grad=1e-3, eps_dup=1.0, log_delta=-1e9, sigma_s=20.0),
}


def _run(orc, name):
    kw = dict(RUNS[name])
    wl = inputs.appendix_d(name, kw.pop("d"), kw.pop("N"), **kw)
    o = orc.Oracle(wl, threads=8)
    for _ in range(wl.hp.n_osc):
        o.step()
    return wl, o.modes()


def test_cycle_finds_all_121_rastrigin_maxima_in_2d(orc):
    """every local maximum of the 2-d Rastrigin function on [-5.12, 5.12]^2 sits next to a lattice point of
    {-5..5}^2 ("regular grid of local maxima"); the best one is the printed f(0) = 0"""
    _, (x, f, _) = _run(orc, "rastrigin")
    assert len(f) == 121 and abs(f[0]) < 1e-6 and np.max(np.abs(x[0])) < 1e-4
    cells = {tuple(np.rint(r).astype(int)) for r in x}
    assert len(cells) == 121 and np.max(np.abs(x - np.rint(x))) < 0.03


def test_cycle_collapses_trid_to_the_printed_optimum(orc):
    """Trid is unimodal: one mode at theta*_i = i (d + 1 - i), f* = d (d + 4)(d - 1)/6 = 50 at d = 6"""
    _, (x, f, _) = _run(orc, "trid")
    i = np.arange(1, 7)
    assert len(f) == 1 and abs(f[0] - 50.0) < 1e-6 and np.max(np.abs(x[0] - i * (7 - i))) < 1e-3


def test_cycle_finds_the_2_pow_d_styblinski_tang_maxima(orc):
    """separable with two maxima per coordinate (roots of 4 t^3 - 32 t + 5 with negative curvature of -f): 2^d modes"""
    _, (x, f, _) = _run(orc, "styblinski_tang")
    r = np.roots([4.0, 0.0, -32.0, 5.0]).real
    tops = np.sort(r)[[0, 2]]                                            # -2.9035 and 2.7468
    assert len(f) == 16
    assert np.max(np.min(np.abs(x[:, :, None] - tops[None, None, :]), axis=2)) < 1e-3
    assert abs(f[0] - 4 * 39.16616570377142) < 1e-5


def test_cycle_finds_the_schwefel_global_maximum(orc):
    _, (x, f, _) = _run(orc, "schwefel")
    assert abs(f[0]) < 1e-3 and np.max(np.abs(x[0] - 420.9687)) < 1e-2  # PAPER.md:619 "near theta_i = 420.97"
    assert len(f) > 20
