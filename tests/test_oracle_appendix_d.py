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
