"""GPU <-> oracle parity on the Appendix-D benchmark functions, through the
C ABI: a1 (value + FD gradient) on seeded uniform populations over the printed domains, the printed optima, and
free-running cycles whose mode sets are known in closed form."""
import numpy as np
import pytest

from paper_2606_26164_b200 import inputs

import parity as PT
from test_oracle_appendix_d import RUNS

pytestmark = pytest.mark.gpu

# (function, d, N, fd_h): d spans the three padded widths (8 / 32 / 64) and ragged tails
A1 = [("rastrigin", 2, 300, 1e-3), ("rastrigin", 64, 261, 1e-3), ("ackley", 5, 300, 1e-3), ("ackley", 33, 130, 1e-3),
      ("schwefel", 2, 300, 1e-2), ("schwefel", 64, 140, 1e-2), ("styblinski_tang", 7, 300, 1e-3),
      ("styblinski_tang", 40, 130, 1e-3), ("michalewicz", 2, 300, 1e-3), ("michalewicz", 64, 140, 1e-3),
      ("trid", 6, 300, 1e-2), ("trid", 64, 140, 0.25), ("bukin6", 2, 515, 1e-3)]


@pytest.fixture(scope="module")
def B():
    from paper_2606_26164_b200 import binding
    binding.load_library()
    return binding


@pytest.mark.parametrize("name,d,N,h", A1)
def test_a1_value_and_fd_gradient(orc, B, name, d, N, h):
    wl = inputs.appendix_d(name, d, N, fd_h=h)
    o, g = orc.Oracle(wl, threads=8), B.Chisao(wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0]); g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL); g.phase(B.PH_RELEASE_EVAL)
    fo, fg = o.get(orc.F), g.get(B.F).astype(np.float64)
    assert np.all(np.abs(fg - fo) <= PT.f_tol(fo)), float(np.max(np.abs(fg - fo) / np.maximum(np.abs(fo), 1)))
    go, gg = o.get(orc.G), g.get(B.G).astype(np.float64)
    if name == "bukin6":   # the ridge y = 0.01 x^2 is a kink: compare stencils that do not straddle it
        x = wl.x0.astype(np.float64)
        keep = np.abs(x[:, 1] - 0.01 * x[:, 0] ** 2) > 0.05
        assert keep.sum() > 0.9 * N
        fo, go, gg = fo[keep], go[keep], gg[keep]
    ok, err, tol = PT.grad_ok(gg, go, fo, h)
    assert np.all(ok), (float(np.max(err / tol)), int(np.sum(~ok)))
    assert g.stats().evals[0] == N * (2 * wl.hp.d + 1)


def test_printed_optima_through_the_c_abi(orc, B):
    """the paper's printed optima evaluated by the CUDA evaluator (centre value of a release step)"""
    cases = [("rastrigin", 16, np.zeros(16), 0.0), ("ackley", 16, np.zeros(16), 0.0),
             ("schwefel", 16, np.full(16, 420.96875), 0.0), ("bukin6", 2, np.array([-10.0, 1.0]), 0.0),
             ("trid", 10, np.arange(1, 11) * (11.0 - np.arange(1, 11)), 10 * 14 * 9 / 6.0)]
    for name, d, xs, fs in cases:
        wl = inputs.appendix_d(name, d, 4)
        wl.x0[:] = xs.astype(np.float32)[None, :]
        g, o = B.Chisao(wl), orc.Oracle(wl)
        g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0]); o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
        g.phase(B.PH_RELEASE_EVAL); o.phase(orc.PH_RELEASE_EVAL)
        fg, fo = g.get(B.F).astype(np.float64), o.get(orc.F)
        assert np.all(np.abs(fg - fo) <= 1e-5 * max(abs(fs), 1.0)), (name, fg, fo)
        assert np.all(np.abs(fg - fs) <= 1e-3 * max(abs(fs), 1.0)), (name, fg)   # Schwefel's printed constant: ~2e-4 d


@pytest.mark.parametrize("name", ["rastrigin", "trid", "styblinski_tang", "schwefel"])
def test_free_running_cycles_recover_the_oracles_modes(orc, B, name):
    kw = dict(RUNS[name])
    wl = inputs.appendix_d(name, kw.pop("d"), kw.pop("N"), **kw)
    o, g = orc.Oracle(wl, threads=8), B.Chisao(wl)
    for _ in range(wl.hp.n_osc):
        o.step(); g.step()
    xo, fo, _ = o.modes()
    xg, fg, _, n = g.modes()
    scale = float(np.max(np.abs(wl.hp.hi)))
    tol = 1e-3 * max(1.0, scale / 5.0)                                   # 1e-3 L2 on a domain of width ~10 (north_star)
    both = PT.match_modes(xg, xo, tol)
    assert both >= 0.95 * max(n, len(fo)), (both, n, len(fo))
    assert abs(float(fg[0]) - fo[0]) <= 1e-4 * max(abs(fo[0]), 1.0)
    if name in ("rastrigin", "trid", "styblinski_tang"):
        assert n == len(fo) == {"rastrigin": 121, "trid": 1, "styblinski_tang": 16}[name]


def test_validation_of_appendix_d_objectives(B):
    wl = inputs.appendix_d("bukin6", 2, 8)
    wl3 = inputs.appendix_d("trid", 3, 8)
    wl3.obj.id = inputs.OBJ_BUKIN6
    with pytest.raises(B.ChisaoError) as ei:
        B.Chisao(wl3)
    assert ei.value.code == B.E_INVALID
    wl.obj.id = 12
    with pytest.raises(B.ChisaoError):
        B.Chisao(wl)
