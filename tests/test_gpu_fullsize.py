"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times: the CUDA path runs the
whole population; outputs of sampled rows are recomputed one by one by the oracle from the same inputs."""
import numpy as np
import pytest

from paper_2606_26164_b200 import inputs

import parity as PT

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_26164_b200 import binding
    binding.load_library()
    return binding


def _subset_oracle(orc, wl, rows, x_rows):
    """an oracle over the sampled rows only (noise-free runs: draws are keyed by sample index)"""
    sub = inputs.config(int(wl.name[1:]), N=len(rows), noise=0.0)
    sub.hp = type(wl.hp)(**{**wl.hp.__dict__, "N": len(rows)})
    sub.x0 = np.ascontiguousarray(x_rows, np.float32)
    return orc.Oracle(sub, threads=8)


@pytest.mark.parametrize("c,nrows", [(5, 48), (4, 64), (3, 96), (2, 256)])
def test_full_size_eval_and_lbfgs_iteration_on_sampled_rows(orc, B, c, nrows):
    wl = inputs.config(c, noise=0.0)
    hp = wl.hp
    N = hp.N
    g = B.Chisao(wl)
    g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    g.phase(B.PH_RELEASE_EVAL)
    rng = np.random.default_rng(c)
    rows = np.sort(np.concatenate([rng.choice(N - 2, nrows - 2, replace=False), [N - 2, N - 1]]))  # incl. the tail tile
    x = g.get(B.X)
    o = _subset_oracle(orc, wl, rows, x[rows])
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    fo, fg = o.get(orc.F), g.get(B.F)[rows].astype(np.float64)
    assert np.all(np.abs(fg - fo) <= PT.f_tol(fo))
    ok, err, tol = PT.grad_ok(g.get(B.G)[rows].astype(np.float64), o.get(orc.G), fo, hp.fd_h)
    assert np.all(ok), float(np.max(err / tol))
    assert g.stats().evals[0] == N * (2 * hp.d + 1)
    # three L-BFGS iterations at full N; the third is checked on the sampled rows from the GPU's own state
    g.phase(B.PH_LBFGS_ITER, 1); g.phase(B.PH_LBFGS_ITER, 2)
    S, Y = g.get(B.HIST_S)[:, rows], g.get(B.HIST_Y)[:, rows]
    for fo_, fg_ in ((orc.X, B.X), (orc.F, B.F), (orc.G, B.G)):
        o.set(fo_, g.get(fg_)[rows].astype(np.float64))
    o.set(orc.HIST_S, S.astype(np.float64)); o.set(orc.HIST_Y, Y.astype(np.float64))
    o.set(orc.HIST_LEN, g.get(B.HIST_LEN)[rows]); o.set(orc.STALLED, g.get(B.STALLED)[rows])
    g.phase(B.PH_LBFGS_ITER, 3); o.phase(orc.PH_LBFGS_ITER, 3)
    safe = (o.get(orc.LS_MARGIN) > PT.LS_MARGIN_MIN) & (o.get(orc.ASC_MARGIN) > PT.REL_MARGIN_MIN)
    assert safe.sum() >= 0.9 * nrows
    assert np.array_equal(g.get(B.LS_B)[rows][safe], o.get(orc.LS_B)[safe])
    po, pg = o.get(orc.P), g.get(B.P)[rows].astype(np.float64)
    assert np.all(np.linalg.norm(pg - po, axis=1)[safe] <= 1e-4 * np.linalg.norm(po, axis=1)[safe] + 1e-30)
    xo = o.get(orc.X)
    assert np.all(np.max(np.abs(g.get(B.X)[rows] - xo), axis=1)[safe] <= PT.x_tol(xo, hp.lo, hp.hi)[safe])
    # properties that hold at any size
    xg = g.get(B.X)
    assert np.isfinite(xg).all() and np.all(xg >= hp.lo[None, :]) and np.all(xg <= hp.hi[None, :])
    ln = g.get(B.HIST_LEN)
    assert ln.min() >= 0 and ln.max() <= min(3, hp.lbfgs_m)


def test_full_size_c5_cycle_with_noise_invariants(B):
    """one complete noisy C5 cycle at N = 65536: counts are consistent, frozen rows do not move."""
    wl = inputs.config(5, n_osc=3)
    hp = wl.hp
    g = B.Chisao(wl)
    st = g.step()
    assert st.n_stuck + st.n_active == hp.N and st.k_lost >= 0
    ev = list(st.evals)
    assert ev[0] == hp.N * (2 * hp.d + 1)
    assert ev[2] % (2 * hp.d) == 0 and ev[1] >= ev[2] // (2 * hp.d)
    assert ev[5] == hp.n_cloud * hp.hlc_M * st.n_active and ev[6] == hp.n_anti * 2 * hp.d * st.n_active
    x = g.get(B.X)
    assert np.isfinite(x).all() and np.all(np.abs(x) <= 10.0)
