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


def test_full_size_c5_stick_dedup_reseed_teacher_forced(orc, B):
    """a3, a4, a5 at BASELINE.json's full C5 size (N = 65536, d = 64), teacher-forced from a seeded synthetic
    post-convergence state (inputs.synthetic_converged_state: ~34 000 samples in 300 tight clusters, exact f ties,
    gradient norms straddling eps_grad, non-finite entries): the ordered scan runs 64 blocks through the single-CTA
    offset kernel, k_dedup tiles ~30 000 stuck rows, k_reseed scores ~30 000 slots x 4 candidates against the modes.
    Flags, lists (through the counts and the removed mask), K_lost, reseed sources and candidates are compared
    exactly with the oracle on the same state; new rows by rule 4."""
    wl = inputs.config(5)
    hp = wl.hp
    N = hp.N
    x, f, gr = inputs.synthetic_converged_state(wl, frac_clustered=0.65)     # > 50 % of the population stuck in 300 clusters
    o, g = orc.Oracle(wl, threads=16), B.Chisao(wl)
    ctrl = [3, 1, 0, 0, 0, 0, 0, 0]
    for fo_, fg_, val in ((orc.X, B.X, x), (orc.F, B.F, f), (orc.G, B.G, gr), (orc.CTRL, B.CTRL, ctrl)):
        o.set(fo_, val); g.set(fg_, val)
    # a3: Eq. 3 on identical inputs -> identical flags (no arithmetic beyond comparisons of fp32 values)
    o.phase(orc.PH_STICK); g.phase(B.PH_STICK)
    so, sg = o.stats(), g.stats()
    assert sg.f_max == np.float32(so.f_max)
    assert np.array_equal(g.get(B.STUCK), o.get(orc.STUCK))
    assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
    assert 0.5 * N < sg.n_stuck < 40000 and not g.get(B.STUCK)[[5, 17, 33, 41]].any()
    # a4: Eq. 4, every pair decided by fp32 differences of fp32 coordinates on both sides; pairs whose L-inf distance is
    # within rounding of eps_dup are excluded (protocol rule 3)
    o.phase(orc.PH_DEDUP); g.phase(B.PH_DEDUP)
    so, sg = o.stats(), g.stats()
    rem_o, rem_g = o.get(orc.REMOVED).astype(bool), g.get(B.REMOVED).astype(bool)
    diff = np.flatnonzero(rem_o != rem_g)
    if len(diff):                                            # only threshold pairs may differ: check each of them
        st0 = np.flatnonzero(o.get(orc.STUCK).astype(bool) | rem_o)
        xs = x.astype(np.float64)
        for i in diff[:50]:
            D = np.max(np.abs(xs[st0] - xs[i][None, :]), axis=1)
            assert np.any(np.abs(D - hp.eps_dup) <= 1e-6 * 10.0), int(i)
    assert len(diff) <= max(2, 0.005 * sg.n_stuck), len(diff)
    if not len(diff):
        assert np.array_equal(g.get(B.STUCK), o.get(orc.STUCK))
        assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
        assert sg.k_lost > 20000 and 200 <= sg.n_stuck <= 2000
    # a5 from identical flags (the oracle's): Repulse Monkey on ~30 000 removed slots
    g.set(B.STUCK, o.get(orc.STUCK)); g.set(B.REMOVED, o.get(orc.REMOVED))
    if len(diff):
        g.phase(B.PH_DEDUP)                                  # rebuild the lists from the oracle's flags
        assert np.array_equal(g.get(B.REMOVED).astype(bool), rem_o)
    o.phase(orc.PH_RESEED); g.phase(B.PH_RESEED)
    so, sg = o.stats(), g.stats()
    assert sg.reseed_strategy == so.reseed_strategy == 1
    assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
    assert np.array_equal(g.get(B.RS_SRC), o.get(orc.RS_SRC))
    safe, n_other = PT.rm_candidates_ok(orc, o, g.get(B.RS_CAND), rem_o)
    print(f"C5 full size: {n_other} of {int(rem_o.sum())} Repulse-Monkey slots kept another candidate than the oracle's, all "
          f"scoring within 1e-5 of it")
    assert n_other <= 0.02 * rem_o.sum()     # d = 64: rays are short against the distance to the modes, the C candidates score alike
    xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
    tol = PT.x_tol(xo, hp.lo, hp.hi)
    assert np.all(np.max(np.abs(xg - xo), axis=1)[safe] <= tol[safe])
    assert np.array_equal(xg[~rem_o], x.astype(np.float64)[~rem_o])          # nobody else moves
    assert np.all(xg >= hp.lo[None, :]) and np.all(xg <= hp.hi[None, :])
    assert not g.get(B.REMOVED).any() and not g.get(B.STUCK)[rem_o].any()


@pytest.mark.parametrize("c,nrows", [(5, 40), (4, 64), (3, 96), (2, 256)])
def test_full_size_hlc_and_anti_steps_on_sampled_rows(orc, B, c, nrows):
    """a6, a7 at BASELINE.json's full sizes, in the launch configuration bench.py times, WITH the configured evaluation
    noise: the CUDA path runs the whole population (every 7th sample frozen); the oracle runs the same population with
    every row frozen except the sampled ones (phases 5-6 skip frozen rows; draws and noise are keyed
    by the sample index, so the sampled rows see the same Philox words on both sides).  Positions are re-synchronised
    oracle -> CUDA between the units (teacher forcing)."""
    wl = inputs.config(c)
    hp = wl.hp
    N, d = hp.N, hp.d
    rng = np.random.default_rng(100 + c)
    rows = np.sort(np.concatenate([rng.choice(N - 2, nrows - 2, replace=False), [N - 2, N - 1]]))
    stuck_g = np.zeros(N, np.uint8); stuck_g[::7] = 1; stuck_g[rows] = 0
    stuck_o = np.ones(N, np.uint8); stuck_o[rows] = 0
    o, g = orc.Oracle(wl, threads=16), B.Chisao(wl)
    ctrl = [2, 1, 0, 0, 0, 0, 0, 0]
    o.set(orc.CTRL, ctrl); g.set(B.CTRL, ctrl)
    o.set(orc.STUCK, stuck_o); g.set(B.STUCK, stuck_g)
    x0 = wl.x0.astype(np.float64)
    # a6: one Hands-Like-Clouds step
    o.phase(orc.PH_HLC_STEP, 1); g.phase(B.PH_HLC_STEP, 1)
    fo, fg = o.get(orc.HLC_F)[rows], g.get(B.HLC_F)[rows].astype(np.float64)
    assert np.all(np.abs(fg - fo) <= PT.F_REL * np.maximum(np.abs(fo), 1.0)), float(np.max(np.abs(fg - fo) / np.maximum(np.abs(fo), 1.0)))
    gho, ghg = o.get(orc.GHAT)[rows], g.get(B.GHAT)[rows].astype(np.float64)
    floor = 8 * PT.EPS32 * np.max(np.abs(fo), axis=1) * 5.5 / hp.sigma_s
    err = np.max(np.abs(ghg - gho), axis=1)
    tol = PT.G_REL * np.max(np.abs(gho), axis=1) + floor
    assert np.all(err <= tol), float(np.max(err / tol))
    xo_all = o.get(orc.X)
    xo, xg = xo_all[rows], g.get(B.X).astype(np.float64)
    step = np.max(np.abs(xo - x0[rows]), axis=1)
    xt = PT.x_tol(xo, hp.lo, hp.hi, step, grad_inside=True) + hp.eta_hlc * floor
    assert np.all(np.max(np.abs(xg[rows] - xo), axis=1) <= xt)
    frozen = stuck_g.astype(bool)
    assert np.array_equal(xg[frozen], x0[frozen])                            # frozen rows bit-identical
    assert g.stats().evals[5] == int((stuck_g == 0).sum()) * hp.hlc_M
    # a7: two anti-convergence steps from the oracle's positions
    xs = g.get(B.X); xs[rows] = xo.astype(np.float32)
    g.set(B.X, xs)
    for t in (1, 2):
        v0 = o.get(orc.V)[rows].copy(); xb = o.get(orc.X)[rows].copy()
        o.phase(orc.PH_ANTI_STEP, t); g.phase(B.PH_ANTI_STEP, t)
        vo, vg = o.get(orc.V)[rows], g.get(B.V)[rows].astype(np.float64)
        xo, xg = o.get(orc.X)[rows], g.get(B.X).astype(np.float64)
        vprev = np.zeros_like(v0) if t == 1 else v0
        g_used = (hp.mu * vprev - vo) / hp.alpha_anti
        floor = PT.fd_floor(np.abs(o.values(xb)), hp.fd_h, wl.obj.sigma_noise) * 4
        vtol = hp.alpha_anti * (PT.G_REL * np.max(np.abs(g_used), axis=1) + floor) + 4 * PT.EPS32 * np.max(np.abs(vo), axis=1)
        ev = np.max(np.abs(vg - vo), axis=1)
        assert np.all(ev <= vtol), (t, float(np.max(ev / vtol)))
        assert np.all(np.max(np.abs(xg[rows] - xo), axis=1) <= PT.x_tol(xo, hp.lo, hp.hi) + vtol)
        assert np.array_equal(xg[frozen], x0[frozen])                        # "Stuck samples are excluded" PAPER.md:129
        xs = g.get(B.X); xs[rows] = xo.astype(np.float32); g.set(B.X, xs)
        vs = g.get(B.V); vs[rows] = vo.astype(np.float32); g.set(B.V, vs)
    assert g.stats().evals[6] == 2 * int((stuck_g == 0).sum()) * 2 * d
