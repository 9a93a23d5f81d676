"""GPU <-> oracle parity, teacher-forced per phase; all calls go through
the C ABI (paper_2606_26164_b200.binding -> libchisao.so).  Sizes span several 256-point tiles and a ragged
tail; C1..C5 are BASELINE.json's configs at reduced N (the full-size checks are in test_gpu_fullsize.py)."""
import numpy as np
import pytest

from paper_2606_26164_b200 import inputs

import parity as PT

pytestmark = pytest.mark.gpu

CASES = [(1, 256), (2, 777), (3, 300), (4, 261), (5, 200)]


@pytest.fixture(scope="module")
def B():
    from paper_2606_26164_b200 import binding
    binding.load_library()
    return binding


def _pair(orc, B, wl):
    return orc.Oracle(wl, threads=8), B.Chisao(wl)


@pytest.mark.parametrize("c,N", CASES)
def test_a1_eval_and_fd_gradient(orc, B, c, N):
    """a1: f within 1e-5 relative, FD gradient within 1e-3 relative + fp32 floor (north_star)."""
    wl = inputs.config(c, N=N)
    o, g = _pair(orc, B, wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0]); g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL); g.phase(B.PH_RELEASE_EVAL)
    fo, fg = o.get(orc.F), g.get(B.F).astype(np.float64)
    assert np.all(np.abs(fg - fo) <= PT.f_tol(fo)), float(np.max(np.abs(fg - fo) / np.maximum(np.abs(fo), 1)))
    ok, err, tol = PT.grad_ok(g.get(B.G).astype(np.float64), o.get(orc.G), fo, wl.hp.fd_h, wl.obj.sigma_noise)
    assert np.all(ok), (float(np.max(err / tol)), int(np.sum(~ok)))
    # release: flags and history cleared; evaluation counter = N (2d + 1)   (Eq. 8 structure)
    assert not g.get(B.STUCK).any() and not g.get(B.HIST_LEN).any()
    assert g.stats().evals[0] == N * (2 * wl.hp.d + 1) == o.stats().evals[0]


@pytest.mark.parametrize("c,N", CASES)
def test_a2_lbfgs_iterations_teacher_forced(orc, B, c, N, resident=None, wl=None, n_it=8):
    """a2: direction, accepted trial, updated position, curvature pair, history bookkeeping, per iteration.  C1 and C2 run
    Phase 1 in its history-resident form (one launch, (s, y) in registers) by default; `resident` forces a form."""
    if wl is None:
        wl = inputs.config(c, N=N)
    hp = wl.hp
    o, g = _pair(orc, B, wl)
    if resident is not None:
        g.set_option(B.OPT_LBFGS_RESIDENT, int(resident))
    if c:
        assert g.lbfgs_resident() == ((c in (1, 2)) if resident is None else resident)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    n_dec = n_excl = 0
    for it in range(1, min(hp.n_conv, n_it) + 1):
        PT.sync_oracle_to_gpu(o, g, orc, B)
        x0 = o.get(orc.X).copy(); len0 = o.get(orc.HIST_LEN).copy(); f0 = o.get(orc.F).copy()
        o.phase(orc.PH_LBFGS_ITER, it); g.phase(B.PH_LBFGS_ITER, it)
        bo, bg = o.get(orc.LS_B), g.get(B.LS_B)
        po, pg = o.get(orc.P), g.get(B.P).astype(np.float64)
        active = bo != -2
        assert np.array_equal(bg == -2, ~active)           # skip decisions (Eq. 3 gradient test on equal inputs)
        # direction: ||dp||_2 <= 1e-4 ||p||_2 wherever the ascent test is not marginal
        safe_dir = active & (o.get(orc.ASC_MARGIN) > PT.REL_MARGIN_MIN)
        dn = np.linalg.norm(pg - po, axis=1); pn = np.linalg.norm(po, axis=1)
        assert np.all(dn[safe_dir] <= 1e-4 * pn[safe_dir] + 1e-30), float(np.max(dn[safe_dir] / (pn[safe_dir] + 1e-30)))
        # accepted trial index: exact away from the Armijo threshold
        safe = safe_dir & (o.get(orc.LS_MARGIN) > PT.LS_MARGIN_MIN)
        n_dec += int(active.sum()); n_excl += int((active & ~safe).sum())
        assert np.array_equal(bg[safe], bo[safe]), int(np.sum(bg[safe] != bo[safe]))
        # updated position (rule 4) and value
        xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
        tol = PT.x_tol(xo, hp.lo, hp.hi)
        ex = np.max(np.abs(xg - xo), axis=1)
        assert np.all(ex[safe] <= tol[safe]), float(np.max(ex[safe] / tol[safe]))
        assert np.array_equal(xg[~active], x0[~active])
        fo, fg = o.get(orc.F), g.get(B.F).astype(np.float64)
        acc = safe & (bo >= 0)
        assert np.all(np.abs(fg - fo)[acc] <= 2 * PT.f_tol(fo)[acc])
        assert np.array_equal(fg[safe & (bo < 0)], f0[safe & (bo < 0)])
        # new gradient at the accepted point
        ok, err, gtol = PT.grad_ok(g.get(B.G).astype(np.float64), o.get(orc.G), fo, hp.fd_h, wl.obj.sigma_noise)
        assert np.all(ok[acc]), float(np.max(err[acc] / gtol[acc]))
        # history: length exact away from the curvature threshold; newest pair values
        safe_h = acc & (o.get(orc.CURV_MARGIN) > PT.REL_MARGIN_MIN)
        lo_, lg_ = o.get(orc.HIST_LEN), g.get(B.HIST_LEN)
        assert np.array_equal(lg_[safe_h], lo_[safe_h])
        assert np.array_equal(lg_[safe & (bo < 0)], lo_[safe & (bo < 0)])
        So, Sg = o.get(orc.HIST_S), g.get(B.HIST_S).astype(np.float64)
        Yo, Yg = o.get(orc.HIST_Y), g.get(B.HIST_Y).astype(np.float64)
        rows = np.nonzero(safe_h & (lo_ > 0))[0]
        if len(rows):
            newest = lo_[rows] - 1
            so, sg = So[newest, rows], Sg[newest, rows]
            yo, yg = Yo[newest, rows], Yg[newest, rows]
            assert np.all(np.max(np.abs(sg - so), axis=1) <= 2 * tol[rows])
            ytol = PT.G_REL * np.max(np.abs(yo), axis=1) + 2 * gtol[rows] + 2e-3 * np.max(np.abs(o.get(orc.G)[rows]), axis=1)
            assert np.all(np.max(np.abs(yg - yo), axis=1) <= ytol)
        assert np.array_equal(g.get(B.STALLED)[safe], o.get(orc.STALLED)[safe])
        assert np.all(len0[~active] == lg_[~active])
    # decisions inside the fp32 uncertainty band are counted, not compared, and their share is capped (protocol rule 3:
    # 0.5 % of the decisions).  C1 alone gets 5 %: its samples converge within these 8 iterations, and a nearly converged
    # sample's decrease per step is below the fp32 resolution of f (2e-5 relative on the Armijo difference), so its
    # decisions sit inside the band by construction (measured counts: DESIGN.md section 5).
    cap = 0.05 if c == 1 else (0.01 if c == 0 else PT.MAX_EXCLUDED_FRACTION)   # (custom small workloads: a few hundred decisions)
    print(f"C{c}: {n_excl} of {n_dec} L-BFGS decisions inside the fp32 band ({n_excl / max(n_dec, 1):.4%}, cap {cap:.1%})")
    assert n_excl <= max(2, cap * n_dec), (n_excl, n_dec)


@pytest.mark.parametrize("kind,d,N,m", [("quad", 64, 203, 4), ("quad", 48, 157, 4), ("quad", 64, 130, 16), ("gmm_full", 40, 300, 6),
                                        ("gmm_full", 64, 99, 10)])
def test_a2_wrapped_rings_on_the_quad_step_kernel(orc, B, kind, d, N, m):
    """The four-lanes-per-sample form of the two-loop kernel (32 < d <= 64, d % 4 = 0: k_lbfgs_step_quad) under the a2
    protocol for MORE iterations than the history holds: rings wrap (head != 0, the oldest pair dropped), N is not a
    multiple of the eight samples of a tile, d = 48 / 40 take the predicated (non-64) chunk path, m = 4 / 6 / 16 the other
    instantiations; samples go stationary on the way, so partly active tiles (copies per sample and row) occur too."""
    if kind == "quad":
        obj = inputs.quad(d, 500 + d, lam_max=30.0)
        wl = inputs.custom(obj, 4.0, N, seed=40 + d + m, fd_h=1e-2, eps_grad=0.5, n_conv=14, lbfgs_m=m)
    else:
        obj = inputs.gmm_full(d, 3, 3.0, 77 + d)
        wl = inputs.custom(obj, 4.0, N, seed=40 + d + m, fd_h=1e-2, eps_grad=0.5, n_conv=14, lbfgs_m=m)
    test_a2_lbfgs_iterations_teacher_forced(orc, B, 0, N, wl=wl, n_it=14 if m < 14 else 8)


@pytest.mark.parametrize("kind,d,N,m", [("gmm_full", 40, 400, 4), ("quad", 64, 300, 4), ("gmm_full", 64, 250, 6)])
def test_fused_quad_step_kernel_inside_a_cycle_follows_the_unit_sequence(B, kind, d, N, m):
    """Inside chisao_step the iterations it > m of a pass run the quad step kernel with the update of iteration it - 1 fused
    in front (the pair it stores goes to HBM and, from registers, into the shared-memory copy of the history); iterations
    2 .. m run the half-warp form with the history staged through shared memory.  The unit sequence chisao_phase runs
    (RELEASE_EVAL, n_conv x LBFGS_ITER, STICK) uses the stand-alone forms (direction kernel, separate update kernel), which
    the a2 tests compare with the oracle step by step.  Same evaluator, same line search, fp32 on both sides: the two
    Phase-1 passes differ by the summation order of a few dots, so after n_conv = 14 iterations (m = 4 / 6: wrapped rings)
    positions, values and flags agree closely -- a wrong row, plane or pair in the fused kernel would not."""
    if kind == "quad":
        wl = inputs.custom(inputs.quad(d, 600 + d, lam_max=30.0), 4.0, N, seed=50 + d, fd_h=1e-2, eps_grad=0.05, n_conv=14,
                           lbfgs_m=m, n_osc=3, phase_mask=0)
    else:
        wl = inputs.custom(inputs.gmm_full(d, 3, 3.0, 88 + d), 4.0, N, seed=50 + d, fd_h=1e-2, eps_grad=1e-2, n_conv=14,
                           lbfgs_m=m, n_osc=3, phase_mask=0)
    hp = wl.hp
    a, b = B.Chisao(wl), B.Chisao(wl)
    sa = a.step()                                            # phases 1-2 of cycle 1 (phases 3-6 masked off)
    b.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    b.phase(B.PH_RELEASE_EVAL)
    for it in range(1, hp.n_conv + 1):
        b.phase(B.PH_LBFGS_ITER, it)
    b.phase(B.PH_STICK)
    sb = b.stats()
    xa, xb = a.get(B.X).astype(np.float64), b.get(B.X).astype(np.float64)
    fa, fb = a.get(B.F).astype(np.float64), b.get(B.F).astype(np.float64)
    dx = np.max(np.abs(xa - xb), axis=1)
    close = dx <= 1e-3 * 4.0
    assert close.mean() >= 0.95, (float(close.mean()), float(np.max(dx)))   # (a differing Armijo decision sends a sample elsewhere for a while)
    assert np.all(np.abs(fa - fb)[close] <= 5e-3 * np.maximum(np.abs(fb[close]), 1.0))   # (|grad f| up to ~1 at these points, dx up to 4e-3)
    assert np.array_equal(a.get(B.HIST_LEN)[close] > 0, b.get(B.HIST_LEN)[close] > 0)
    assert int(a.get(B.HIST_LEN).max()) == m                 # the rings did fill
    assert abs(sa.n_stuck - sb.n_stuck) <= max(2, 0.02 * N), (sa.n_stuck, sb.n_stuck)
    assert abs(sa.f_max - sb.f_max) <= 1e-4 * max(abs(sb.f_max), 1.0)
    assert list(sa.evals)[0] == list(sb.evals)[0]


def _converged_pair(orc, B, wl, n_conv=None):
    o, g = _pair(orc, B, wl)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL)
    for it in range(1, (n_conv or wl.hp.n_conv) + 1):
        o.phase(orc.PH_LBFGS_ITER, it)
    return o, g


@pytest.mark.parametrize("c,N,n_conv", [(1, 256, 20), (2, 777, 10), (3, 300, 120), (5, 200, 18), (4, 130, 5)])
def test_a3_stick_and_a4_dedup(orc, B, c, N, n_conv):
    """a3: f_max, Eq. 3 flags exact away from the thresholds; a4: Eq. 4 removed mask, K_lost, counts."""
    wl = inputs.config(c, N=N)
    hp = wl.hp
    o, g = _converged_pair(orc, B, wl, n_conv)
    PT.sync_oracle_to_gpu(o, g, orc, B)
    o.phase(orc.PH_STICK); g.phase(B.PH_STICK)
    so, sg = o.stats(), g.stats()
    assert abs(sg.f_max - so.f_max) <= 1e-5 * max(abs(so.f_max), 1.0)
    fo, go = o.get(orc.F), o.get(orc.G)
    ginf = np.max(np.abs(go), axis=1)
    thr = so.f_max + hp.log_delta
    near = (np.abs(ginf - hp.eps_grad) <= 1e-6 * ginf) | (np.abs(fo - thr) <= 2e-5 * np.maximum(np.abs(fo), 1.0))
    assert near.sum() <= max(2, 0.005 * N)
    assert np.array_equal(g.get(B.STUCK)[~near], o.get(orc.STUCK)[~near])
    if not near.any():
        assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
    # dedup from identical flags
    g.set(B.STUCK, o.get(orc.STUCK))
    o.phase(orc.PH_DEDUP); g.phase(B.PH_DEDUP)
    so, sg = o.stats(), g.stats()
    x = o.get(orc.X); st0 = (o.get(orc.STUCK) | o.get(orc.REMOVED)).astype(bool)
    # pairs whose L-inf distance is within fp32 rounding of eps_dup are not required to agree
    idx = np.nonzero(st0)[0]
    amb = np.zeros(N, bool)
    if len(idx):
        D = np.max(np.abs(x[idx][:, None, :] - x[idx][None, :, :]), axis=2)
        amb[idx] = np.any(np.abs(D - hp.eps_dup) <= 1e-6 * max(1.0, float(np.abs(x).max())), axis=1)
    assert np.array_equal(g.get(B.REMOVED)[~amb], o.get(orc.REMOVED)[~amb])
    assert np.array_equal(g.get(B.STUCK)[~amb], o.get(orc.STUCK)[~amb])
    if not amb.any():
        assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
        assert sg.n_stuck + sg.k_lost == int(st0.sum())


def test_a4_dedup_many_duplicates_and_ties(orc, B):
    """dense duplicate clusters, exact f ties (lower index survives), phase mask off removes nothing (R-7)."""
    obj = inputs.gmm_iso(3, 2, 0.5, 2.0, 5)
    wl = inputs.custom(obj, 3.0, 1500, eps_dup=0.05, eps_grad=1.0)
    o, g = _pair(orc, B, wl)
    rng = np.random.default_rng(3)
    centres = rng.uniform(-2.5, 2.5, size=(12, 3))
    x = PT.f32(centres[rng.integers(0, 12, 1500)] + rng.uniform(-0.02, 0.02, size=(1500, 3)))
    f = PT.f32(np.round(rng.standard_normal(1500), 1))          # many exact ties
    stuck = (rng.uniform(size=1500) < 0.8).astype(np.uint8)
    for fld_o, fld_g, val in ((orc.X, B.X, x), (orc.F, B.F, f), (orc.STUCK, B.STUCK, stuck)):
        o.set(fld_o, val); g.set(fld_g, val)
    o.phase(orc.PH_DEDUP); g.phase(B.PH_DEDUP)
    assert np.array_equal(g.get(B.REMOVED), o.get(orc.REMOVED))
    assert np.array_equal(g.get(B.STUCK), o.get(orc.STUCK))
    so, sg = o.stats(), g.stats()
    assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
    assert sg.k_lost > 500
    # survivors are pairwise >= eps_dup apart (invariant) and a second application removes nothing
    surv = x[g.get(B.STUCK).astype(bool)]
    D = np.max(np.abs(surv[:, None, :] - surv[None, :, :]), axis=2) + np.eye(len(surv))
    assert D.min() >= 0.05
    g.phase(B.PH_DEDUP)
    assert g.stats().k_lost == 0


@pytest.mark.parametrize("strategy", [1, 2, 3])
def test_a5_reseed_via_dedup(orc, B, strategy):
    """a5 through the real pipeline: a crafted stuck set with duplicates -> DEDUP -> RESEED on both sides."""
    obj = inputs.gmm_diag(8, 16, 5.0, 1002)
    wl = inputs.custom(obj, 5.0, 640, eps_dup=0.05, eps_grad=1.0, reseed_cands=4, seed=77)
    hp = wl.hp
    o, g = _pair(orc, B, wl)
    N, d = 640, 8
    rng = np.random.default_rng(20 + strategy)
    centres = rng.uniform(-4.5, 4.5, size=(25, d))
    x = PT.f32(rng.uniform(-5, 5, size=(N, d)))
    stuck = np.zeros(N, np.uint8)
    n_dup = 200 if strategy == 1 else N - 3
    dup = rng.choice(N, n_dup, replace=False)
    x[dup] = PT.f32(centres[rng.integers(0, 25, n_dup)] + rng.uniform(-0.01, 0.01, size=(n_dup, d)))
    stuck[dup] = 1
    f = PT.f32(rng.standard_normal(N))
    ctrl = [2, 1 if strategy != 3 else 0, 0, 0, 0, 0, int(stuck.sum()), N - int(stuck.sum())]
    for fo, fg, val in ((orc.X, B.X, x), (orc.F, B.F, f), (orc.STUCK, B.STUCK, stuck), (orc.CTRL, B.CTRL, ctrl)):
        o.set(fo, val); g.set(fg, val)
    g.set(B.V, np.ones((N, d), np.float32)); o.set(orc.V, np.ones((N, d)))
    g.set(B.HIST_LEN, np.full(N, 2, np.int32)); o.set(orc.HIST_LEN, np.full(N, 2, np.int32))
    o.phase(orc.PH_DEDUP); g.phase(B.PH_DEDUP)
    removed = o.get(orc.REMOVED).astype(bool)
    assert np.array_equal(g.get(B.REMOVED).astype(bool), removed)
    o.phase(orc.PH_RESEED); g.phase(B.PH_RESEED)
    so, sg = o.stats(), g.stats()
    assert sg.reseed_strategy == so.reseed_strategy == strategy
    assert (sg.n_stuck, sg.k_lost, sg.n_active) == (so.n_stuck, so.k_lost, so.n_active)
    src_o, src_g = o.get(orc.RS_SRC), g.get(B.RS_SRC)
    assert np.array_equal(src_g, src_o)
    if strategy == 1:
        safe, n_other = PT.rm_candidates_ok(orc, o, g.get(B.RS_CAND), removed)
        print(f"RM: {n_other} of {int(removed.sum())} slots kept another candidate than the oracle's (all within 1e-5 of its score)")
        assert n_other <= max(2, 0.01 * removed.sum())       # protocol rule 3 (d = 8)
    else:
        safe = removed
        assert np.array_equal(g.get(B.RS_CAND)[safe], o.get(orc.RS_CAND)[safe])
    xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
    tol = PT.x_tol(xo, hp.lo, hp.hi)
    assert np.all(np.max(np.abs(xg - xo), axis=1)[safe] <= tol[safe])
    assert np.array_equal(xg[~removed], x[~removed])                       # nobody else moves
    assert np.all(xg >= hp.lo[None, :]) and np.all(xg <= hp.hi[None, :])   # inside Theta
    assert not g.get(B.REMOVED).any() and not g.get(B.STUCK)[removed].any()  # "marked as unstuck" PAPER.md:111
    assert not g.get(B.HIST_LEN)[removed].any() and not g.get(B.V)[removed].any()
    assert np.all(g.get(B.HIST_LEN)[~removed] == 2)
    if strategy == 2:
        Q = g.get(B.GR_Q).astype(np.float64)
        assert np.allclose(Q.T @ Q, np.eye(d), atol=5e-6)
        assert np.allclose(Q, o.gr_basis(2), atol=2e-5)


@pytest.mark.parametrize("c,N,baseline", [(1, 256, 1), (2, 500, 1), (3, 300, 1), (4, 140, 1), (5, 150, 1), (2, 300, 0), (5, 150, 0)])
def test_a6_hlc_step(orc, B, c, N, baseline):
    """a6: every f_k within 1e-5 relative, ghat within 1e-3 relative + floor, x by rule 4; stuck rows frozen."""
    wl = inputs.config(c, N=N, hlc_baseline=baseline)
    hp = wl.hp
    o, g = _converged_pair(orc, B, wl, 3)
    o.phase(orc.PH_STICK)
    stuck = o.get(orc.STUCK).copy(); stuck[::7] = 1            # make sure some rows are frozen
    o.set(orc.STUCK, stuck)
    for t in (1, 2):
        PT.sync_oracle_to_gpu(o, g, orc, B, with_history=False)
        x0 = o.get(orc.X).copy()
        o.phase(orc.PH_HLC_STEP, t); g.phase(B.PH_HLC_STEP, t)
        act = stuck == 0
        fo, fg = o.get(orc.HLC_F), g.get(B.HLC_F).astype(np.float64)
        assert np.all(np.abs(fg - fo)[act] <= PT.F_REL * np.maximum(np.abs(fo[act]), 1.0))
        gho, ghg = o.get(orc.GHAT), g.get(B.GHAT).astype(np.float64)
        u_inf = 5.5
        floor = 8 * PT.EPS32 * np.max(np.abs(fo), axis=1) * u_inf / hp.sigma_s
        err = np.max(np.abs(ghg - gho), axis=1)
        tol = PT.G_REL * np.max(np.abs(gho), axis=1) + floor
        assert np.all(err[act] <= tol[act]), float(np.max(err[act] / tol[act]))
        xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
        step = np.max(np.abs(xo - x0), axis=1)
        xt = PT.x_tol(xo, hp.lo, hp.hi, step, grad_inside=True) + hp.eta_hlc * floor
        assert np.all(np.max(np.abs(xg - xo), axis=1)[act] <= xt[act])
        assert np.array_equal(xg[~act], x0[~act])              # frozen rows bit-identical
    assert g.stats().evals[5] == 2 * int((stuck == 0).sum()) * hp.hlc_M


@pytest.mark.parametrize("c,N", [(1, 256), (2, 500), (3, 300), (4, 140), (5, 150)])
def test_a7_anti_convergence_step(orc, B, c, N):
    """a7: Eq. 6 with the FD gradient computed inside the unit; v and x; stuck rows frozen."""
    wl = inputs.config(c, N=N)
    hp = wl.hp
    o, g = _converged_pair(orc, B, wl, 3)
    o.phase(orc.PH_STICK)
    stuck = o.get(orc.STUCK).copy(); stuck[::5] = 1
    o.set(orc.STUCK, stuck)
    act = stuck == 0
    for t in (1, 2, 3):
        PT.sync_oracle_to_gpu(o, g, orc, B, with_history=False)
        x0 = o.get(orc.X).copy(); v0 = o.get(orc.V).copy()
        o.phase(orc.PH_ANTI_STEP, t); g.phase(B.PH_ANTI_STEP, t)
        vo, vg = o.get(orc.V), g.get(B.V).astype(np.float64)
        xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
        # the gradient inside the step: recover it from the oracle's update for the tolerance
        vprev = np.zeros_like(v0) if t == 1 else v0
        g_used = (hp.mu * vprev - vo) / hp.alpha_anti
        f_here = np.abs(o.get(orc.F))
        floor = PT.fd_floor(f_here, hp.fd_h, wl.obj.sigma_noise) * 4
        vtol = hp.alpha_anti * (PT.G_REL * np.max(np.abs(g_used), axis=1) + floor) + 4 * PT.EPS32 * np.max(np.abs(vo), axis=1)
        assert np.all(np.max(np.abs(vg - vo), axis=1)[act] <= vtol[act]), float(np.max((np.max(np.abs(vg - vo), axis=1) / vtol)[act]))
        xt = PT.x_tol(xo, hp.lo, hp.hi) + vtol
        assert np.all(np.max(np.abs(xg - xo), axis=1)[act] <= xt[act])
        assert np.array_equal(xg[~act], x0[~act])              # "Stuck samples are excluded" PAPER.md:129
    assert g.stats().evals[6] == 3 * int(act.sum()) * 2 * hp.d


@pytest.mark.parametrize("c,N,M", [(2, 300, 6), (3, 130, 3), (5, 70, 3), (1, 256, 10)])
def test_a6_hlc_step_paper_form_eq5(orc, B, c, N, M):
    """NEXT-2: Hands Like Clouds as the paper writes it (Eq. 5): mean of M finite-difference gradients
    at Gaussian-perturbed points (hlc_baseline = 2): ghat within 1e-3 relative + FD floor, x by rule 4, stuck rows
    frozen, M 2d evaluations per active sample."""
    wl = inputs.config(c, N=N, hlc_baseline=2, hlc_M=M)
    hp = wl.hp
    o, g = _converged_pair(orc, B, wl, 2)
    o.phase(orc.PH_STICK)
    stuck = o.get(orc.STUCK).copy(); stuck[::6] = 1
    o.set(orc.STUCK, stuck)
    act = stuck == 0
    PT.sync_oracle_to_gpu(o, g, orc, B, with_history=False)
    x0 = o.get(orc.X).copy()
    o.phase(orc.PH_HLC_STEP, 2); g.phase(B.PH_HLC_STEP, 2)
    gho, ghg = o.get(orc.GHAT), g.get(B.GHAT).astype(np.float64)
    floor = PT.fd_floor(np.abs(o.get(orc.F)) + 50.0 * hp.sigma_s ** 2, hp.fd_h, wl.obj.sigma_noise) * 4
    err = np.max(np.abs(ghg - gho), axis=1)
    tol = PT.G_REL * np.max(np.abs(gho), axis=1) + floor
    assert np.all(err[act] <= tol[act]), float(np.max(err[act] / tol[act]))
    xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
    xt = PT.x_tol(xo, hp.lo, hp.hi) + hp.eta_hlc * tol
    assert np.all(np.max(np.abs(xg - xo), axis=1)[act] <= xt[act])
    assert np.array_equal(xg[~act], x0[~act])
    assert g.stats().evals[5] == int(act.sum()) * M * 2 * hp.d == o.stats().evals[5]


@pytest.mark.parametrize("c,N,form", [(2, 500, 1), (5, 150, 1), (3, 200, 2)])
def test_a6_hlc_sigma_auto_estimate(orc, B, c, N, form):
    """NEXT-4 / PAPER.md:120: sigma = c std({x_i : not stuck_i}) (sigma_s = -0.1 selects c = 0.1; R-18): the scale
    matches the oracle to fp32 rounding, and the step taken with it stays within the HLC tolerances."""
    wl = inputs.config(c, N=N, sigma_s=-0.1, hlc_baseline=form, hlc_M=8)
    hp = wl.hp
    o, g = _converged_pair(orc, B, wl, 2)
    o.phase(orc.PH_STICK)
    stuck = o.get(orc.STUCK).copy(); stuck[::4] = 1
    o.set(orc.STUCK, stuck)
    act = stuck == 0
    PT.sync_oracle_to_gpu(o, g, orc, B, with_history=False)
    x0 = o.get(orc.X).copy()
    o.phase(orc.PH_HLC_STEP, 1); g.phase(B.PH_HLC_STEP, 1)
    so, sg = float(o.get(orc.SIGMA)[0]), float(g.get(B.SIGMA)[0])
    assert so > 0 and abs(sg - so) <= 4 * PT.EPS32 * so
    gho, ghg = o.get(orc.GHAT), g.get(B.GHAT).astype(np.float64)
    fscale = np.max(np.abs(o.get(orc.HLC_F)), axis=1) if form == 1 else np.abs(o.get(orc.F)) + 50.0 * so ** 2
    floor = 8 * PT.EPS32 * (fscale + 6 * wl.obj.sigma_noise + 1.0) * (5.5 / so if form == 1 else 4.0 / (2 * hp.fd_h))
    err = np.max(np.abs(ghg - gho), axis=1)
    tol = PT.G_REL * np.max(np.abs(gho), axis=1) + floor
    assert np.all(err[act] <= tol[act]), float(np.max(err[act] / tol[act]))
    xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
    assert np.all(np.max(np.abs(xg - xo), axis=1)[act] <= (PT.x_tol(xo, hp.lo, hp.hi) + hp.eta_hlc * tol)[act])
    assert np.array_equal(xg[~act], x0[~act])
    # everybody frozen: sigma = 0 and nothing moves on either side
    g.set(B.STUCK, np.ones(N, np.uint8)); x1 = g.get(B.X).copy()
    g.phase(B.PH_HLC_STEP, 2)
    assert float(g.get(B.SIGMA)[0]) == 0.0 and np.array_equal(g.get(B.X), x1)


def test_ablation_switches_phase_mask(orc, B):
    """PAPER.md:498-509 (Table 7 rows): phase_mask bit p off disables phase p on both sides -- no removal (3), no
    reseeding (4), no HLC move (5), no anti-convergence move (6); the other phases still run."""
    obj = inputs.gmm_diag(8, 16, 5.0, 1002)
    for off in (3, 4, 5, 6):
        wl = inputs.custom(obj, 5.0, 300, eps_dup=0.5, eps_grad=1.0, seed=5, phase_mask=0xFFFFFFFF & ~(1 << off))
        o, g = _pair(orc, B, wl)
        rng = np.random.default_rng(off)
        x = PT.f32(rng.uniform(-5, 5, size=(300, 8))); x[100:200] = PT.f32(x[100] + rng.uniform(-0.01, 0.01, size=(100, 8)))
        stuck = np.zeros(300, np.uint8); stuck[100:220] = 1
        f = PT.f32(rng.standard_normal(300))
        for fo, fg, val in ((orc.X, B.X, x), (orc.F, B.F, f), (orc.STUCK, B.STUCK, stuck), (orc.CTRL, B.CTRL, [1, 1, 0, 0, 0, 0, 120, 180])):
            o.set(fo, val); g.set(fg, val)
        o.phase(orc.PH_DEDUP); g.phase(B.PH_DEDUP)
        assert np.array_equal(g.get(B.REMOVED), o.get(orc.REMOVED))
        assert (g.get(B.REMOVED).sum() == 0) == (off == 3)
        o.phase(orc.PH_RESEED); g.phase(B.PH_RESEED)
        assert g.stats().reseed_strategy == o.stats().reseed_strategy
        assert (g.stats().reseed_strategy == 0) == (off in (3, 4))
        x1 = g.get(B.X).copy()
        g.phase(B.PH_HLC_STEP, 1)
        moved = not np.array_equal(g.get(B.X), x1)
        assert moved == (off != 5)
        x2 = g.get(B.X).copy()
        g.phase(B.PH_ANTI_STEP, 1)
        assert (not np.array_equal(g.get(B.X), x2)) == (off != 6)


def test_tensor_evaluator_selection_and_tf32_fallback(orc, B, monkeypatch):
    """chisao_get_info: which evaluator chisao_init chose; the tf32 hi/lo form (forced by CHISAO_TC_TF32, or chosen
    when the box radius leaves fp16's range) passes the same a1 parity as the fp16 hi/lo form"""
    for c, want in ((5, 3), (4, 5), (3, 4), (1, 0)):
        g = B.Chisao(inputs.config(c, N=64))
        assert g.evaluator() == want, (c, g.evaluator())
        g.close()
    # random-Fourier objective: exact fixed-point contraction on the tensor cores at d <= 32, K <= 256; the fp64-phase
    # FFMA evaluator otherwise (or when CHISAO_RFF_FP64 is set), same tolerances
    for d, K, want in ((32, 256, 4), (33, 16, 0), (8, 257, 0)):
        g = B.Chisao(inputs.custom(inputs.rff(d, K, 5), 5.0, 64))
        assert g.evaluator() == want, (d, K, g.evaluator())
        g.close()
    monkeypatch.setenv("CHISAO_RFF_FP64", "1")
    g = B.Chisao(inputs.config(3, N=64))
    assert g.evaluator() == 0
    g.close()
    test_a1_eval_and_fd_gradient(orc, B, 3, 200)
    monkeypatch.delenv("CHISAO_RFF_FP64")
    monkeypatch.setenv("CHISAO_TC_TF32", "1")
    g = B.Chisao(inputs.config(5, N=64))
    assert g.evaluator() == 2
    g.close()
    test_a1_eval_and_fd_gradient(orc, B, 5, 200)
    g = B.Chisao(inputs.config(4, N=64))
    assert g.evaluator() == 1                                # QUAD: 3xTF32 with A = x - c
    g.close()
    test_a1_eval_and_fd_gradient(orc, B, 4, 200)
    test_quad_values_near_the_optimum(orc, B, "tf32", monkeypatch)
    monkeypatch.delenv("CHISAO_TC_TF32")
    # a box of radius 9000 > 2^13: fp16 would overflow -> tf32 operands, same tolerances
    wl = inputs.custom(inputs.gmm_full(40, 3, 3.0, 77), 9000.0, 300, seed=5, fd_h=4.0)
    o, g = _pair(orc, B, wl)
    assert g.evaluator() == 2
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0]); g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL); g.phase(B.PH_RELEASE_EVAL)
    fo, fg = o.get(orc.F), g.get(B.F).astype(np.float64)
    assert np.all(np.abs(fg - fo) <= PT.f_tol(fo)), float(np.max(np.abs(fg - fo) / np.maximum(np.abs(fo), 1)))
    ok, err, tol = PT.grad_ok(g.get(B.G).astype(np.float64), o.get(orc.G), fo, wl.hp.fd_h)
    assert np.all(ok), float(np.max(err / tol))


@pytest.mark.parametrize("form", ["f16", "tf32"])
def test_quad_values_near_the_optimum(orc, B, form, monkeypatch):
    """QUAD (C4): f = -1/2 |W (x - c)|^2 -> 0 at the optimum, where the 1e-5 max(|f|, 1) bar is an ABSOLUTE 1e-5 on values
    that span twelve orders of magnitude.  Samples sit at distances 1e-6 .. 6 from c (along random directions, along the
    stiffest and along the softest direction of W).  Both operand forms (scaled fp16 hi / lo on kind::f16, the default;
    tf32 hi / lo) must meet the bar; both keep the RELATIVE accuracy of the product, which is asserted as well, and the
    FD gradient follows rule 2."""
    if form == "tf32":
        monkeypatch.setenv("CHISAO_TC_TF32", "1")
    wl = inputs.config(4, N=768)
    hp = wl.hp
    rng = np.random.default_rng(31)
    c = np.asarray(wl.obj.means, np.float64).reshape(-1)[:hp.d]
    W = np.asarray(wl.obj.mats, np.float64).reshape(hp.d, hp.d)
    _, _, vt = np.linalg.svd(W)
    dirs = rng.standard_normal((hp.N, hp.d))
    dirs[0::3] = vt[0] * np.sign(rng.standard_normal((len(dirs[0::3]), 1)))      # stiffest direction of W
    dirs[1::3] = vt[-1] * np.sign(rng.standard_normal((len(dirs[1::3]), 1)))     # softest
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    radius = 10.0 ** rng.uniform(-6.0, np.log10(6.0), hp.N)
    wl.x0 = np.clip(c + dirs * radius[:, None], hp.lo, hp.hi).astype(np.float32)
    o, g = _pair(orc, B, wl)
    assert g.evaluator() == (5 if form == "f16" else 1)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, 0]); g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
    o.phase(orc.PH_RELEASE_EVAL); g.phase(B.PH_RELEASE_EVAL)
    fo, fg = o.get(orc.F), g.get(B.F).astype(np.float64)
    assert fo.min() < -1e3 and fo.max() > -1e-9                 # the values do span the range
    assert np.all(np.abs(fg - fo) <= PT.f_tol(fo)), float(np.max(np.abs(fg - fo) / np.maximum(np.abs(fo), 1)))
    # relative: 22-bit operands in a 64-term product of condition <= kappa; far looser than what is measured (~1e-6)
    assert np.all(np.abs(fg - fo) <= 2e-5 * np.abs(fo) + 1e-30), float(np.max(np.abs(fg - fo) / np.abs(fo)))
    ok, err, tol = PT.grad_ok(g.get(B.G).astype(np.float64), o.get(orc.G), fo, hp.fd_h)
    assert np.all(ok), float(np.max(err / tol))


@pytest.mark.parametrize("case", ["c1", "c2", "c3", "c4", "diag33", "rastrigin5", "c4_two_groups", "c3_two_groups"])
def test_line_search_forms_are_bit_identical(B, case):
    """The tile-local line search (one launch for every trial of a tile, CHISAO_OPT_LS_TILE_LOCAL = 1) and the
    per-trial launches on compacted worklists run the same arithmetic per sample: after every L-BFGS iteration the
    whole state is bit-identical (and the evaluation counters are equal)."""
    wl = {"c1": lambda: inputs.config(1), "c2": lambda: inputs.config(2, N=1500), "c3": lambda: inputs.config(3, N=700),
          "c4": lambda: inputs.config(4, N=600),
          # (tiles of one group of 128 below 148 tiles of 256; above, both groups of a CTA hold points)
          "c4_two_groups": lambda: inputs.config(4, N=148 * 256 + 77, n_conv=3),
          "c3_two_groups": lambda: inputs.config(3, N=148 * 256 + 77, n_conv=3),
          "diag33": lambda: inputs.custom(inputs.gmm_diag(33, 5, 3.0, 9), 4.0, 300, fd_h=1e-2, eps_grad=1e-3, n_conv=6, lbfgs_m=4),
          "rastrigin5": lambda: inputs.appendix_d("rastrigin", 5, 400, fd_h=1e-3, eps_grad=1e-3)}[case]()
    a, b = B.Chisao(wl), B.Chisao(wl)
    a.set_option(B.OPT_LS_TILE_LOCAL, 1); b.set_option(B.OPT_LS_TILE_LOCAL, 0)
    for g in (a, b):
        if g.lbfgs_resident():
            g.set_option(B.OPT_LBFGS_RESIDENT, 0)          # the two line-search forms belong to the spill form of Phase 1
    assert a.ls_tile_local() and not b.ls_tile_local()
    for g in (a, b):
        g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
        g.phase(B.PH_RELEASE_EVAL)
    retried = False
    for it in range(1, 4 if case.endswith("two_groups") else 7):
        a.phase(B.PH_LBFGS_ITER, it); b.phase(B.PH_LBFGS_ITER, it)
        for fld in (B.X, B.F, B.G, B.LS_B, B.HIST_LEN, B.HIST_S, B.HIST_Y, B.STALLED, B.XT):
            assert np.array_equal(a.get(fld), b.get(fld), equal_nan=True), (it, fld)
        assert list(a.stats().evals)[:7] == list(b.stats().evals)[:7]
        retried |= bool((a.get(B.LS_B) > 0).any())
    assert retried                                         # some samples needed more than one trial
    # whole cycles through chisao_step (graph submission) agree as well
    wl.hp.n_osc = 3
    a, b = B.Chisao(wl), B.Chisao(wl)
    a.set_option(B.OPT_LS_TILE_LOCAL, 1); b.set_option(B.OPT_LS_TILE_LOCAL, 0)
    for g in (a, b):
        if g.lbfgs_resident():
            g.set_option(B.OPT_LBFGS_RESIDENT, 0)
    for k in range(3):
        sa, sb = a.step(), b.step()
        for fld in (B.X, B.F, B.G, B.STUCK):
            assert np.array_equal(a.get(fld), b.get(fld), equal_nan=True), (k, fld)
        assert list(sa.evals)[:7] == list(sb.evals)[:7]
    assert a.launch_count() < b.launch_count()


def test_gmm_full_keeps_the_per_trial_line_search(B):
    g = B.Chisao(inputs.config(5, N=64))
    assert not g.ls_tile_local()
    with pytest.raises(B.ChisaoError) as ei:
        g.set_option(B.OPT_LS_TILE_LOCAL, 1)
    assert ei.value.code == B.E_INVALID
    for c in (1, 2, 3, 4):
        assert B.Chisao(inputs.config(c, N=64)).ls_tile_local()


@pytest.mark.parametrize("kind,d,N", [("quad", 50, 1000), ("rff", 24, 2000), ("quad", 33, 1400), ("rff", 5, 5000), ("rff", 32, 3001),
                                      ("quad", 64, 1001)])
def test_anti_step_in_place_update_on_multi_tile_persistent_ctas(orc, B, kind, d, N):
    """Eq. 6 rewrites x and v in place from the FD kernel's epilogue.  On the tensor-core evaluators the two groups of
    128 points of a CTA run unsynchronised, so the 2d stencil points of a sample must never straddle them (a row could
    be read half-updated by the group that lags): >= 3 tiles per persistent CTA, 2d not a divisor of 128, a large alpha
    (a torn row would be far off) and the normal position tolerance."""
    obj = inputs.quad(d, 71 + d, lam_max=50.0) if kind == "quad" else inputs.rff(d, 64, 72 + d)
    wl = inputs.custom(obj, 4.0, N, seed=321 + d, fd_h=5e-2, eps_grad=1e-3, alpha_anti=2e-2 if kind == "rff" else 2e-3, mu=0.9)
    o, g = orc.Oracle(wl, threads=8), B.Chisao(wl)
    assert g.evaluator() in (5, 4)
    o.set(orc.CTRL, [1, 1, 0, 0, 0, 0, 0, N]); g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, N])
    for t in (1, 2, 3):
        PT.sync_oracle_to_gpu(o, g, orc, B, with_history=False)
        v0 = o.get(orc.V).copy()
        o.phase(orc.PH_ANTI_STEP, t); g.phase(B.PH_ANTI_STEP, t)
        vo, vg = o.get(orc.V), g.get(B.V).astype(np.float64)
        xo, xg = o.get(orc.X), g.get(B.X).astype(np.float64)
        vprev = np.zeros_like(v0) if t == 1 else v0
        g_used = (wl.hp.mu * vprev - vo) / wl.hp.alpha_anti
        fscale = np.abs(o.values(xo)) + 1.0
        floor = PT.fd_floor(fscale, wl.hp.fd_h) * 4
        vtol = wl.hp.alpha_anti * (PT.G_REL * np.max(np.abs(g_used), axis=1) + floor) + 4 * PT.EPS32 * np.max(np.abs(vo), axis=1)
        ev = np.max(np.abs(vg - vo), axis=1)
        assert np.all(ev <= vtol), (t, int(np.sum(ev > vtol)), float(np.max(ev / vtol)))
        ex = np.max(np.abs(xg - xo), axis=1)
        xt = PT.x_tol(xo, wl.hp.lo, wl.hp.hi) + vtol
        assert np.all(ex <= xt), (t, int(np.sum(ex > xt)), float(np.max(ex / xt)))
    assert g.stats().evals[6] == 3 * N * 2 * d


@pytest.mark.parametrize("c,N", [(1, 256), (2, 777)])
def test_a2_spill_form_at_small_d(orc, B, c, N):
    """the spill form of Phase 1 (history in HBM, launches per iteration) on the configurations whose default is the
    resident form: same teacher-forced check"""
    test_a2_lbfgs_iterations_teacher_forced(orc, B, c, N, resident=False)


def test_resident_form_selection(B):
    for c, want in ((1, True), (2, True), (3, False), (4, False), (5, False)):
        assert B.Chisao(inputs.config(c, N=64)).lbfgs_resident() == want
    g = B.Chisao(inputs.config(4, N=64))
    with pytest.raises(B.ChisaoError) as ei:
        g.set_option(B.OPT_LBFGS_RESIDENT, 1)
    assert ei.value.code == B.E_INVALID
    # d = 3 is not a power of two: spill form; d = 16 with a small diagonal mixture: resident
    assert not B.Chisao(inputs.custom(inputs.gmm_diag(3, 3, 2.0, 43), 3.0, 64)).lbfgs_resident()
    assert B.Chisao(inputs.custom(inputs.gmm_diag(16, 3, 2.0, 43), 3.0, 64)).lbfgs_resident()


@pytest.mark.parametrize("case", ["c1", "c2", "diag16", "iso1", "rastrigin4"])
def test_resident_pass_whole_cycles_against_the_oracle(orc, B, case):
    """chisao_step with Phase 1 as ONE launch (release + f, g + n_conv iterations + Phase 2's partials): per cycle the
    evaluation counters of the start evaluation are exact, the stuck counts follow the oracle's (free-running fp32 / fp64
    trajectories: small differences allowed where samples sit at the thresholds), and the two forms of Phase 1 agree
    with each other to the same degree."""
    wl = {"c1": lambda: inputs.config(1, n_osc=4), "c2": lambda: inputs.config(2, N=1500, n_osc=4, noise=0.0),
          "diag16": lambda: inputs.custom(inputs.gmm_diag(16, 5, 3.0, 9), 4.0, 300, fd_h=1e-2, eps_grad=1e-3, n_conv=25, lbfgs_m=12, n_osc=3, hlc_baseline=1),
          "iso1": lambda: inputs.custom(inputs.gmm_iso(1, 3, 0.4, 2.0, 5), 3.0, 200, fd_h=1e-3, eps_grad=1e-3, n_conv=15, lbfgs_m=3, n_osc=3, hlc_baseline=1),
          "rastrigin4": lambda: inputs.appendix_d("rastrigin", 4, 400, fd_h=1e-3, eps_grad=1e-3, n_osc=3, hlc_baseline=1)}[case]()
    hp = wl.hp
    a, b, o = B.Chisao(wl), B.Chisao(wl), orc.Oracle(wl, threads=8)
    b.set_option(B.OPT_LBFGS_RESIDENT, 0)
    assert a.lbfgs_resident() and not b.lbfgs_resident()
    prev = [0, 0]
    for k in range(hp.n_osc):
        sa, sb, so = a.step(), b.step(), o.step()
        for q, st in enumerate((sa, sb)):
            assert st.evals[0] - prev[q] == hp.N * (2 * hp.d + 1)           # release + f, g at the start positions
            prev[q] = st.evals[0]
            assert st.evals[2] % (2 * hp.d) == 0 and st.evals[1] >= st.evals[2] // (2 * hp.d)
            assert abs(st.n_stuck - so.n_stuck) <= max(2, 0.03 * hp.N), (k, q, st.n_stuck, so.n_stuck)
            assert abs(st.f_max - so.f_max) <= 1e-4 * max(abs(so.f_max), 1.0) + (0 if wl.obj.sigma_noise == 0 else 1.0)
        xa = a.get(B.X)
        assert np.isfinite(xa).all() and np.all(xa >= hp.lo[None, :]) and np.all(xa <= hp.hi[None, :])
    assert a.launch_count() < 0.5 * b.launch_count()
    xo, fo, _ = o.modes()
    for g_ in (a, b):
        xg, fg, _, n = g_.modes()
        pair, only_g, only_o, text = PT.mode_set_report(xg, fg, xo, fo, 2e-3 if case != "rastrigin4" else 5e-3)
        assert len(only_g) <= max(1, 0.1 * len(fo)) and len(only_o) <= max(1, 0.1 * len(fo)), text
