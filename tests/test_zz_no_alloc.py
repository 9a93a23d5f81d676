"""chisao_stick_test_static (include/chisao.h): the allocation-free Phase 2 entry point against the context path
(CHISAO_PH_STICK on a chisao_ctx with a caller-allocated workspace) on the same inputs.  Eq. 3 decides
bytes from fp32 comparisons that both paths take in the same precision and order-independent maxima, so the bar is
bit-exact: flags, count and f_max.  The file name keeps it last in pytest's collection order."""
import numpy as np
import pytest

from paper_2606_26164_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2606_26164_b200 import binding
    binding.load_library()
    return binding


def _state(N, d, eps_grad, log_delta, seed, f_top):
    """gradients with about half of the rows under eps_grad, values spread over 3 |log delta| below f_top, a NaN gradient
    row, a +inf and a NaN value (none of them may be stuck or count towards f_max)"""
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((N, d)).astype(np.float32)
    scale = np.where(rng.random(N) < 0.5, 0.2, 3.0) * eps_grad / np.maximum(np.max(np.abs(g), axis=1), 1e-6)
    g = (g * scale[:, None]).astype(np.float32)
    f = (f_top - 3.0 * abs(log_delta) * rng.random(N)).astype(np.float32)
    if N >= 16:
        g[3, d - 1] = np.nan
        f[5] = np.inf
        f[7] = np.nan
        f[11] = f_top                      # the maximum itself is there
    return g, f


def _context_path(B, c, N, g, f):
    """the existing path: state into a context, the stick unit, flags / count / f_max back"""
    ctx = B.Chisao(inputs.config(c, N=N))
    ctx.set(B.G, g); ctx.set(B.F, f)
    ctx.phase(B.PH_STICK)
    st = ctx.stats()
    out = ctx.get(B.STUCK).copy(), int(st.n_stuck), np.float32(st.f_max)
    ctx.close()
    return out


@pytest.mark.parametrize("c,sizes", [(2, (4096 + 37, 1500)), (5, (2049, 2049)), (2, (262144, 333))])
def test_static_stick_test_matches_the_context_path_on_two_calls_in_a_row(B, c, sizes):
    import torch
    hp = inputs.config(c, N=8).hp
    d = hp.d
    # call 2 has a LOWER f_max (and in two cases a smaller N) than call 1: a stale f_max or stale per-sample norms left in
    # the shared static scratch by call 1 would change its flags
    cases = [_state(sizes[0], d, hp.eps_grad, hp.log_delta, 11 + c, f_top=5.0),
             _state(sizes[1], d, hp.eps_grad, hp.log_delta, 23 + c, f_top=5.0 - 10.0 * abs(hp.log_delta))]
    want = [_context_path(B, c, g.shape[0], g, f) for g, f in cases]
    dev = torch.device("cuda:0")
    bufs = []
    for g, f in cases:
        N = g.shape[0]
        bufs.append((torch.from_numpy(g).to(dev), torch.from_numpy(f).to(dev),
                     torch.full((N,), 7, dtype=torch.uint8, device=dev),          # outputs start with garbage
                     torch.full((1,), -5, dtype=torch.int32, device=dev), torch.full((1,), 1e30, dtype=torch.float32, device=dev)))
    # first call on the device looks up the scratch address (module load); the calls measured below must not allocate
    B.stick_test_static(*bufs[0][:2], hp.eps_grad, hp.log_delta, *bufs[0][2:])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(dev)[0]
    for _ in range(2):                                            # two rounds of (call 1, call 2) back to back on one stream
        for gt, ft, st, ns, fm in bufs:
            st.fill_(7); ns.fill_(-5); fm.fill_(1e30)
            B.stick_test_static(gt, ft, hp.eps_grad, hp.log_delta, st, ns, fm)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info(dev)[0] == free_before      # no cudaMalloc behind the entry point
        for (gt, ft, st, ns, fm), (stuck_w, n_w, fmax_w) in zip(bufs, want):
            stuck = st.cpu().numpy()
            assert set(np.unique(stuck)) <= {0, 1}
            assert np.array_equal(stuck, stuck_w)                  # bytes: bit-exact
            assert int(ns.item()) == n_w == int(stuck_w.sum())
            assert np.float32(fm.item()) == fmax_w
    # the test is not vacuous: both classes occur, and the special rows are not stuck
    for stuck_w, _, _ in want:
        assert 0 < stuck_w.sum() < stuck_w.size
        assert stuck_w[3] == 0 and stuck_w[5] == 0 and stuck_w[7] == 0 and stuck_w[11] in (0, 1)


def test_static_stick_test_optional_outputs_and_empty_population(B):
    import torch
    dev = torch.device("cuda:0")
    hp = inputs.config(2, N=8).hp
    g, f = _state(777, hp.d, hp.eps_grad, hp.log_delta, 5, f_top=-2.0)
    stuck_w, n_w, fmax_w = _context_path(B, 2, 777, g, f)
    gt, ft = torch.from_numpy(g).to(dev), torch.from_numpy(f).to(dev)
    st = torch.empty(777, dtype=torch.uint8, device=dev)
    B.stick_test_static(gt, ft, hp.eps_grad, hp.log_delta, st)      # no count, no f_max asked for
    assert np.array_equal(st.cpu().numpy(), stuck_w)
    # N = 0 between two calls: count 0, f_max = -inf, and the next call is unaffected
    ns = torch.full((1,), 9, dtype=torch.int32, device=dev); fm = torch.zeros(1, device=dev)
    B.stick_test_static(torch.empty((0, hp.d), device=dev), torch.empty(0, device=dev), hp.eps_grad, hp.log_delta,
                        torch.empty(0, dtype=torch.uint8, device=dev), ns, fm)
    assert int(ns.item()) == 0 and fm.item() == -np.inf
    B.stick_test_static(gt, ft, hp.eps_grad, hp.log_delta, st, ns, fm)
    assert np.array_equal(st.cpu().numpy(), stuck_w) and int(ns.item()) == n_w and np.float32(fm.item()) == fmax_w


def test_static_stick_test_rejects_sizes_beyond_the_static_scratch(B):
    import torch
    dev = torch.device("cuda:0")
    N = B.STATIC_MAX_N + 1
    g = torch.zeros((N, 1), device=dev); f = torch.zeros(N, device=dev)
    st = torch.full((N,), 3, dtype=torch.uint8, device=dev)
    with pytest.raises(B.ChisaoError) as ei:
        B.stick_test_static(g, f, 1e-3, -2.3, st)
    assert ei.value.code == -1 and "CHISAO_STATIC_MAX_N" in str(ei.value) and str(N) in str(ei.value)
    torch.cuda.synchronize()
    assert int(st.min().item()) == 3                               # nothing was launched
    with pytest.raises(B.ChisaoError):
        B.stick_test_static(torch.zeros((4, 65), device=dev), torch.zeros(4, device=dev), 1e-3, -2.3,
                            torch.zeros(4, dtype=torch.uint8, device=dev))   # d beyond CHISAO_MAX_D
