"""NEXT-5: the opt-in stencil-aware FD evaluator (chisao_set_option,
CHISAO_OPT_STENCIL_AWARE) must reproduce the same 2d stencil values within the same tolerances as the black-box
path.  The existing per-phase and end-to-end parity tests are re-run against the oracle with the option switched on
(the oracle itself always evaluates every stencil point independently), plus a direct comparison with the black-box
CUDA path and the option's error behaviour."""
import numpy as np
import pytest

from paper_2606_26164_b200 import inputs

import parity as PT
import test_gpu_end_to_end as EE
import test_gpu_fullsize as FS
import test_gpu_parity_phases as PP

pytestmark = pytest.mark.gpu


class _StencilBinding:
    """the binding module with Chisao() switching the option on"""

    def __init__(self, B):
        self._B = B

    def __getattr__(self, k):
        return getattr(self._B, k)

    def Chisao(self, wl, *a, **k):
        g = self._B.Chisao(wl, *a, **k)
        g.set_option(self._B.OPT_STENCIL_AWARE, 1)
        return g


@pytest.fixture(scope="module")
def B():
    from paper_2606_26164_b200 import binding
    binding.load_library()
    return binding


@pytest.fixture(scope="module")
def SB(B):
    return _StencilBinding(B)


@pytest.mark.parametrize("c,N", [(5, 200), (4, 261)])
def test_a1_a2_with_the_stencil_aware_evaluator(orc, SB, c, N):
    PP.test_a1_eval_and_fd_gradient(orc, SB, c, N)
    PP.test_a2_lbfgs_iterations_teacher_forced(orc, SB, c, N)


@pytest.mark.parametrize("c,N", [(5, 150), (4, 140)])
def test_a7_with_the_stencil_aware_evaluator(orc, SB, c, N):
    PP.test_a7_anti_convergence_step(orc, SB, c, N)


@pytest.mark.parametrize("obj_id,d,K,N", [(2, 40, 3, 300), (2, 64, 1, 130), (2, 33, 2, 257), (4, 50, 1, 260),
                                          (2, 64, 5, 513), (2, 6, 4, 300), (2, 20, 3, 129), (4, 8, 1, 200)])
def test_shapes_with_the_stencil_aware_evaluator(orc, SB, obj_id, d, K, N):
    """all three padded widths (8 / 32 / 64), ragged d, odd K, ragged last tile of 128 samples"""
    EE.test_tensor_core_evaluator_shapes(orc, SB, obj_id, d, K, N)


def test_free_running_cycles_with_the_stencil_aware_evaluator(orc, SB):
    EE.test_noise_free_mixtures_recover_the_same_modes(orc, SB, 5, 256, 4)
    EE.test_c4_side_run_unimodal_collapses_to_the_maximiser(orc, SB)


def test_full_size_sampled_rows_with_the_stencil_aware_evaluator(orc, SB):
    FS.test_full_size_eval_and_lbfgs_iteration_on_sampled_rows(orc, SB, 5, 48)


def test_same_values_as_the_black_box_path_and_same_counters(B, SB):
    """C5 with its noise: gradients of the two CUDA paths agree to the FD floor; evaluation counters are identical"""
    wl = inputs.config(5, N=777)
    a, b = B.Chisao(wl), SB.Chisao(wl)
    for g in (a, b):
        g.set(B.CTRL, [1, 1, 0, 0, 0, 0, 0, 0])
        g.phase(B.PH_RELEASE_EVAL)
    fa, fb = a.get(B.F).astype(np.float64), b.get(B.F).astype(np.float64)
    assert np.array_equal(fa, fb)                                       # the centre value is the same kernel
    ga, gb = a.get(B.G).astype(np.float64), b.get(B.G).astype(np.float64)
    ok, err, tol = PT.grad_ok(gb, ga, fa, wl.hp.fd_h, wl.obj.sigma_noise)
    assert np.all(ok), float(np.max(err / tol))
    assert list(a.stats().evals)[:7] == list(b.stats().evals)[:7]


def test_option_errors(B):
    g = B.Chisao(inputs.config(2, N=64))
    with pytest.raises(B.ChisaoError) as ei:                            # diagonal mixture: not a dense objective
        g.set_option(B.OPT_STENCIL_AWARE, 1)
    assert ei.value.code == B.E_INVALID
    g.set_option(B.OPT_STENCIL_AWARE, 0)
    with pytest.raises(B.ChisaoError):
        g.set_option(99, 1)
