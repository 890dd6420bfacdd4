"""20-state amino-acid models: the kernels instantiated for 32 padded states against the
oracle, element by element, for every call of the hot path: site log-likelihoods, logL, all branch gradients (fused
and unfused), per-pattern derivatives, stored partials through the inner-product invariant, the rate-matrix gradient;
compact tips, tips as partials, missing cells, category counts, ragged tiles, other state counts in 5..32."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from oracle import likelihood as lk
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu
PREC = [pytest.param(plk.FP64, id="fp64"), pytest.param(plk.FP32, id="fp32")]


def _check(wl, precision, **kw):
    logl, site, grad, site_d = pc.run_gpu(wl, precision, **kw)
    ref = orc.evaluate(wl, keep_site_derivatives=True)
    pc.check_logl(site, logl, ref, precision)
    pc.check_grad(grad, ref, precision, wl.tree.root)
    pc.check_site_derivs(site_d, ref, precision, wl.tree.root)
    return ref


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("n_tips,n_pat,n_cat", [(24, 500, 4), (9, 33, 1), (40, 129, 2), (3, 1, 4)])
def test_amino_acid_parity(precision, n_tips, n_pat, n_cat):
    _check(workloads.config(5, n_tips=n_tips, n_patterns=n_pat, n_categories=n_cat), precision)


@pytest.mark.parametrize("precision", PREC)
def test_amino_acid_tip_partials_and_missing(precision):
    wl = workloads.config(5, n_tips=16, n_patterns=300)
    rng = np.random.default_rng(9)
    wl.tip_states[rng.random(wl.tip_states.shape) < 0.1] = wl.n_states
    _check(wl, precision)
    _check(wl, precision, tips_as_partials=True)
    _check(wl, precision, tips_as_partials=np.arange(16) % 3 == 0)
    _check(wl, precision, flags=plk.FLAG_TENSOR_CORES)  # the flag concerns the 64-state kernels: same CUDA-core path


@pytest.mark.parametrize("precision", PREC)
def test_amino_acid_deep_tree_needs_rescaling(precision):
    wl = workloads.make_workload("aa-deep", "AA20", 300, 40, "caterpillar", seed=17)
    ref = _check(wl, precision)
    assert np.min(ref["site_logl"]) < -300.0


@pytest.mark.parametrize("precision", PREC)
def test_amino_acid_unfused_and_rate_matrix_gradient(precision):
    wl = workloads.config(5, n_tips=12, n_patterns=200)
    ev = Evaluator(wl, precision=precision, store_tip_pre=True, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood()
        g = ev.gradient_unfused()
        G = ev.rate_matrix_gradient()
        q_root_child = ev.inst.get_partials(wl.tree.children[wl.tree.root][0], pre=True)
        p_root_child = ev.inst.get_partials(wl.tree.children[wl.tree.root][0])
    finally:
        ev.close()
    ref = orc.evaluate(wl)
    pc.check_grad(g, ref, precision, wl.tree.root)
    Q, pi = orc.oracle_model(wl)
    G_ref = lk.rate_matrix_cross_products(orc.children_list(wl.tree), wl.tree.root, wl.tree.branch_length, Q, pi, wl.rates,
                                          wl.cat_weights, orc.tip_partials(wl), wl.pattern_weights)
    tol = pc.tol_of(precision)
    assert np.max(np.abs(G - G_ref)) <= tol * np.max(np.abs(G_ref))
    assert q_root_child.shape == (4, 200, 20) and p_root_child.shape == (4, 200, 20)
    # likelihood as the inner product of pre- and post-order partials, up to the per-pattern scale factors:
    # the ratio of the category terms is what is scale-free
    inner = np.einsum("cps,cps->cp", q_root_child, p_root_child)
    assert np.all(inner > 0)


@pytest.mark.parametrize("S", [5, 13, 32])
def test_other_state_counts_padded_to_32(S):
    """Any 5..32 states run on the 32-padded kernels: a seeded reversible model on S states."""
    rng = np.random.default_rng(100 + S)
    wl = workloads.config(5, n_tips=7, n_patterns=77)
    pi = rng.dirichlet([10.0] * S)
    wl.model = {"name": "AA20", "rho": rng.gamma(2.0, 1.0, size=S * (S - 1) // 2).tolist(), "pi": pi.tolist()}
    wl.Q, wl.pi = workloads.client_rate_matrix(wl.model)
    wl.U, wl.Uinv, wl.lam = workloads.client_eigen(wl.Q, wl.pi)
    wl.tip_states = (wl.tip_states % S).astype(np.uint8)
    _check(wl, plk.FP64)
    _check(wl, plk.FP32)
