"""GPU parity of plk_rate_matrix_gradient against oracle.likelihood.
rate_matrix_cross_products, element by element, plus the chain rule to model parameters through
plk_chain_rule_rate_matrix.  Tolerances: fp64 1e-10 and fp32 1e-4, relative to the conditioning scale of each element,
A_ij = the same sum with every term's absolute value (G_ij is a score at the simulating parameters and cancels like the
branch gradients do) -- taken from the oracle's per-pattern terms."""
import numpy as np
import pytest

import oracle_runner as orc
from oracle import likelihood as lk
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu


def _oracle_G(wl, t=None):
    Q, pi = orc.oracle_model(wl)
    t = wl.tree.branch_length if t is None else t
    tips = orc.tip_partials(wl)
    G = lk.rate_matrix_cross_products(orc.children_list(wl.tree), wl.tree.root, np.asarray(t), Q, pi, wl.rates,
                                      wl.cat_weights, tips, wl.pattern_weights)
    # conditioning scale: |G| with the absolute value of every pattern's term = the cross products of all-positive
    # partials weighted the same way; an upper bound that needs no second code path: sum_p omega_p |...| >= |G_ij|
    Gabs = G if np.all(wl.pattern_weights >= 0) else lk.rate_matrix_cross_products(
        orc.children_list(wl.tree), wl.tree.root, np.asarray(t), Q, pi, wl.rates, wl.cat_weights, tips,
        np.abs(wl.pattern_weights))
    return G, np.maximum(np.abs(Gabs), np.max(np.abs(Gabs)) * 1e-3), Q


CASES = [pytest.param(0, None, 700, 4, plk.FP64, 0, id="hky8-fp64"),
         pytest.param(1, 24, 1237, 4, plk.FP64, 0, id="gtr24-fp64"),
         pytest.param(1, 24, 1237, 4, plk.FP32, 0, id="gtr24-fp32"),
         pytest.param(1, 24, 333, 3, plk.FP64, 0, id="gtr24-3cat-fp64"),
         pytest.param(2, 12, 150, 4, plk.FP64, 0, id="gy94-fp64"),
         pytest.param(2, 12, 150, 4, plk.FP32, 0, id="gy94-fp32"),
         pytest.param(2, 12, 150, 4, plk.FP64, plk.FLAG_TENSOR_CORES, id="gy94-fp64-tensor-partials"),
         pytest.param(2, 12, 33, 2, plk.FP32, plk.FLAG_TENSOR_CORES, id="gy94-fp32-tensor-partials"),
         # k_cross_tc: several pattern tiles with a ragged tail, more units than one wave would hold branch ranges for
         pytest.param(2, 12, 1003, 4, plk.FP64, plk.FLAG_TENSOR_CORES, id="gy94-1003-fp64-tensor"),
         pytest.param(2, 12, 1003, 4, plk.FP32, plk.FLAG_TENSOR_CORES, id="gy94-1003-fp32-tensor"),
         pytest.param(2, 6, 4100, 3, plk.FP64, plk.FLAG_TENSOR_CORES, id="gy94-4100-3cat-fp64-tensor"),
         pytest.param(2, 6, 4100, 3, plk.FP32, plk.FLAG_TENSOR_CORES, id="gy94-4100-3cat-fp32-tensor")]


_full = {}


@pytest.mark.parametrize("cfg,precision,flags", [pytest.param(2, plk.FP64, plk.FLAG_TENSOR_CORES, id="cfg2-fp64-tensor"),
                                                 pytest.param(2, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg2-fp32-tensor"),
                                                 pytest.param(2, plk.FP64, 0, id="cfg2-fp64-cuda"),
                                                 pytest.param(1, plk.FP64, 0, id="cfg1-fp64"),
                                                 pytest.param(1, plk.FP32, 0, id="cfg1-fp32"),
                                                 pytest.param(3, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg3-fp32-tensor")])
def test_full_size_configs(cfg, precision, flags):
    """BASELINE configs[1] / configs[2] / configs[3] (oracle: ~70 s on one core) at full size, in the launch configuration bench.py --rate-matrix-gradient times
    (k_cross_tc: several waves of units, branch ranges; k_cross4: branch ranges in blockIdx.y), every element of G
    against the oracle on all patterns."""
    if cfg not in _full:
        _full.clear()
        wl = workloads.config(cfg)
        _full[cfg] = (wl,) + _oracle_G(wl)
    wl, G_ref, scale, Q = _full[cfg]
    ev = Evaluator(wl, precision=precision, flags=flags, store_tip_pre=True, eigen=orc.oracle_eigen(wl))
    try:
        ev.log_likelihood(want_site=False)
        ev.gradient_unfused()
        G = ev.rate_matrix_gradient()
        G2 = ev.rate_matrix_gradient()
    finally:
        ev.close()
    err = np.max(np.abs(G - G_ref) / scale)
    assert err <= (1e-10 if precision == plk.FP64 else 1e-4), f"rate-matrix gradient err / scale = {err:.3e}"
    assert np.array_equal(G, G2)


@pytest.mark.parametrize("precision", [plk.FP64, plk.FP32])
def test_tensor_kernel_with_tips_given_as_partials(precision):
    """k_cross_tc with single-category tip partials (the operand kind staged once for all categories) instead of
    compact states: same oracle, same bars."""
    wl = workloads.config(2, n_tips=10, n_patterns=530, n_categories=4)
    ev = Evaluator(wl, precision=precision, flags=plk.FLAG_TENSOR_CORES, store_tip_pre=True, tips_as_partials=True,
                   eigen=orc.oracle_eigen(wl))
    try:
        ev.log_likelihood()
        ev.gradient_unfused()
        G = ev.rate_matrix_gradient()
    finally:
        ev.close()
    G_ref, scale, _ = _oracle_G(wl)
    err = np.max(np.abs(G - G_ref) / scale)
    assert err <= (1e-10 if precision == plk.FP64 else 1e-4), f"rate-matrix gradient err / scale = {err:.3e}"


@pytest.mark.parametrize("cfg,n_tips,n_pat,n_cat,precision,flags", CASES)
def test_rate_matrix_gradient_matches_oracle(cfg, n_tips, n_pat, n_cat, precision, flags):
    wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_pat, n_categories=n_cat) if cfg else workloads.config(0, n_patterns=n_pat)
    ev = Evaluator(wl, precision=precision, flags=flags, store_tip_pre=True, eigen=orc.oracle_eigen(wl))
    try:
        ev.log_likelihood()
        ev.gradient_unfused()  # stores the pre-order partials of every node, tips included
        G = ev.rate_matrix_gradient()
        G2 = ev.rate_matrix_gradient()
    finally:
        ev.close()
    G_ref, scale, Q = _oracle_G(wl)
    tol = 1e-10 if precision == plk.FP64 else 1e-4
    err = np.max(np.abs(G - G_ref) / scale)
    assert err <= tol, f"rate-matrix gradient err / scale = {err:.3e}"
    assert np.array_equal(G, G2)  # fixed-order reductions
    # exact where the approximation is exact: sum_ij G_ij Q_ij = sum_b t_b g_b (tests/test_oracle_substitution_gradient.py)
    ref = orc.evaluate(wl)
    euler = float(np.dot(wl.tree.branch_length, ref["grad"]))
    assert abs(np.sum(G * Q) - euler) <= tol * float(np.dot(wl.tree.branch_length, ref["cond"]))
    # chain rule through the C ABI (host helper) against numpy
    rng = np.random.default_rng(3)
    dQ = rng.normal(size=(5, wl.n_states, wl.n_states))
    assert np.allclose(plk.chain_rule_rate_matrix(G, dQ), np.einsum("ij,kij->k", G, dQ), rtol=1e-13, atol=0)


def test_errors():
    wl = workloads.config(0, n_patterns=50)
    ev = Evaluator(wl)  # tips' pre-order partials are not stored
    try:
        ev.log_likelihood()
        ev.gradient()
        with pytest.raises(plk.PlkError) as e:
            ev.rate_matrix_gradient()
        assert e.value.status == plk.ERR_UNINITIALIZED
        with pytest.raises(plk.PlkError) as e:
            ev.inst.rate_matrix_gradient([wl.tree.n_tips], [wl.tree.n_tips], [-1.0])
        assert e.value.status == plk.ERR_OUT_OF_RANGE
    finally:
        ev.close()
