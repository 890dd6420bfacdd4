"""The two caching variants of PAPER.md:101 on the GPU (-m gpu), against the oracle:
(a) PLK_FLAG_CACHE_RATE_PRODUCTS -- Q p_k stored during plk_update_partials, plk_branch_derivatives reads it;
(b) plk_update_partials_on_the_fly -- the post-order pass in one launch, no transition matrix formed."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from oracle import caching as och
from oracle import likelihood as lk
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu

CACHE_CASES = [
    pytest.param(1, 24, 3000, 4, plk.FP64, False, id="gtr-24x3000-fp64"),
    pytest.param(1, 24, 3000, 4, plk.FP32, False, id="gtr-24x3000-fp32"),
    pytest.param(1, 12, 777, 3, plk.FP64, True, id="gtr-12x777-c3-fp64-tip-partials"),
    pytest.param(2, 8, 300, 4, plk.FP64, False, id="gy94-8x300-fp64"),
    pytest.param(2, 8, 300, 4, plk.FP32, False, id="gy94-8x300-fp32"),
    pytest.param(2, 6, 97, 2, plk.FP64, True, id="gy94-6x97-c2-fp64-tip-partials"),
    pytest.param(5, 8, 300, 4, plk.FP64, False, id="aa-8x300-fp64"),
    pytest.param(5, 8, 300, 4, plk.FP32, True, id="aa-8x300-fp32-tip-partials"),
]


@pytest.mark.parametrize("cfg,n_tips,n_pat,n_cat,precision,tap", CACHE_CASES)
def test_cached_rate_products_gradient_matches_oracle(cfg, n_tips, n_pat, n_cat, precision, tap):
    wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_pat, n_categories=n_cat)
    ref = orc.evaluate(wl, keep_site_derivatives=True)
    root = wl.tree.root
    flags = plk.FLAG_CACHE_RATE_PRODUCTS | plk.FLAG_SITE_DERIVATIVES
    ev = Evaluator(wl, precision=precision, flags=flags, tips_as_partials=tap, store_tip_pre=True, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood()
        grad, site_d = ev.gradient_unfused(want_site=True)
        pc.check_logl(site, logl, ref, precision)
        pc.check_grad(grad, ref, precision, root)
        pc.check_site_derivs(site_d, ref, precision, root)
        # the cache itself: Qp_k = Q p_k element by element, with the ORACLE's Q applied to the stored p_k
        Q = orc.oracle_model(wl)[0]
        tol = 1e-12 if precision == plk.FP64 else 2e-6
        nodes = [root, wl.tree.n_tips] + ([0] if tap else [])
        for k in nodes:
            p = ev.inst.get_partials(k)
            qp = ev.inst.get_partials(k, pre=2)
            want = np.matmul(p, Q.T)
            assert np.max(np.abs(qp - want)) <= tol * np.max(np.abs(p)) * np.max(np.abs(Q)) * wl.n_states
        # a second evaluation at other branch lengths refreshes every cached product
        rng = np.random.default_rng(11)
        t2 = np.asarray(wl.tree.branch_length) * np.exp(rng.normal(0.0, 0.3, size=wl.tree.n_nodes))
        ref2 = orc.evaluate(wl, branch_lengths=t2)
        ev.log_likelihood(t2)
        pc.check_grad(ev.gradient_unfused(), ref2, precision, root)
    finally:
        ev.close()


def test_cached_rate_products_state_machine():
    wl = workloads.config(0, n_patterns=200)
    ev = Evaluator(wl, precision=plk.FP64, store_tip_pre=True)  # flag absent
    try:
        with pytest.raises(plk.PlkError) as e:
            ev.inst.cache_rate_products(0, [wl.tree.root])
        assert e.value.status == plk.ERR_UNSUPPORTED
    finally:
        ev.close()
    ev = Evaluator(wl, precision=plk.FP64, flags=plk.FLAG_CACHE_RATE_PRODUCTS, store_tip_pre=True)
    try:
        ev.log_likelihood()
        g0 = ev.gradient_unfused()
        k = wl.tree.n_tips  # an internal node: overwrite its partials -> its cached product is stale
        ev.inst.set_partials(k, ev.inst.get_partials(k))
        with pytest.raises(plk.PlkError) as e:
            ev.gradient_unfused()
        assert e.value.status == plk.ERR_UNINITIALIZED
        ev.inst.cache_rate_products(0, [k])
        assert np.array_equal(ev.gradient_unfused(), g0)
        with pytest.raises(plk.PlkError) as e:
            ev.inst.get_partials(0, pre=2)  # a compact tip has no cached product
        assert e.value.status == plk.ERR_UNSUPPORTED
    finally:
        ev.close()


OTF_CASES = [
    pytest.param(2, 8, 1, 1, plk.FP64, False, id="gy94-8x1-c1-fp64"),
    pytest.param(2, 32, 1, 4, plk.FP64, False, id="gy94-32x1-c4-fp64"),
    pytest.param(2, 32, 1, 4, plk.FP32, False, id="gy94-32x1-c4-fp32"),
    pytest.param(2, 200, 3, 4, plk.FP32, False, id="gy94-200x3-c4-fp32-deep"),
    pytest.param(2, 200, 3, 4, plk.FP64, False, id="gy94-200x3-c4-fp64-deep"),
    pytest.param(2, 12, 75, 5, plk.FP64, True, id="gy94-12x75-c5-fp64-tip-partials"),
    pytest.param(5, 16, 40, 4, plk.FP64, False, id="aa-16x40-fp64"),
    pytest.param(5, 16, 40, 9, plk.FP32, True, id="aa-16x40-c9-fp32-tip-partials"),
]


@pytest.mark.parametrize("cfg,n_tips,n_pat,n_cat,precision,tap", OTF_CASES)
def test_on_the_fly_post_order_matches_oracle(cfg, n_tips, n_pat, n_cat, precision, tap):
    wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_pat, n_categories=n_cat)
    ref = orc.evaluate(wl)
    # the oracle's own on-the-fly recursion (oracle/caching.py) on the same inputs
    U, Uinv, lam = orc.oracle_eigen(wl)
    Q, pi = orc.oracle_model(wl)
    p_fly, log_m = och.post_order_on_the_fly(orc.children_list(wl.tree), wl.tree.root, U, Uinv, lam, wl.rates,
                                             np.asarray(wl.tree.branch_length), orc.tip_partials(wl))
    site_fly = lk.site_log_likelihoods(p_fly[wl.tree.root], pi, wl.cat_weights, log_m)
    tol = pc.tol_of(precision)
    ev = Evaluator(wl, precision=precision, flags=plk.FLAG_ON_THE_FLY_MATRICES, tips_as_partials=tap,
                   eigen=(U, Uinv, lam))
    try:
        n0 = ev.inst.kernel_launch_count()
        logl, site = ev.log_likelihood_on_the_fly()
        # ONE post-order launch + the root reduction (site kernel + sum kernel; one kernel when its grid is one block)
        root_blocks = -(-wl.n_patterns * (1 if wl.n_states == 4 else (8 if wl.n_states <= 32 else 16)) // 128)
        assert ev.inst.kernel_launch_count() - n0 == (2 if root_blocks == 1 else 3)
        pc.check_logl(site, logl, ref, precision)
        assert np.max(np.abs(site - site_fly) / np.abs(site_fly)) <= tol
        # repeatable bit for bit (fixed arithmetic order per ticket, whatever CTA takes it)
        for _ in range(3):
            logl2, site2 = ev.log_likelihood_on_the_fly()
            assert logl2 == logl and np.array_equal(site2, site)
        # the buffers it leaves are the ones the matrix-based pass leaves: the fused gradient runs on top of them
        ev.inst.update_transition_matrices(0, ev.matrix_idx, np.asarray(wl.tree.branch_length)[ev.matrix_idx])
        pc.check_grad(ev.gradient(), ref, precision, wl.tree.root)
        # and against the matrix-based post-order pass of the library (different rounding order only)
        logl3, site3 = ev.log_likelihood()
        assert np.max(np.abs(site3 - site) / np.abs(site)) <= tol
        # new branch lengths
        rng = np.random.default_rng(3)
        t2 = np.asarray(wl.tree.branch_length) * np.exp(rng.normal(0.0, 0.3, size=wl.tree.n_nodes))
        ref2 = orc.evaluate(wl, branch_lengths=t2, gradient=False)
        logl4, site4 = ev.log_likelihood_on_the_fly(t2)
        pc.check_logl(site4, logl4, ref2, precision)
    finally:
        ev.close()


def test_on_the_fly_errors():
    wl = workloads.config(2, n_tips=4, n_patterns=2)
    ev = Evaluator(wl, precision=plk.FP64)
    try:
        with pytest.raises(plk.PlkError) as e:
            ev.log_likelihood_on_the_fly()
        assert e.value.status == plk.ERR_UNSUPPORTED  # flag absent
    finally:
        ev.close()
    ev = Evaluator(wl, precision=plk.FP64, flags=plk.FLAG_ON_THE_FLY_MATRICES)
    try:
        t = np.asarray(wl.tree.branch_length).copy()
        t[0] = -0.5
        with pytest.raises(plk.PlkError) as e:
            ev.log_likelihood_on_the_fly(t)
        assert e.value.status == plk.ERR_OUT_OF_RANGE
    finally:
        ev.close()
    with pytest.raises(plk.PlkError) as e:  # nucleotide instances: the variant is for large state spaces
        plk.Instance(4, 4, 10, 1, flags=plk.FLAG_ON_THE_FLY_MATRICES)
    assert e.value.status == plk.ERR_UNSUPPORTED
