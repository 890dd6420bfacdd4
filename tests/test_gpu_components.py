"""GPU parity of the individual C-ABI calls (-m gpu): transition matrices, stored partials + scale factors, pre-order
partials, the unfused derivative call, edge / degenerate cases and error codes."""
import numpy as np
import pytest

import oracle_runner as orc
from oracle import likelihood as lk
from oracle import models
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,n_pat", [(0, 64), (2, 40)], ids=["hky4", "gy94_61"])
@pytest.mark.parametrize("precision", [plk.FP64, plk.FP32], ids=["fp64", "fp32"])
def test_transition_and_rate_matrices(cfg, n_pat, precision):
    """S8a step 1: P = U diag(exp(lam r t)) U^-1 for every branch x category; Q rebuilt from the eigensystem."""
    wl = workloads.config(cfg, n_patterns=n_pat)
    ev = Evaluator(wl, precision=precision)
    try:
        ev.log_likelihood()
        Q, pi = orc.oracle_model(wl)
        U, Uinv, lam = models.eigen_decomposition(Q, pi)
        tol = 1e-12 if precision == plk.FP64 else 3e-7
        for k in (0, 1, wl.tree.n_tips, wl.tree.n_nodes - 2):
            ref = lk.transition_matrices(U, Uinv, lam, wl.rates, wl.tree.branch_length[k])
            got = ev.inst.get_transition_matrix(k)
            assert np.max(np.abs(got - ref)) <= tol
        assert np.max(np.abs(ev.inst.get_rate_matrix(0) - Q)) <= 1e-13
    finally:
        ev.close()


@pytest.mark.parametrize("cfg,n_pat", [(0, 300), (2, 70)], ids=["hky4", "gy94_61"])
@pytest.mark.parametrize("precision", [plk.FP64, plk.FP32], ids=["fp64", "fp32"])
def test_stored_partials_match_oracle(cfg, n_pat, precision):
    """S8a steps 2-3 and 5: p_k * exp(cumulated log factors) and q_k (up to its per-pattern factor) equal the
    oracle's unscaled recursion at every internal node; likelihood = <q_k, p_k> at every node."""
    wl = workloads.config(cfg, n_patterns=n_pat)
    ev = Evaluator(wl, precision=precision, store_tip_pre=True)
    # fp64: both sides rebuild P = U diag(exp) U^-1 in fp64 with different summation orders; with |U| up to
    # pi_min^-1/2 ~ 1e2 for the codon model that is ~1e-12 per matrix entry, compounded over the ~10 levels between a
    # tip and the root of the 32-taxon tree (measured on B200: 1.3e-11 at 61 states, 2e-13 at 4 states)
    tol = (1e-11 if wl.n_states == 4 else 1e-10) if precision == plk.FP64 else 2e-5
    try:
        logl, site = ev.log_likelihood()
        ev.gradient_unfused()
        Q, pi = orc.oracle_model(wl)
        ch = orc.children_list(wl.tree)
        U, Uinv, lam = models.eigen_decomposition(Q, pi)
        Pm = {k: lk.transition_matrices(U, Uinv, lam, wl.rates, wl.tree.branch_length[k])
              for k in range(wl.tree.n_nodes) if k != wl.tree.root}
        p_ref, _ = lk.post_order(ch, wl.tree.root, Pm, orc.tip_partials(wl), wl.n_categories, rescale=False)
        q_ref, _ = lk.pre_order(ch, wl.tree.root, Pm, p_ref, pi, rescale=False)
        N = wl.tree.n_tips
        for k in (N, N + 1, wl.tree.root - 1, wl.tree.root):
            got = ev.inst.get_partials(k)
            # the library's stored values are proportional to the unscaled ones, per pattern
            ratio = np.sum(got, axis=(0, 2)) / np.sum(p_ref[k], axis=(0, 2))
            assert np.max(np.abs(got - p_ref[k] * ratio[None, :, None])) <= tol * np.max(got)
        for k in (0, N - 1, N, wl.tree.root - 1):
            got = ev.inst.get_partials(k, pre=True)
            ratio = np.sum(got, axis=(0, 2)) / np.sum(q_ref[k], axis=(0, 2))
            assert np.max(np.abs(got - q_ref[k] * ratio[None, :, None]) / np.max(got, axis=(0, 2))[None, :, None]) <= tol
            # inner-product invariant at node k, using the GPU's own post-order partials
            pk = ev.inst.get_partials(k)
            pr = np.sum(pk, axis=(0, 2)) / np.sum(p_ref[k], axis=(0, 2))
            lik = np.einsum("c,cps,cps->p", wl.cat_weights, got, pk) / (ratio * pr)
            assert np.max(np.abs(np.log(lik) - site)) <= (1e-10 if precision == plk.FP64 else 1e-4)
    finally:
        ev.close()


def test_scale_factors_accumulate_to_site_logl():
    """S8a steps 3-4: sum of the stored log factors + log of the scaled root sum = site log-likelihood."""
    wl = workloads.config(4, n_tips=128, n_patterns=200)
    ev = Evaluator(wl, precision=plk.FP64)
    try:
        logl, site = ev.log_likelihood()
        cum = sum(ev.inst.get_scale_factors(int(k)) for k in ev.scale_idx)
        root = ev.inst.get_partials(wl.tree.root)
        lik = np.einsum("c,cps,s->p", wl.cat_weights, root, wl.pi)
        assert np.max(np.abs(np.log(lik) + cum - site)) <= 1e-10 * np.max(np.abs(site))
        assert np.any(cum != 0.0)
    finally:
        ev.close()


@pytest.mark.parametrize("cfg,n_pat", [(0, 200), (2, 45)], ids=["hky4", "gy94_61"])
@pytest.mark.parametrize("precision", [plk.FP64, plk.FP32], ids=["fp64", "fp32"])
def test_unfused_equals_fused_and_no_level_batch(cfg, n_pat, precision):
    wl = workloads.config(cfg, n_patterns=n_pat)
    out = []
    for flags, unfused in ((0, False), (0, True), (plk.FLAG_NO_LEVEL_BATCH, False)):
        ev = Evaluator(wl, precision=precision, flags=flags, store_tip_pre=unfused)
        try:
            logl, site = ev.log_likelihood()
            g = ev.gradient_unfused() if unfused else ev.gradient()
            out.append((logl, site, g))
        finally:
            ev.close()
    tol = 1e-12 if precision == plk.FP64 else 1e-5
    for logl, site, g in out[1:]:
        assert np.array_equal(site, out[0][1])  # same kernels, same order: bit-identical site values
        assert np.allclose(g, out[0][2], rtol=tol, atol=tol * np.max(np.abs(out[0][2])))


def test_repeatable_bitwise():
    """Deterministic reductions (SURVEY section 7 hard part 8): two evaluations give identical bits."""
    wl = workloads.config(1, n_patterns=1500)
    ev = Evaluator(wl, precision=plk.FP64)
    try:
        a = ev.log_likelihood()
        ga = ev.gradient()
        b = ev.log_likelihood()
        gb = ev.gradient()
        assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(ga, gb)
    finally:
        ev.close()


@pytest.mark.parametrize("arm", [0, plk.FLAG_NO_TCGEN05], ids=["tcgen05", "mma_sync"])
def test_tensor_fp32_unfused_no_level_batch_and_repeatable(arm):
    """fp32 tensor path (tcgen05 / TMEM kernels and the mma.sync arm): plk_update_pre_partials (no gradient slots, tip
    pre-order partials stored) + plk_branch_derivatives agrees with the fused call; one launch per operation agrees
    with level batching bit for bit; two evaluations give identical bits (fixed summation order)."""
    wl = workloads.config(2, n_tips=10, n_patterns=300)
    base = plk.FLAG_TENSOR_CORES | arm
    out = []
    for flags, unfused in ((base, False), (base, True), (base | plk.FLAG_NO_LEVEL_BATCH, False)):
        ev = Evaluator(wl, precision=plk.FP32, flags=flags, store_tip_pre=unfused)
        try:
            logl, site = ev.log_likelihood()
            g = ev.gradient_unfused() if unfused else ev.gradient()
            if not unfused and flags == base:
                logl2, site2 = ev.log_likelihood()
                g2 = ev.gradient()
                assert logl == logl2 and np.array_equal(site, site2) and np.array_equal(g, g2)
            out.append((logl, site, g))
        finally:
            ev.close()
    for logl, site, g in out[1:]:
        assert np.array_equal(site, out[0][1])
        assert np.allclose(g, out[0][2], rtol=1e-5, atol=1e-5 * np.max(np.abs(out[0][2])))
    ref = orc.evaluate(wl)
    strict, rel_cond, norm = orc.gradient_errors(out[1][2], ref)
    assert rel_cond <= 1e-4 and norm <= 1e-4


def test_tip_states_u8_matches_int32():
    """plk_set_tip_states_u8 (byte states, asynchronous copy) gives the same bits as plk_set_tip_states."""
    wl = workloads.config(1, n_tips=16, n_patterns=700)
    ev = Evaluator(wl, precision=plk.FP64)
    try:
        a = ev.log_likelihood()
        ga = ev.gradient()
        u8 = np.ascontiguousarray(np.minimum(wl.tip_states, 255).astype(np.uint8))
        for k in range(wl.tree.n_tips):
            ev.inst.set_tip_states_u8(k, u8[k])
        b = ev.log_likelihood()
        gb = ev.gradient()
        assert a[0] == b[0] and np.array_equal(a[1], b[1]) and np.array_equal(ga, gb)
    finally:
        ev.close()
