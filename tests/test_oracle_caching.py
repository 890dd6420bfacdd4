"""Pins for oracle/caching.py (no GPU): the two caching variants of PAPER.md:101 -- (a) Q p_k cached during the
post-order traversal, the gradient step reading S values instead of applying Q; (b) transition matrices applied on the
fly from the eigendecomposition, never formed.  Both reach results with a plain definition, so the pins are the ones
of the main oracle: the printed worked examples W1 / W2 (tests/golden/), brute-force enumeration over
all internal-state assignments with scipy's expm, central differences of that brute-force likelihood, the JC69
two-taxon closed form, and the sum over all patterns = 1.  No expected value comes from oracle/ or the CUDA path."""
import itertools

import numpy as np
import pytest

import golden_io
from oracle import caching as ch
from oracle import likelihood as lk
from oracle import models
from test_oracle_likelihood import T3, T4, T5, TREE3, TREE4, TREE5, _gamma4, _tips, brute_force_site_likelihood

G = golden_io.load("model_constants.txt")
W1 = golden_io.load("w1_nucleotide.txt")
W2 = golden_io.load("w2_codon.txt")


def _cached_gradient(tree, root, t, Q, pi, rates, w, tips, rescale=True):
    """logl [Pn] and d [n_nodes, Pn] through the cached-product path (a)."""
    U, Uinv, lam = models.eigen_decomposition(Q, pi)
    P = {k: lk.transition_matrices(U, Uinv, lam, rates, t[k]) for k in range(len(tree)) if k != root}
    p, Qp, log_m = ch.post_order_with_rate_products(tree, root, P, tips, len(rates), Q, rescale=rescale)
    logl = lk.site_log_likelihoods(p[root], pi, w, log_m)
    q, _ = lk.pre_order(tree, root, P, p, pi, rescale=rescale)
    d = np.zeros((len(tree), logl.shape[0]))
    for k in range(len(tree)):
        if k != root:
            d[k] = ch.branch_site_derivatives_cached(q[k], Qp[k], p[k], rates, w)[0]
    return logl, d


def _on_the_fly_logl(tree, root, t, Q, pi, rates, w, tips, rescale=True):
    U, Uinv, lam = models.eigen_decomposition(Q, pi)
    p, log_m = ch.post_order_on_the_fly(tree, root, U, Uinv, lam, rates, t, tips, rescale=rescale)
    return lk.site_log_likelihoods(p[root], pi, w, log_m)


def _worked(gold, tree, root, t, Q, pi, S, parse):
    n_tips = (len(tree) + 1) // 2
    n_cases = len([k for k in gold if k.endswith(".tips")])
    for cn, (rates, w) in {"c1": (np.ones(1), np.ones(1)), "c4": _gamma4()}.items():
        for i in range(n_cases):
            tips = _tips([[parse(x)] for x in gold[f"case{i}.tips"]], S)
            logl, d = _cached_gradient(tree, root, t, Q, pi, rates, w, tips)
            assert abs(logl[0] - gold[f"case{i}.{cn}.logl"][0]) < 2e-12
            assert np.abs(d[: 2 * n_tips - 2, 0] - np.array(gold[f"case{i}.{cn}.grad"])).max() < 2e-12
            fly = _on_the_fly_logl(tree, root, t, Q, pi, rates, w, tips)
            assert abs(fly[0] - gold[f"case{i}.{cn}.logl"][0]) < 2e-12


def test_worked_example_w1_both_variants():
    Q, pi = models.hky(2.0, [0.1, 0.2, 0.3, 0.4])
    _worked(W1, TREE4, 6, T4, Q, pi, 4, lambda x: int(x))


def test_worked_example_w2_both_variants():
    Q, pi = models.gy94(2.0, 0.3, (0.1, 0.2, 0.3, 0.4), (0.4, 0.3, 0.2, 0.1), (0.25,) * 4)
    cod = models.codon_states()
    _worked(W2, TREE3, 4, T3, Q, pi, 61, lambda x: 61 if x == "---" else cod.index(x))


def _random_gtr(seed):
    rng = np.random.default_rng(seed)
    return models.gtr(rng.gamma(2.0, 1.0, size=6), rng.dirichlet([10.0] * 4))


def test_on_the_fly_equals_brute_force_enumeration():
    """5 taxa, GTR, 4 categories, one missing tip: the plain sum over 4^4 internal assignments with scipy expm."""
    Q, pi = _random_gtr(3)
    rates, w = _gamma4()
    rng = np.random.default_rng(4)
    for _ in range(6):
        states = [int(z) for z in rng.integers(0, 4, size=5)]
        states[int(rng.integers(0, 5))] = 4 if rng.random() < 0.5 else states[0]
        want = brute_force_site_likelihood(TREE5, 8, T5, Q, pi, rates, w, states)
        for rescale in (True, False):
            got = _on_the_fly_logl(TREE5, 8, T5, Q, pi, rates, w, _tips([[z] for z in states], 4), rescale=rescale)
            assert abs(got[0] - np.log(want)) < 1e-13 * abs(np.log(want)) + 1e-13


def test_on_the_fly_sums_to_one_over_all_patterns():
    Q, pi = _random_gtr(5)
    rates, w = _gamma4()
    pats = np.array(list(itertools.product(range(4), repeat=4))).T  # [tip][256 patterns]
    logl = _on_the_fly_logl(TREE4, 6, T4, Q, pi, rates, w, _tips(pats, 4))
    assert abs(np.exp(logl).sum() - 1.0) < 1e-12


def test_jc69_closed_form_both_variants():
    """Two taxa under JC69 (SURVEY 8(c) pins): printed values at t = (0.1, 0.25), same / different tip states."""
    Q, pi = models.hky(1.0, [0.25] * 4)
    tree = [(-1, -1), (-1, -1), (0, 1)]
    t = np.array([0.1, 0.25, 0.0])
    tips = _tips([[0, 0], [0, 2]], 4)
    logl, d = _cached_gradient(tree, 2, t, Q, pi, np.ones(1), np.ones(1), tips)
    fly = _on_the_fly_logl(tree, 2, t, Q, pi, np.ones(1), np.ones(1), tips)
    for got in (logl, fly):
        assert abs(got[0] - G["jc69.same"][0]) < 1e-13 and abs(got[1] - G["jc69.diff"][0]) < 1e-13
    for k in (0, 1):
        assert abs(d[k, 0] - G["jc69.same"][1]) < 1e-13 and abs(d[k, 1] - G["jc69.diff"][1]) < 1e-13


def test_cached_gradient_equals_central_differences_of_the_brute_force_likelihood():
    """Every branch of the 4-taxon tree, GTR + 4 categories: (log l(t_k + h) - log l(t_k - h)) / 2h with l from the
    brute-force enumeration (scipy expm) -- nothing of the oracle on the expected side."""
    Q, pi = _random_gtr(7)
    rates, w = _gamma4()
    states = [2, 0, 3, 4]  # tip 3 missing
    _, d = _cached_gradient(TREE4, 6, T4, Q, pi, rates, w, _tips([[z] for z in states], 4))
    for k in range(6):
        h = 1e-6
        tp, tm = T4.copy(), T4.copy()
        tp[k] += h
        tm[k] -= h
        fd = (np.log(brute_force_site_likelihood(TREE4, 6, tp, Q, pi, rates, w, states)) -
              np.log(brute_force_site_likelihood(TREE4, 6, tm, Q, pi, rates, w, states))) / (2 * h)
        assert abs(d[k, 0] - fd) < 2e-8 * max(1.0, abs(fd))
    assert d[3, 0] == pytest.approx(0.0, abs=1e-14)  # branch above the all-missing tip


def test_cached_product_carries_the_rescaling_factor():
    """Qp_k is formed from the rescaled p_k: it is Q p_k exactly (no extra factor), and num / den is the same with
    rescaling on and off."""
    Q, pi = _random_gtr(9)
    rates, w = _gamma4()
    rng = np.random.default_rng(10)
    pats = rng.integers(0, 5, size=(5, 40))
    tips = _tips(pats, 4)
    U, Uinv, lam = models.eigen_decomposition(Q, pi)
    P = {k: lk.transition_matrices(U, Uinv, lam, rates, T5[k]) for k in range(9) if k != 8}
    p, Qp, _ = ch.post_order_with_rate_products(TREE5, 8, P, tips, 4, Q)
    for k in range(9):
        for c in range(4):
            for pat in (0, 17, 39):
                want = np.array([sum(Q[s, x] * p[k][c, pat, x] for x in range(4)) for s in range(4)])
                assert np.allclose(Qp[k][c, pat], want, rtol=0, atol=1e-15)
    _, d_on = _cached_gradient(TREE5, 8, T5, Q, pi, rates, w, tips, rescale=True)
    _, d_off = _cached_gradient(TREE5, 8, T5, Q, pi, rates, w, tips, rescale=False)
    assert np.abs(d_on - d_off).max() < 1e-12 * np.abs(d_off).max()
