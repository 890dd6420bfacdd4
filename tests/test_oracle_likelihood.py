"""Pins for oracle/likelihood.py (no GPU): brute-force enumeration, sum over all patterns = 1, JC69 closed form,
central finite differences, the pre/post inner-product invariant, pulley, worked examples W1/W2
(tests/golden/), rescaling on/off and a deep tree where unscaled fp64 underflows (checked in log space).
None of the expected values comes from oracle/ itself or from the CUDA path."""
import itertools

import numpy as np
import pytest

import golden_io
from oracle import likelihood as lk
from oracle import models

G = golden_io.load("model_constants.txt")
W1 = golden_io.load("w1_nucleotide.txt")
W2 = golden_io.load("w2_codon.txt")

# ((0,1)4,(2,3)5)6 and a 5-taxon unbalanced one (((0,1)5,2)6,(3,4)7)8
TREE4 = [(-1, -1)] * 4 + [(0, 1), (2, 3), (4, 5)]
T4 = np.array([0.1, 0.2, 0.3, 0.4, 0.05, 0.15, 0.0])
TREE5 = [(-1, -1)] * 5 + [(0, 1), (5, 2), (3, 4), (6, 7)]
T5 = np.array([0.11, 0.07, 0.31, 0.02, 0.45, 0.09, 0.13, 0.21, 0.0])
TREE3 = [(-1, -1)] * 3 + [(1, 2), (0, 3)]
T3 = np.array([0.1, 0.2, 0.3, 0.05, 0.0])


def _gamma4():
    return models.discrete_gamma(0.5, 4), np.full(4, 0.25)


def _tips(states_per_tip, S):
    """states_per_tip: [n_tips][P] codes -> dict tip -> [P, S]"""
    return {k: lk.tip_partials_from_states(np.asarray(s), S) for k, s in enumerate(states_per_tip)}


def brute_force_site_likelihood(children, root, t, Q, pi, rates, cat_w, tip_states):
    """The plain definition: sum over every assignment of states to internal nodes of pi[root] * prod over branches
    of expm(Q r t)[parent state, child state], averaged over categories.  Uses scipy expm, not the oracle."""
    from scipy.linalg import expm

    S = Q.shape[0]
    n = len(children)
    internal = [k for k in range(n) if children[k][0] >= 0]
    total = 0.0
    for c, r in enumerate(rates):
        P = {k: expm(Q * r * t[k]) for k in range(n) if k != root}
        acc = 0.0
        for assign in itertools.product(range(S), repeat=len(internal)):
            st = dict(zip(internal, assign))
            term = pi[st[root]]
            for m in internal:
                for ch in children[m]:
                    if children[ch][0] >= 0:
                        term *= P[ch][st[m], st[ch]]
                    else:
                        z = tip_states[ch]
                        term *= P[ch][st[m], z] if z < S else P[ch][st[m], :].sum()
            acc += term
        total += cat_w[c] * acc
    return total


@pytest.mark.parametrize("tree,t", [(TREE4, T4), (TREE5, T5)])
def test_pruning_equals_brute_force_nucleotide(tree, t):
    rng = np.random.default_rng(11)
    Q, pi = models.gtr(rng.gamma(2, 1, 6), rng.dirichlet([10] * 4))
    rates, w = _gamma4()
    n_tips = (len(tree) + 1) // 2
    root = len(tree) - 1
    pats = [rng.integers(0, 4, n_tips) for _ in range(4)] + [np.array([0, 4, 2, 4, 1][:n_tips])]
    states = np.stack(pats, axis=1)
    r = lk.evaluate(tree, root, t, Q, pi, rates, w, _tips(states, 4), np.ones(states.shape[1]), gradient=False)
    for p in range(states.shape[1]):
        bf = brute_force_site_likelihood(tree, root, t, Q, pi, rates, w, states[:, p])
        assert abs(np.exp(r["site_logl"][p]) - bf) <= 1e-13 * bf


def test_pruning_equals_brute_force_codon():
    rng = np.random.default_rng(12)
    Q, pi = models.gy94(2.0, 0.3, rng.dirichlet([10] * 4), rng.dirichlet([10] * 4), rng.dirichlet([10] * 4))
    rates, w = np.array([0.4, 1.6]), np.array([0.5, 0.5])
    states = np.array([[14, 3], [14, 61], [20, 7]])
    r = lk.evaluate(TREE3, 4, T3, Q, pi, rates, w, _tips(states, 61), np.ones(2), gradient=False)
    for p in range(2):
        bf = brute_force_site_likelihood(TREE3, 4, T3, Q, pi, rates, w, states[:, p])  # 61^2 terms
        # 1e-11: the brute force multiplies scipy-expm entries of size ~1e-4 whose absolute error is ~1e-16
        assert abs(np.exp(r["site_logl"][p]) - bf) <= 1e-11 * bf


def test_sum_over_all_patterns_is_one_nucleotide():
    rng = np.random.default_rng(13)
    Q, pi = models.hky(2.0, rng.dirichlet([10] * 4))
    rates, w = _gamma4()
    allp = np.array(list(itertools.product(range(4), repeat=5))).T  # [5, 1024]
    r = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, _tips(allp, 4), np.ones(allp.shape[1]), gradient=False)
    assert abs(np.exp(r["site_logl"]).sum() - 1.0) < 1e-12
    # and the gradient of a constant is zero: sum_p l_p * d log l_p / dt_k = 0 for every branch
    rr = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, _tips(allp, 4), np.exp(r["site_logl"]), gradient=True)
    assert np.abs(rr["grad"]).max() < 1e-13


def test_sum_over_all_patterns_is_one_codon():
    Q, pi = models.gy94(2.0, 0.3, (0.1, 0.2, 0.3, 0.4), (0.4, 0.3, 0.2, 0.1), (0.25,) * 4)
    rates, w = _gamma4()
    allp = np.array(list(itertools.product(range(61), repeat=2))).T  # [2, 3721]
    tree = [(-1, -1), (-1, -1), (0, 1)]
    r = lk.evaluate(tree, 2, np.array([0.3, 0.7, 0.0]), Q, pi, rates, w, _tips(allp, 61), np.ones(3721), gradient=False)
    assert abs(np.exp(r["site_logl"]).sum() - 1.0) < 1e-12


def test_jc69_two_taxon_closed_form():
    Q, pi = models.hky(1.0, [0.25] * 4)
    tree = [(-1, -1), (-1, -1), (0, 1)]
    t = np.array([0.1, 0.25, 0.0])
    states = np.array([[2, 1], [2, 3]])  # same, different
    r = lk.evaluate(tree, 2, t, Q, pi, np.ones(1), np.ones(1), _tips(states, 4), np.ones(2), keep_site_derivatives=True)
    # printed values
    assert abs(r["site_logl"][0] - G["jc69.same"][0]) < 1e-13
    assert abs(r["site_logl"][1] - G["jc69.diff"][0]) < 1e-13
    for k in (0, 1):
        assert abs(r["site_derivs"][k, 0] - G["jc69.same"][1]) < 1e-13
        assert abs(r["site_derivs"][k, 1] - G["jc69.diff"][1]) < 1e-13
    # the formula itself, with rate categories: average l over r_c T
    rates, w = _gamma4()
    T = 0.35
    e = np.exp(-4.0 * rates * T / 3.0)
    same = np.sum(w * 0.25 * (0.25 + 0.75 * e))
    diff = np.sum(w * 0.25 * (0.25 - 0.25 * e))
    dsame = np.sum(w * 0.25 * 0.75 * e * (-4.0 * rates / 3.0)) / same
    ddiff = np.sum(w * 0.25 * -0.25 * e * (-4.0 * rates / 3.0)) / diff
    r = lk.evaluate(tree, 2, t, Q, pi, rates, w, _tips(states, 4), np.ones(2), keep_site_derivatives=True)
    assert np.allclose(r["site_logl"], np.log([same, diff]), rtol=0, atol=1e-14)
    assert np.allclose(r["site_derivs"][0], [dsame, ddiff], rtol=1e-13)
    assert np.allclose(r["site_derivs"][1], [dsame, ddiff], rtol=1e-13)


def _worked(gold, tree, root, t, Q, pi, S, parse):
    n_tips = (len(tree) + 1) // 2
    n_cases = len([k for k in gold if k.endswith(".tips")])
    for cn, (rates, w) in {"c1": (np.ones(1), np.ones(1)), "c4": _gamma4()}.items():
        for i in range(n_cases):
            tips = [parse(x) for x in gold[f"case{i}.tips"]]
            r = lk.evaluate(tree, root, t, Q, pi, rates, w, _tips([[z] for z in tips], S), np.ones(1))
            assert abs(r["logL"] - gold[f"case{i}.{cn}.logl"][0]) < 2e-12
            assert np.abs(r["grad"][: 2 * n_tips - 2] - np.array(gold[f"case{i}.{cn}.grad"])).max() < 2e-12


def test_worked_example_w1():
    Q, pi = models.hky(2.0, [0.1, 0.2, 0.3, 0.4])
    _worked(W1, TREE4, 6, T4, Q, pi, 4, lambda x: int(x))


def test_weighted_sums_and_conditioning_from_the_printed_w1_values():
    """evaluate() on all five W1 patterns at once with pattern weights != 1: logL = sum_p omega_p logl_p,
    grad_k = sum_p omega_p d_kp and cond_k = A_k = sum_p omega_p |d_kp| must equal the same sums
    formed from the PRINTED per-pattern values (tests/golden/w1_nucleotide.txt).  Patterns 0, 2, 4 have negative and
    positive derivatives on the same branch, so dropping the weight, the absolute value or the sign shows."""
    Q, pi = models.hky(2.0, [0.1, 0.2, 0.3, 0.4])
    omega = np.array([3.0, 1.0, 7.0, 2.0, 5.0])
    for cn, (rates, w) in {"c1": (np.ones(1), np.ones(1)), "c4": _gamma4()}.items():
        tips = np.array([[int(x) for x in W1[f"case{i}.tips"]] for i in range(5)]).T  # [tip][pattern]
        d = np.array([W1[f"case{i}.{cn}.grad"] for i in range(5)])                      # [pattern][branch 0..5]
        ll = np.array([W1[f"case{i}.{cn}.logl"][0] for i in range(5)])
        r = lk.evaluate(TREE4, 6, T4, Q, pi, rates, w, _tips(tips, 4), omega, chunk=2, keep_site_derivatives=True)
        assert abs(r["logL"] - np.dot(omega, ll)) < 1e-11
        assert np.abs(r["grad"][:6] - omega @ d).max() < 1e-11
        assert np.abs(r["cond"][:6] - omega @ np.abs(d)).max() < 1e-11
        assert np.all(r["cond"][:6] > np.abs(r["grad"][:6]) + 1.0)  # mixed signs: A_k is not |g_k|
        assert r["grad"][6] == 0.0 and r["cond"][6] == 0.0
        assert np.abs(r["site_derivs"][:6].T - d).max() < 2e-12


def test_worked_example_w2():
    Q, pi = models.gy94(2.0, 0.3, (0.1, 0.2, 0.3, 0.4), (0.4, 0.3, 0.2, 0.1), (0.25,) * 4)
    cod = models.codon_states()
    _worked(W2, TREE3, 4, T3, Q, pi, 61, lambda x: cod.index(x) if x in cod else 61)


def _random_case(S, seed, n_pat=6):
    rng = np.random.default_rng(seed)
    if S == 4:
        Q, pi = models.gtr(rng.gamma(2, 1, 6), rng.dirichlet([10] * 4))
    else:
        Q, pi = models.gy94(2.0, 0.3, rng.dirichlet([10] * 4), rng.dirichlet([10] * 4), rng.dirichlet([10] * 4))
    states = rng.integers(0, S, size=(5, n_pat))
    states[1, 0] = S  # one missing tip cell
    states[:, 1] = states[0, 1]  # one constant column
    wts = rng.integers(1, 11, size=n_pat).astype(float)
    return Q, pi, states, wts


@pytest.mark.parametrize("S", [4, 61])
def test_gradient_equals_central_differences_every_branch(S):
    Q, pi, states, wts = _random_case(S, 21)
    rates, w = _gamma4()
    tips = _tips(states, S)
    r = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, tips, wts)
    # step 1e-4 * max(t, 1e-2): FD round-off ~ eps |logL| / h ~ 1e-8, truncation ~ h^2 f''' / 6 far below that
    fd = lk.finite_difference_gradient(TREE5, 8, T5, Q, pi, rates, w, tips, wts, rel_step=1e-4)
    assert np.abs(r["grad"][:8] - fd[:8]).max() <= 2e-7 * np.abs(fd[:8]).max()
    # pulley: the two root children share one effective branch under a reversible model
    assert abs(r["grad"][6] - r["grad"][7]) < 1e-12 * max(1.0, abs(r["grad"][6]))
    # Euler identity: sum_k t_k g_k = d logL / d log mu for a global branch-length scale mu (FD on mu)
    h = 1e-6
    up = lk.evaluate(TREE5, 8, T5 * (1 + h), Q, pi, rates, w, tips, wts, gradient=False)["logL"]
    dn = lk.evaluate(TREE5, 8, T5 * (1 - h), Q, pi, rates, w, tips, wts, gradient=False)["logL"]
    assert abs(np.dot(T5, r["grad"]) - (up - dn) / (2 * h)) < 1e-6 * max(1.0, abs(np.dot(T5, r["grad"])))


def test_gradient_above_all_missing_tip_is_zero():
    Q, pi, states, wts = _random_case(4, 22)
    states[3, :] = 4
    r = lk.evaluate(TREE5, 8, T5, Q, pi, *_gamma4(), _tips(states, 4), wts)
    assert abs(r["grad"][3]) < 1e-14


@pytest.mark.parametrize("S", [4, 61])
def test_inner_product_of_pre_and_post_equals_likelihood_at_every_node(S):
    """the likelihood is the inner product of the post- and pre-order partials (at any node)."""
    Q, pi, states, _ = _random_case(S, 23)
    rates, w = _gamma4()
    U, Uinv, lam = models.eigen_decomposition(Q, pi)
    P = {k: lk.transition_matrices(U, Uinv, lam, rates, T5[k]) for k in range(8)}
    tips = _tips(states, S)
    for rescale in (True, False):
        p, log_m = lk.post_order(TREE5, 8, P, tips, 4, rescale=rescale)
        site = lk.site_log_likelihoods(p[8], pi, w, log_m)
        q, log_mq = lk.pre_order(TREE5, 8, P, p, pi, rescale=rescale)
        parent = {c: i for i, ch in enumerate(TREE5) for c in ch if c >= 0}
        for k in range(9):
            inner = sum(w[c] * np.sum(q[k][c] * p[k][c], axis=1) for c in range(4))
            # Restoring scale factors: q_k and p_k are built from the *rescaled* partials of every internal node
            # except the ancestors of k (an ancestor's own partial is never used on the way to k), each exactly
            # once, plus q's own factors log_mq[k].
            anc = set()
            m = k
            while m in parent:
                m = parent[m]
                anc.add(m)
            used = sum(v for kk, v in log_m.items() if kk not in anc)
            assert np.abs(np.log(inner) + log_mq[k] + used - site).max() < 1e-12, (k, rescale)


def test_child_order_and_rerooting_leave_logl_unchanged():
    Q, pi, states, wts = _random_case(4, 24)
    rates, w = _gamma4()
    tips = _tips(states, 4)
    a = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, tips, wts)
    swapped = [(-1, -1)] * 5 + [(1, 0), (2, 5), (4, 3), (7, 6)]
    b = lk.evaluate(swapped, 8, T5, Q, pi, rates, w, tips, wts)
    assert abs(a["logL"] - b["logL"]) < 1e-12 * abs(a["logL"])
    assert np.abs(a["grad"] - b["grad"]).max() < 1e-11
    t2 = T5.copy()
    t2[6], t2[7] = T5[6] + T5[7] - 0.01, 0.01  # slide the root along its edge
    c = lk.evaluate(TREE5, 8, t2, Q, pi, rates, w, tips, wts, gradient=False)
    assert abs(a["logL"] - c["logL"]) < 1e-12 * abs(a["logL"])


def test_rescaling_on_off_agree_and_chunking_is_invisible():
    Q, pi, states, wts = _random_case(4, 25, n_pat=50)
    rates, w = _gamma4()
    tips = _tips(states, 4)
    a = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, tips, wts, rescale=True, keep_site_derivatives=True)
    b = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, tips, wts, rescale=False, chunk=7, keep_site_derivatives=True)
    assert np.abs(a["site_logl"] - b["site_logl"]).max() < 1e-13
    assert np.abs(a["site_derivs"] - b["site_derivs"]).max() < 1e-12
    assert np.abs(a["grad"] - b["grad"]).max() < 1e-11


def _log_space_caterpillar(n_tips, t, Q, pi, state):
    """Independent log-space pruning on the caterpillar ((((0,1),2),3),...) with every tip in `state`, one category,
    via scipy expm + logsumexp: log p_k[s] = log P[s,z] + logsumexp_x(log P[s,x] + log p_prev[x])."""
    from scipy.linalg import expm
    from scipy.special import logsumexp

    logP = np.log(expm(Q * t))
    cur = logP[:, state] + logP[:, state]
    for _ in range(2, n_tips):
        cur = logP[:, state] + logsumexp(logP + cur[None, :], axis=1)
    return logsumexp(np.log(pi) + cur)


def test_rescaling_is_necessary_on_a_deep_tree():
    n = 1500
    Q, pi = models.hky(2.0, [0.1, 0.2, 0.3, 0.4])
    children = [(-1, -1)] * n
    prev = 0
    for tip in range(1, n):
        children.append((prev, tip))
        prev = len(children) - 1
    root = len(children) - 1
    t = np.full(len(children), 0.7)
    t[root] = 0.0
    tips = _tips([[0]] * n, 4)
    one = np.ones(1)
    with np.errstate(under="ignore"):
        off = lk.evaluate(children, root, t, Q, pi, one, one, tips, one, gradient=False, rescale=False)
    on = lk.evaluate(children, root, t, Q, pi, one, one, tips, one, gradient=False, rescale=True)
    assert off["logL"] == -np.inf
    ref = _log_space_caterpillar(n, 0.7, Q, pi, 0)
    assert ref < -1000.0 and abs(on["logL"] - ref) < 1e-10 * abs(ref)
