"""Pins for oracle.likelihood.rate_matrix_cross_products / substitution_parameter_gradient (PAPER.md:29,
:45-47).  The paper prints no formula; DESIGN.md section 2 reading 14 derives the first-order approximation.  None of
the expected values below comes from the function under test:

  * exactness where the approximation is exact -- the direction dQ = Q (overall rate mu, Q(mu) = mu Q_0) commutes with
    Q, so sum_ij G_ij Q_ij must equal d logL / d mu, taken by CENTRAL DIFFERENCES of the (separately pinned) oracle
    likelihood, and also sum_b t_b g_b (Euler identity with the branch-length gradient).  A transposed G, a missing
    t_b, r_c, w_c or omega_p each break it;
  * element by element -- on a 3-taxon tree with short branches, G_ij against central differences, with respect to the
    single element Q_ij, of a BRUTE-FORCE likelihood built on scipy.linalg.expm (no eigendecomposition, no pruning);
    the discrepancy is the dropped commutator term, O(t) relative, and must shrink in proportion when all branch
    lengths are scaled down;
  * model parameters -- kappa of HKY, the exchangeabilities of GTR and omega of GY94 by the chain rule, against
    central differences of the oracle likelihood in those parameters: within 0.3 % / 3 % at branch lengths 1000 / 100
    times shorter than the configs' (first order: the error scales with them), within 30 % at the configs' own scale
    (the size of the dropped commutator term there; the approximation is what the paper's method computes)."""
import itertools

import numpy as np
import pytest

from oracle import likelihood as lk
from oracle import models

TREE3 = [(-1, -1)] * 3 + [(1, 2), (0, 3)]
T3 = np.array([0.1, 0.2, 0.3, 0.05, 0.0])
TREE5 = [(-1, -1)] * 5 + [(0, 1), (5, 2), (3, 4), (6, 7)]
T5 = np.array([0.11, 0.07, 0.31, 0.02, 0.45, 0.09, 0.13, 0.21, 0.0])


def _gamma4():
    return models.discrete_gamma(0.5, 4), np.full(4, 0.25)


def _tips(states, S):
    return {k: lk.tip_partials_from_states(np.asarray(s), S) for k, s in enumerate(states)}


def _logl(tree, root, t, Q, pi, rates, w, tips, omega):
    return lk.evaluate(tree, root, t, Q, pi, rates, w, tips, omega, gradient=False)["logL"]


@pytest.mark.parametrize("S", [4, 61])
def test_exact_in_the_commuting_direction(S):
    rng = np.random.default_rng(5 + S)
    if S == 4:
        Q, pi = models.gtr(rng.gamma(2, 1, 6), rng.dirichlet([10] * 4))
    else:
        Q, pi = models.gy94(2.0, 0.3, rng.dirichlet([10] * 4), rng.dirichlet([10] * 4), rng.dirichlet([10] * 4))
    rates, w = _gamma4()
    states = rng.integers(0, S, size=(5, 7))
    states[2, 3] = S  # a missing cell
    omega = rng.integers(1, 11, size=7).astype(float)
    tips = _tips(states, S)
    G = lk.rate_matrix_cross_products(TREE5, 8, T5, Q, pi, rates, w, tips, omega)
    h = 1e-6
    fd = (_logl(TREE5, 8, T5, Q * (1 + h), pi, rates, w, tips, omega) -
          _logl(TREE5, 8, T5, Q * (1 - h), pi, rates, w, tips, omega)) / (2 * h)
    assert abs(np.sum(G * Q) - fd) <= 1e-6 * abs(fd)  # limited by the finite difference itself
    g = lk.evaluate(TREE5, 8, T5, Q, pi, rates, w, tips, omega)["grad"]
    assert abs(np.sum(G * Q) - np.dot(T5, g)) <= 1e-11 * abs(fd)
    assert abs(np.sum(G.T * Q) - fd) > 1e-3 * abs(fd)  # the transposed matrix does not satisfy it


def _brute_force_logl(tree, root, t, Q, pi, rates, cat_w, states, omega):
    """log-likelihood by the plain sum over internal states with scipy's expm for an ARBITRARY (non-reversible) Q."""
    from scipy.linalg import expm

    S = Q.shape[0]
    n = len(tree)
    internal = [k for k in range(n) if tree[k][0] >= 0]
    total = 0.0
    for p in range(states.shape[1]):
        lik = 0.0
        for c, r in enumerate(rates):
            Pm = {k: expm(Q * r * t[k]) for k in range(n) if k != root}
            acc = 0.0
            for assign in itertools.product(range(S), repeat=len(internal)):
                st = dict(zip(internal, assign))
                term = pi[st[root]]
                for m in internal:
                    for ch in tree[m]:
                        term *= Pm[ch][st[m], st[ch]] if tree[ch][0] >= 0 else Pm[ch][st[m], states[ch, p]]
                acc += term
            lik += cat_w[c] * acc
        total += omega[p] * np.log(lik)
    return total


def test_elementwise_against_brute_force_and_first_order_convergence():
    Q, pi = models.hky(2.0, [0.1, 0.2, 0.3, 0.4])
    rates, w = np.array([0.5, 1.5]), np.array([0.4, 0.6])
    states = np.array([[0, 1, 3], [0, 2, 3], [1, 2, 0]])
    omega = np.array([2.0, 1.0, 3.0])
    errs = []
    for eps in (1.0, 0.1, 0.01):
        t = T3 * eps
        G = lk.rate_matrix_cross_products(TREE3, 4, t, Q, pi, rates, w, _tips(states, 4), omega)
        fd = np.zeros((4, 4))
        for i in range(4):
            for j in range(4):
                h = 1e-6
                Qp, Qm = Q.copy(), Q.copy()
                Qp[i, j] += h
                Qm[i, j] -= h
                fd[i, j] = (_brute_force_logl(TREE3, 4, t, Qp, pi, rates, w, states, omega) -
                            _brute_force_logl(TREE3, 4, t, Qm, pi, rates, w, states, omega)) / (2 * h)
        errs.append(np.max(np.abs(G - fd)) / np.max(np.abs(fd)))
    assert errs[0] < 0.2 and errs[1] < 0.03 and errs[2] < 0.003
    assert errs[1] < 0.2 * errs[0] and errs[2] < 0.2 * errs[1]  # first order: the error scales with the branch lengths


def _dq_dtheta(build, theta, h=1e-6):
    """[K, S, S] derivative of the (normalised) rate matrix with respect to each parameter, by central differences."""
    out = []
    for k in range(len(theta)):
        tp, tm = np.array(theta, float), np.array(theta, float)
        tp[k] += h
        tm[k] -= h
        out.append((build(tp)[0] - build(tm)[0]) / (2 * h))
    return np.array(out)


@pytest.mark.parametrize("model", ["HKY", "GTR", "GY94"])
def test_chain_rule_to_model_parameters(model):
    rng = np.random.default_rng(31)
    pi4 = rng.dirichlet([10] * 4)
    f = [rng.dirichlet([10] * 4) for _ in range(3)]
    if model == "HKY":
        theta, build, S = [2.0], (lambda th: models.hky(th[0], pi4)), 4
    elif model == "GTR":
        theta, build, S = list(rng.gamma(2, 1, 6)), (lambda th: models.gtr(th, pi4)), 4
    else:
        theta, build, S = [2.0, 0.3], (lambda th: models.gy94(th[0], th[1], *f)), 61
    Q, pi = build(theta)
    rates, w = _gamma4()
    states = rng.integers(0, S, size=(5, 12))
    if model == "GY94":
        # Codons that differ at two or three positions have Q_ij = 0: there P_ij(t) is itself second order in t and the
        # first-order approximation of dP has an O(1) relative error however short the branch (two tips moved to
        # different neighbours of one codon already make such a pair).  Columns as short-branch data look: one codon
        # per column and at most ONE tip moved to a single-nucleotide neighbour (a state with Q_ij > 0).
        for col in range(states.shape[1]):
            base = int(states[0, col])
            nb = np.nonzero(Q[base] > 0)[0]
            states[:, col] = base
            if rng.random() < 0.75:
                states[int(rng.integers(5)), col] = int(rng.choice(nb))
    omega = rng.integers(1, 11, size=12).astype(float)
    tips = _tips(states, S)
    dQ = _dq_dtheta(build, theta)
    for scale, tol in ((0.001, 0.003), (0.01, 0.03), (1.0, 0.3)):
        t = T5 * scale
        G = lk.rate_matrix_cross_products(TREE5, 8, t, Q, pi, rates, w, tips, omega)
        approx = lk.substitution_parameter_gradient(G, dQ)
        fd = np.zeros(len(theta))
        for k in range(len(theta)):
            h = 1e-5 * max(abs(theta[k]), 1.0)
            tp, tm = np.array(theta, float), np.array(theta, float)
            tp[k] += h
            tm[k] -= h
            Qp, _ = build(tp)
            Qm, _ = build(tm)
            fd[k] = (_logl(TREE5, 8, t, Qp, pi, rates, w, tips, omega) - _logl(TREE5, 8, t, Qm, pi, rates, w, tips, omega)) / (2 * h)
        print(model, scale, float(np.max(np.abs(approx - fd)) / np.max(np.abs(fd))))
        assert np.max(np.abs(approx - fd)) <= tol * np.max(np.abs(fd)), (model, scale, approx, fd)
