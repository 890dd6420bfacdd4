"""Pins for oracle/models.py (no GPU).  Every expected value is a property fixed by the mathematics or a value
printed in SURVEY.md section 8(c) ("What pins each part", rows 1 and 7) and stored under tests/golden/."""
import numpy as np
import pytest
from scipy.linalg import expm

import golden_io
from oracle import likelihood as lk
from oracle import models

G = golden_io.load("model_constants.txt")
F1, F2, F3 = (0.1, 0.2, 0.3, 0.4), (0.4, 0.3, 0.2, 0.1), (0.25, 0.25, 0.25, 0.25)


def _all_models():
    rng = np.random.default_rng(7)
    return {
        "hky": models.hky(2.0, rng.dirichlet([10.0] * 4)),
        "gtr": models.gtr(rng.gamma(2.0, 1.0, size=6), rng.dirichlet([10.0] * 4)),
        "gy94": models.gy94(2.0, 0.3, rng.dirichlet([10.0] * 4), rng.dirichlet([10.0] * 4), rng.dirichlet([10.0] * 4)),
    }


@pytest.mark.parametrize("name", ["hky", "gtr", "gy94"])
def test_rate_matrix_invariants(name):
    Q, pi = _all_models()[name]
    S = Q.shape[0]
    assert S == (61 if name == "gy94" else 4)
    assert abs(pi.sum() - 1.0) < 1e-14
    assert np.abs(Q.sum(axis=1)).max() < 1e-14  # rows sum to 0
    assert np.abs(pi @ Q).max() < 1e-15  # stationarity
    flux = pi[:, None] * Q
    assert np.abs(flux - flux.T).max() < 1e-16  # detailed balance
    assert abs(-(pi * np.diag(Q)).sum() - 1.0) < 1e-14  # one expected substitution per unit time
    off = Q - np.diag(np.diag(Q))
    assert off.min() >= 0.0


def test_hky_printed_values():
    Q, _ = models.hky(2.0, [0.1, 0.2, 0.3, 0.4])
    assert np.allclose(Q[0], G["hky.q_row0"], rtol=0, atol=2e-15)
    lam = np.sort(np.linalg.eigvals(Q).real)[::-1]
    assert np.allclose(lam, G["hky.eigenvalues"], rtol=0, atol=5e-15)


def test_hky_is_gtr_special_case():
    pi = np.array([0.1, 0.2, 0.3, 0.4])
    Qh, _ = models.hky(3.5, pi)
    Qg, _ = models.gtr([1.0, 3.5, 1.0, 1.0, 3.5, 1.0], pi)  # AC AG AT CG CT GT: AG and CT are transitions
    assert np.abs(Qh - Qg).max() < 1e-15


def test_gtr_exchangeability_order():
    """rho order AC, AG, AT, CG, CT, GT: q_ij / pi_j recovers rho_ij up to the common normalisation."""
    pi = np.array([0.1, 0.2, 0.3, 0.4])
    rho = np.array([1.0, 2.0, 3.0, 4.0, 5.0, 6.0])
    Q, _ = models.gtr(rho, pi)
    R = Q / pi[None, :]
    got = np.array([R[0, 1], R[0, 2], R[0, 3], R[1, 2], R[1, 3], R[2, 3]])
    assert np.allclose(got / got[0], rho, rtol=1e-14)


def test_gy94_printed_values():
    Q, pi = models.gy94(2.0, 0.3, F1, F2, F3)
    cod = models.codon_states()
    idx = {c: i for i, c in enumerate(cod)}
    assert abs(pi[idx["ATG"]] - G["gy94.pi_ATG"][0]) < 1e-16
    assert abs(Q[idx["AAA"], idx["AAG"]] - G["gy94.q_AAA_AAG"][0]) < 1e-14
    assert abs(Q[idx["AAA"], idx["AAA"]] - G["gy94.q_AAA_AAA"][0]) < 1e-14
    _, _, lam = models.eigen_decomposition(Q, pi)
    lam = np.sort(lam)
    assert abs(lam[0] - G["gy94.lambda_min"][0]) < 1e-13
    assert abs(lam[-1]) < 1e-14
    assert abs(lam[-2] - G["gy94.lambda_largest_nonzero"][0]) < 1e-13


def test_codon_state_order_and_census():
    cod = models.codon_states()
    assert len(cod) == 61 and len(set(cod)) == 61
    assert [cod.index(c) for c in ("AAA", "ATG", "TGG", "TTT")] == [int(v) for v in G["codon.index_checks"]]
    assert all(c not in cod for c in ("TAA", "TAG", "TGA"))
    # census of ordered one-nucleotide neighbour pairs from the *rate matrix* (kappa, omega chosen to be separable)
    kappa, omega = 2.0, 0.3
    Q, pi = models.gy94(kappa, omega, [0.25] * 4, [0.25] * 4, [0.25] * 4)
    R = Q / pi[None, :]
    base = np.min(R[R > 0]) / omega  # smallest class is nonsyn-transversion = omega * base
    counts = {}
    for i in range(61):
        for j in range(61):
            if i != j and R[i, j] > 0:
                key = round(R[i, j] / base, 6)
                counts[key] = counts.get(key, 0) + 1
    total, syn_ts, syn_tv, non_ts, non_tv = [int(v) for v in G["codon.neighbour_census"]]
    assert sum(counts.values()) == total
    assert counts[round(kappa, 6)] == syn_ts
    assert counts[1.0] == syn_tv
    assert counts[round(kappa * omega, 6)] == non_ts
    assert counts[round(omega, 6)] == non_tv


def test_genetic_code_spot_checks():
    code = models.genetic_code()
    assert len(code) == 64 and sum(1 for v in code.values() if v == "*") == 3
    assert code["ATG"] == "M" and code["TGG"] == "W" and code["AAA"] == "K" and code["TTT"] == "F"
    assert code["GGG"] == "G" and code["CTG"] == "L" and code["ATA"] == "I" and code["AGA"] == "R"
    # degeneracy classes of the standard code: 2 singletons (M, W), 3 six-fold (L, S, R), 5 four-fold, 1 three-fold (I)
    from collections import Counter
    deg = Counter(Counter(v for v in code.values() if v != "*").values())
    assert deg == {1: 2, 2: 9, 3: 1, 4: 5, 6: 3}


def test_discrete_gamma():
    r = models.discrete_gamma(0.5, 4)
    assert np.allclose(r, G["gamma.rates"], rtol=1e-11)
    assert abs(r.mean() - 1.0) < 1e-14
    for alpha, n in ((0.5, 8), (2.0, 4), (1.0, 5)):
        rr = models.discrete_gamma(alpha, n)
        assert abs(rr.mean() - 1.0) < 1e-13 and np.all(np.diff(rr) > 0)
    # alpha -> infinity: all rates -> 1
    assert np.abs(models.discrete_gamma(1e6, 4) - 1.0).max() < 5e-3
    # brute-force quadrature of the bin means for alpha = 2 (smooth density)
    from scipy import integrate, stats
    a, n = 2.0, 4
    cuts = np.concatenate([[0.0], stats.gamma.ppf(np.arange(1, n) / n, a=a, scale=1 / a), [np.inf]])
    ref = [n * integrate.quad(lambda x: x * stats.gamma.pdf(x, a=a, scale=1 / a), cuts[i], cuts[i + 1])[0] for i in range(n)]
    assert np.allclose(models.discrete_gamma(a, n), ref, rtol=1e-9)


@pytest.mark.parametrize("name", ["hky", "gtr", "gy94"])
def test_transition_matrices(name):
    Q, pi = _all_models()[name]
    U, Uinv, lam = models.eigen_decomposition(Q, pi)
    S = Q.shape[0]
    assert np.abs(U @ Uinv - np.eye(S)).max() < 1e-12
    assert np.abs(U @ np.diag(lam) @ Uinv - Q).max() < 1e-13
    rates = np.array([0.3, 1.0, 2.5])
    P0 = lk.transition_matrices(U, Uinv, lam, rates, 0.0)
    assert np.abs(P0 - np.eye(S)[None]).max() < 1e-13
    for t in (0.01, 0.1, 1.3):
        P = lk.transition_matrices(U, Uinv, lam, rates, t)
        assert P.shape == (3, S, S)
        assert np.abs(P.sum(axis=2) - 1.0).max() < 1e-13
        for c, r in enumerate(rates):
            assert np.abs(P[c] - expm(Q * r * t)).max() < 1e-13  # library routine, different algorithm (Pade)
    Ps = lk.transition_matrices(U, Uinv, lam, rates, 0.2)
    Pt = lk.transition_matrices(U, Uinv, lam, rates, 0.5)
    Pst = lk.transition_matrices(U, Uinv, lam, rates, 0.7)
    for c in range(3):
        assert np.abs(Ps[c] @ Pt[c] - Pst[c]).max() < 1e-13  # Chapman-Kolmogorov
    Pinf = lk.transition_matrices(U, Uinv, lam, np.ones(1), 1e4)[0]
    assert np.abs(Pinf - pi[None, :]).max() < 1e-12  # rows -> stationary distribution


def test_general_reversible_20_states():
    """SURVEY 8(f)-2 (PAPER.md:59 amino-acid models): the S-state reversible model reduces to GTR at S = 4 (same
    exchangeability order AC, AG, AT, CG, CT, GT), and at S = 20 satisfies the defining properties -- rows sum to 0,
    detailed balance pi_i q_ij = pi_j q_ji, pi Q = 0, unit normalisation, q_ij / pi_j symmetric and equal to the given
    exchangeability up to the common normalisation -- and its eigendecomposition reconstructs it."""
    rng = np.random.default_rng(77)
    rho4, pi4 = rng.gamma(2, 1, 6), rng.dirichlet([10] * 4)
    assert np.array_equal(models.general_reversible(rho4, pi4)[0], models.gtr(rho4, pi4)[0])
    rho, pi = rng.gamma(2, 1, 190), rng.dirichlet([10] * 20)
    Q, pi_out = models.general_reversible(rho, pi)
    assert Q.shape == (20, 20) and np.array_equal(pi_out, pi)
    assert np.max(np.abs(Q.sum(axis=1))) < 1e-14 and np.max(np.abs(pi @ Q)) < 1e-15
    F = pi[:, None] * Q
    assert np.max(np.abs(F - F.T)) < 1e-16
    assert abs(-np.sum(pi * np.diag(Q)) - 1.0) < 1e-14
    ratio = Q / pi[None, :]
    mu = ratio[0, 1] / rho[0]
    assert abs(ratio[0, 19] / rho[18] - mu) < 1e-13 * mu and abs(ratio[1, 2] / rho[19] - mu) < 1e-13 * mu
    assert abs(ratio[18, 19] / rho[189] - mu) < 1e-13 * mu
    U, Uinv, lam = models.eigen_decomposition(Q, pi)
    assert np.max(np.abs(U @ np.diag(lam) @ Uinv - Q)) < 1e-13 and np.max(np.abs(U @ Uinv - np.eye(20))) < 1e-13
    assert abs(np.max(lam)) < 1e-14 and np.all(np.sort(lam)[:-1] < 0)
