"""Oracle, step 1 of SURVEY.md section 8(c): substitution model -> (Q, pi) -> eigendecomposition; discrete gamma.

TEST INFRASTRUCTURE (see oracle/__init__.py).  The paper names the models only (HKY PAPER.md:65, GY94 PAPER.md:65,
GTR PAPER.md:81) and says transition matrices come from "numerical eigendecomposition of the infinitesimal rate
matrix".  Definitions follow SURVEY.md 8(c) rows 3-7 ("readings"), pinned in
tests/test_oracle_models.py: rows sum to 0, pi Q = 0, detailed balance, unit normalisation, the printed HKY row /
eigenvalues, the printed GY94 entries / extreme eigenvalues, the 526 = 62+72+116+276 neighbour-pair census.
"""
import numpy as np

STATES_NUC = "ACGT"  # state codes 0..3

# NCBI translation table 1, written in the conventional T,C,A,G order (first base slowest).
_BASES_TCAG = "TCAG"
_AMINO_TCAG = "FFLLSSSSYY**CC*WLLLLPPPPHHQQRRRRIIIMTTTTNNKKSSRRVVVVAAAADDEEGGGG"


def genetic_code():
    """dict codon (str over ACGT) -> amino-acid letter or '*'."""
    code = {}
    n = 0
    for a in _BASES_TCAG:
        for b in _BASES_TCAG:
            for c in _BASES_TCAG:
                code[a + b + c] = _AMINO_TCAG[n]
                n += 1
    return code


def codon_states():
    """The 61 sense codons in state order: lexicographic with A<C<G<T, stop codons dropped (8(c) row 7)."""
    code = genetic_code()
    allc = [a + b + c for a in STATES_NUC for b in STATES_NUC for c in STATES_NUC]
    return [c for c in allc if code[c] != "*"]


def _transition(x, y):
    purine = "AG"
    return (x in purine) == (y in purine)  # x != y assumed: A<->G or C<->T


def _finish(R, pi):
    """Off-diagonal rates R -> Q with zero row sums, scaled so that -sum_i pi_i Q_ii = 1 (8(c) row 3)."""
    Q = np.array(R, dtype=np.float64)
    for i in range(Q.shape[0]):
        Q[i, i] = 0.0
        Q[i, i] = -np.sum(Q[i, :])
    mu = -np.sum(pi * np.diag(Q))
    return Q / mu


def hky(kappa, pi):
    """HKY85: q_ij = kappa pi_j for transitions (A<->G, C<->T), pi_j for transversions (8(c) row 4)."""
    pi = np.asarray(pi, dtype=np.float64)
    R = np.zeros((4, 4))
    for i, x in enumerate(STATES_NUC):
        for j, y in enumerate(STATES_NUC):
            if i != j:
                R[i, j] = (kappa if _transition(x, y) else 1.0) * pi[j]
    return _finish(R, pi), pi


def gtr(rho, pi):
    """GTR: q_ij = rho_ij pi_j, rho symmetric, given in the order AC, AG, AT, CG, CT, GT (8(c) row 5)."""
    pi = np.asarray(pi, dtype=np.float64)
    rac, rag, rat, rcg, rct, rgt = [float(r) for r in rho]
    sym = np.array([[0.0, rac, rag, rat], [rac, 0.0, rcg, rct], [rag, rcg, 0.0, rgt], [rat, rct, rgt, 0.0]])
    return _finish(sym * pi[None, :], pi), pi


def general_reversible(rho_upper, pi):
    """General time-reversible model on S = len(pi) states (the 20-state amino-acid models the paper's tensor-core
    claim covers): q_ij = rho_ij pi_j with rho symmetric, its S(S-1)/2 upper-triangle
    entries given row by row ((0,1), (0,2), ..., (S-2,S-1)).  GTR (8(c) row 5) is the case S = 4."""
    pi = np.asarray(pi, dtype=np.float64)
    S = pi.shape[0]
    rho = np.asarray(rho_upper, dtype=np.float64)
    assert rho.shape[0] == S * (S - 1) // 2
    sym = np.zeros((S, S))
    n = 0
    for i in range(S):
        for j in range(i + 1, S):
            sym[i, j] = sym[j, i] = rho[n]
            n += 1
    return _finish(sym * pi[None, :], pi), pi


def gy94(kappa, omega, f1, f2, f3):
    """GY94 with F3x4 frequencies (8(c) row 6): q_ij = 0 unless codons i, j differ at exactly one position; then
    pi_j, times kappa for a transition, times omega for a non-synonymous change.  pi_j ~ f1[n1] f2[n2] f3[n3]
    renormalised over the 61 sense codons."""
    code = genetic_code()
    cod = codon_states()
    f = [np.asarray(f1, float), np.asarray(f2, float), np.asarray(f3, float)]
    pi = np.array([f[0][STATES_NUC.index(c[0])] * f[1][STATES_NUC.index(c[1])] * f[2][STATES_NUC.index(c[2])] for c in cod])
    pi = pi / np.sum(pi)
    S = len(cod)
    R = np.zeros((S, S))
    for i in range(S):
        for j in range(S):
            if i == j:
                continue
            where = [k for k in range(3) if cod[i][k] != cod[j][k]]
            if len(where) != 1:
                continue
            k = where[0]
            q = pi[j]
            if _transition(cod[i][k], cod[j][k]):
                q = q * kappa
            if code[cod[i]] != code[cod[j]]:
                q = q * omega
            R[i, j] = q
    return _finish(R, pi), pi


def rate_matrix(model):
    """Dispatch on the raw-parameter dict used by the workloads ({"name": "HKY"|"GTR"|"GY94", ...})."""
    name = model["name"]
    if name == "HKY":
        return hky(model["kappa"], model["pi"])
    if name == "GTR":
        return gtr(model["rho"], model["pi"])
    if name == "AA20":
        return general_reversible(model["rho"], model["pi"])
    if name == "GY94":
        return gy94(model["kappa"], model["omega"], model["f1"], model["f2"], model["f3"])
    raise ValueError(name)


def eigen_decomposition(Q, pi):
    """Reversible Q: A = Pi^{1/2} Q Pi^{-1/2} is symmetric, A = V L V^T, so Q = U diag(L) Uinv with
    U = Pi^{-1/2} V and Uinv = V^T Pi^{1/2} (8(c) step 1).  Returns (U, Uinv, lam)."""
    root = np.sqrt(pi)
    A = np.diag(root) @ Q @ np.diag(1.0 / root)
    A = (A + A.T) / 2.0
    lam, V = np.linalg.eigh(A)
    U = np.diag(1.0 / root) @ V
    Uinv = V.T @ np.diag(root)
    return U, Uinv, lam


def discrete_gamma(alpha, n_cat):
    """Equal-probability discrete gamma with shape = rate = alpha and bin-mean rates (8(c) row 1).

    Bin c is (x_{c}, x_{c+1}) with x the c/n quantiles; its mean rate is n * integral of t f(t) dt over the bin,
    and integral_0^x t f(t) dt = P(alpha + 1, alpha x) (regularised lower incomplete gamma)."""
    from scipy.special import gammainc, gammaincinv

    probs = np.arange(1, n_cat) / float(n_cat)
    x = gammaincinv(alpha, probs) / alpha  # quantiles of Gamma(shape alpha, rate alpha)
    cum = np.concatenate([[0.0], gammainc(alpha + 1.0, alpha * x), [1.0]])
    return n_cat * np.diff(cum)
