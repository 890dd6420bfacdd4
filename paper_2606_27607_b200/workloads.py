"""Seeded synthetic workloads (the *client side* of the library) -- shared input data, no method arithmetic.

This module plays the role that BEAST X plays in the paper's benchmarks (section 3.1): it owns the
tree, the branch lengths, the substitution model and the alignment, and hands them to a likelihood library.  It
serves both the CUDA path and the CPU oracle with *inputs only*:

  * a random rooted binary tree (coalescent or Yule topology), branch lengths iid Exp(mean 0.1);
  * a substitution model (HKY / GTR / GY94-F3x4) as raw parameters, plus what a client must compute before it
    can call the library's `plk_set_eigen_decomposition` (the rate matrix and its eigendecomposition:
    "numerical eigendecomposition of the infinitesimal rate matrix", is client-side);
  * discrete-gamma category rates and weights;
  * site patterns simulated down the tree, integer pattern weights, a tip-ambiguity mask.

It contains none of the method's steps (no pruning, no rescaling, no root reduction, no pre-order pass, no
gradient).  Transition probabilities needed to *simulate* data come from
scipy.linalg.expm, a library routine, not from the library's or the oracle's eigen-reconstruction.
The oracle never imports this module; it rebuilds Q from the raw model parameters with its own code
(oracle/models.py), so a mistake here shows up as a parity failure rather than cancelling out.

Recipes follow SURVEY.md section 8(c) rows 1, 4-7, 12-15 and section 8(d); they stand in for the paper's own
alignments and BEAST XMLs, which are external and not available.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Tuple

import numpy as np

BASE_SEED = 20260627  # seed = BASE_SEED + config index

NUCLEOTIDES = "ACGT"
# Standard genetic code (NCBI translation table 1), codons in lexicographic A<C<G<T order, idx64 = 16 n1 + 4 n2 + n3.
_AA_TABLE_ACGT = (
    "KNKN" "TTTT" "RSRS" "IIMI"  # A**
    "QHQH" "PPPP" "RRRR" "LLLL"  # C**
    "EDED" "AAAA" "GGGG" "VVVV"  # G**
    "*Y*Y" "SSSS" "*CWC" "LFLF"  # T**
)


# --------------------------------------------------------------------------------------------------------------
# Trees
# --------------------------------------------------------------------------------------------------------------
@dataclass
class Tree:
    """Rooted binary tree.  Tips are 0..N-1, internal nodes N..2N-2 numbered in a post-order (children before
    parents), root = 2N-2.  `branch_length[k]` is the branch above node k (root entry is 0 and unused)."""

    n_tips: int
    children: np.ndarray  # int32 [2N-1, 2], -1 for tips
    parent: np.ndarray  # int32 [2N-1], -1 for root
    branch_length: np.ndarray  # float64 [2N-1]

    @property
    def n_nodes(self) -> int:
        return 2 * self.n_tips - 1

    @property
    def root(self) -> int:
        return 2 * self.n_tips - 2

    def internal_nodes(self) -> range:
        return range(self.n_tips, 2 * self.n_tips - 1)

    def levels(self) -> np.ndarray:
        """level[k] = 0 for tips, 1 + max(level of children) otherwise."""
        lvl = np.zeros(self.n_nodes, dtype=np.int32)
        for k in self.internal_nodes():
            a, b = self.children[k]
            lvl[k] = 1 + max(lvl[a], lvl[b])
        return lvl


def _relabel_postorder(n_tips: int, children_of: Dict[int, Tuple[int, int]], root: int, tip_ids: List[int]) -> Tree:
    """Relabel an arbitrary labelled binary tree: tips -> 0..N-1 (in the order of `tip_ids`), internals in post-order."""
    n_nodes = 2 * n_tips - 1
    new_id = {t: i for i, t in enumerate(tip_ids)}
    nxt = n_tips
    stack = [(root, False)]
    while stack:
        node, done = stack.pop()
        if node not in children_of:
            continue
        if done:
            new_id[node] = nxt
            nxt += 1
        else:
            stack.append((node, True))
            a, b = children_of[node]
            stack.append((b, False))
            stack.append((a, False))
    children = -np.ones((n_nodes, 2), dtype=np.int32)
    parent = -np.ones(n_nodes, dtype=np.int32)
    for node, (a, b) in children_of.items():
        k = new_id[node]
        children[k] = (new_id[a], new_id[b])
        parent[new_id[a]] = k
        parent[new_id[b]] = k
    assert nxt == n_nodes and new_id[root] == n_nodes - 1
    return Tree(n_tips, children, parent, np.zeros(n_nodes))


def coalescent_topology(n_tips: int, rng: np.random.Generator) -> Tree:
    """start with N lineages, merge a uniformly random pair until one remains."""
    live = list(range(n_tips))
    children_of: Dict[int, Tuple[int, int]] = {}
    nxt = n_tips
    while len(live) > 1:
        i, j = rng.choice(len(live), size=2, replace=False)
        a, b = live[int(i)], live[int(j)]
        children_of[nxt] = (a, b)
        live = [x for x in live if x != a and x != b] + [nxt]
        nxt += 1
    return _relabel_postorder(n_tips, children_of, live[0], list(range(n_tips)))


def yule_topology(n_tips: int, rng: np.random.Generator) -> Tree:
    """start with one leaf, split a uniformly random leaf until there are N."""
    leaves = [0]
    children_of: Dict[int, Tuple[int, int]] = {}
    nxt = 1
    while len(leaves) < n_tips:
        i = int(rng.integers(len(leaves)))
        node = leaves.pop(i)
        children_of[node] = (nxt, nxt + 1)
        leaves += [nxt, nxt + 1]
        nxt += 2
    return _relabel_postorder(n_tips, children_of, 0, sorted(leaves))


def caterpillar_topology(n_tips: int) -> Tree:
    """Maximally unbalanced tree ((((0,1),2),3),...): the deep input used to show that rescaling is necessary."""
    children_of: Dict[int, Tuple[int, int]] = {}
    prev = 0
    nxt = n_tips
    for t in range(1, n_tips):
        children_of[nxt] = (prev, t)
        prev = nxt
        nxt += 1
    return _relabel_postorder(n_tips, children_of, prev, list(range(n_tips)))


def draw_branch_lengths(tree: Tree, rng: np.random.Generator, mean: float = 0.1) -> None:
    t = rng.exponential(mean, size=tree.n_nodes)
    t[tree.root] = 0.0
    tree.branch_length = t


# --------------------------------------------------------------------------------------------------------------
# Substitution models (client side: parameters -> Q -> eigendecomposition handed to the library)
# --------------------------------------------------------------------------------------------------------------
def sense_codons() -> List[str]:
    """61 sense codons, lexicographic A<C<G<T, stops TAA/TAG/TGA removed."""
    out = []
    for i in range(64):
        if _AA_TABLE_ACGT[i] != "*":
            out.append(NUCLEOTIDES[i // 16] + NUCLEOTIDES[(i // 4) % 4] + NUCLEOTIDES[i % 4])
    return out


def _amino_acid(codon: str) -> str:
    i = 16 * NUCLEOTIDES.index(codon[0]) + 4 * NUCLEOTIDES.index(codon[1]) + NUCLEOTIDES.index(codon[2])
    return _AA_TABLE_ACGT[i]


def _is_transition(a: str, b: str) -> bool:
    return {a, b} in ({"A", "G"}, {"C", "T"})


def client_rate_matrix(model: dict) -> Tuple[np.ndarray, np.ndarray]:
    """Model parameters -> (Q, pi), Q normalised to one expected substitution per unit time."""
    name = model["name"]
    if name == "AA20":  # 20-state reversible model: exchangeabilities (upper triangle, row by row) x frequencies
        pi = np.asarray(model["pi"], dtype=np.float64)
        S = len(pi)
        R = np.zeros((S, S))
        R[np.triu_indices(S, 1)] = model["rho"]
        Q = (R + R.T) * pi[None, :]
    elif name in ("HKY", "GTR"):
        pi = np.asarray(model["pi"], dtype=np.float64)
        R = np.zeros((4, 4))
        if name == "HKY":
            for i in range(4):
                for j in range(4):
                    if i != j:
                        R[i, j] = model["kappa"] if _is_transition(NUCLEOTIDES[i], NUCLEOTIDES[j]) else 1.0
        else:
            pairs = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]  # AC AG AT CG CT GT
            for (i, j), r in zip(pairs, model["rho"]):
                R[i, j] = R[j, i] = r
        Q = R * pi[None, :]
    elif name == "GY94":
        codons = sense_codons()
        f = [np.asarray(model["f1"], float), np.asarray(model["f2"], float), np.asarray(model["f3"], float)]
        pi = np.array([np.prod([f[k][NUCLEOTIDES.index(c[k])] for k in range(3)]) for c in codons])
        pi = pi / pi.sum()
        S = len(codons)
        Q = np.zeros((S, S))
        for i, ci in enumerate(codons):
            for j, cj in enumerate(codons):
                diff = [k for k in range(3) if ci[k] != cj[k]]
                if len(diff) != 1:
                    continue
                k = diff[0]
                rate = pi[j]
                if _is_transition(ci[k], cj[k]):
                    rate *= model["kappa"]
                if _amino_acid(ci) != _amino_acid(cj):
                    rate *= model["omega"]
                Q[i, j] = rate
    else:
        raise ValueError(f"unknown model {name}")
    np.fill_diagonal(Q, 0.0)
    np.fill_diagonal(Q, -Q.sum(axis=1))
    Q = Q / (-(pi * np.diag(Q)).sum())
    return Q, pi


def client_eigen(Q: np.ndarray, pi: np.ndarray) -> Tuple[np.ndarray, np.ndarray, np.ndarray]:
    """Eigendecomposition of a reversible Q through its symmetrised form: Q = U diag(lam) Uinv (client-side)."""
    s = np.sqrt(pi)
    A = (s[:, None] * Q) / s[None, :]
    A = 0.5 * (A + A.T)
    lam, V = np.linalg.eigh(A)
    U = V / s[:, None]
    Uinv = V.T * s[None, :]
    return np.ascontiguousarray(U), np.ascontiguousarray(Uinv), lam


def discrete_gamma_rates(alpha: float, n_cat: int) -> np.ndarray:
    """Equal-weight discrete gamma, shape = rate = alpha, bin-MEAN rates; mean is exactly 1."""
    from scipy.special import gammainc
    from scipy.stats import gamma as gamma_dist

    cuts = gamma_dist.ppf(np.arange(1, n_cat) / n_cat, a=alpha, scale=1.0 / alpha)
    # integral_0^x t f(t) dt for Gamma(shape a, rate a) equals the regularised incomplete gamma P(a+1, a x)
    upper = np.concatenate([gammainc(alpha + 1.0, cuts * alpha), [1.0]])
    lower = np.concatenate([[0.0], upper[:-1]])
    return (upper - lower) * n_cat


# --------------------------------------------------------------------------------------------------------------
# Alignment simulation
# --------------------------------------------------------------------------------------------------------------
def _sample_rows(cdf_rows: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    u = rng.random(cdf_rows.shape[0])
    idx = (u[:, None] >= cdf_rows).sum(axis=1)
    return np.minimum(idx, cdf_rows.shape[1] - 1).astype(np.uint8)


def simulate_columns(tree: Tree, Q: np.ndarray, pi: np.ndarray, rates: np.ndarray, cat_weights: np.ndarray,
                     n_sites: int, rng: np.random.Generator) -> np.ndarray:
    """Simulate `n_sites` alignment columns down the tree: root state ~ pi, site category ~ w,
    child state ~ row of expm(Q r_c t_b).  Returns uint8 [N, n_sites] tip states."""
    from scipy.linalg import expm

    S = Q.shape[0]
    cat = np.sort(rng.choice(len(rates), size=n_sites, p=cat_weights))
    bounds = np.searchsorted(cat, np.arange(len(rates) + 1))
    state = np.zeros((tree.n_nodes, n_sites), dtype=np.uint8)
    pi_cdf = np.cumsum(pi)
    pi_cdf[-1] = 1.0
    state[tree.root] = _sample_rows(np.broadcast_to(pi_cdf, (n_sites, S)), rng)
    for node in range(tree.n_nodes - 2, -1, -1):  # parents have larger ids than children
        par = tree.parent[node]
        for c in range(len(rates)):
            lo, hi = bounds[c], bounds[c + 1]
            if hi == lo:
                continue
            Pm = expm(Q * (rates[c] * tree.branch_length[node]))
            cdf = np.cumsum(np.clip(Pm, 0.0, None), axis=1)
            cdf /= cdf[:, -1:]
            state[node, lo:hi] = _sample_rows(cdf[state[par, lo:hi]], rng)
    tips = state[: tree.n_tips]
    perm = rng.permutation(n_sites)  # undo the category sort so columns are exchangeable
    return np.ascontiguousarray(tips[:, perm])


def simulate_distinct_columns(tree, Q, pi, rates, cat_weights, n_patterns, rng) -> np.ndarray:
    """configs[0]: keep drawing until `n_patterns` distinct columns exist (order of first occurrence)."""
    seen = {}
    cols = []
    while len(cols) < n_patterns:
        batch = simulate_columns(tree, Q, pi, rates, cat_weights, max(256, n_patterns), rng)
        for j in range(batch.shape[1]):
            key = batch[:, j].tobytes()
            if key not in seen:
                seen[key] = True
                cols.append(batch[:, j])
                if len(cols) == n_patterns:
                    break
    return np.ascontiguousarray(np.stack(cols, axis=1))


# --------------------------------------------------------------------------------------------------------------
# Workloads = BASELINE.json configs
# --------------------------------------------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    tree: Tree
    model: dict  # raw parameters; the oracle rebuilds Q from these with its own code
    Q: np.ndarray  # client's rate matrix (for simulation and plk_set_rate_matrix)
    pi: np.ndarray
    U: np.ndarray
    Uinv: np.ndarray
    lam: np.ndarray
    rates: np.ndarray
    cat_weights: np.ndarray
    tip_states: np.ndarray  # uint8 [N, P]; value S = missing / fully ambiguous
    pattern_weights: np.ndarray  # float64 [P]
    seed: int
    notes: Dict[str, str] = field(default_factory=dict)

    @property
    def n_states(self) -> int:
        return self.Q.shape[0]

    @property
    def n_patterns(self) -> int:
        return self.tip_states.shape[1]

    @property
    def n_categories(self) -> int:
        return len(self.rates)

    def perturbed_branch_lengths(self, sigma: float = 0.5) -> np.ndarray:
        """seeded factor exp(N(0, sigma^2)) per branch -- evaluation away from the truth."""
        rng = np.random.default_rng(self.seed + 7919)
        t = self.tree.branch_length * np.exp(rng.normal(0.0, sigma, size=self.tree.n_nodes))
        t[self.tree.root] = 0.0
        return t


def draw_model(name: str, rng: np.random.Generator) -> dict:
    if name == "HKY":
        return {"name": "HKY", "kappa": 2.0, "pi": rng.dirichlet([10.0] * 4).tolist()}
    if name == "GTR":
        rho = rng.gamma(2.0, 1.0, size=6).tolist()
        return {"name": "GTR", "rho": rho, "pi": rng.dirichlet([10.0] * 4).tolist()}
    if name == "AA20":
        return {"name": "AA20", "rho": rng.gamma(2.0, 1.0, size=190).tolist(), "pi": rng.dirichlet([10.0] * 20).tolist()}
    if name == "GY94":
        return {"name": "GY94", "kappa": 2.0, "omega": 0.3,
                "f1": rng.dirichlet([10.0] * 4).tolist(), "f2": rng.dirichlet([10.0] * 4).tolist(),
                "f3": rng.dirichlet([10.0] * 4).tolist()}
    raise ValueError(name)


def make_workload(name: str, model_name: str, n_tips: int, n_patterns: int, topology: str, seed: int,
                  n_cat: int = 4, alpha: float = 0.5, ambiguity: float = 0.0, distinct: bool = False,
                  tree: Optional[Tree] = None) -> Workload:
    rng = np.random.default_rng(seed)
    if tree is None:
        if topology == "coalescent":
            tree = coalescent_topology(n_tips, rng)
        elif topology == "yule":
            tree = yule_topology(n_tips, rng)
        elif topology == "caterpillar":
            tree = caterpillar_topology(n_tips)
        else:
            raise ValueError(topology)
        draw_branch_lengths(tree, rng)
    model = draw_model(model_name, rng)
    Q, pi = client_rate_matrix(model)
    U, Uinv, lam = client_eigen(Q, pi)
    rates = discrete_gamma_rates(alpha, n_cat) if n_cat > 1 else np.ones(1)
    cat_w = np.full(n_cat, 1.0 / n_cat)
    if distinct:
        tips = simulate_distinct_columns(tree, Q, pi, rates, cat_w, n_patterns, rng)
    else:
        tips = simulate_columns(tree, Q, pi, rates, cat_w, n_patterns, rng)
    if ambiguity > 0.0:
        mask = rng.random(tips.shape) < ambiguity
        tips = np.where(mask, np.uint8(Q.shape[0]), tips).astype(np.uint8)
    weights = rng.integers(1, 11, size=n_patterns).astype(np.float64)
    return Workload(name, tree, model, Q, pi, U, Uinv, lam, rates, cat_w, np.ascontiguousarray(tips), weights, seed)


def config(index: int, n_tips: Optional[int] = None, n_patterns: Optional[int] = None,
           n_categories: int = 4) -> Workload:
    """BASELINE.json configs[index]; `n_tips`/`n_patterns` override the size (sweep points of configs[4], reduced
    parity cases).  Recipes: SURVEY.md section 8(d)."""
    seed = BASE_SEED + index
    if index == 0:
        return make_workload("cfg0_hky_8x1000", "HKY", n_tips or 8, n_patterns or 1000, "coalescent", seed, distinct=True)
    if index == 1:
        return make_workload("cfg1_gtr_128x100000", "GTR", n_tips or 128, n_patterns or 100_000, "yule", seed,
                             n_cat=n_categories, ambiguity=0.05)
    if index == 2:
        return make_workload("cfg2_gy94_32x10000", "GY94", n_tips or 32, n_patterns or 10_000, "coalescent", seed,
                             n_cat=n_categories)
    if index == 3:
        return make_workload("cfg3_gy94_256x20000", "GY94", n_tips or 256, n_patterns or 20_000, "coalescent", seed,
                             n_cat=n_categories)
    if index == 5:  # not a BASELINE config: the 20-state amino-acid shape of SURVEY 8(f)-2
        return make_workload("aa20_64x20000", "AA20", n_tips or 64, n_patterns or 20_000, "coalescent", seed,
                             n_cat=n_categories)
    if index == 4:
        n = n_tips or 512
        p = n_patterns or 500_000
        return make_workload(f"cfg4_hky_{n}x{p}", "HKY", n, p, "coalescent", seed + 1000 * n + (p % 997))
    raise ValueError(index)


SWEEP_TAXA = (8, 32, 128, 512)
SWEEP_PATTERNS = (100, 1_000, 10_000, 100_000, 500_000)


# --------------------------------------------------------------------------------------------------------------
# Raw alignments for the encode/compress step
# --------------------------------------------------------------------------------------------------------------
def random_alignment(kind: str, n_taxa: int, n_sites: int, seed: int, dup_fraction: float = 0.5,
                     gap_fraction: float = 0.03, lower_fraction: float = 0.2) -> List[bytes]:
    """Seeded character alignment with many duplicated columns, gaps/ambiguity codes and lower-case letters.
    `n_sites` counts nucleotide columns for kind='nuc' and codon columns for kind='codon'."""
    rng = np.random.default_rng(seed)
    if kind == "nuc":
        alphabet = [b"A", b"C", b"G", b"T", b"U"]
        junk = [b"-", b"N", b"?", b"R", b"Y"]
    else:
        alphabet = [c.encode() for c in sense_codons()]
        junk = [b"---", b"NNN", b"A-G", b"AN?", b"RAT"]
    n_base = max(1, int(n_sites * (1.0 - dup_fraction)))
    base_cols = []
    for _ in range(n_base):
        col = []
        for _t in range(n_taxa):
            tok = junk[int(rng.integers(len(junk)))] if rng.random() < gap_fraction else alphabet[int(rng.integers(len(alphabet)))]
            if rng.random() < lower_fraction:
                tok = tok.lower()
            col.append(tok)
        base_cols.append(col)
    pick = np.concatenate([np.arange(n_base), rng.integers(n_base, size=n_sites - n_base)])
    rng.shuffle(pick)
    return [b"".join(base_cols[j][t] for j in pick) for t in range(n_taxa)]
