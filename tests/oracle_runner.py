"""Test helper: run the CPU oracle on a `workloads.Workload` (inputs only are shared; the oracle rebuilds Q, pi and
the eigendecomposition from the raw model parameters with its own code)."""
import numpy as np

from oracle import likelihood as lk
from oracle import models


def children_list(tree):
    return [tuple(int(x) for x in tree.children[k]) for k in range(tree.n_nodes)]


def oracle_model(wl):
    Q, pi = models.rate_matrix(wl.model)
    return Q, pi


def tip_partials(wl, lo=0, hi=None):
    S = wl.n_states
    hi = wl.n_patterns if hi is None else hi
    return {k: lk.tip_partials_from_states(wl.tip_states[k, lo:hi], S) for k in range(wl.tree.n_tips)}


def evaluate(wl, branch_lengths=None, gradient=True, keep_site_derivatives=False, lo=0, hi=None, rescale=True):
    Q, pi = oracle_model(wl)
    t = wl.tree.branch_length if branch_lengths is None else branch_lengths
    hi = wl.n_patterns if hi is None else hi
    return lk.evaluate(children_list(wl.tree), wl.tree.root, np.asarray(t), Q, pi, wl.rates, wl.cat_weights,
                       tip_partials(wl, lo, hi), wl.pattern_weights[lo:hi], gradient=gradient, rescale=rescale,
                       keep_site_derivatives=keep_site_derivatives)


def gradient_errors(g_gpu, ref):
    """The three figures of SURVEY 8(c) row 18: strict element-wise, relative to A_k, vector 2-norm."""
    g = ref["grad"]
    # a derivative that is exactly 0 (branch above an all-missing tip: Q.1 = 0) comes out of the fp64 oracle as
    # round-off (~1e-15); such entries have no relative error and are left to the /A_k and 2-norm figures
    nz = np.abs(g) > 1e-13 * max(float(np.max(np.abs(g))), 1e-300)
    d = np.abs(g_gpu - g)
    strict = float(np.max(d[nz] / np.abs(g[nz]))) if nz.any() else 0.0
    cond = ref["cond"]
    cz = cond > 1e-13 * max(float(np.max(cond)), 1e-300)  # A_k of an analytically-zero branch is round-off too
    rel_cond = float(np.max(d[cz] / cond[cz])) if cz.any() else 0.0
    norm = float(np.linalg.norm(g_gpu - g) / max(np.linalg.norm(g), 1e-300))
    return strict, rel_cond, norm
