"""Test helper: run the CPU oracle on a `workloads.Workload` (inputs only are shared; the oracle rebuilds Q, pi and
the eigendecomposition from the raw model parameters with its own code).

`evaluate` runs in this process; `evaluate_pool` splits the pattern axis into chunks (patterns are conditionally
independent) and runs `oracle.likelihood.evaluate` on them in a pool of worker processes, so that the
FULL-size configs of BASELINE.json can be compared with the GPU on every pattern in well under a minute.  The
workers execute nothing but oracle/ code; sums over chunks are taken in chunk order."""
import multiprocessing as mp
import os
from concurrent.futures import ProcessPoolExecutor

import numpy as np

from oracle import likelihood as lk
from oracle import models


def children_list(tree):
    return [tuple(int(x) for x in tree.children[k]) for k in range(tree.n_nodes)]


def oracle_model(wl):
    Q, pi = models.rate_matrix(wl.model)
    return Q, pi


def tip_partials(wl, lo=0, hi=None, idx=None):
    S = wl.n_states
    hi = wl.n_patterns if hi is None else hi
    cols = slice(lo, hi) if idx is None else np.asarray(idx)
    return {k: lk.tip_partials_from_states(wl.tip_states[k, cols], S) for k in range(wl.tree.n_tips)}


def evaluate(wl, branch_lengths=None, gradient=True, keep_site_derivatives=False, lo=0, hi=None, rescale=True, idx=None):
    """Oracle on patterns lo..hi-1, or on the pattern subset `idx` (any order)."""
    Q, pi = oracle_model(wl)
    t = wl.tree.branch_length if branch_lengths is None else branch_lengths
    hi = wl.n_patterns if hi is None else hi
    w = wl.pattern_weights[lo:hi] if idx is None else wl.pattern_weights[np.asarray(idx)]
    return lk.evaluate(children_list(wl.tree), wl.tree.root, np.asarray(t), Q, pi, wl.rates, wl.cat_weights,
                       tip_partials(wl, lo, hi, idx), w, gradient=gradient, rescale=rescale,
                       keep_site_derivatives=keep_site_derivatives)


def oracle_eigen(wl):
    """The oracle's own eigendecomposition (U, Uinv, lam) of the oracle's own Q."""
    Q, pi = oracle_model(wl)
    return models.eigen_decomposition(Q, pi)


def oracle_transition_matrices(wl, branch_lengths=None):
    """{node: [C, S, S]} as the oracle forms them (8(c) step 2)."""
    U, Uinv, lam = oracle_eigen(wl)
    t = wl.tree.branch_length if branch_lengths is None else branch_lengths
    return {k: lk.transition_matrices(U, Uinv, lam, wl.rates, t[k]) for k in range(wl.tree.n_nodes) if k != wl.tree.root}


def _chunk_job(job):
    (children, root, t, model, rates, cat_w, states, weights, n_states, gradient, keep) = job
    try:  # one BLAS thread per worker: the pool is the parallelism
        from threadpoolctl import threadpool_limits

        limiter = threadpool_limits(limits=1)
    except Exception:  # pragma: no cover
        limiter = None
    Q, pi = models.rate_matrix(model)
    tips = {k: lk.tip_partials_from_states(states[k], n_states) for k in range(states.shape[0])}
    out = lk.evaluate(children, root, t, Q, pi, rates, cat_w, tips, weights, gradient=gradient,
                      keep_site_derivatives=keep)
    del limiter
    return out


def evaluate_pool(wl, branch_lengths=None, gradient=True, keep_site_derivatives=False, chunk=2048, workers=None,
                  lo=0, hi=None):
    """`evaluate` over patterns lo..hi-1 by pattern chunks in `workers` processes (default: all host cores).
    Returns the same dict (site_logl, logL, grad, cond, optionally site_derivs) plus "workers"."""
    hi = wl.n_patterns if hi is None else hi
    workers = workers or (os.cpu_count() or 1)
    t = np.asarray(wl.tree.branch_length if branch_lengths is None else branch_lengths, dtype=np.float64)
    children, root = children_list(wl.tree), int(wl.tree.root)
    jobs = [(children, root, t, wl.model, wl.rates, wl.cat_weights, np.ascontiguousarray(wl.tip_states[:, a:min(hi, a + chunk)]),
             wl.pattern_weights[a:min(hi, a + chunk)], wl.n_states, gradient, keep_site_derivatives)
            for a in range(lo, hi, chunk)]
    workers = max(1, min(workers, len(jobs)))
    if workers == 1:
        parts = [_chunk_job(j) for j in jobs]
    else:
        # spawn: the parent may hold a CUDA context and BLAS threads, neither of which survives a fork cleanly
        # (ProcessPoolExecutor raises BrokenProcessPool if a worker cannot start; mp.Pool would respawn forever)
        with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as pool:
            parts = list(pool.map(_chunk_job, jobs, chunksize=1))
    out = {"site_logl": np.concatenate([p["site_logl"] for p in parts]), "workers": workers}
    out["logL"] = float(np.sum(wl.pattern_weights[lo:hi] * out["site_logl"]))
    if gradient:
        out["grad"] = np.sum([p["grad"] for p in parts], axis=0)
        out["cond"] = np.sum([p["cond"] for p in parts], axis=0)
        if keep_site_derivatives:
            out["site_derivs"] = np.concatenate([p["site_derivs"] for p in parts], axis=1)
    return out


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
