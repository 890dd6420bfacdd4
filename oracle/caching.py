"""Oracle for the two caching variants of PAPER.md:101 (section 4, "improve the caching strategies during post- and
pre-order traversals").  TEST INFRASTRUCTURE (see oracle/__init__.py): plain fp64 numpy, written
in the paper's order, sharing no code with the CUDA path.

(a) Cached rate products.  "Since the infinitesimal rate matrix is already available during the post-order
    traversal, the product of the infinitesimal rate matrix and the post-order partial likelihood vector at each node
    could be cached directly thus reducing memory burden from S^2 elements of the infinitesimal rate matrix to S
    partial likelihoods."  During the post-order traversal every node k also stores  Qp_k[c,p,.] = Q p_k[c,p,.];
    the sandwich of the gradient step then needs no matrix:
        num_p = sum_c w_c r_c  q_k[c,p] . Qp_k[c,p],      den_p = sum_c w_c  q_k[c,p] . p_k[c,p].
    Qp_k is formed from the RESCALED p_k, so it carries the same per-pattern factor and num / den is unchanged.

(b) Transition matrices on the fly.  "for phylogeographic problems that typically have a large state-space size but
    only a single site pattern, the transition probability matrices are not reused, and it is more efficient to form
    the transition probability matrix on-the-fly while calculating the likelihood ... through Felsenstein's pruning
    algorithm."  Reading (reading 15): the S x S matrix P = U diag(exp(lambda r_c t)) U^-1 is
    never formed or stored; its three factors are applied to the child's partial one after the other,
        P p = U ( exp(lambda r_c t) o ( U^-1 p ) ),
    two matrix-vector products (4 S^2 flops) per child edge, pattern and category instead of the 2 S^3 flops of the
    matrix plus 2 S^2 of its use.  The result is the pruning recursion's, up to rounding order.

Both give results that have a plain definition (the log-likelihood, the branch-length derivative), so they are
pinned in tests/test_oracle_caching.py by the same independent facts as oracle/likelihood.py: the worked examples
W1 / W2 (tests/golden/), brute-force enumeration with scipy's expm, the JC69 closed form and central differences.
"""
import numpy as np

from .likelihood import _post_order_sequence


# ------------------------------------------------------------------------------------------ (a) cached Q p_k
def post_order_with_rate_products(children, root, P, tip_partials, n_categories, Q, rescale=True):
    """Felsenstein pruning as in likelihood.post_order, and at every node -- tips included -- the cached
    product Qp_k[c,p,s] = sum_x Q[s,x] p_k[c,p,x] of the rate matrix with the node's (rescaled) post-order partial
    (PAPER.md:101).  Returns (p, Qp, log_m)."""
    p, Qp, log_m = {}, {}, {}
    for k in range(len(children)):
        if children[k][0] < 0:
            p[k] = np.repeat(tip_partials[k][None, :, :], n_categories, axis=0)
            Qp[k] = np.stack([p[k][c] @ Q.T for c in range(n_categories)])
    for k in _post_order_sequence(children, root):
        i, j = children[k]
        pk = np.stack([(p[i][c] @ P[i][c].T) * (p[j][c] @ P[j][c].T) for c in range(n_categories)])
        if rescale:
            m = pk.max(axis=(0, 2))
            safe = np.where(m > 0.0, m, 1.0)
            pk = pk / safe[None, :, None]
            log_m[k] = np.log(safe)
        else:
            log_m[k] = np.zeros(pk.shape[1])
        p[k] = pk
        Qp[k] = np.stack([pk[c] @ Q.T for c in range(n_categories)])  # cached while Q is at hand
    return p, Qp, log_m


def branch_site_derivatives_cached(qk, Qpk, pk, rates, cat_weights):
    """d_{k,p} = num_p / den_p from the cached product: num_p = sum_c w_c r_c q_k[c,p] . Qp_k[c,p],
    den_p = sum_c w_c q_k[c,p] . p_k[c,p]: S values read per (node, pattern, category), no matrix."""
    num = np.zeros(qk.shape[1])
    den = np.zeros(qk.shape[1])
    for c in range(qk.shape[0]):
        num = num + cat_weights[c] * rates[c] * np.sum(qk[c] * Qpk[c], axis=1)
        den = den + cat_weights[c] * np.sum(qk[c] * pk[c], axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        return num / den, num, den


# ------------------------------------------------------------------------------------------ (b) matrices on the fly
def apply_branch_on_the_fly(U, Uinv, lam, rate, t, v):
    """(exp(Q rate t) v)[p,s] for row vectors v [Pn, S] without forming the matrix:
    y = U^-1 v;  y_i *= exp(lambda_i rate t);  result = U y."""
    y = v @ Uinv.T                      # y[p,i] = sum_x Uinv[i,x] v[p,x]
    y = y * np.exp(lam * (rate * t))[None, :]
    return y @ U.T                      # out[p,s] = sum_i U[s,i] y[p,i]


def post_order_on_the_fly(children, root, U, Uinv, lam, rates, branch_lengths, tip_partials, rescale=True):
    """Felsenstein pruning with the transition matrix of every child edge applied on the fly from the
    eigendecomposition -- no P_{b,c} is formed.  Same outputs as likelihood.post_order."""
    C = len(rates)
    p, log_m = {}, {}
    for k in range(len(children)):
        if children[k][0] < 0:
            p[k] = np.repeat(tip_partials[k][None, :, :], C, axis=0)
    for k in _post_order_sequence(children, root):
        i, j = children[k]
        pk = np.stack([apply_branch_on_the_fly(U, Uinv, lam, rates[c], branch_lengths[i], p[i][c]) *
                       apply_branch_on_the_fly(U, Uinv, lam, rates[c], branch_lengths[j], p[j][c]) for c in range(C)])
        if rescale:
            m = pk.max(axis=(0, 2))
            safe = np.where(m > 0.0, m, 1.0)
            pk = pk / safe[None, :, None]
            log_m[k] = np.log(safe)
        else:
            log_m[k] = np.zeros(pk.shape[1])
        p[k] = pk
    return p, log_m
