"""Oracle, steps 2-8 of SURVEY.md section 8(c): transition matrices, post-order pruning with per-pattern
rescaling, root log-likelihood, pre-order partials, branch-length gradient, central finite differences.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Plain fp64 numpy, one node at a time, arrays in the paper-facing
layout [category c, pattern p, state s]; the only library primitive is a matrix product (np.matmul) used for the
S x S matrix-vector products, one per (node, category).  No blocking, fusion or reordering beyond a loop over
chunks of independent patterns (to bound host memory) in `evaluate`.

Also the approximate gradient with respect to the elements of the rate matrix and its chain rule
to substitution-model parameters, see `rate_matrix_cross_products`.

Passages followed: PAPER.md:27 (Felsenstein's pruning algorithm gives the likelihood of the data on a tree);
PAPER.md:43 (a pre-order traversal complements the post-order one; the likelihood is the inner product of post- and
pre-order partials; the gradient w.r.t. all branch-length-specific parameters takes one pre-order traversal);
PAPER.md:101 (transition matrices from the eigendecomposition of Q, cached for reuse across patterns; the gradient
is a sandwich of pre-order partial, rate matrix Q and post-order partial).  The paper is silent on rate categories,
rescaling, pattern weights and missing data; readings are SURVEY.md 8(c) rows 1, 2, 8-11, 14, 15.

Notation: p_k post-order partial of node k, q_k pre-order partial, P_{k,c} = exp(Q r_c t_k)
transition matrix of the branch above k in category c with P[parent state, child state], pi root frequencies,
w_c category weights, r_c category rates, omega_p pattern weights, m_k[p] rescaling factor.
"""
import numpy as np


# ---------------------------------------------------------------------------------------------- step 2
def transition_matrices(U, Uinv, lam, rates, t):
    """P_c = U diag(exp(lam r_c t)) Uinv for every category c (8(c) step 2).  No clamping."""
    return np.stack([U @ np.diag(np.exp(lam * (r * t))) @ Uinv for r in rates])


def tip_partials_from_states(states, n_states):
    """[P] state codes -> [P, S] one-hot rows; code S (or above) = missing -> all ones (8(c) step 3, row 15)."""
    states = np.asarray(states)
    out = np.zeros((states.shape[0], n_states))
    for p in range(states.shape[0]):
        if states[p] >= n_states:
            out[p, :] = 1.0
        else:
            out[p, states[p]] = 1.0
    return out


def _matvec(M, v):
    """(M v)[c,p,s] = sum_x M[c,s,x] v[c,p,x]"""
    return np.matmul(v, np.swapaxes(M, 1, 2))


def _matvec_transposed(M, v):
    """(M^T v)[c,p,s] = sum_x M[c,x,s] v[c,p,x]"""
    return np.matmul(v, M)


def _post_order_sequence(children, root):
    order = []
    stack = [(root, False)]
    while stack:
        node, expanded = stack.pop()
        if children[node][0] < 0:
            continue
        if expanded:
            order.append(node)
        else:
            stack.append((node, True))
            stack.append((children[node][1], False))
            stack.append((children[node][0], False))
    return order


# ---------------------------------------------------------------------------------------------- steps 3-4
def post_order(children, root, P, tip_partials, n_categories, rescale=True):
    """Felsenstein pruning (8(a) step 2) with per-pattern rescaling (8(a) step 3).

    children[k] = (i, j) or (-1, -1) for tips; P[k] = [C, S, S]; tip_partials[k] = [Pn, S] for tips.
    Returns (p, log_m): p[k] = [C, Pn, S] for every node, log_m[k] = [Pn] natural-log factors (internal nodes)."""
    p = {}
    log_m = {}
    for k in range(len(children)):
        if children[k][0] < 0:
            p[k] = np.repeat(tip_partials[k][None, :, :], n_categories, axis=0)
    for k in _post_order_sequence(children, root):
        i, j = children[k]
        pk = _matvec(P[i], p[i]) * _matvec(P[j], p[j])
        if rescale:
            m = pk.max(axis=(0, 2))
            safe = np.where(m > 0.0, m, 1.0)  # m == 0: leave the zeros; site log-likelihood becomes -inf
            pk = pk / safe[None, :, None]
            log_m[k] = np.log(safe)
        else:
            log_m[k] = np.zeros(pk.shape[1])
        p[k] = pk
    return p, log_m


# ---------------------------------------------------------------------------------------------- step 5
def site_log_likelihoods(p_root, pi, cat_weights, log_m):
    """log l_p = log(sum_c w_c sum_s pi_s p_root[c,p,s]) + sum_k log m_k[p]   (8(a) step 4)."""
    lik = np.zeros(p_root.shape[1])
    for c in range(p_root.shape[0]):
        lik = lik + cat_weights[c] * (p_root[c] @ pi)
    cum = np.zeros(p_root.shape[1])
    for k in log_m:
        cum = cum + log_m[k]
    with np.errstate(divide="ignore"):
        return np.log(lik) + cum


# ---------------------------------------------------------------------------------------------- step 6
def pre_order(children, root, P, p, pi, rescale=True):
    """Pre-order partials (8(a) step 5): q_root = pi for every (c, p); for child k of m with sibling j
    q_k[c,p,s] = sum_x P_k[c][x,s] ( q_m[c,p,x] * sum_y P_j[c][x,y] p_j[c,p,y] ).
    Each q_k is rescaled per pattern by its own maximum; the log factors are returned only so that tests can
    check the inner-product invariant -- the gradient does not need them (they cancel in num/den)."""
    C, Pn, S = p[root].shape
    q = {root: np.broadcast_to(pi[None, None, :], (C, Pn, S)).copy()}
    log_mq = {root: np.zeros(Pn)}
    for m in reversed(_post_order_sequence(children, root)):
        i, j = children[m]
        for k, sib in ((i, j), (j, i)):
            u = q[m] * _matvec(P[sib], p[sib])
            qk = _matvec_transposed(P[k], u)
            if rescale:
                mx = qk.max(axis=(0, 2))
                safe = np.where(mx > 0.0, mx, 1.0)
                qk = qk / safe[None, :, None]
                log_mq[k] = log_mq[m] + np.log(safe)
            else:
                log_mq[k] = log_mq[m].copy()
            q[k] = qk
    return q, log_mq


# ---------------------------------------------------------------------------------------------- step 7
def branch_site_derivatives(qk, pk, Q, rates, cat_weights):
    """d_{k,p} = num_p / den_p with num_p = sum_c w_c r_c q_k[c,p]^T Q p_k[c,p] and den_p = sum_c w_c q_k[c,p]^T
    p_k[c,p]  (PAPER.md:101 sandwich; 8(a) step 6).  Scale factors of q_k and p_k cancel."""
    num = np.zeros(qk.shape[1])
    den = np.zeros(qk.shape[1])
    for c in range(qk.shape[0]):
        Qp = pk[c] @ Q.T  # (Q p)[p, s] = sum_x Q[s,x] p[p,x]
        num = num + cat_weights[c] * rates[c] * np.sum(qk[c] * Qp, axis=1)
        den = den + cat_weights[c] * np.sum(qk[c] * pk[c], axis=1)
    with np.errstate(divide="ignore", invalid="ignore"):
        return num / den, num, den


# ---------------------------------------------------------------------------------------------- 8(f)-1
def rate_matrix_cross_products(children, root, branch_lengths, Q, pi, rates, cat_weights, tip_partials,
                               pattern_weights, eigen=None):
    """Approximate gradient of logL with respect to every ELEMENT of the rate matrix ("the gradient
    w.r.t. elements of the rate matrix ... exploiting a first-order approximation of the derivative of the matrix
    exponential"; DESIGN.md section 2 reading 14).

    The likelihood of pattern p is, for ANY branch b (node b below its parent m, sibling j),
        l_p = sum_c w_c u_b[c,p]^T P_{b,c} p_b[c,p],   u_b = q_m o (P_j p_j),   q_b = P_{b,c}^T u_b
    and P_{b,c} = exp(Q r_c t_b) enters l_p once per branch, so d l_p / d Q_ij = sum_b sum_c w_c u_b^T (d P_{b,c} / d Q_ij) p_b.
    First-order approximation (the commutator terms of the exact integral are dropped):
        d exp(Q tau) / d Q_ij  ~=  tau exp(Q tau) E_ij           (E_ij = unit matrix element, tau = r_c t_b)
    which turns the sandwich into an outer product of the pre- and post-order partials of the SAME node:
        G_ij = sum_b t_b sum_p omega_p ( sum_c w_c r_c q_b[c,p,i] p_b[c,p,j] ) / ( sum_c w_c q_b[c,p]^T p_b[c,p] ).
    It is exact in every direction dQ that commutes with Q (e.g. dQ = Q: the derivative with respect to an overall
    rate).  Per-pattern scale factors of q_b and p_b cancel in the quotient.  Returns G [S, S] (diagonal included: the
    chain rule below decides how the diagonal depends on the parameters)."""
    from .models import eigen_decomposition

    n_nodes = len(children)
    n_tips = (n_nodes + 1) // 2
    C = len(rates)
    S = Q.shape[0]
    U, Uinv, lam = eigen if eigen is not None else eigen_decomposition(Q, pi)
    P = {k: transition_matrices(U, Uinv, lam, rates, branch_lengths[k]) for k in range(n_nodes) if k != root}
    tips = {k: tip_partials[k] for k in range(n_tips)}
    p, _ = post_order(children, root, P, tips, C)
    q, _ = pre_order(children, root, P, p, pi)
    G = np.zeros((S, S))
    for b in range(n_nodes):
        if b == root:
            continue
        den = np.zeros(p[b].shape[1])
        for c in range(C):
            den = den + cat_weights[c] * np.sum(q[b][c] * p[b][c], axis=1)
        for c in range(C):
            scale = pattern_weights * (cat_weights[c] * rates[c] * branch_lengths[b]) / den  # [Pn]
            G = G + (q[b][c] * scale[:, None]).T @ p[b][c]  # sum_p scale_p q[p, i] p[p, j]
    return G


def substitution_parameter_gradient(G, dQ):
    """Chain rule: d logL / d theta_k ~= sum_ij G_ij dQ_ij / d theta_k, dQ [K, S, S] (O(K S^2))."""
    return np.einsum("ij,kij->k", G, np.asarray(dQ))


# ---------------------------------------------------------------------------------------------- driver
def evaluate(children, root, branch_lengths, Q, pi, rates, cat_weights, tip_partials, pattern_weights,
             gradient=True, rescale=True, chunk=8192, keep_site_derivatives=False, eigen=None):
    """Whole evaluation on all patterns, chunk by chunk (patterns are independent).

    tip_partials: dict/list tip -> [P, S].  Returns a dict with
      site_logl [P], logL, and if `gradient`: grad [n_nodes] (0 at the root), cond [n_nodes] = A_k = sum_p
      omega_p |d_{k,p}| (8(c) step 7), and optionally site_derivs [n_nodes, P]."""
    from .models import eigen_decomposition

    n_nodes = len(children)
    n_tips = (n_nodes + 1) // 2
    C = len(rates)
    U, Uinv, lam = eigen if eigen is not None else eigen_decomposition(Q, pi)
    P = {k: transition_matrices(U, Uinv, lam, rates, branch_lengths[k]) for k in range(n_nodes) if k != root}
    n_pat = tip_partials[0].shape[0]
    site_logl = np.zeros(n_pat)
    grad = np.zeros(n_nodes)
    cond = np.zeros(n_nodes)
    site_derivs = np.zeros((n_nodes, n_pat)) if (gradient and keep_site_derivatives) else None
    for lo in range(0, n_pat, chunk):
        hi = min(n_pat, lo + chunk)
        tips = {k: tip_partials[k][lo:hi] for k in range(n_tips)}
        p, log_m = post_order(children, root, P, tips, C, rescale=rescale)
        site_logl[lo:hi] = site_log_likelihoods(p[root], pi, cat_weights, log_m)
        if gradient:
            q, _ = pre_order(children, root, P, p, pi, rescale=rescale)
            w = pattern_weights[lo:hi]
            for k in range(n_nodes):
                if k == root:
                    continue
                d, _, _ = branch_site_derivatives(q[k], p[k], Q, rates, cat_weights)
                grad[k] += np.sum(w * d)
                cond[k] += np.sum(w * np.abs(d))
                if site_derivs is not None:
                    site_derivs[k, lo:hi] = d
    out = {"site_logl": site_logl, "logL": float(np.sum(pattern_weights * site_logl))}
    if gradient:
        out["grad"] = grad
        out["cond"] = cond
        if site_derivs is not None:
            out["site_derivs"] = site_derivs
    return out


# ---------------------------------------------------------------------------------------------- step 8
def finite_difference_gradient(children, root, branch_lengths, Q, pi, rates, cat_weights, tip_partials,
                               pattern_weights, rel_step=1e-6):
    """Central differences (logL(t_k + h) - logL(t_k - h)) / 2h, h = rel_step * max(t_k, 1e-2), every branch
    (8(c) step 8; the O(N^2) numerical gradient the paper's method replaces)."""
    from .models import eigen_decomposition

    eig = eigen_decomposition(Q, pi)
    g = np.zeros(len(children))
    for k in range(len(children)):
        if k == root:
            continue
        h = rel_step * max(branch_lengths[k], 1e-2)
        vals = []
        for sgn in (+1.0, -1.0):
            t = np.array(branch_lengths, dtype=np.float64)
            t[k] = t[k] + sgn * h
            vals.append(evaluate(children, root, t, Q, pi, rates, cat_weights, tip_partials, pattern_weights,
                                 gradient=False, eigen=eig)["logL"])
        g[k] = (vals[0] - vals[1]) / (2.0 * h)
    return g
