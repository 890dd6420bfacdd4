"""Client-side driver: turns a tree + model + alignment (a `workloads.Workload`) into calls of the library, the way
a tree-inference package drives BEAGLE (SURVEY.md section 3 call stack).

Only bookkeeping lives here -- which buffer holds which node, the post-order operation list, the pre-order operation
list.  Every number is computed by libplk.so.  Buffer convention used by this client: node k uses partials buffer
k, pre-order buffer k, matrix buffer k (the branch above k) and scale buffer k.
"""
from __future__ import annotations

from typing import Optional

import numpy as np

from . import plk


def post_order_ops(tree) -> np.ndarray:
    """One plk_op per internal node, children before parents (tree ids are already in post-order)."""
    ops = np.zeros(tree.n_tips - 1, dtype=plk.OP_DTYPE)
    for i, k in enumerate(tree.internal_nodes()):
        a, b = tree.children[k]
        ops[i] = (k, k, a, a, b, b)
    return ops


def pre_order_ops(tree, store_tips: bool = False) -> np.ndarray:
    """One plk_pre_op per non-root node, parents before children.  Tip pre-order partials are not stored unless
    `store_tips` (the fused gradient does not need them; SURVEY 8(d) "tip q never stored")."""
    ops = np.zeros(2 * tree.n_tips - 2, dtype=plk.PRE_OP_DTYPE)
    i = 0
    for m in reversed(tree.internal_nodes()):
        a, b = tree.children[m]
        for k, j in ((a, b), (b, a)):
            dest = k if (store_tips or k >= tree.n_tips) else -1
            ops[i] = (dest, m, k, j, j, k)
            i += 1
    return ops


class Evaluator:
    """Holds one library instance loaded with a workload; evaluates logL and the branch-length gradient."""

    def __init__(self, wl, precision=plk.FP64, flags=0, tips_as_partials=False, device="cuda:0",
                 stream=None, store_tip_pre: bool = False, eigen=None):
        """`tips_as_partials`: False (all tips compact states), True (all tips one-hot / all-ones partials) or a
        boolean sequence per tip (mixed).  `eigen`: (U, Uinv, lam) handed to plk_set_eigen_decomposition instead of the
        workload's own (the eigendecomposition is a client-side input)."""
        self.wl = wl
        self.eigen = eigen
        tree = wl.tree
        self.tree = tree
        N = tree.n_tips
        S = wl.n_states
        self.inst = plk.Instance(
            N, S, wl.n_patterns, wl.n_categories,
            compact_buffer_count=N - int(np.sum(np.broadcast_to(np.asarray(tips_as_partials, dtype=bool), (N,)))),
            preorder_slot_count=0 if store_tip_pre else N,  # root + internal nodes (N-1) rounded up
            precision=precision, flags=flags, device=device, stream=stream)
        self.tips_as_partials = np.broadcast_to(np.asarray(tips_as_partials, dtype=bool), (N,)).copy()
        self.ops = post_order_ops(tree)
        self.pre_ops = pre_order_ops(tree, store_tips=store_tip_pre)
        self.branch_nodes = self.pre_ops["node_post"].copy()  # gradient order of pre_order_gradient
        self.matrix_idx = np.array([k for k in range(tree.n_nodes) if k != tree.root], dtype=np.int32)
        self.scale_idx = np.arange(N, 2 * N - 1, dtype=np.int32)
        self.upload_model()
        self.upload_tips()

    # -- set-up
    def upload_model(self):
        wl, inst = self.wl, self.inst
        inst.set_pattern_weights(wl.pattern_weights)
        inst.set_state_frequencies(wl.pi)
        inst.set_category_rates(wl.rates)
        inst.set_category_weights(wl.cat_weights)
        U, Uinv, lam = self.eigen if self.eigen is not None else (wl.U, wl.Uinv, wl.lam)
        inst.set_eigen_decomposition(0, U, Uinv, lam)
        inst.set_rate_matrix(0, wl.Q)

    def upload_tips(self):
        wl, inst = self.wl, self.inst
        S = wl.n_states
        for k in range(self.tree.n_tips):
            if self.tips_as_partials[k]:
                st = wl.tip_states[k]
                part = np.zeros((wl.n_patterns, S))
                known = st < S
                part[np.nonzero(known)[0], st[known]] = 1.0
                part[~known, :] = 1.0
                inst.set_tip_partials(k, part)
                if inst.cfg.flags & plk.FLAG_CACHE_RATE_PRODUCTS:  # Q p_k cached next to the partials
                    inst.cache_rate_products(0, [k])
            else:
                inst.set_tip_states(k, wl.tip_states[k].astype(np.int32))

    # -- evaluation with host inputs / outputs
    def log_likelihood(self, branch_lengths: Optional[np.ndarray] = None, want_site=True, allow_nonfinite=False,
                       matrices=None):
        """`matrices`: {node: [C, S, S]} transition matrices supplied by the client (plk_set_transition_matrix)
        instead of being formed from the eigendecomposition and `branch_lengths`."""
        t = self.tree.branch_length if branch_lengths is None else branch_lengths
        if matrices is not None:
            for k in self.matrix_idx:
                self.inst.set_transition_matrix(int(k), matrices[int(k)])
        else:
            self.inst.update_transition_matrices(0, self.matrix_idx, np.asarray(t)[self.matrix_idx])
        self.inst.update_partials(self.ops)
        return self.inst.root_log_likelihoods(self.tree.root, self.scale_idx, want_site, allow_nonfinite)

    def log_likelihood_on_the_fly(self, branch_lengths: Optional[np.ndarray] = None, want_site=True):
        """The same through plk_update_partials_on_the_fly: no transition matrix is formed; needs
        FLAG_ON_THE_FLY_MATRICES."""
        t = np.asarray(self.tree.branch_length if branch_lengths is None else branch_lengths, dtype=np.float64)
        bl = np.stack([t[self.ops["child1"]], t[self.ops["child2"]]], axis=1)
        self.inst.update_partials_on_the_fly(0, self.ops, bl)
        return self.inst.root_log_likelihoods(self.tree.root, self.scale_idx, want_site)

    def gradient(self, want_site=False):
        """After log_likelihood(): d logL / d t_k for every node k (0 at the root), fused pre-order + derivative."""
        g, site = self.inst.pre_order_gradient(0, self.tree.root, self.pre_ops, want_site)
        grad = np.zeros(self.tree.n_nodes)
        grad[self.branch_nodes] = g
        if want_site:
            full = np.zeros((self.tree.n_nodes, self.wl.n_patterns))
            full[self.branch_nodes] = site
            return grad, full
        return grad

    def gradient_unfused(self, want_site=False):
        """Same through plk_update_pre_partials + plk_branch_derivatives (needs store_tip_pre=True)."""
        self.inst.update_pre_partials(self.tree.root, self.pre_ops)
        nodes = self.matrix_idx
        g, site = self.inst.branch_derivatives(0, nodes, nodes, want_site)
        grad = np.zeros(self.tree.n_nodes)
        grad[nodes] = g
        if want_site:
            full = np.zeros((self.tree.n_nodes, self.wl.n_patterns))
            full[nodes] = site
            return grad, full
        return grad

    def rate_matrix_gradient(self, branch_lengths: Optional[np.ndarray] = None):
        """After log_likelihood() and a pre-order pass that stored EVERY node's pre-order partials
        (gradient_unfused(), store_tip_pre=True): the S x S approximate gradient with respect to the rate-matrix
        elements (plk_rate_matrix_gradient)."""
        t = self.tree.branch_length if branch_lengths is None else branch_lengths
        nodes = self.matrix_idx
        return self.inst.rate_matrix_gradient(nodes, nodes, np.asarray(t)[nodes])

    # -- device-resident step used by bench.py: nothing but launches, outputs stay on the device
    def make_device_io(self, out=None):
        """`out`: optional fp64 device tensor [1 + 2N-2] that receives [logL, gradient] (one buffer, so that a
        multi-GPU caller can all-reduce it as it is: sharded.py)."""
        torch = self.inst.torch
        dev = self.inst.device
        t = np.asarray(self.tree.branch_length)[self.matrix_idx]
        self.d_t = torch.from_numpy(np.ascontiguousarray(t)).to(dev)
        if out is None:
            out = torch.zeros(1 + len(self.pre_ops), dtype=torch.float64, device=dev)
        self.d_out = out
        self.d_logl = out[:1]
        self.d_grad = out[1:]

    def step_matrices(self):
        self.inst.update_transition_matrices_device(0, self.matrix_idx, self.d_t)

    def step_post(self):
        self.inst.update_partials(self.ops)

    def step_root(self):
        self.inst.root_log_likelihoods_device(self.tree.root, self.scale_idx, self.d_logl)

    def step_pre_gradient(self):
        self.inst.pre_order_gradient_device(0, self.tree.root, self.pre_ops, self.d_grad)

    def step_device(self):
        self.step_matrices()
        self.step_post()
        self.step_root()
        self.step_pre_gradient()

    def step_evaluate(self):
        """The same evaluation as step_device() through plk_evaluate_device: ONE library call, replayed from a cached
        CUDA graph from its third use (needs a non-default stream; otherwise it runs eagerly)."""
        self.inst.evaluate_device(0, self.matrix_idx, self.d_t, self.ops, self.tree.root, self.scale_idx, self.tree.root,
                                  self.pre_ops, self.d_out)

    def evaluate(self, branch_lengths: Optional[np.ndarray] = None):
        """(logL, gradient per node) through plk_evaluate: host branch lengths in, host results out."""
        t = self.tree.branch_length if branch_lengths is None else branch_lengths
        logl, g = self.inst.evaluate(0, self.matrix_idx, np.asarray(t)[self.matrix_idx], self.ops, self.tree.root,
                                     self.scale_idx, self.tree.root, self.pre_ops)
        grad = np.zeros(self.tree.n_nodes)
        grad[self.branch_nodes] = g
        return logl, grad

    def close(self):
        self.inst.destroy()
