"""Multi-GPU pattern sharding (section 3.3).

"Partitioning the sequence alignment into conditionally independent blocks running on separate GPUs", "one BEAGLE
instance per GPU": site patterns are conditionally independent given the tree and the model, so rank r of G holds
the whole tree, every transition matrix and 1/G of every partials buffer -- a contiguous range of the pattern axis
-- and runs the unchanged single-GPU path (libplk.so) on it.  The only exchange step of the method is the sum of the
per-rank results: logL and the 2N-2 branch derivatives, 1 + (2N-2) fp64 values (<= 8 KB at N = 512), ONE all-reduce
per evaluation (torch.distributed: NCCL over NVLink on GPUs, gloo in the CPU tests).  It is latency-bound and
topology-insensitive; there is nothing to overlap it with except the next evaluation's matrix update.

One process per GPU.  The result buffer is one device tensor laid out [logL, g_0 .. g_{2N-3}] so that the root
reduction and the gradient reduction write straight into the tensor that is all-reduced (no packing kernel).
"""
from __future__ import annotations

import copy
from typing import Callable, Optional, Tuple

import numpy as np

PATTERN_ALIGN = 128  # shard boundaries fall on multiples of the largest pattern tile of the kernels


def pattern_range(rank: int, world: int, n_patterns: int, align: int = PATTERN_ALIGN) -> Tuple[int, int]:
    """Contiguous range [lo, hi) of rank `rank`: the pattern axis is cut into `align`-sized blocks that are dealt out
    as evenly as possible (the first `rem` ranks get one block more); the ragged tail belongs to the last non-empty
    rank.  Ranges are disjoint, ordered by rank and cover 0..n_patterns-1; a rank may be empty when
    n_patterns < world * align."""
    if not (0 <= rank < world) or n_patterns < 0:
        raise ValueError("bad rank / world / pattern count")
    n_blocks = (n_patterns + align - 1) // align
    base, rem = divmod(n_blocks, world)
    b0 = rank * base + min(rank, rem)
    b1 = b0 + base + (1 if rank < rem else 0)
    return min(b0 * align, n_patterns), min(b1 * align, n_patterns)


def shard_workload(wl, lo: int, hi: int):
    """The same tree, model and categories with patterns lo..hi-1 only (a view of the alignment; inputs, not method)."""
    sub = copy.copy(wl)
    sub.tip_states = np.ascontiguousarray(wl.tip_states[:, lo:hi])
    sub.pattern_weights = np.ascontiguousarray(wl.pattern_weights[lo:hi])
    sub.name = f"{wl.name}[{lo}:{hi}]"
    return sub


class ShardedEvaluator:
    """Rank `rank` of `world`: owns patterns pattern_range(rank, world, P) of the workload, evaluates them with one
    library instance on its GPU and all-reduces [logL, gradient].  `dist` is torch.distributed (already initialised)
    or None for world == 1.  `make_local(sub_workload)` builds the per-rank evaluator; the default is the CUDA
    `client.Evaluator` (the CPU tests of the exchange logic pass a stand-in)."""

    def __init__(self, wl, rank: int, world: int, dist=None, device=None, make_local: Optional[Callable] = None,
                 **evaluator_kwargs):
        import torch

        self.torch = torch
        self.rank, self.world, self.dist = rank, world, dist
        self.lo, self.hi = pattern_range(rank, world, wl.n_patterns)
        self.n_branches = 2 * wl.tree.n_tips - 2
        self.device = torch.device(device if device is not None else "cpu")
        self.result = torch.zeros(1 + self.n_branches, dtype=torch.float64, device=self.device)
        self.local = None
        if self.hi > self.lo:
            sub = shard_workload(wl, self.lo, self.hi)
            if make_local is None:
                from .client import Evaluator

                self.local = Evaluator(sub, device=str(self.device), **evaluator_kwargs)
                self.local.make_device_io(out=self.result)
            else:
                self.local = make_local(sub)

    def evaluate_device(self):
        """One evaluation: local device step (results land in self.result), then the one all-reduce.  Asynchronous on
        the GPU; returns the result tensor [logL, g...] (valid on every rank after the collective)."""
        if self.local is None:
            self.result.zero_()  # empty shard contributes nothing
        elif hasattr(self.local, "step_device"):
            self.local.step_device()
        else:
            self.result.copy_(self.torch.as_tensor(self.local(), dtype=self.torch.float64))
        if self.world > 1 and self.dist is not None:  # dist None: the caller sums the shards itself (tests)
            self.dist.all_reduce(self.result, op=self.dist.ReduceOp.SUM)
        return self.result

    def evaluate(self):
        """(logL, gradient in the order of client.pre_order_ops) on the host."""
        r = self.evaluate_device().cpu().numpy()
        return float(r[0]), r[1:].copy()

    def close(self):
        if self.local is not None and hasattr(self.local, "close"):
            self.local.close()
