"""Pattern sharding on the CUDA path (-m gpu): the per-rank evaluators of a 2- and a 3-way split run one after the
other on the one GPU of this box (no rank waits on another: B200_PROFILING.md), their [logL, gradient] buffers are
summed as the all-reduce would, and the total is compared with the oracle on all patterns.  The collective itself
is covered by tests/test_sharding_host.py (gloo, world size 2)."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from paper_2606_27607_b200 import plk, sharded, workloads
from paper_2606_27607_b200.client import pre_order_ops

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("cfg,n_pat,precision,flags", [(1, 5000, plk.FP64, 0), (1, 5000, plk.FP32, 0),
                                                       (2, 700, plk.FP64, plk.FLAG_TENSOR_CORES),
                                                       (2, 700, plk.FP32, plk.FLAG_TENSOR_CORES)],
                         ids=["nuc-fp64", "nuc-fp32", "codon-fp64", "codon-fp32"])
def test_shards_sum_to_the_full_evaluation(world, cfg, n_pat, precision, flags):
    wl = workloads.config(cfg, n_patterns=n_pat)
    ref = orc.evaluate(wl)
    total = np.zeros(1 + 2 * wl.tree.n_tips - 2)
    covered = 0
    for rank in range(world):
        ev = sharded.ShardedEvaluator(wl, rank, world, device="cuda:0", precision=precision, flags=flags,
                                      eigen=orc.oracle_eigen(wl))
        try:
            logl, grad = ev.evaluate()  # world > 1 but dist is None is never reached: see below
        finally:
            ev.close()
        total += np.concatenate([[logl], grad])
        covered += ev.hi - ev.lo
    assert covered == n_pat
    nodes = pre_order_ops(wl.tree)["node_post"]
    g = np.zeros(wl.tree.n_nodes)
    g[nodes] = total[1:]
    assert abs(total[0] - ref["logL"]) <= pc.tol_of(precision) * abs(ref["logL"])
    pc.check_grad(g, ref, precision, wl.tree.root)
