"""Multi-GPU pattern sharding (paper_2606_27607_b200/sharded.py): the host-side logic on
CPU -- the partition of the pattern axis, and the exchange step (ONE all-reduce of [logL, gradient]) run by two
`gloo` ranks.  The per-rank compute is played by the oracle on the rank's pattern range (there is no CPU product
path); what is under test is the partition, the buffer layout and the collective, against the oracle on all
patterns.  The CUDA per-rank path on sub-ranges is covered by tests/test_gpu_sharding.py."""
import os
import socket
import sys

import numpy as np
import pytest

from paper_2606_27607_b200 import sharded, workloads


@pytest.mark.parametrize("P", [0, 1, 127, 128, 129, 1000, 100_000, 500_000])
@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_pattern_ranges_partition_the_axis(P, world):
    ranges = [sharded.pattern_range(r, world, P) for r in range(world)]
    assert ranges[0][0] == 0 and ranges[-1][1] == P
    for (a0, a1), (b0, b1) in zip(ranges, ranges[1:]):
        assert a1 == b0 and a0 <= a1
    sizes = [hi - lo for lo, hi in ranges]
    assert all(lo % sharded.PATTERN_ALIGN == 0 for lo, _ in ranges if lo < P)
    nonempty = [s for s in sizes if s > 0]
    if len(nonempty) > 1:  # balanced to within one tile block (+ the ragged tail)
        assert max(nonempty) - min(nonempty) <= 2 * sharded.PATTERN_ALIGN
    with pytest.raises(ValueError):
        sharded.pattern_range(world, world, P)


def _rank_main(rank, world, port, n_patterns, out_dir):
    sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__))))
    import torch.distributed as dist

    import oracle_runner as orc

    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = workloads.config(1, n_tips=10, n_patterns=n_patterns)
    from paper_2606_27607_b200.client import pre_order_ops

    nodes = pre_order_ops(wl.tree)["node_post"]

    def make_local(sub):
        def run():  # stands in for the per-GPU instance: [logL, gradient in pre-order-op order] of this shard
            ref = orc.evaluate(sub)
            return np.concatenate([[ref["logL"]], ref["grad"][nodes]])
        return run

    ev = sharded.ShardedEvaluator(wl, rank, world, dist=dist, make_local=make_local)
    logl, grad = ev.evaluate()
    np.save(os.path.join(out_dir, f"rank{rank}.npy"), np.concatenate([[logl], grad, [ev.lo, ev.hi]]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n_patterns", [300, 100])  # 100 < 2 * 128: rank 1 owns an EMPTY shard
def test_two_gloo_ranks_all_reduce_to_the_full_result(tmp_path, n_patterns):
    import torch.multiprocessing as tmp

    import oracle_runner as orc
    from paper_2606_27607_b200.client import pre_order_ops

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    tmp.spawn(_rank_main, args=(2, port, n_patterns, str(tmp_path)), nprocs=2, join=True)
    wl = workloads.config(1, n_tips=10, n_patterns=n_patterns)
    ref = orc.evaluate(wl)
    nodes = pre_order_ops(wl.tree)["node_post"]
    r0, r1 = (np.load(tmp_path / f"rank{r}.npy") for r in range(2))
    assert np.array_equal(r0[:-2], r1[:-2]), "every rank must hold the same reduced result"
    assert (r0[-2], r1[-1]) == (0, n_patterns) and r0[-1] == r1[-2]
    assert abs(r0[0] - ref["logL"]) <= 1e-12 * abs(ref["logL"])
    assert np.all(np.abs(r0[1:-2] - ref["grad"][nodes]) <= 1e-12 * ref["cond"][nodes] + 1e-300)
