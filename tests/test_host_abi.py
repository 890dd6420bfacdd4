"""No-GPU checks of the C-ABI library: it builds, loads, exports every symbol include/plk.h declares, its host-only
entry points (level scheduler, encode/compress, arena sizing, error strings) behave, and compute calls fail loudly
(PLK_ERR_CUDA) instead of falling back when there is no device."""
import os
import re

import numpy as np
import pytest

from oracle import encode as oracle_encode
from paper_2606_27607_b200 import build, plk, workloads
from paper_2606_27607_b200.client import post_order_ops, pre_order_ops

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    build.build()


def test_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "plk.h")).read()
    declared = set(re.findall(r"PLK_API[^;(]*?\b(plk_\w+)\s*\(", header))
    assert len(declared) >= 30
    assert declared == set(plk.EXPORTED)
    lib = plk.lib()
    for name in declared:
        assert getattr(lib, name) is not None


def test_error_strings_and_arena_bytes():
    assert plk.error_string(0) == "success"
    assert "range" in plk.error_string(plk.ERR_OUT_OF_RANGE)
    cfg = plk.Config(8, 4, 1000, 4, 15, 8, 0, 15, 0, 15, 1, 15, plk.FP64, 0)
    small = plk.arena_bytes(cfg)
    assert small >= 7 * 4 * 1000 * 4 * 8
    cfg.precision = plk.FP32
    assert plk.arena_bytes(cfg) < small
    cfg.state_count = 100
    assert plk.arena_bytes(cfg) == 0


def test_no_device_fails_loudly():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(plk.PlkError) as e:
        plk.Instance(4, 4, 10, 4)
    assert e.value.status == plk.ERR_CUDA


def test_schedule_levels_match_tree_levels():
    """Level of an op = level of its node in the tree minus 1 (cherries first): SURVEY 8(a) level structure."""
    rng = np.random.default_rng(3)
    for n in (2, 8, 33, 128):
        tree = workloads.coalescent_topology(n, rng)
        ops = post_order_ops(tree)
        n_levels, level = plk.schedule_levels(ops)
        lv = tree.levels()
        assert n_levels == lv[tree.root]
        assert np.array_equal(level, lv[ops["dest"]] - 1)
        # shuffled (but still valid) order gives the same levels per dest
        pre = pre_order_ops(tree)
        n_pre, plevel, partner = plk.schedule_pre_levels(pre)
        depth = np.zeros(tree.n_nodes, dtype=int)
        for k in range(tree.n_nodes - 2, -1, -1):
            depth[k] = depth[tree.parent[k]] + 1
        assert np.array_equal(plevel, depth[pre["node_post"]] - 1)
        assert n_pre == depth.max()
        for i, j in enumerate(partner):  # the two children of one parent are partners
            assert j >= 0 and partner[j] == i and pre["parent_pre"][i] == pre["parent_pre"][j] and i != j


def test_schedule_rejects_bad_lists():
    ops = np.array([(4, 0, 0, 0, 1, 1), (4, 1, 2, 2, 3, 3)], dtype=plk.OP_DTYPE)  # duplicate dest
    assert plk.lib().plk_schedule_levels(ops.ctypes.data, 2, None) == plk.ERR_OUT_OF_RANGE
    ops = np.array([(4, 0, 4, 0, 1, 1)], dtype=plk.OP_DTYPE)  # dest is its own child
    assert plk.lib().plk_schedule_levels(ops.ctypes.data, 1, None) == plk.ERR_OUT_OF_RANGE
    # write-after-read: op 1 overwrites buffer 5 that op 0 reads -> must sit in a later level
    ops = np.array([(6, 0, 5, 0, 1, 1), (5, 1, 2, 2, 3, 3)], dtype=plk.OP_DTYPE)
    n, level = plk.schedule_levels(ops)
    assert n == 2 and level.tolist() == [0, 1]


@pytest.mark.parametrize("kind,okind", [("nuc", oracle_encode.NUC), ("codon", oracle_encode.CODON)])
def test_encode_and_compress_bit_exact(kind, okind):
    """S8a step 0: library arrays equal the oracle's bit for bit (integer work)."""
    for seed, taxa, sites in ((1, 3, 50), (2, 17, 4000), (3, 64, 1), (4, 5, 1000)):
        seqs = workloads.random_alignment(kind, taxa, sites, seed)
        s, w, m = plk.encode_and_compress(plk.NUCLEOTIDE if kind == "nuc" else plk.CODON, seqs)
        rs, rw, rm = oracle_encode.encode_and_compress(okind, seqs)
        assert s.dtype == rs.dtype and np.array_equal(s, rs)
        assert np.array_equal(w, rw) and np.array_equal(m, rm)


def test_encode_errors():
    lib = plk.lib()
    with pytest.raises(plk.PlkError) as e:
        plk.encode_and_compress(plk.CODON, [b"ATGTAA", b"ATGAAA"])
    assert e.value.status == plk.ERR_STOP_CODON
    with pytest.raises(plk.PlkError) as e:
        plk.encode_and_compress(plk.CODON, [b"ATGA", b"ATGA"])
    assert e.value.status == plk.ERR_OUT_OF_RANGE
    s, w, m = plk.encode_and_compress(plk.NUCLEOTIDE, [b"", b""])
    assert s.shape == (2, 0) and w.size == 0 and m.size == 0
    assert lib.plk_destroy(None) == 0


def test_chain_rule_rate_matrix_host_helper():
    """plk_chain_rule_rate_matrix: out[k] = sum_ab G[a][b] dQ[k][a][b]; no device needed."""
    rng = np.random.default_rng(11)
    G = rng.normal(size=(61, 61))
    dQ = rng.normal(size=(7, 61, 61))
    out = plk.chain_rule_rate_matrix(G, dQ)
    assert np.allclose(out, [np.sum(G * dQ[k]) for k in range(7)], rtol=1e-13, atol=0)
    assert plk.chain_rule_rate_matrix(G, np.zeros((0, 61, 61))).shape == (0,)
