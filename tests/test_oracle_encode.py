"""Pins for oracle/encode.py (no GPU): hand-made alignments whose answer is written out by hand, codon index checks
from SURVEY.md 8(c) row 7, and the expand-shuffle-compress round trip."""
import numpy as np
import pytest

from oracle import encode


def test_nucleotide_hand_made():
    seqs = ["ACGTAC-acgua", "ACGTACNACGTA", "AAGTAAAAAGTA"]
    #        012345678901 ; columns: 0 AAA,1 CCA,2 GGG,3 TTT,4 AAA,5 CCA,6 -NA,7 aAA,8 cCA,9 gGG,10 uTT,11 aAA
    states, weights, s2p = encode.encode_and_compress(encode.NUC, seqs)
    assert states.dtype == np.uint8 and weights.dtype == np.float64 and s2p.dtype == np.int64
    assert states.tolist() == [[0, 1, 2, 3, 4], [0, 1, 2, 3, 4], [0, 0, 2, 3, 0]]
    assert weights.tolist() == [4.0, 3.0, 2.0, 2.0, 1.0]
    assert s2p.tolist() == [0, 1, 2, 3, 0, 1, 4, 0, 1, 2, 3, 0]


def test_codon_hand_made_and_index_checks():
    assert encode.encode_sequence(encode.CODON, "AAAATGTGGTTT") == [0, 14, 55, 60]
    assert encode.encode_sequence(encode.CODON, "aaaAuGugg") == [0, 14, 55]
    assert encode.encode_sequence(encode.CODON, "---A-GNNNAAR") == [61, 61, 61, 61]
    # the three stops sit at 64-triplet indices 48, 50, 56 -> sense indices around them
    assert encode.encode_sequence(encode.CODON, "TAC") == [48]  # idx64 49 minus one stop before it
    assert encode.encode_sequence(encode.CODON, "TAT") == [49]  # idx64 51 minus two stops
    assert encode.encode_sequence(encode.CODON, "TGC") == [54]  # idx64 57 minus three stops
    seqs = ["ATGAAAATG---", "ATGAAGATGAAA"]
    states, weights, s2p = encode.encode_and_compress(encode.CODON, seqs)
    assert states.tolist() == [[14, 0, 61], [14, 2, 0]]
    assert weights.tolist() == [2.0, 1.0, 1.0]
    assert s2p.tolist() == [0, 1, 0, 2]


def test_errors():
    with pytest.raises(encode.StopCodonError):
        encode.encode_sequence(encode.CODON, "ATGTAA")
    with pytest.raises(ValueError):
        encode.encode_sequence(encode.CODON, "ATGA")
    with pytest.raises(ValueError):
        encode.encode_and_compress(encode.NUC, ["ACG", "AC"])


def test_expand_shuffle_compress_round_trip():
    rng = np.random.default_rng(5)
    n_taxa, n_pat = 6, 40
    cols = set()
    while len(cols) < n_pat:
        cols.add(tuple(rng.integers(0, 5, n_taxa)))
    cols = sorted(cols)
    mult = rng.integers(1, 6, n_pat)
    sites = [c for c, m in zip(cols, mult) for _ in range(m)]
    order = rng.permutation(len(sites))
    letters = "ACGT-"
    seqs = ["".join(letters[sites[j][t]] for j in order) for t in range(n_taxa)]
    states, weights, s2p = encode.encode_and_compress(encode.NUC, seqs)
    assert states.shape == (n_taxa, n_pat) and weights.sum() == len(sites)
    got = {tuple(states[:, k]): weights[k] for k in range(n_pat)}
    assert got == {c: float(m) for c, m in zip(cols, mult)}
    # first-occurrence order and site map
    firsts = [int(np.argmax(s2p == k)) for k in range(n_pat)]
    assert firsts == sorted(firsts)
    for site in range(len(sites)):
        assert tuple(states[:, s2p[site]]) == sites[order[site]]
