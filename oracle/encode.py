"""Oracle, step 0 of SURVEY.md section 8(a): tip-state encoding and unique-site-pattern compression.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Integer work, compared bit-for-bit with the library's
plk_encode_and_compress.  The paper only names the result ("unique site patterns"); the rules
are the readings of SURVEY.md 8(c) rows 7, 16, 17.  Written as explicit per-site Python loops on purpose.
Pins (tests/test_oracle_encode.py): hand-made alignments with known duplicates, gaps and lower case; the
expand-shuffle-compress round trip; AAA->0, ATG->14, TGG->55, TTT->60.
"""
import numpy as np

NUC = 0
CODON = 1

_NUC_CODE = {"A": 0, "C": 1, "G": 2, "T": 3, "U": 3}


class StopCodonError(ValueError):
    pass


def _codon_index_table():
    """sense-codon index for each of the 64 triplets (16 n1 + 4 n2 + n3, A<C<G<T); -1 for the three stops."""
    stops = {"TAA", "TAG", "TGA"}
    table = {}
    nxt = 0
    for a in "ACGT":
        for b in "ACGT":
            for c in "ACGT":
                if a + b + c in stops:
                    table[a + b + c] = -1
                else:
                    table[a + b + c] = nxt
                    nxt += 1
    assert nxt == 61
    return table


def encode_sequence(kind, seq):
    """One sequence (str or bytes) -> list of state codes; missing = 4 (nucleotide) or 61 (codon)."""
    if isinstance(seq, bytes):
        seq = seq.decode("ascii")
    seq = seq.upper()
    if kind == NUC:
        return [_NUC_CODE.get(ch, 4) for ch in seq]
    if len(seq) % 3 != 0:
        raise ValueError("codon sequence length not divisible by 3")
    table = _codon_index_table()
    out = []
    for i in range(0, len(seq), 3):
        triplet = seq[i:i + 3].replace("U", "T")
        if all(ch in "ACGT" for ch in triplet):
            idx = table[triplet]
            if idx < 0:
                raise StopCodonError(f"stop codon {triplet} at codon site {i // 3}")
            out.append(idx)
        else:
            out.append(61)
    return out


def encode_and_compress(kind, seqs):
    """Returns (states uint8 [taxa, n_patterns], weights float64 [n_patterns], site_to_pattern int64 [sites]).
    Patterns are numbered in order of first occurrence along the alignment; weight = multiplicity (row 17)."""
    codes = [encode_sequence(kind, s) for s in seqs]
    n_sites = len(codes[0])
    for c in codes:
        if len(c) != n_sites:
            raise ValueError("sequences differ in length")
    first = {}
    columns = []
    weights = []
    site_to_pattern = np.zeros(n_sites, dtype=np.int64)
    for site in range(n_sites):
        col = tuple(c[site] for c in codes)
        if col not in first:
            first[col] = len(columns)
            columns.append(col)
            weights.append(0.0)
        k = first[col]
        weights[k] += 1.0
        site_to_pattern[site] = k
    states = np.array(columns, dtype=np.uint8).T.reshape(len(seqs), len(columns))
    return np.ascontiguousarray(states), np.array(weights, dtype=np.float64), site_to_pattern
