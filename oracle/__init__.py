"""CPU oracle for the BEAGLE-4.1 hot path -- TEST INFRASTRUCTURE, not a product path.

Plain, slow, fp64 numpy restatement of what the library computes (PAPER.md:27 Felsenstein pruning; PAPER.md:43
post- + pre-order traversal, likelihood as inner product, O(N) gradient; PAPER.md:101 transition matrices from an
eigendecomposition, gradient as the `pre . Q . post` sandwich), in the order and notation of SURVEY.md section
8(a)/(c).  The paper prints no equations; the formulas are the textbook definitions of the works it cites and are
pinned in tests/test_oracle_*.py by brute-force enumeration, the sum-over-all-patterns = 1 invariant, the JC69
closed form, central finite differences, scipy's expm and the worked examples in tests/golden/.

Rules (task statement, section 3):
  * only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this;
  * it shares no code with paper_2606_27607_b200/ (the CUDA path) and neither imports the other;
  * no expected value stored anywhere comes from the CUDA path.

Pins: every function in models.py / likelihood.py / caching.py / encode.py is pinned; the
fp32 / tensor-core GPU modes have no pin of their own -- they are compared with this fp64 oracle at 1e-4.
"""
from . import caching, encode, likelihood, models  # noqa: F401
