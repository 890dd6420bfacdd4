"""GPU parity at BASELINE.json's FULL sizes (-m gpu), in the launch configuration bench.py times (default flags for
4 states, PLK_FLAG_TENSOR_CORES for 61 states).  The oracle cannot evaluate 10^5 patterns x 128 taxa in seconds, but
patterns are conditionally independent, so it can evaluate SAMPLED patterns one by one: three windows
of the pattern axis (the first tile, a window straddling tile boundaries in the middle, the ragged tail) give
per-pattern log-likelihoods and per-pattern branch derivatives for every branch, compared element by element.
What is not sampled is checked through properties that hold at any size: logL and the gradient are exactly the
weighted sums of the per-pattern outputs, the two root-child derivatives coincide (reversible model), everything
is finite, and a second evaluation is bitwise identical."""
import numpy as np
import pytest

import oracle_runner as orc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu

CASES = [
    pytest.param(1, plk.FP64, 0, id="cfg1-fp64"),
    pytest.param(1, plk.FP32, 0, id="cfg1-fp32"),
    pytest.param(2, plk.FP64, plk.FLAG_TENSOR_CORES, id="cfg2-fp64-tensor"),
    pytest.param(2, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg2-fp32-tensor"),
    pytest.param(2, plk.FP64, 0, id="cfg2-fp64-cuda"),
    pytest.param(3, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg3-fp32-tensor"),
]


def _windows(P):
    mid = P // 2 - 17
    return [(0, 64), (mid, mid + 64), (P - 50, P)]


@pytest.mark.parametrize("cfg,precision,flags", CASES)
def test_full_size_sampled_patterns_and_invariants(cfg, precision, flags):
    wl = workloads.config(cfg)
    P, root = wl.n_patterns, wl.tree.root
    ev = Evaluator(wl, precision=precision, flags=flags | plk.FLAG_SITE_DERIVATIVES)
    try:
        logl, site = ev.log_likelihood()
        grad, site_d = ev.gradient(want_site=True)
        logl2, _ = ev.log_likelihood(want_site=False)
        grad2 = ev.gradient()
        launches = ev.inst.kernel_launch_count()
    finally:
        ev.close()
    assert launches > 0
    fp64 = precision == plk.FP64
    tol = 1e-10 if fp64 else 1e-4
    # ---- sampled patterns against the oracle
    for lo, hi in _windows(P):
        ref = orc.evaluate(wl, lo=lo, hi=hi, keep_site_derivatives=True)
        rel = np.max(np.abs(site[lo:hi] - ref["site_logl"]) / np.abs(ref["site_logl"]))
        assert rel <= tol, f"site logL window [{lo},{hi}) rel err {rel:.3e}"
        d_ref = ref["site_derivs"]  # [n_nodes, hi - lo]: the oracle saw only the window
        floor = 1e-6 * np.max(np.abs(d_ref))
        for k in range(wl.tree.n_nodes):
            if k == root:
                continue
            scale = max(np.max(np.abs(d_ref[k])), floor)
            err = np.max(np.abs(site_d[k, lo:hi] - d_ref[k]))
            assert err <= (1e-9 if fp64 else 2e-4) * scale, f"site derivative branch {k} window [{lo},{hi}): {err / scale:.3e}"
    # ---- properties over ALL patterns
    w = wl.pattern_weights
    assert np.all(np.isfinite(site)) and np.all(np.isfinite(site_d)) and np.isfinite(logl)
    assert abs(logl - float(np.dot(w, site))) <= 1e-12 * abs(logl)
    A = np.abs(site_d) @ w  # A_k from the library's own per-pattern derivatives
    g_sum = site_d @ w
    nz = np.arange(wl.tree.n_nodes) != root
    assert np.all(np.abs(grad[nz] - g_sum[nz]) <= 1e-12 * A[nz] + 1e-300)
    assert grad[root] == 0.0
    a, b = wl.tree.children[root]
    assert abs(grad[a] - grad[b]) <= (1e-10 if fp64 else 1e-4) * max(A[a], A[b])
    # ---- repeatability (fixed-order reductions, no atomics)
    assert logl2 == logl and np.array_equal(grad2, grad)
