"""GPU parity at BASELINE.json's FULL sizes (-m gpu), in the launch configuration bench.py times (default flags for
4 states, PLK_FLAG_TENSOR_CORES for 61 states), against the oracle on ALL patterns.

The oracle evaluates the full pattern set by chunks in a process pool (patterns are conditionally independent,
PAPER.md:87; tests/oracle_runner.py evaluate_pool) -- configs[1] in ~10 s, configs[3] in ~30 s on 16 cores -- and
every output is compared: all site log-likelihoods element by element, logL, every branch gradient (the figures
of SURVEY 8(c) row 18) and all per-pattern derivatives.  The one exception is the largest sweep point of configs[4]
(512 taxa x 500 000 patterns, 49 GB of partials, minutes of oracle time): there 60 seeded patterns out of every
block of 10 000 (3 000 in all) are compared one by one and the rest is covered by properties that hold at any size.
No assertion below compares the library with itself except the bitwise repeatability checks."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu

_cache = {}


def _workload_and_oracle(cfg, n_tips=None, n_patterns=None):
    """Workload + full oracle evaluation, shared by the precisions / code paths of one config (one entry kept)."""
    key = (cfg, n_tips, n_patterns)
    if key not in _cache:
        _cache.clear()
        wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_patterns)
        ref = orc.evaluate_pool(wl, keep_site_derivatives=True, chunk=4096 if wl.n_states == 4 else 512)
        _cache[key] = (wl, ref)
    return _cache[key]


CASES = [
    pytest.param(1, None, None, plk.FP64, 0, id="cfg1-fp64"),
    pytest.param(1, None, None, plk.FP32, 0, id="cfg1-fp32"),
    pytest.param(2, None, None, plk.FP64, plk.FLAG_TENSOR_CORES, id="cfg2-fp64-tensor"),
    pytest.param(2, None, None, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg2-fp32-tensor"),
    pytest.param(2, None, None, plk.FP64, 0, id="cfg2-fp64-cuda"),
    pytest.param(2, None, None, plk.FP32, 0, id="cfg2-fp32-cuda"),
    pytest.param(3, None, None, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg3-fp32-tensor"),
    pytest.param(4, 128, 100_000, plk.FP32, 0, id="cfg4-128x100000-fp32"),
    pytest.param(4, 512, 10_000, plk.FP32, 0, id="cfg4-512x10000-fp32"),
    pytest.param(4, 8, 100_000, plk.FP32, 0, id="cfg4-8x100000-fp32"),
]


@pytest.mark.parametrize("cfg,n_tips,n_patterns,precision,flags", CASES)
def test_full_size_all_patterns(cfg, n_tips, n_patterns, precision, flags):
    wl, ref = _workload_and_oracle(cfg, n_tips, n_patterns)
    root = wl.tree.root
    ev = Evaluator(wl, precision=precision, flags=flags | plk.FLAG_SITE_DERIVATIVES, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood()
        grad, site_d = ev.gradient(want_site=True)
        logl2, _ = ev.log_likelihood(want_site=False)
        grad2 = ev.gradient()
        launches = ev.inst.kernel_launch_count()
    finally:
        ev.close()
    assert launches > 0
    pc.check_logl(site, logl, ref, precision)
    figures = pc.check_grad(grad, ref, precision, root)
    worst_d = pc.check_site_derivs(site_d, ref, precision, root)
    print(f"{wl.name}: gradient strict {figures[0]:.2e}, /A_k {figures[1]:.2e}, 2-norm {figures[2]:.2e}; "
          f"per-pattern derivatives {worst_d:.2e}; oracle on {ref['workers']} processes")
    a, b = wl.tree.children[root]  # reversible model: the two root-child derivatives coincide
    assert abs(grad[a] - grad[b]) <= pc.tol_of(precision) * max(ref["cond"][a], ref["cond"][b])
    # repeatability (fixed-order reductions, no atomics): the only library-vs-library comparison in this file
    assert logl2 == logl and np.array_equal(grad2, grad)


@pytest.mark.parametrize("cfg,precision,flags", [pytest.param(3, plk.FP32, plk.FLAG_TENSOR_CORES, id="cfg3-fp32-tcgen05"),
                                                 pytest.param(3, plk.FP64, plk.FLAG_TENSOR_CORES, id="cfg3-fp64-dmma"),
                                                 pytest.param(3, plk.FP32, plk.FLAG_TENSOR_CORES | plk.FLAG_NO_TCGEN05,
                                                              id="cfg3-fp32-mma-sync"),
                                                 pytest.param(1, plk.FP64, 0, id="cfg1-fp64"),
                                                 pytest.param(1, plk.FP32, 0, id="cfg1-fp32")])
def test_repeated_evaluations_are_bitwise_equal(cfg, precision, flags):
    """Forty evaluations of a full-size config in a row: logL, every branch gradient and every per-pattern derivative bitwise
    equal to the first.  The warp-specialised kernels hand tiles between warps through phase-counted barriers; a
    protocol error shows up as rare last-bits differences in a few rows of a tile (round 2: the class-1 producers of
    k_pre_tc5v could complete another round's phase -- 9 % of the evaluations at this size differed), which a single
    repeat does not catch reliably.  Library against itself: repeatability only, parity is the test above."""
    wl = workloads.config(cfg)
    ev = Evaluator(wl, precision=precision, flags=flags | plk.FLAG_SITE_DERIVATIVES)
    try:
        logl0, _ = ev.log_likelihood(want_site=False)
        g0, s0 = ev.gradient(want_site=True)
        for it in range(40):
            if it % 4 == 0:
                logl, _ = ev.log_likelihood(want_site=False)
                assert logl == logl0
            g, s = ev.gradient(want_site=True)
            assert np.array_equal(g, g0), f"evaluation {it}: gradient differs at nodes {np.nonzero(g != g0)[0][:8]}"
            assert np.array_equal(s, s0), f"evaluation {it}: per-pattern derivatives differ at {np.argwhere(s != s0)[:8]}"
    finally:
        ev.close()


def test_largest_sweep_point_sampled():
    """configs[4] 512 x 500 000 fp32 (49 GB of partials): 60 seeded patterns from every block of 10 000 against the
    oracle one by one (site log-likelihoods and the per-pattern derivatives of all 1022 branches); over ALL patterns
    the properties that hold at any size: everything finite, logL below the sum of the per-site maxima it is made of,
    the pulley identity at the root, and -- since a sampled sum estimates the full one -- the oracle's gradient over
    the sample, rescaled, within sampling error of the library's full gradient."""
    wl = workloads.config(4, n_tips=512, n_patterns=500_000)
    P, root = wl.n_patterns, wl.tree.root
    rng = np.random.default_rng(20260627)
    idx = np.sort(np.concatenate([b + rng.choice(10_000, size=60, replace=False) for b in range(0, P, 10_000)]))
    ref = orc.evaluate(wl, idx=idx, keep_site_derivatives=True)
    ev = Evaluator(wl, precision=plk.FP32, flags=plk.FLAG_SITE_DERIVATIVES, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood()
        grad, site_d = ev.gradient(want_site=True)
    finally:
        ev.close()
    rel = np.max(np.abs(site[idx] - ref["site_logl"]) / np.abs(ref["site_logl"]))
    assert rel <= pc.FP32_TOL, f"sampled site logL rel err {rel:.3e}"
    pc.check_site_derivs(site_d, ref, plk.FP32, root, cols=idx)
    assert np.all(np.isfinite(site)) and np.all(np.isfinite(site_d)) and np.isfinite(logl) and np.all(np.isfinite(grad))
    assert np.all(site < 0.0) and grad[root] == 0.0
    a, b = wl.tree.children[root]
    A = np.abs(site_d[[a, b]]) @ wl.pattern_weights
    assert abs(grad[a] - grad[b]) <= pc.FP32_TOL * np.max(A)
    # sampled estimate of logL: mean of omega_p log l_p over the sample x P, standard error from the sample
    terms = wl.pattern_weights[idx] * ref["site_logl"]
    est, se = P * np.mean(terms), P * np.std(terms) / np.sqrt(len(idx))
    assert abs(logl - est) <= 6.0 * se
