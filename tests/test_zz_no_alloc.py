"""plk_root_log_likelihoods_static_device (-m gpu): the root reduction with its scratch in the library's file-scope
`static __device__` array -- the one entry point for callers that must not allocate (README "No-allocation entry point").

Collected last on purpose (file name): its result is compared with the existing path (plk_root_log_likelihoods), which
the other test files compare with the oracle; here additionally with the oracle directly.  Both paths launch the same
kernels in the same order, so the results are bitwise equal; the assertion uses the suite's tolerances (1e-10 fp64,
1e-4 fp32) as the stated bar and then the stronger equality.  Two calls in a row per instance, and instances of
different shapes one after the other: the array is shared and keeps the previous call's contents."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu

CASES = [
    pytest.param(1, 24, 5000, plk.FP64, 0, id="gtr-24x5000-fp64"),        # 40 blocks
    pytest.param(0, None, 333, plk.FP32, 0, id="hky-8x333-fp32"),          # 3 blocks after 40: stale entries behind
    pytest.param(2, 8, 300, plk.FP64, plk.FLAG_TENSOR_CORES, id="gy94-8x300-fp64-dmma"),   # deferred rescaling
    pytest.param(2, 8, 300, plk.FP32, plk.FLAG_TENSOR_CORES, id="gy94-8x300-fp32-tcgen05"),
    pytest.param(5, 8, 200, plk.FP64, 0, id="aa-8x200-fp64"),
]


@pytest.mark.parametrize("cfg,n_tips,n_pat,precision,flags", CASES)
def test_static_scratch_root_matches_existing_path_twice(cfg, n_tips, n_pat, precision, flags):
    import torch

    wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_pat)
    ref = orc.evaluate(wl, gradient=False)
    tol = pc.tol_of(precision)
    ev = Evaluator(wl, precision=precision, flags=flags, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood()  # existing path: plk_root_log_likelihoods (scratch in the arena)
        pc.check_logl(site, logl, ref, precision)
        d_sum = torch.zeros(1, dtype=torch.float64, device="cuda:0")
        d_site = torch.zeros(wl.n_patterns, dtype=torch.float64, device="cuda:0")
        n0 = ev.inst.kernel_launch_count()
        for call in range(2):  # two calls in a row on the shared array
            d_sum.fill_(float("nan"))
            d_site.fill_(float("nan"))
            ev.inst.root_log_likelihoods_static_device(wl.tree.root, ev.scale_idx, d_sum, d_site)
            torch.cuda.synchronize()
            got, got_site = float(d_sum.cpu()[0]), d_site.cpu().numpy()
            assert abs(got - logl) <= tol * abs(logl), (call, got, logl)
            assert np.max(np.abs(got_site - site) / np.abs(site)) <= tol
            assert got == logl and np.array_equal(got_site, site)  # same kernels, same order
            pc.check_logl(got_site, got, ref, precision)
        assert ev.inst.kernel_launch_count() - n0 == 4  # k_root + k_sum_rows per call: the CUDA path ran
        # without the per-pattern output, and after new branch lengths (the existing path re-evaluated next to it)
        rng = np.random.default_rng(2)
        t2 = np.asarray(wl.tree.branch_length) * np.exp(rng.normal(0.0, 0.3, size=wl.tree.n_nodes))
        logl2, _ = ev.log_likelihood(t2, want_site=False)
        ev.inst.root_log_likelihoods_static_device(wl.tree.root, ev.scale_idx, d_sum)
        torch.cuda.synchronize()
        assert float(d_sum.cpu()[0]) == logl2
    finally:
        ev.close()


def test_static_scratch_limits_and_errors():
    import torch

    # 61 states: G = 16 threads per pattern -> ceil(P / 8) blocks; P = 8 * 8192 fits exactly, one more pattern does not
    p_fit = 8 * plk.STATIC_SCRATCH_DOUBLES
    d_sum = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    for P, fits in ((p_fit, True), (p_fit + 1, False)):
        inst = plk.Instance(2, 61, P, 1, preorder_buffer_count=0, precision=plk.FP32)
        try:
            with pytest.raises(plk.PlkError) as e:
                inst.root_log_likelihoods_static_device(2, np.zeros(0, dtype=np.int32), d_sum)
            # inside the limit the call gets as far as the state checks (nothing was set up: _UNINITIALIZED)
            assert e.value.status == (plk.ERR_UNINITIALIZED if fits else plk.ERR_STATIC_SCRATCH_LIMIT)
            if not fits:
                assert "static scratch" in str(e.value)
                assert inst.kernel_launch_count() == 0  # rejected before anything was launched
        finally:
            inst.destroy()
    wl = workloads.config(0, n_patterns=64)
    ev = Evaluator(wl, precision=plk.FP64)
    try:
        ev.log_likelihood()
        with pytest.raises(plk.PlkError) as e:  # too many scale buffers for the on-stack list
            ev.inst.root_log_likelihoods_static_device(wl.tree.root, np.zeros(plk.STATIC_SCALE_MAX + 1, dtype=np.int32), d_sum)
        assert e.value.status == plk.ERR_STATIC_SCRATCH_LIMIT
        with pytest.raises(plk.PlkError) as e:
            ev.inst.root_log_likelihoods_static_device(wl.tree.root, [10_000], d_sum)
        assert e.value.status == plk.ERR_OUT_OF_RANGE
        with pytest.raises(plk.PlkError) as e:
            ev.inst.root_log_likelihoods_static_device(0, ev.scale_idx, d_sum)  # a compact tip is no root
        assert e.value.status == plk.ERR_OUT_OF_RANGE
    finally:
        ev.close()
