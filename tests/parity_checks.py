"""Shared by the -m gpu parity tests: run libplk.so through its C ABI on a workload and compare with the oracle.

Tolerances (BASELINE.json north_star):
  fp64          site log-likelihoods, logL, per-pattern derivatives (norm-wise per branch) and EVERY branch gradient
                (strict, element-wise) within 1e-10 relative -- with the library given the same eigendecomposition
                (U, U^-1, lambda) as the oracle.  The eigendecomposition is a client-side INPUT of the library
                (plk_set_eigen_decomposition), so "the same seeded inputs" includes
                it.  Two different fp64 eigendecompositions of the same Q give transition matrices that differ by
                ~1e-12, which the cancellation in g_k = sum_p omega_p d_kp (a score at the truth) amplifies beyond
                1e-10 on some branches; tests/test_gpu_parity.py::test_fp64_residual_is_the_eigendecomposition
                measures exactly that (oracle's matrices: 6e-13, oracle's eigensystem: 7e-12, independent
                eigensystem: 1.7e-10 at configs[1] full size).
  fp32 / tensor site log-likelihoods and logL within 1e-4 relative; per-pattern derivatives within 1e-4 norm-wise per
                branch; gradients |dg_k| <= 1e-4 A_k for every branch and ||dg|| <= 1e-4 ||g||; every branch beyond
                strict 1e-4 must have cancellation ratio A_k / |g_k| > 100.
"""
import numpy as np

import oracle_runner as orc
from paper_2606_27607_b200 import plk
from paper_2606_27607_b200.client import Evaluator

FP64_TOL = 1e-10
FP32_TOL = 1e-4


def tol_of(precision):
    return FP64_TOL if precision == plk.FP64 else FP32_TOL


def run_gpu(wl, precision, flags=0, tips_as_partials=False, t=None, eigen="oracle", want_site=True, matrices=None):
    """One full evaluation through the C ABI.  eigen = "oracle": hand the oracle's (U, U^-1, lambda) to
    plk_set_eigen_decomposition; "client": the workload's own, independently computed one."""
    ev = Evaluator(wl, precision=precision, flags=flags | (plk.FLAG_SITE_DERIVATIVES if want_site else 0),
                   tips_as_partials=tips_as_partials, eigen=orc.oracle_eigen(wl) if eigen == "oracle" else None)
    try:
        logl, site = ev.log_likelihood(t, matrices=matrices)
        out = ev.gradient(want_site=want_site)
        launches = ev.inst.kernel_launch_count()
    finally:
        ev.close()
    assert launches > 0, "no kernel was launched"
    grad, site_d = out if want_site else (out, None)
    return logl, site, grad, site_d


def check_logl(site_gpu, logl_gpu, ref, precision):
    tol = tol_of(precision)
    rel = np.max(np.abs(site_gpu - ref["site_logl"]) / np.abs(ref["site_logl"]))
    assert rel <= tol, f"site logL rel err {rel:.3e} > {tol}"
    assert abs(logl_gpu - ref["logL"]) <= tol * abs(ref["logL"]), "logL"


def check_grad(g_gpu, ref, precision, root):
    """fp64: strict 1e-10 on every branch.  fp32: the three figures of SURVEY 8(c) row 18."""
    strict, rel_cond, norm = orc.gradient_errors(g_gpu, ref)
    assert g_gpu[root] == 0.0
    g = ref["grad"]
    gmax = np.max(np.abs(g))
    nz = np.abs(g) > 1e-13 * gmax  # analytically-zero derivatives (all-missing tip) are round-off on both sides
    d = np.abs(g_gpu - g)
    assert np.all(d[~nz] <= 1e-13 * gmax), "analytically-zero derivative is not ~0"
    if precision == plk.FP64:
        assert strict <= FP64_TOL, f"fp64 gradient strict rel err {strict:.3e}"
        assert norm <= FP64_TOL and rel_cond <= FP64_TOL
    else:
        assert rel_cond <= FP32_TOL, f"fp32 gradient err / A_k = {rel_cond:.3e}"
        assert norm <= FP32_TOL, f"fp32 gradient 2-norm rel err {norm:.3e}"
        bad = (d > FP32_TOL * np.abs(g)) & nz  # beyond strict tolerance: must be a heavy-cancellation branch
        assert np.all(ref["cond"][bad] > 100.0 * np.abs(g[bad]))
    return strict, rel_cond, norm


def check_site_derivs(site_d, ref, precision, root, cols=None):
    """Per-pattern derivatives, norm-wise per branch (last sentence): max_p |dd_kp| <= tol *
    max_p |d_kp|.  d_kp = num / den is a quotient whose numerator is a sum of terms of both signs (Q has a negative
    diagonal), so a single d_kp can be small by cancellation; the norm over the patterns of a branch absorbs that,
    but it degenerates when a branch has one pattern (P = 1) or is analytically zero (branch above an all-missing
    tip: pure round-off on both sides).  Hence a floor: a branch whose largest |d_kp| is below 1e-3 of the largest
    branch's is measured against that floor."""
    tol = tol_of(precision)
    sd = ref["site_derivs"]
    got = site_d if cols is None else site_d[:, cols]
    scale = np.max(np.abs(sd), axis=1)
    scale[root] = 0.0
    scale = np.maximum(scale, 1e-3 * np.max(scale))
    err = np.max(np.abs(got - sd), axis=1) / scale
    err[root] = 0.0
    k = int(np.argmax(err))
    assert err[k] <= tol, f"site derivative branch {k}: {err[k]:.3e} > {tol}"
    return float(err[k])
