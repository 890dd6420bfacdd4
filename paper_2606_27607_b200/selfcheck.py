"""Install / sanitizer check of libplk.so: every kernel family once, on small seeded inputs.

    python -m paper_2606_27607_b200.selfcheck [--quick]
    compute-sanitizer --tool memcheck python -m paper_2606_27607_b200.selfcheck --quick

Runs a full evaluation (matrices -> post-order -> root -> pre-order + gradient, fused and unfused) through every
launch shape, staging scheme and codon path the library has (the flag arms of include/plk.h) and checks that all
arms of one precision agree with the first one (they compute the same numbers in different orders).  No oracle is
involved: this is the product checking itself for consistency, sized so that it finishes under compute-sanitizer
(memcheck / racecheck / initcheck / synccheck) in minutes.  Parity with the paper's method is tests/'s job.
"""
import sys

import numpy as np

from . import build, plk, workloads
from .client import Evaluator

NUC_ARMS = [("default", 0), ("level", plk.FLAG_LEVEL_BATCH_ONLY), ("walk", plk.FLAG_PATTERN_WALK_ONLY),
            ("level-ldg", plk.FLAG_LEVEL_BATCH_ONLY | plk.FLAG_NO_TMA), ("walk-ldg", plk.FLAG_PATTERN_WALK_ONLY | plk.FLAG_NO_TMA),
            ("level-no-pdl", plk.FLAG_LEVEL_BATCH_ONLY | plk.FLAG_NO_PDL), ("per-op", plk.FLAG_NO_LEVEL_BATCH)]
CODON_ARMS = [("cuda-core", 0), ("tensor", plk.FLAG_TENSOR_CORES),
              ("tensor-mma.sync", plk.FLAG_TENSOR_CORES | plk.FLAG_NO_TCGEN05)]


def _one(wl, precision, flags, tips_as_partials=False, unfused=False):
    ev = Evaluator(wl, precision=precision, flags=flags, tips_as_partials=tips_as_partials, store_tip_pre=unfused)
    try:
        logl, site = ev.log_likelihood()
        grad = ev.gradient_unfused() if unfused else ev.gradient()
        n = ev.inst.kernel_launch_count()
    finally:
        ev.close()
    if not (np.isfinite(logl) and np.all(np.isfinite(site)) and np.all(np.isfinite(grad))):
        raise AssertionError("non-finite result")
    return logl, site, grad, n


def run(quick=False):
    build.build()
    n_nuc, n_cod = (700, 150) if quick else (5000, 600)
    mixed = None
    cases = []
    wl4 = workloads.config(1, n_tips=12, n_patterns=n_nuc)
    wl61 = workloads.config(2, n_tips=8, n_patterns=n_cod)
    wl20 = workloads.config(5, n_tips=8, n_patterns=n_cod)
    mixed = np.arange(wl4.tree.n_tips) % 3 == 0  # every third tip as partials, the others compact
    for prec, pname in ((plk.FP64, "fp64"), (plk.FP32, "fp32")):
        for name, flags in NUC_ARMS:
            cases.append((f"nuc-{pname}-{name}", wl4, prec, flags, False, False))
        cases.append((f"nuc-{pname}-tip-partials", wl4, prec, 0, True, False))
        cases.append((f"nuc-{pname}-mixed-tips-level", wl4, prec, plk.FLAG_LEVEL_BATCH_ONLY, mixed, False))
        cases.append((f"nuc-{pname}-unfused", wl4, prec, 0, False, True))
        for name, flags in CODON_ARMS:
            cases.append((f"codon-{pname}-{name}", wl61, prec, flags, False, False))
        cases.append((f"codon-{pname}-tensor-tip-partials", wl61, prec, plk.FLAG_TENSOR_CORES, True, False))
        cases.append((f"codon-{pname}-unfused", wl61, prec, 0, False, True))
        cases.append((f"amino-{pname}", wl20, prec, 0, False, False))
        cases.append((f"amino-{pname}-tip-partials", wl20, prec, 0, True, False))
        cases.append((f"amino-{pname}-unfused", wl20, prec, 0, False, True))
    base = {}
    worst = 0.0
    total = 0
    for name, wl, prec, flags, tap, unfused in cases:
        logl, site, grad, n = _one(wl, prec, flags, tap, unfused)
        total += n
        key = (id(wl), prec)
        if key not in base:
            base[key] = (logl, site, grad)
        b = base[key]
        tol = 1e-9 if prec == plk.FP64 else 2e-4
        e_site = float(np.max(np.abs(site - b[1]) / np.abs(b[1])))
        e_grad = float(np.linalg.norm(grad - b[2]) / np.linalg.norm(b[2]))
        worst = max(worst, e_site / tol, e_grad / tol)
        print(f"{name:40s} logL {logl:.9f}  vs first arm: site {e_site:.1e} grad {e_grad:.1e}  launches {n}")
        if e_site > tol or e_grad > tol:
            raise AssertionError(f"{name}: arms disagree (site {e_site:.2e}, grad {e_grad:.2e}, tol {tol})")
    print(f"selfcheck ok: {len(cases)} arms, {total} kernel launches")


if __name__ == "__main__":
    run(quick="--quick" in sys.argv)
