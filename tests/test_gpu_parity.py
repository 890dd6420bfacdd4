"""GPU parity (-m gpu): libplk.so through its C ABI (via the thin binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances and what "the same inputs" means: tests/parity_checks.py (fp64 strict
1e-10 on every branch with the oracle's eigendecomposition handed to plk_set_eigen_decomposition; fp32 / tensor
1e-4 relative to A_k and in the 2-norm).  Sizes are reduced so that the oracle finishes in seconds but still span
several pattern tiles and a ragged tail (tile = 128 patterns for 4 states, 32 for 61 states); the full sizes are in
tests/test_gpu_full_size.py."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator, pre_order_ops

pytestmark = pytest.mark.gpu

FP64_TOL = pc.FP64_TOL
FP32_TOL = pc.FP32_TOL


def _run_case(wl, precision, flags=0, tips_as_partials=False, t=None, eigen="oracle"):
    logl, site, grad, site_d = pc.run_gpu(wl, precision, flags, tips_as_partials, t, eigen=eigen)
    ref = orc.evaluate(wl, t, keep_site_derivatives=True)
    pc.check_logl(site, logl, ref, precision)
    pc.check_grad(grad, ref, precision, wl.tree.root)
    pc.check_site_derivs(site_d, ref, precision, wl.tree.root)
    return ref, grad


PREC = [pytest.param(plk.FP64, id="fp64"), pytest.param(plk.FP32, id="fp32")]


def test_config0_full():
    """BASELINE configs[0] at full size: HKY, 8 taxa, 1000 distinct patterns, 4 gamma categories, fp64."""
    _run_case(workloads.config(0), plk.FP64)


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("as_partials", [False, True], ids=["compact", "tip-partials"])
def test_config1_reduced(precision, as_partials):
    """configs[1] shape (GTR, 128 taxa, Yule, 5% ambiguity) at 3000 patterns = 23 tiles of 128 + a tail of 56."""
    _run_case(workloads.config(1, n_patterns=3000), precision, tips_as_partials=as_partials)


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("shape", [plk.FLAG_LEVEL_BATCH_ONLY, plk.FLAG_PATTERN_WALK_ONLY], ids=["level", "walk"])
@pytest.mark.parametrize("n_cat", [1, 2, 3, 4, 6, 8])
@pytest.mark.parametrize("staging", [0, plk.FLAG_NO_TMA], ids=["tma", "ldg"])
def test_nucleotide_launch_shapes_and_category_counts(precision, shape, n_cat, staging):
    """Both launch shapes of the 4-state kernels (one launch per level / one pattern-walk launch) and both staging
    schemes (TMA ring / register-staged; 3 and 6 categories always run register-staged) for every lane mapping
    (1, 2 or 4 lanes per pattern); 1237 patterns = a ragged last tile for each."""
    _run_case(workloads.config(1, n_tips=24, n_patterns=1237, n_categories=n_cat), precision, flags=shape | staging)


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("n_pat", [1, 7, 8, 33, 5000])
def test_nucleotide_walk_small_and_ragged_pattern_counts(precision, n_pat):
    """Walk shape with fewer own tiles than pipeline stages (the producer's extra dependency wait), a single
    pattern, and a pattern count that leaves CTAs with ranges of different length."""
    _run_case(workloads.config(1, n_tips=40, n_patterns=n_pat), precision, flags=plk.FLAG_PATTERN_WALK_ONLY)


@pytest.mark.parametrize("precision", PREC)
def test_gradient_launch_chain_matches_plain_launches(precision):
    """4-state gradient pass: the programmatic dependent launch chain (the item classes of a dependency level
    overlap one another's tail; a level still waits for the one before it) against plain stream-ordered launches
    (PLK_FLAG_NO_PDL).  Same kernels, fixed summation order: the gradients must be bitwise equal, repeatedly (an
    ordering bug would show as a stale q_parent).  Deep tree = many short levels."""
    wl = workloads.config(1, n_tips=96, n_patterns=20000)
    _, g_plain = _run_case(wl, precision, flags=plk.FLAG_NO_PDL | plk.FLAG_LEVEL_BATCH_ONLY)
    ev = Evaluator(wl, precision=precision, flags=plk.FLAG_LEVEL_BATCH_ONLY, eigen=orc.oracle_eigen(wl))
    try:
        for _ in range(20):
            ev.log_likelihood()
            assert np.array_equal(ev.gradient(), g_plain)
    finally:
        ev.close()


@pytest.mark.parametrize("precision", PREC)
def test_config1_perturbed_branch_lengths(precision):
    wl = workloads.config(1, n_patterns=2000)
    ref, grad = _run_case(wl, precision, t=wl.perturbed_branch_lengths())
    if precision == plk.FP32:  # away from the truth strict 1e-4 holds on all well-conditioned branches
        g = ref["grad"]
        ok = np.abs(g) > 1e-3 * ref["cond"]
        assert np.max(np.abs(grad[ok] - g[ok]) / np.abs(g[ok])) <= FP32_TOL


@pytest.mark.parametrize("precision", PREC)
def test_config2_reduced_cuda_cores(precision):
    """configs[2] shape (GY94, 61 states, 32 taxa) at 500 patterns = 15 tiles of 32 + a tail of 20; CUDA-core path."""
    _run_case(workloads.config(2, n_patterns=500), precision)


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("n_pat", [500, 64, 129, 1])
def test_config2_reduced_tensor_cores(precision, n_pat):
    """configs[2] on the tensor pipe (fp64: DMMA m8n8k4, fp32: split-TF32 m16n8k8): 500 patterns = several tiles of
    64 / 128 + a ragged tail; exactly one fp64 tile; one fp32 tile + 1; a single pattern."""
    _run_case(workloads.config(2, n_patterns=n_pat), precision, flags=plk.FLAG_TENSOR_CORES)


@pytest.mark.parametrize("precision", PREC)
def test_config2_tensor_cores_tip_partials(precision):
    """Tips supplied as partials (KIND_BCAST operands go through the contraction instead of the column gather)."""
    _run_case(workloads.config(2, n_tips=12, n_patterns=300), precision, flags=plk.FLAG_TENSOR_CORES,
              tips_as_partials=True)


@pytest.mark.parametrize("arm", [0, plk.FLAG_NO_TCGEN05], ids=["tcgen05", "mma_sync"])
def test_config3_reduced_tensor_cores(arm):
    """configs[3] shape (GY94, 256 taxa, 510 branches, level-batched) at 150 patterns, fp32 tensor path: post-order on
    tcgen05 / TMEM (default) and on the legacy mma.sync arm."""
    _run_case(workloads.config(3, n_patterns=150), plk.FP32, flags=plk.FLAG_TENSOR_CORES | arm)


@pytest.mark.parametrize("n_pat", [500, 129])
def test_config2_fp32_mma_sync_arm(n_pat):
    """The comparison arm PLK_FLAG_NO_TCGEN05 (split-TF32 m16n8k8 post-order) stays parity-green."""
    _run_case(workloads.config(2, n_patterns=n_pat), plk.FP32, flags=plk.FLAG_TENSOR_CORES | plk.FLAG_NO_TCGEN05)


@pytest.mark.parametrize("n_cat,n_pat", [(1, 257), (2, 128), (3, 300), (5, 77), (8, 1000)])
def test_tcgen05_category_counts_and_tiles(n_cat, n_pat):
    """tcgen05 post-order kernel: category counts other than 4 (the pending-exponent fetch handles C > 4 separately),
    exactly one / two tiles, ragged tails, more work items than CTAs (8 categories x 8 tiles x 31 operations)."""
    _run_case(workloads.config(2, n_patterns=n_pat, n_categories=n_cat), plk.FP32, flags=plk.FLAG_TENSOR_CORES)


def test_tcgen05_missing_states_and_deep_tree():
    """One-hot / all-ones tip rows on the tensor pipe (10 % missing cells) and a 200-taxon caterpillar-like depth
    where the deferred power-of-two rescaling is necessary in fp32."""
    wl = workloads.config(2, n_tips=20, n_patterns=200)
    rng = np.random.default_rng(7)
    wl.tip_states[rng.random(wl.tip_states.shape) < 0.1] = wl.n_states
    _run_case(wl, plk.FP32, flags=plk.FLAG_TENSOR_CORES)
    _run_case(workloads.config(3, n_tips=200, n_patterns=140), plk.FP32, flags=plk.FLAG_TENSOR_CORES)


def test_config3_reduced_cuda_cores():
    """configs[3] shape (GY94, 256 taxa, 510 branches, level-batched) at 150 patterns, fp32."""
    _run_case(workloads.config(3, n_patterns=150), plk.FP32)


@pytest.mark.parametrize("n_tips,n_patterns", [(8, 100), (32, 1000), (128, 777), (512, 300)])
def test_config4_sweep_points(n_tips, n_patterns):
    """configs[4]: HKY fp32 sweep, small points + a deep 512-taxon tree (rescaling is necessary in fp32 there)."""
    _run_case(workloads.config(4, n_tips=n_tips, n_patterns=n_patterns), plk.FP32)


# ---- what the fp64 tolerance rests on ---------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n_pat,flags", [(2, 500, 0), (2, 500, plk.FLAG_TENSOR_CORES), (2, 3000, plk.FLAG_TENSOR_CORES),
                                             (1, 20000, 0)],
                         ids=["cfg2-cuda", "cfg2-dmma", "cfg2-dmma-3000", "cfg1-20000"])
def test_fp64_residual_is_the_eigendecomposition(cfg, n_pat, flags):
    """Three evaluations of the same workload in fp64, differing only in where the transition matrices come from:
      (i)   the oracle's own matrices handed in through plk_set_transition_matrix  -> the kernels' arithmetic alone:
            every gradient within 1e-11 strict, site log-likelihoods within 1e-13;
      (ii)  the oracle's (U, U^-1, lambda) through plk_set_eigen_decomposition      -> adds k_transition's summation
            order: strict 1e-10 on every branch (the parity criterion of north_star);
      (iii) the workload's independently computed eigensystem of the same Q         -> two valid fp64
            eigendecompositions differ by ~1e-15 / eigenvalue gap, the matrices by ~1e-12, and the cancellation in
            g_k = sum_p omega_p d_kp (A_k / |g_k| up to 1e4) lifts some branches above 1e-10 strict; bounded here in
            the A_k-relative form of SURVEY 8(c) row 18: |dg_k| <= 1e-10 A_k and ||dg|| <= 1e-10 ||g|| (measured
            |dg_k| / A_k: 1e-12 typically, 1.9e-11 at 129 patterns).
    (Measured on B200 at configs[1] full size: 5.6e-13 / 6.8e-12 / 1.7e-10 strict.)"""
    wl = workloads.config(cfg, n_patterns=n_pat)
    ref = orc.evaluate_pool(wl, keep_site_derivatives=True, chunk=1024)
    root = wl.tree.root
    # (i)
    logl, site, grad, site_d = pc.run_gpu(wl, plk.FP64, flags, matrices=orc.oracle_transition_matrices(wl))
    strict, rel_cond, norm = orc.gradient_errors(grad, ref)
    assert np.max(np.abs(site - ref["site_logl"]) / np.abs(ref["site_logl"])) <= 1e-13
    assert strict <= 1e-11 and rel_cond <= 1e-14
    # (ii)
    logl, site, grad, site_d = pc.run_gpu(wl, plk.FP64, flags, eigen="oracle")
    pc.check_logl(site, logl, ref, plk.FP64)
    pc.check_grad(grad, ref, plk.FP64, root)
    pc.check_site_derivs(site_d, ref, plk.FP64, root)
    # (iii)
    logl, site, grad, site_d = pc.run_gpu(wl, plk.FP64, flags, eigen="client")
    pc.check_logl(site, logl, ref, plk.FP64)
    strict, rel_cond, norm = orc.gradient_errors(grad, ref)
    g, d = ref["grad"], np.abs(grad - ref["grad"])
    bad = d > FP64_TOL * np.abs(g)
    assert np.all(d <= FP64_TOL * ref["cond"] + 1e-13 * np.max(np.abs(g))) and norm <= FP64_TOL
    assert np.all(ref["cond"][bad] > 50.0 * np.abs(g[bad])), "beyond strict 1e-10 without heavy cancellation"


# ---- mixed operand kinds, partial branch lists, launch-chain stress -----------------------
@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("flags", [0, plk.FLAG_LEVEL_BATCH_ONLY, plk.FLAG_PATTERN_WALK_ONLY, plk.FLAG_NO_TMA],
                         ids=["auto", "level", "walk", "ldg"])
def test_mixed_tip_kinds(precision, flags):
    """Some tips as partials, the others as compact states: one gradient call then mixes the class-specialised kernels
    (tile of 32 x rows) with the general one (tile of 32), whose partial-sum rows have different lengths."""
    wl = workloads.config(1, n_tips=24, n_patterns=1237)
    as_partials = np.arange(wl.tree.n_tips) % 3 == 0
    _run_case(wl, precision, flags=flags, tips_as_partials=as_partials)
    wl = workloads.config(1, n_tips=3, n_patterns=333)  # ((A, B) compact, C partials): the smallest mix
    _run_case(wl, precision, flags=flags, tips_as_partials=np.array([False, False, True]))


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("cfg,n_tips,n_pat,flags", [(1, 24, 1237, 0), (1, 24, 1237, plk.FLAG_PATTERN_WALK_ONLY),
                                                    (2, 10, 150, 0), (2, 10, 150, plk.FLAG_TENSOR_CORES)],
                         ids=["nuc-auto", "nuc-walk", "codon-cuda", "codon-tensor"])
def test_gradient_for_a_subset_of_branches(precision, cfg, n_tips, n_pat, flags):
    """plk_pre_order_gradient with derivatives requested for only some branches: ops whose sibling op is absent run
    unpaired (one child of the item has no slot), ops that only propagate q carry no gradient slot."""
    wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_pat)
    tree = wl.tree
    ev = Evaluator(wl, precision=precision, flags=flags, eigen=orc.oracle_eigen(wl))
    try:
        ev.log_likelihood()
        full = pre_order_ops(tree)
        # keep every op that stores q (internal children: the traversal below them needs it) and every third tip op
        keep = [i for i, o in enumerate(full) if o["dest_pre"] >= 0 or o["node_post"] % 3 == 0]
        ops = full[keep]
        g, _ = ev.inst.pre_order_gradient(0, tree.root, ops)
    finally:
        ev.close()
    ref = orc.evaluate(wl)
    nodes = ops["node_post"]
    d = np.abs(g - ref["grad"][nodes])
    if precision == plk.FP64:
        nz = np.abs(ref["grad"][nodes]) > 1e-13 * np.max(np.abs(ref["grad"]))
        assert np.all(d[nz] <= FP64_TOL * np.abs(ref["grad"][nodes][nz]))
    else:
        assert np.all(d <= FP32_TOL * ref["cond"][nodes] + 1e-30)


@pytest.mark.parametrize("precision", PREC)
@pytest.mark.parametrize("topology,n_tips,n_pat,n_cat", [("caterpillar", 40, 9000, 4), ("yule", 200, 4000, 4),
                                                         ("coalescent", 17, 30011, 4), ("yule", 64, 5000, 2)])
def test_launch_chain_stress(precision, topology, n_tips, n_pat, n_cat):
    """The programmatic-dependent-launch chain of the 4-state gradient pass over several tree shapes (a caterpillar
    has one item per level: every launch is the first of its level; wide Yule levels mix all three item classes)
    and category counts: bitwise equal to plain launches, ten times over."""
    wl = workloads.make_workload("chain", "HKY", n_tips, n_pat, topology, seed=4242 + n_tips, n_cat=n_cat)
    _, g_plain = _run_case(wl, precision, flags=plk.FLAG_NO_PDL | plk.FLAG_LEVEL_BATCH_ONLY)
    ev = Evaluator(wl, precision=precision, flags=plk.FLAG_LEVEL_BATCH_ONLY, eigen=orc.oracle_eigen(wl))
    try:
        for _ in range(10):
            ev.log_likelihood()
            assert np.array_equal(ev.gradient(), g_plain)
    finally:
        ev.close()
