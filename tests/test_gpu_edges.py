"""GPU edge / degenerate cases and error behaviour of the C ABI (-m gpu)."""
import numpy as np
import pytest

import oracle_runner as orc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu


def _compare(wl, precision, t=None, flags=0, strict_tol=1e-10, cond_tol=None):
    """Site log-likelihoods and gradient against the oracle (the oracle's eigendecomposition is handed to the
    library: tests/parity_checks.py)."""
    ev = Evaluator(wl, precision=precision, flags=flags, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood(t)
        g = ev.gradient()
    finally:
        ev.close()
    ref = orc.evaluate(wl, t)
    tol = 1e-10 if precision == plk.FP64 else 1e-4
    assert np.max(np.abs(site - ref["site_logl"]) / np.abs(ref["site_logl"])) <= tol
    strict, rel_cond, norm = orc.gradient_errors(g, ref)
    gmax = np.max(np.abs(ref["grad"]))
    zero = np.abs(ref["grad"]) <= 1e-13 * gmax  # analytically-zero derivatives: round-off on both sides
    assert np.all(np.abs(g[zero]) <= 1e-13 * gmax)
    if precision == plk.FP64:
        assert strict <= strict_tol, f"strict {strict:.3e}"
        if cond_tol is not None:
            assert rel_cond <= cond_tol
    else:
        assert rel_cond <= 1e-4 and norm <= 1e-4
    return site, g, ref


@pytest.mark.parametrize("precision", [plk.FP64, plk.FP32], ids=["fp64", "fp32"])
@pytest.mark.parametrize("model,n_tips,n_pat,n_cat", [("HKY", 2, 1, 1), ("HKY", 3, 129, 1), ("GY94", 2, 1, 1),
                                                      ("GY94", 3, 33, 2), ("GTR", 5, 128, 8)])
def test_minimal_sizes(precision, model, n_tips, n_pat, n_cat):
    """Smallest trees (2 and 3 tips), a single pattern, a single category, one-past-a-tile pattern counts."""
    wl = workloads.make_workload("tiny", model, n_tips, n_pat, "coalescent", seed=99 + n_tips + n_pat, n_cat=n_cat)
    _compare(wl, precision)


@pytest.mark.parametrize("model", ["HKY", "GY94"])
def test_all_missing_tip_and_zero_branch(model):
    """A tip that is missing at every pattern has derivative 0 on its branch (SURVEY 8(c) pins); t = 0 gives P = I."""
    wl = workloads.make_workload("edge", model, 6, 70, "yule", seed=5)
    wl.tip_states[2, :] = wl.n_states
    t = wl.tree.branch_length.copy()
    t[4] = 0.0
    t[wl.tree.n_tips] = 0.0
    site, g, ref = _compare(wl, plk.FP64, t)
    assert abs(g[2]) <= 1e-12 * np.max(np.abs(g))


def test_root_children_pulley():
    """Reversible model: the derivatives of the two root-child branches are equal."""
    wl = workloads.config(0, n_patterns=400)
    ev = Evaluator(wl)
    try:
        ev.log_likelihood()
        g = ev.gradient()
    finally:
        ev.close()
    a, b = wl.tree.children[wl.tree.root]
    assert abs(g[a] - g[b]) <= 1e-9 * max(abs(g[a]), 1.0)


@pytest.mark.parametrize("precision,n_tips", [(plk.FP64, 1500), (plk.FP32, 400)], ids=["fp64-1500", "fp32-400"])
def test_deep_caterpillar_needs_rescaling(precision, n_tips):
    """Deep tree: unscaled arithmetic underflows (oracle with rescale=False gives -inf), the library stays finite
    and matches the rescaled oracle."""
    wl = workloads.make_workload("deep", "HKY", n_tips, 40, "caterpillar", seed=31)
    site, g, ref = _compare(wl, precision, strict_tol=1e-10, cond_tol=1e-12)
    assert np.all(np.isfinite(site))
    if precision == plk.FP64:
        unscaled = orc.evaluate(wl, gradient=False, rescale=False)
        assert np.any(np.isneginf(unscaled["site_logl"]))
    else:
        assert np.min(ref["site_logl"]) < -120.0  # beyond the fp32 range (exp(-87))


def test_error_codes():
    wl = workloads.config(0, n_patterns=50)
    with pytest.raises(plk.PlkError) as e:
        plk.Instance(4, 70, 10, 4)
    assert e.value.status == plk.ERR_UNSUPPORTED
    with pytest.raises(plk.PlkError) as e:
        plk.Instance(1, 4, 10, 4)
    assert e.value.status == plk.ERR_OUT_OF_RANGE
    ev = Evaluator(wl)
    inst = ev.inst
    try:
        with pytest.raises(plk.PlkError) as e:
            inst.set_tip_states(99, np.zeros(50, dtype=np.int32))
        assert e.value.status == plk.ERR_OUT_OF_RANGE
        with pytest.raises(plk.PlkError) as e:  # negative branch length
            inst.update_transition_matrices(0, [0], [-0.1])
        assert e.value.status == plk.ERR_OUT_OF_RANGE
        with pytest.raises(plk.PlkError) as e:  # matrices not computed yet
            inst.update_partials(ev.ops)
        assert e.value.status == plk.ERR_UNINITIALIZED
        ev.log_likelihood()
        bad = ev.ops.copy()
        bad["child1"][0] = 1000
        with pytest.raises(plk.PlkError) as e:
            inst.update_partials(bad)
        assert e.value.status == plk.ERR_OUT_OF_RANGE
        dup = ev.ops.copy()
        dup["dest"][1] = dup["dest"][0]
        with pytest.raises(plk.PlkError) as e:
            inst.update_partials(dup)
        assert e.value.status == plk.ERR_OUT_OF_RANGE
        with pytest.raises(plk.PlkError) as e:  # site derivatives were not reserved at creation
            inst.pre_order_gradient(0, wl.tree.root, ev.pre_ops, want_site=True)
        assert e.value.status == plk.ERR_UNSUPPORTED
        with pytest.raises(plk.PlkError) as e:
            inst.get_partials(wl.tree.root, pre=True)
        assert e.value.status == plk.ERR_UNINITIALIZED
    finally:
        ev.close()
    # impossible data: a site whose likelihood is 0 -> _FLOATING_POINT, site value -inf
    inst = plk.Instance(2, 4, 3, 1)
    try:
        inst.set_pattern_weights(np.ones(3))
        inst.set_state_frequencies(np.full(4, 0.25))
        inst.set_category_weights([1.0])
        inst.set_category_rates([1.0])
        inst.set_tip_states(0, [0, 1, 2])
        inst.set_tip_states(1, [0, 1, 3])
        eye = np.eye(4)[None]
        inst.set_transition_matrix(0, eye)
        inst.set_transition_matrix(1, eye)
        ops = np.array([(2, 0, 0, 0, 1, 1)], dtype=plk.OP_DTYPE)
        inst.update_partials(ops)
        with pytest.raises(plk.PlkError) as e:
            inst.root_log_likelihoods(2, [0])
        assert e.value.status == plk.ERR_FLOATING_POINT
        logl, site = inst.root_log_likelihoods(2, [0], allow_nonfinite=True)
        assert np.isneginf(site[2]) and np.allclose(site[:2], np.log(0.25))
    finally:
        inst.destroy()
