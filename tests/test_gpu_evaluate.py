"""plk_evaluate / plk_evaluate_device (-m gpu): steps 1-6 in one call, replayed from a cached CUDA graph.

Every use of a call signature -- the eager first ones, the captured one and the graph replays -- must give the oracle's
log-likelihood and gradient (the graph launches the same kernels with the same arguments), also after the inputs the
graph reads from device memory (branch lengths, tip states) have changed, and after a change that is baked into the
launch parameters (the rate matrix) has invalidated the graph."""
import numpy as np
import pytest

import oracle_runner as orc
import parity_checks as pc
from paper_2606_27607_b200 import plk, workloads
from paper_2606_27607_b200.client import Evaluator

pytestmark = pytest.mark.gpu

CASES = [
    pytest.param(0, None, 600, plk.FP64, 0, id="cfg0-fp64"),
    pytest.param(0, None, 600, plk.FP32, 0, id="cfg0-fp32"),
    pytest.param(4, 8, 100, plk.FP32, 0, id="cfg4-8x100-fp32"),
    pytest.param(1, 24, 3000, plk.FP64, 0, id="gtr-24x3000-fp64"),
    pytest.param(1, 24, 3000, plk.FP32, plk.FLAG_LEVEL_BATCH_ONLY, id="gtr-24x3000-fp32-level"),
    pytest.param(2, 8, 300, plk.FP64, plk.FLAG_TENSOR_CORES, id="gy94-8x300-fp64-dmma"),
    pytest.param(2, 8, 300, plk.FP32, plk.FLAG_TENSOR_CORES, id="gy94-8x300-fp32-tcgen05"),
    pytest.param(2, 8, 300, plk.FP64, 0, id="gy94-8x300-fp64-cuda"),
    pytest.param(5, 8, 300, plk.FP64, 0, id="aa-8x300-fp64"),
]


def _check(logl, grad, ref, precision, root):
    tol = pc.tol_of(precision)
    assert abs(logl - ref["logL"]) <= tol * abs(ref["logL"])
    pc.check_grad(grad, ref, precision, root)


@pytest.mark.parametrize("cfg,n_tips,n_pat,precision,flags", CASES)
def test_evaluate_matches_oracle_on_every_use(cfg, n_tips, n_pat, precision, flags):
    import torch

    wl = workloads.config(cfg, n_tips=n_tips, n_patterns=n_pat)
    ref = orc.evaluate(wl)
    root = wl.tree.root
    stream = torch.cuda.Stream()  # a graph needs a capturable (non-default) stream
    with torch.cuda.stream(stream):
        ev = Evaluator(wl, precision=precision, flags=flags, stream=stream, eigen=orc.oracle_eigen(wl))
        try:
            ev.make_device_io()
            results = []
            for _ in range(6):  # eager, eager (bindings settled), captured, replayed x 3
                ev.step_evaluate()
                stream.synchronize()
                out = ev.d_out.cpu().numpy()
                grad = np.zeros(wl.tree.n_nodes)
                grad[ev.branch_nodes] = out[1:]
                _check(float(out[0]), grad, ref, precision, root)
                results.append(out.copy())
            # fixed-order reductions: eager, captured and replayed evaluations are bitwise equal
            for r in results[1:]:
                assert np.array_equal(r, results[0])
            n0 = ev.inst.kernel_launch_count()
            ev.step_evaluate()
            per_eval = ev.inst.kernel_launch_count() - n0
            assert per_eval > 0  # the replay accounts for the kernels of the graph
            # new branch lengths: read from device memory by the graph -> same graph, new result
            rng = np.random.default_rng(5)
            t2 = np.asarray(wl.tree.branch_length) * np.exp(rng.normal(0.0, 0.3, size=wl.tree.n_nodes))
            ref2 = orc.evaluate(wl, branch_lengths=t2)
            ev.d_t.copy_(torch.from_numpy(np.ascontiguousarray(t2[ev.matrix_idx])))
            ev.step_evaluate()
            stream.synchronize()
            out = ev.d_out.cpu().numpy()
            grad = np.zeros(wl.tree.n_nodes)
            grad[ev.branch_nodes] = out[1:]
            _check(float(out[0]), grad, ref2, precision, root)
            # host variant (plk_evaluate): its own signature (library staging buffers), eager -> captured -> replayed
            for _ in range(4):
                logl, g = ev.evaluate(t2)
                _check(logl, g, ref2, precision, root)
            logl, g = ev.evaluate()
            _check(logl, g, ref, precision, root)
        finally:
            ev.close()


def test_model_change_invalidates_the_graph():
    """The 4-state gradient kernels take Q by value (a launch parameter baked into the graph): after
    plk_set_rate_matrix / plk_set_eigen_decomposition the old graph must not be replayed."""
    import torch

    wl = workloads.config(0, n_patterns=500)
    wl2 = workloads.config(0, n_patterns=500)
    wl2.model = dict(wl2.model)
    wl2.model["kappa"] = 5.0
    ref2 = orc.evaluate(wl2)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ev = Evaluator(wl, precision=plk.FP64, stream=stream)
        try:
            ev.make_device_io()
            for _ in range(4):
                ev.step_evaluate()
            ev.inst.set_eigen_decomposition(0, *orc.oracle_eigen(wl2))
            ev.inst.set_rate_matrix(0, orc.oracle_model(wl2)[0])
            ev.inst.set_state_frequencies(orc.oracle_model(wl2)[1])
            for _ in range(4):
                ev.step_evaluate()
                stream.synchronize()
                out = ev.d_out.cpu().numpy()
                grad = np.zeros(wl.tree.n_nodes)
                grad[ev.branch_nodes] = out[1:]
                _check(float(out[0]), grad, ref2, plk.FP64, wl.tree.root)
        finally:
            ev.close()


def test_default_stream_runs_eagerly_and_errors_propagate():
    wl = workloads.config(0, n_patterns=200)
    ref = orc.evaluate(wl)
    ev = Evaluator(wl, precision=plk.FP64, eigen=orc.oracle_eigen(wl))  # torch's current stream = legacy default
    try:
        for _ in range(4):
            logl, g = ev.evaluate()
            _check(logl, g, ref, plk.FP64, wl.tree.root)
        t = np.asarray(wl.tree.branch_length).copy()
        t[0] = -1.0
        with pytest.raises(plk.PlkError) as e:
            ev.evaluate(t)
        assert e.value.status == plk.ERR_OUT_OF_RANGE
        bad = ev.ops.copy()
        bad["child1"][0] = 10_000
        with pytest.raises(plk.PlkError):
            ev.inst.evaluate(0, ev.matrix_idx, np.asarray(wl.tree.branch_length)[ev.matrix_idx], bad, wl.tree.root,
                             ev.scale_idx, wl.tree.root, ev.pre_ops)
    finally:
        ev.close()


@pytest.mark.parametrize("n_pat", [3001, 2048])  # staged pitched copy / one linear copy (P a multiple of the slot pitch)
def test_set_all_tip_states_u8_matches_per_tip_upload(n_pat):
    """plk_set_all_tip_states_u8: the whole alignment in one call.  Uploading the columns in reversed order must give
    the reversed per-pattern log-likelihoods of the per-tip upload (patterns are independent), which the
    other tests compare with the oracle."""
    wl = workloads.config(1, n_tips=24, n_patterns=n_pat)
    ref = orc.evaluate(wl, gradient=False)
    ev = Evaluator(wl, precision=plk.FP64, eigen=orc.oracle_eigen(wl))
    try:
        logl, site = ev.log_likelihood()
        pc.check_logl(site, logl, ref, plk.FP64)
        rev = np.ascontiguousarray(np.minimum(wl.tip_states, 255).astype(np.uint8)[:, ::-1])
        ev.inst.set_all_tip_states_u8(rev)
        ev.inst.set_pattern_weights(wl.pattern_weights[::-1].copy())
        logl2, site2 = ev.log_likelihood()
        assert np.array_equal(site2, site[::-1])
        assert abs(logl2 - logl) <= 1e-12 * abs(logl)
        # a prefix of the tips only: the others keep their states
        fwd = np.ascontiguousarray(np.minimum(wl.tip_states, 255).astype(np.uint8))
        ev.inst.set_all_tip_states_u8(fwd[:10])
        for k in range(10, wl.tree.n_tips):
            ev.inst.set_tip_states_u8(k, fwd[k])
        ev.inst.set_pattern_weights(wl.pattern_weights)
        logl3, site3 = ev.log_likelihood()
        assert np.array_equal(site3, site) and logl3 == logl
    finally:
        ev.close()
    ev = Evaluator(wl, precision=plk.FP64, tips_as_partials=True)
    try:
        with pytest.raises(plk.PlkError) as e:  # tips bound as partials cannot become compact states
            ev.inst.set_all_tip_states_u8(fwd)
        assert e.value.status == plk.ERR_OUT_OF_RANGE
    finally:
        ev.close()


def test_more_signatures_than_cached_plans():
    """The library caches at most 8 evaluation graphs per instance and then drops them all: twelve different call
    signatures (the same evaluation with the branch list rotated), each used often enough to be captured and replayed,
    must all give the same result as the first."""
    import torch

    wl = workloads.config(0, n_patterns=300)
    ref = orc.evaluate(wl)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        ev = Evaluator(wl, precision=plk.FP64, stream=stream, eigen=orc.oracle_eigen(wl))
        try:
            t = np.asarray(wl.tree.branch_length)
            first = None
            for rot in range(12):
                idx = np.roll(ev.matrix_idx, rot)
                for use in range(4):
                    logl, g = ev.inst.evaluate(0, idx, t[idx], ev.ops, wl.tree.root, ev.scale_idx, wl.tree.root, ev.pre_ops)
                    grad = np.zeros(wl.tree.n_nodes)
                    grad[ev.branch_nodes] = g
                    _check(logl, grad, ref, plk.FP64, wl.tree.root)
                    if first is None:
                        first = (logl, g.copy())
                    assert logl == first[0] and np.array_equal(g, first[1])
        finally:
            ev.close()
