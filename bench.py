"""bench.py -- throughput of the whole hot path on synthetic seeded workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--precision fp64|fp32] [--tensor]
                    [--impl ours|reference] [--no-extras]

One "step" = one full evaluation as an HMC step needs it: transition matrices for all 2N-2 branches,
post-order partials over the whole tree with rescaling, root log-likelihood, pre-order partials fused with all 2N-2
branch-length derivatives.  Default workload: BASELINE.json configs[1] (GTR, 128 taxa, 100 000 patterns, 4 gamma
categories, 5% tip ambiguity), fp64.  Prints ONE JSON line (rank 0).  Multi-GPU (--gpus N; the driver launches N
ranks with torchrun, a plain `python bench.py --gpus N` re-launches itself that way): by default N independent
replicas, scaling "weak" (north_star: "no sharding or collectives across GPUs"); with --shard-patterns the pattern
axis is split into N contiguous ranges, one instance per GPU, and logL + the 2N-2 derivatives are summed with ONE
all-reduce per evaluation, scaling "strong".
The oracle (oracle/) is executed only by the cpu_baseline / parity leg and by --impl reference.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "node-pattern-cat updates/s (full logL + all-branch-gradient evaluation)"
UNIT = "updates/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--taxa", type=int, default=None)
    ap.add_argument("--patterns", type=int, default=None)
    ap.add_argument("--precision", choices=["fp64", "fp32"], default="fp64")
    ap.add_argument("--tensor", action="store_true", help="61-state kernels on the tensor pipe")
    ap.add_argument("--shape", choices=["auto", "level", "walk"], default="auto",
                    help="4-state launch shape: one launch per level / one pattern-walk launch / library's choice")
    ap.add_argument("--staging", choices=["tma", "ldg"], default="tma",
                    help="4-state operand staging: TMA ring (cp.async.bulk) / register-staged loads")
    ap.add_argument("--no-pdl", action="store_true",
                    help="4-state gradient pass: plain stream-ordered launches (comparison arm of the programmatic "
                         "dependent launch chain)")
    ap.add_argument("--codon-fp32", choices=["tcgen05", "mma_sync"], default="tcgen05",
                    help="fp32 --tensor codon kernels: tcgen05/TMEM (default) or the legacy mma.sync arm")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--sweep", action="store_true",
                    help="BASELINE configs[4]: HKY fp32, taxa {8,32,128,512} x patterns {1e2..5e5}; prints one JSON "
                         "line with the 20 points instead of the headline line")
    ap.add_argument("--rate-matrix-gradient", action="store_true",
                    help="also time plk_rate_matrix_gradient (SURVEY 8(f)-1) on the chosen workload")
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs / precisions")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shard-patterns", action="store_true",
                    help="N > 1: split the pattern axis over the ranks (one all-reduce of 1 + 2N-2 doubles per "
                         "evaluation) instead of running N independent replicas")
    return ap.parse_args()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return {"hbm_gbs": float(d["hbm_gbs"]), "bf16_tflops": float(d["bf16_tflops"]),
                "bf16_tflops_sustained": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


HBM_NOMINAL_GBS = 8000.0  # the "~8 TB/s" BASELINE.json north_star names (report against both)


def measure_matmul_peaks(device):
    """fp64 and TF32 dense matmul throughput of THIS box, measured the way MEASURED_PEAKS.json measured bf16
    (torch.matmul 8192^3 = cuBLAS, best of 5, CUDA events): the denominators of the codon rooflines (SURVEY 8(d):
    "peaks for fp64 and TF32 are not in MEASURED_PEAKS.json -- measure them in the same run").  A library GEMM used as
    a yardstick only; nothing on the product path calls it."""
    import torch

    out = {}
    n = 8192
    flops = 2.0 * n ** 3
    prev = torch.backends.cuda.matmul.allow_tf32
    try:
        for name, dtype, tf32 in (("fp64_tflops", torch.float64, False), ("tf32_tflops", torch.float32, True),
                                  ("fp32_simt_tflops", torch.float32, False)):
            torch.backends.cuda.matmul.allow_tf32 = tf32
            a = torch.randn(n, n, dtype=dtype, device=device)
            b = torch.randn(n, n, dtype=dtype, device=device)
            c = torch.empty(n, n, dtype=dtype, device=device)
            torch.matmul(a, b, out=c)
            best = None
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                torch.matmul(a, b, out=c)
                e1.record()
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                best = ms if best is None else min(best, ms)
            out[name] = flops / (best * 1e-3) / 1e12
            del a, b, c
    finally:
        torch.backends.cuda.matmul.allow_tf32 = prev
    out["how"] = "torch.matmul 8192^3 (2 n^3 flops), best of 5, CUDA events, this run"
    return out


# ---- algorithmic traffic / work of one evaluation ----------------
def algorithmic(N, P, S, C, w):
    SP = 4 if S == 4 else 64
    W = C * P * SP * w
    scale = 2 * P if S == 4 else C * P * w  # int16 exponents (4-state) / per-category maxima (64-state)
    post_bytes = (2 * N - 3) * W + N * P + 2 * (N - 1) * scale
    pre_bytes = 3 * (N - 2) * W + N * P
    mv = 2 * S * S  # flops of one S x S matrix-vector product
    post_flops = (N - 2) * P * C * mv      # internal child edges only (tip edges are column gathers)
    pre_flops = 3 * (N - 2) * P * C * mv   # recompute P_j p_j, apply P_k^T, apply Q
    return {"W": W, "post_bytes": post_bytes, "pre_bytes": pre_bytes, "post_flops": post_flops,
            "pre_flops": pre_flops, "updates": (N - 1) * P * C, "grad_units": (2 * N - 2) * P * C}


def issued_tensor_flops(N, P, C, precision, kernels):
    """Flops the 64-state tensor-pipe kernels ISSUE per evaluation (padding 61 -> 64, the three split-TF32 passes of
    the fp32 kernels, tip edges that travel through the pipe as one-hot rows), as opposed to the algorithmic count
    above ("report issued flops separately").  Edges: N - 2 internal child edges, N tip edges (compact).
      mma.sync (plk_tc.cuh)    post: internal edges only (tips are column gathers); pre: a_k, Q x_k, M_k^T u_k for every
                               edge with partials; fp32 = 3 passes
      tcgen05 (plk_tc5*.cuh)   post: every edge (one-hot tips: 2 of the 3 passes); pre (plk_tc5_pre2.cuh): a_k and
                               D_k x_k for internal edges (3 passes each) and M_k^T u_k for internal edges (3 passes);
                               tip edges are table gathers on the CUDA cores"""
    mv = 2.0 * 64 * 64 * P * C
    n_int, n_tip = N - 2, N
    passes = 1 if precision == "fp64" else 3
    if kernels == "tcgen05":
        post = mv * (3 * n_int + 2 * n_tip)
        pre = mv * (3 * (2 * n_int) + 3 * n_int)
    else:
        post = mv * passes * n_int
        pre = mv * passes * 3 * n_int
    return {"post": post, "pre": pre}


# ---- nvidia-smi clock sampler (B200_PROFILING.md "clocks DURING the timed region") -------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---- one workload on the GPU -------------------------------------------------------------------------------------
def measure_device(wl, precision, flags, steps, warmup, peaks, sampler=None, device="cuda:0", keep_site=False,
                   shard=None):
    """Device-resident timing: K full evaluations, CUDA events on the launching stream; per-phase events inside.
    shard = (rank, world, dist): this rank evaluates its pattern range and every step ends with the all-reduce of
    [logL, gradient] (sharded.py); the algorithmic work reported is then this rank's share."""
    import torch

    from paper_2606_27607_b200 import plk, sharded
    from paper_2606_27607_b200.client import Evaluator

    prec = plk.FP64 if precision == "fp64" else plk.FP32
    sh = None
    if shard is not None:
        sh = sharded.ShardedEvaluator(wl, shard[0], shard[1], dist=shard[2], device=device, precision=prec, flags=flags)
        ev = sh.local
        assert ev is not None, "empty shard: fewer pattern tiles than ranks"
    else:
        # a stream of its own: plk_evaluate* replays its cached CUDA graph only on a capturable (non-default) stream
        ev = Evaluator(wl, precision=prec, flags=flags, device=device, stream=torch.cuda.Stream(device))
        ev.make_device_io()
        torch.cuda.synchronize()  # set-up ran on torch's current stream; everything below on the instance's
    stream = ev.inst.stream
    d_site = torch.zeros(ev.wl.n_patterns, dtype=torch.float64, device=device) if keep_site else None

    def reduce_step():
        if sh is not None and sh.world > 1:
            sh.dist.all_reduce(sh.result, op=sh.dist.ReduceOp.SUM)

    for _ in range(max(warmup, 3)):
        ev.step_device()
        reduce_step()
    torch.cuda.synchronize()
    l0 = ev.inst.kernel_launch_count()
    marks = [[torch.cuda.Event(enable_timing=True) for _ in range(6)] for _ in range(steps)]
    if sampler is not None:
        sampler.start()
        time.sleep(0.3)
    torch.cuda.synchronize()
    for s in range(steps):
        marks[s][0].record(stream)
        ev.step_matrices()
        marks[s][1].record(stream)
        ev.step_post()
        marks[s][2].record(stream)
        ev.step_root()
        marks[s][3].record(stream)
        ev.step_pre_gradient()
        marks[s][4].record(stream)
        reduce_step()
        marks[s][5].record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler is not None else None
    launches = ev.inst.kernel_launch_count() - l0
    total_ms = marks[0][0].elapsed_time(marks[-1][5])
    # the same evaluation as ONE library call (plk_evaluate_device: eager, captured, then one CUDA-graph launch per use)
    one_call = None
    if sh is None:
        for _ in range(4):
            ev.step_evaluate()
        torch.cuda.synchronize()
        l1 = ev.inst.kernel_launch_count()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(stream)
        for _ in range(steps):
            ev.step_evaluate()
        g1.record(stream)
        torch.cuda.synchronize()
        one_call = {"ms_per_step": g0.elapsed_time(g1) / steps,
                    "launches_per_step": (ev.inst.kernel_launch_count() - l1) / steps,
                    "what": "plk_evaluate_device: steps 1-6 in one call, replayed from the cached CUDA graph"}
    phase = np.zeros(5)
    for s in range(steps):
        for i in range(5):
            phase[i] += marks[s][i].elapsed_time(marks[s][i + 1])
    phase /= steps
    site = None
    logl = float(ev.d_logl.cpu()[0])
    grad = ev.d_grad.cpu().numpy()
    if keep_site:
        # Parity leg (untimed): one more evaluation that also writes the per-pattern log-likelihoods, with the oracle's
        # own eigendecomposition handed to plk_set_eigen_decomposition -- a client-side input, so that
        # "the same inputs" includes it -- next to the timed run's independent one.
        sys.path.insert(0, os.path.join(ROOT, "tests"))
        import oracle_runner as orc

        ev.step_post()
        ev.inst.root_log_likelihoods_device(ev.tree.root, ev.scale_idx, ev.d_logl, d_site)
        torch.cuda.synchronize()
        site = {"client": (d_site.cpu().numpy(), logl, grad)}
        ev.inst.set_eigen_decomposition(0, *orc.oracle_eigen(ev.wl))
        ev.inst.set_rate_matrix(0, ev.wl.Q)
        ev.step_matrices()
        ev.step_post()
        ev.inst.root_log_likelihoods_device(ev.tree.root, ev.scale_idx, ev.d_logl, d_site)
        ev.step_pre_gradient()
        torch.cuda.synchronize()
        site["oracle"] = (d_site.cpu().numpy(), float(ev.d_logl.cpu()[0]), ev.d_grad.cpu().numpy())
        ev.upload_model()  # back to the workload's own model for the end-to-end leg
    N, P, S, C = ev.wl.tree.n_tips, ev.wl.n_patterns, ev.wl.n_states, ev.wl.n_categories
    w = 8 if precision == "fp64" else 4
    alg = algorithmic(N, P, S, C, w)
    ms_step = total_ms / steps
    res = {
        "ms_per_step": ms_step,
        "updates_per_s": alg["updates"] / (ms_step * 1e-3),
        "gradient_evals_per_s": 1e3 / ms_step,
        "bls_gradients_per_s": (2 * N - 2) * 1e3 / ms_step,
        "post_order_updates_per_s": alg["updates"] / (phase[1] * 1e-3),
        "grad_units_per_s": alg["grad_units"] / (phase[3] * 1e-3),
        "phase_ms": {"matrices": phase[0], "post_order": phase[1], "root": phase[2], "pre_order_gradient": phase[3],
                     "all_reduce": phase[4]},
        "post_gbs": alg["post_bytes"] / (phase[1] * 1e-3) / 1e9,
        "pre_gbs": alg["pre_bytes"] / (phase[3] * 1e-3) / 1e9,
        "post_tflops": alg["post_flops"] / (phase[1] * 1e-3) / 1e12,
        "pre_tflops": alg["pre_flops"] / (phase[3] * 1e-3) / 1e12,
        "launches": int(launches), "logL": logl, "grad": grad, "site": site,
        "grad_norm": float(np.linalg.norm(grad)),
        "finite": bool(np.isfinite(logl) and np.all(np.isfinite(grad))),
        "alg": alg, "clocks": clocks, "one_call": one_call,
    }
    return res, ev


def measure_rate_matrix_gradient(wl, precision, flags, steps, peaks, device="cuda:0"):
    """plk_rate_matrix_gradient over every branch, from the pre- and post-order
    partials an evaluation leaves on the device (tips' pre-order partials stored).  Timed per call with CUDA events on
    the instance's stream (the call ends with the 32 KB result read back).  Algorithmic bytes: q_k of every branch and
    p_k of every internal node, read once; flops: 2 S^2 per (branch, pattern, category)."""
    import torch

    from paper_2606_27607_b200 import plk
    from paper_2606_27607_b200.client import Evaluator

    prec = plk.FP64 if precision == "fp64" else plk.FP32
    ev = Evaluator(wl, precision=prec, flags=flags, device=device, store_tip_pre=True)
    try:
        ev.log_likelihood(want_site=False)
        ev.gradient_unfused()
        for _ in range(3):
            G = ev.rate_matrix_gradient()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        stream = torch.cuda.current_stream()
        e0.record(stream)
        for _ in range(steps):
            G = ev.rate_matrix_gradient()
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
    finally:
        ev.close()
    N, P, S, C = wl.tree.n_tips, wl.n_patterns, wl.n_states, wl.n_categories
    w = 8 if precision == "fp64" else 4
    sp = 4 if S == 4 else (32 if S <= 32 else 64)
    n_br, n_int = 2 * N - 2, N - 2
    nbytes = (n_br + n_int) * C * P * sp * w + N * P
    flops = 2.0 * n_br * C * P * S * S
    return {"ms": ms, "branches": n_br, "algorithmic_bytes": nbytes, "hbm_gbs": nbytes / ms / 1e6,
            "frac_hbm": nbytes / ms / 1e6 / peaks["hbm_gbs"], "alg_tflops": flops / ms / 1e9,
            "finite": bool(np.isfinite(G).all()),
            "kernel": "k_cross4" if S == 4 else ("k_cross_tc" if (flags & 1 and sp == 64) else "k_cross64")}


def measure_e2e(ev, wl, steps, warmup):
    """Same evaluation through the host-pointer C-ABI calls a client makes per HMC step: every step uploads the tip
    states (pinned host memory, one pitched copy: plk_set_all_tip_states_u8) and hands HOST branch lengths to
    plk_evaluate, which returns logL and the gradient to the HOST (one upload, the cached graph, one download)."""
    import torch

    N, P = wl.tree.n_tips, wl.n_patterns
    pinned = torch.empty((N, P), dtype=torch.uint8, pin_memory=True)  # one byte per pattern: what the kernels read
    pinned.copy_(torch.from_numpy(np.minimum(wl.tip_states, 255).astype(np.uint8)))
    tips = pinned.numpy()
    t = np.ascontiguousarray(np.asarray(wl.tree.branch_length)[ev.matrix_idx])

    def one():
        ev.inst.set_all_tip_states_u8(tips)
        return ev.inst.evaluate(0, ev.matrix_idx, t, ev.ops, wl.tree.root, ev.scale_idx, wl.tree.root, ev.pre_ops)

    for _ in range(max(3, warmup)):  # eager, captured, replayed; and the clocks are back up after the host-side parity leg
        one()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        logl, g = one()
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / steps
    return dt, N * P + t.size * 8, 8 + g.size * 8


# ---- the oracle on the host cores ------------------------------------------------------------------------------------
def cpu_model_string():
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_time(wl, n_sample, workers=1):
    """The fp64 CPU oracle as it stands on the first `n_sample` patterns of the workload (full evaluation incl. the
    gradient): in this process (workers = 1; `cores` = CPU time / wall time, i.e. the threads numpy's BLAS really
    used) or by pattern chunks in `workers` processes.  Returns (seconds, cores used, patterns, oracle result)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle_runner as orc

    n_sample = min(n_sample, wl.n_patterns)
    c0, t0 = os.times(), time.perf_counter()
    if workers <= 1:
        ref = orc.evaluate(wl, lo=0, hi=n_sample)
        used = None
    else:
        ref = orc.evaluate_pool(wl, lo=0, hi=n_sample, workers=workers, chunk=4096 if wl.n_states == 4 else 512)
        used = ref["workers"]
    dt = time.perf_counter() - t0
    c1 = os.times()
    if used is None:
        cpu = (c1.user - c0.user) + (c1.system - c0.system)
        used = max(1, int(round(cpu / dt)))
    return dt, used, n_sample, ref


def parity_against_oracle(ref, n_used, gpu, wl, branch_nodes):
    """The GPU's outputs on the timed workload against the oracle result of the cpu_baseline leg, on the oracle's
    patterns: every site log-likelihood; when the oracle covered ALL patterns also logL and every branch gradient
    (the three figures of SURVEY 8(c) row 18).  Two GPU evaluations are compared: with the oracle's eigendecomposition
    handed in (the parity criterion: fp64 1e-10 / fp32 1e-4) and with the workload's independently computed one."""
    return {which: _parity_one(ref, n_used, *gpu[which], wl, branch_nodes)
            for which in ("oracle", "client") if which in gpu} | {
        "eigendecomposition": {"oracle": "the oracle's (U, U^-1, lambda) given to plk_set_eigen_decomposition: same inputs",
                               "client": "the workload's own, computed independently (the timed run)"}}


def _parity_one(ref, n_used, gpu_site, gpu_logl, gpu_grad, wl, branch_nodes):
    out = {"patterns": n_used, "of": wl.n_patterns,
           "site_rel": float(np.max(np.abs(gpu_site[:n_used] - ref["site_logl"]) / np.abs(ref["site_logl"]))),
           "logL_rel_on_sample": float(abs(np.dot(wl.pattern_weights[:n_used], gpu_site[:n_used]) - ref["logL"])
                                       / abs(ref["logL"]))}
    if n_used == wl.n_patterns:
        g_ref, cond = ref["grad"][branch_nodes], ref["cond"][branch_nodes]
        d = np.abs(gpu_grad - g_ref)
        nz = np.abs(g_ref) > 1e-13 * np.max(np.abs(g_ref))
        out.update({"logL_rel": float(abs(gpu_logl - ref["logL"]) / abs(ref["logL"])),
                    "grad_strict_rel": float(np.max(d[nz] / np.abs(g_ref[nz]))),
                    "grad_rel_to_A_k": float(np.max(d[cond > 0] / cond[cond > 0])),
                    "grad_2norm_rel": float(np.linalg.norm(gpu_grad - g_ref) / np.linalg.norm(g_ref))})
    return out


def ncu_dram_bytes_per_step(csv_name, kernel_pattern):
    """DRAM bytes (read + write) per evaluation of the kernels whose name matches `kernel_pattern`, from a committed
    ncu launch list (profiles/*.csv, `--metrics gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum`):
    summed over every matching launch of the capture and divided by the number of evaluations in it (= launches of
    k_transition over more than one branch).  None when the list is absent."""
    import csv
    import re

    path = os.path.join(ROOT, "profiles", csv_name)
    if not os.path.exists(path):
        return None
    pat = re.compile(kernel_pattern)
    total, evals, seen = 0.0, 0, set()
    with open(path, newline="") as fh:
        rows = (ln for ln in fh if ln.startswith('"'))
        for row in csv.DictReader(rows):
            name, metric = row["Kernel Name"], row["Metric Name"]
            if metric in ("dram__bytes_read.sum", "dram__bytes_write.sum") and pat.search(name):
                val = float(row["Metric Value"].replace(",", ""))
                unit = row["Metric Unit"].lower()
                total += val * {"byte": 1.0, "kbyte": 1e3, "mbyte": 1e6, "gbyte": 1e9}.get(unit, 1.0)
            if "k_transition" in name and row["ID"] not in seen and row["Grid Size"].replace(" ", "") != "(1,1,1)":
                seen.add(row["ID"])
                evals += 1
    return total / evals if evals else None


# committed launch lists by (workload, precision); the newest capture of each is used
NCU_LISTS = {("cfg1_gtr_128x100000", "fp64"): ["r02_launches_cfg1_fp64.csv", "r01_launches_cfg1_fp64.csv"],
             ("cfg1_gtr_128x100000", "fp32"): ["r02_launches_cfg1_fp32.csv", "r01_launches_cfg1_fp32.csv"],
             ("cfg3_gy94_256x20000", "fp32"): ["r02_launches_cfg3_fp32_tensor.csv", "r01_launches_cfg3_fp32_tensor.csv"],
             ("cfg2_gy94_32x10000", "fp64"): ["r02_launches_cfg2_fp64_tensor.csv"]}
KERNEL_PATTERNS = {"k_pre4_lean+k_grad4_tips": r"k_pre4_lean|k_grad4_tips", "k_post4_walk": r"k_post4_walk",
                   "k_pre_tc5": r"k_pre_tc5", "k_post_tc5": r"k_post_tc5", "k_pre_tc": r"k_pre_tc<",
                   "k_post_tc": r"k_post_tc<"}


def measured_traffic(wl_name, precision, kname):
    for csv_name in NCU_LISTS.get((wl_name, precision), []):
        if kname in KERNEL_PATTERNS:
            v = ncu_dram_bytes_per_step(csv_name, KERNEL_PATTERNS[kname])
            if v:
                return v, "profiles/" + csv_name
    return None, None


ORACLE_1CORE_BUDGET_S = 25.0  # cpu_baseline, one process: the largest pattern prefix that fits this budget
REFERENCE_SAMPLE = {4: 8000, 61: 800}  # --impl reference: patterns per step (a few seconds per step)


def make_workload(args):
    from paper_2606_27607_b200 import workloads

    return workloads.config(args.config, n_tips=args.taxa, n_patterns=args.patterns)


def workload_config(wl, precision, flags, extra=None):
    cfg = {"workload": wl.name, "taxa": wl.tree.n_tips, "patterns": wl.n_patterns, "states": wl.n_states,
           "categories": wl.n_categories, "branches": 2 * wl.tree.n_tips - 2, "precision": precision,
           "codon_path": ("tensor" if flags & 1 else "cuda-core") if wl.n_states != 4 else None,
           "codon_fp32_kernels": (("mma.sync" if flags & 64 else "tcgen05") if (flags & 1 and precision == "fp32"
                                                                                   and wl.n_states != 4) else None),
           "substitution_model": wl.model["name"], "seed": wl.seed,
           "launch_shape": {8: "level", 16: "walk"}.get(flags & 24, "auto") if wl.n_states == 4 else "level",
           "staging": ("ldg" if flags & 32 else "tma") if wl.n_states == 4 else None,
           "dependent_launch": (not flags & 128) if wl.n_states == 4 else None,
           "l2_policy": "inputs exceed L2 (no flush between iterations)"}
    if extra:
        cfg.update(extra)
    return cfg


def run_reference(args):
    """--impl reference: the CPU oracle as it stands (one process), each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args)
    n_sample = REFERENCE_SAMPLE[4 if wl.n_states == 4 else 61]
    N, C = wl.tree.n_tips, wl.n_categories
    for _ in range(min(args.warmup, 1)):
        oracle_time(wl, min(n_sample, 2000 if wl.n_states == 4 else 50))
    times, cores, n_used = [], 1, n_sample
    for _ in range(args.steps):
        dt, cores, n_used, _ = oracle_time(wl, n_sample)
        times.append(dt)
    dt = float(np.mean(times))
    value = (N - 1) * n_used * C / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, args.precision, 0, {"parallelism": "single GPU" if args.gpus == 1 else "replicas only"}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu": cpu_model_string(),
                         "sample": f"first {n_used} of {wl.n_patterns} patterns, full logL + gradient, per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def codon_roofline(name, wl, precision, kernels, res, peaks, mm):
    """Both rooflines of a 64-state run (SURVEY 8(d) "report both, state which binds"): tensor pipe against the
    matmul peak of its precision MEASURED in this run (fp64: DMMA; fp32: TF32), with algorithmic and issued flops
    separately, and HBM against the measured copy rate."""
    N, P, C = wl.tree.n_tips, wl.n_patterns, wl.n_categories
    iss = issued_tensor_flops(N, P, C, precision, kernels)
    peak = mm["fp64_tflops"] if precision == "fp64" else mm["tf32_tflops"]
    ph = res["phase_ms"]
    out = {"workload": wl.name, "precision": precision, "kernels": kernels,
           "peak_tflops": peak, "peak_source": ("fp64" if precision == "fp64" else "tf32") + " torch.matmul 8192^3, this run"}
    for tag, key, alg_fl, alg_by in (("post_order", "post", res["alg"]["post_flops"], res["alg"]["post_bytes"]),
                                     ("pre_order_gradient", "pre", res["alg"]["pre_flops"], res["alg"]["pre_bytes"])):
        t = ph[tag] * 1e-3
        out[tag] = {"ms": ph[tag], "alg_tflops": alg_fl / t / 1e12, "issued_tflops": iss[key] / t / 1e12,
                    "frac_tensor_alg": alg_fl / t / 1e12 / peak, "frac_tensor_issued": iss[key] / t / 1e12 / peak,
                    "hbm_gbs": alg_by / t / 1e9, "frac_hbm": alg_by / t / 1e9 / peaks["hbm_gbs"]}
        out[tag]["binds"] = "tensor" if out[tag]["frac_tensor_issued"] >= out[tag]["frac_hbm"] else "hbm"
    return out


def run_extras(peaks, steps, warmup, mm):
    """The other BASELINE configs / precisions, a few steps each (context for the headline line)."""
    from paper_2606_27607_b200 import workloads

    plan = [("cfg1_fp32", 1, None, None, "fp32", 0), ("cfg0_fp64", 0, None, None, "fp64", 0),
            ("cfg2_fp64_cuda", 2, None, None, "fp64", 0), ("cfg2_fp32_cuda", 2, None, None, "fp32", 0),
            ("cfg2_fp64_tensor", 2, None, None, "fp64", 1), ("cfg2_fp32_tensor", 2, None, None, "fp32", 1),
            ("cfg3_fp32_tensor", 3, None, None, "fp32", 1), ("cfg3_fp32_tensor_mma_sync", 3, None, None, "fp32", 1 | 64),
            ("cfg4_hky_fp32_512x100000", 4, 512, 100_000, "fp32", 0), ("cfg4_hky_fp32_8x100", 4, 8, 100, "fp32", 0)]
    out, codon = {}, []
    cache = {}
    for name, idx, n, p, prec, flags in plan:
        key = (idx, n, p)
        if key not in cache:
            cache.clear()
            cache[key] = workloads.config(idx, n_tips=n, n_patterns=p)
        wl = cache[key]
        try:
            res, ev = measure_device(wl, prec, flags, steps, warmup, peaks)
            ev.close()
        except Exception as exc:  # report, never hide
            out[name] = {"error": repr(exc)}
            continue
        hbm = peaks["hbm_gbs"]
        out[name] = {
            "ms_per_step": round(res["ms_per_step"], 4), "updates_per_s": res["updates_per_s"],
            "post_order_updates_per_s": res["post_order_updates_per_s"],
            "gradient_evals_per_s": res["gradient_evals_per_s"],
            "phase_ms": {k: round(v, 4) for k, v in res["phase_ms"].items()},
            "post_hbm_frac": res["post_gbs"] / hbm, "pre_hbm_frac": res["pre_gbs"] / hbm,
            "post_hbm_frac_of_8TBs": res["post_gbs"] / HBM_NOMINAL_GBS, "pre_hbm_frac_of_8TBs": res["pre_gbs"] / HBM_NOMINAL_GBS,
            "post_alg_tflops": res["post_tflops"], "pre_alg_tflops": res["pre_tflops"],
            "launches_per_step": res["launches"] / steps, "finite": res["finite"],
            "one_call_ms_per_step": round(res["one_call"]["ms_per_step"], 4) if res["one_call"] else None,
        }
        if flags & 1 and mm is not None:
            codon.append(codon_roofline(name, wl, prec, "mma.sync" if (prec == "fp64" or flags & 64) else "tcgen05",
                                        res, peaks, mm))
        if name in ("cfg1_fp32", "cfg2_fp64_tensor", "cfg3_fp32_tensor"):
            try:
                out[name]["rate_matrix_gradient"] = measure_rate_matrix_gradient(wl, prec, flags, max(3, steps // 2), peaks)
            except Exception as exc:
                out[name]["rate_matrix_gradient"] = {"error": repr(exc)}
    return out, codon


def run_sweep(peaks, steps, warmup):
    """BASELINE configs[4]: likelihood and gradient throughput per (taxa, patterns) point, HKY fp32, 4 categories."""
    from paper_2606_27607_b200 import workloads

    points = []
    for n in (8, 32, 128, 512):
        for p in (100, 1_000, 10_000, 100_000, 500_000):
            wl = workloads.config(4, n_tips=n, n_patterns=p)
            res, ev = measure_device(wl, "fp32", 0, steps, warmup, peaks)
            ev.close()
            ph = res["phase_ms"]
            lik_ms = ph["matrices"] + ph["post_order"] + ph["root"]
            points.append({
                "taxa": n, "patterns": p, "ms_per_step": round(res["ms_per_step"], 4),
                "likelihood_ms": round(lik_ms, 4), "gradient_ms": round(ph["pre_order_gradient"], 4),
                "likelihood_updates_per_s": res["alg"]["updates"] / (lik_ms * 1e-3),
                "gradient_units_per_s": res["grad_units_per_s"],
                "gradient_evals_per_s": res["gradient_evals_per_s"],
                "post_hbm_frac": round(res["post_gbs"] / peaks["hbm_gbs"], 4),
                "pre_hbm_frac": round(res["pre_gbs"] / peaks["hbm_gbs"], 4),
                "launches_per_step": res["launches"] / steps, "finite": res["finite"],
                "one_call_ms_per_step": round(res["one_call"]["ms_per_step"], 4)})
            del wl
    print(json.dumps({"sweep": "configs[4] HKY fp32", "unit": UNIT, "steps": steps, "points": points}))


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without a launcher: start N ranks of this very command line with torchrun (what the
    driver does itself), so that --gpus N never silently measures one GPU."""
    import torch

    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible")
    import socket

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    args = parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and world == 1 and args.impl == "ours":
        respawn_under_torchrun(args)
    if args.impl == "ours" and world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if args.impl == "reference":
        run_reference(args)
        return
    if args.sweep:
        from paper_2606_27607_b200 import build

        build.build()
        run_sweep(load_peaks(), max(3, min(args.steps, 10)), 3)
        return
    import torch

    from paper_2606_27607_b200 import build, plk

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if rank == 0:
        build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    device = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    build.build()
    peaks = load_peaks()
    wl = make_workload(args)
    flags = plk.FLAG_TENSOR_CORES if args.tensor else 0
    flags |= {"auto": 0, "level": plk.FLAG_LEVEL_BATCH_ONLY, "walk": plk.FLAG_PATTERN_WALK_ONLY}[args.shape]
    flags |= plk.FLAG_NO_TMA if args.staging == "ldg" else 0
    flags |= plk.FLAG_NO_TCGEN05 if args.codon_fp32 == "mma_sync" else 0
    flags |= plk.FLAG_NO_PDL if args.no_pdl else 0
    sampler = ClockSampler(local_rank) if rank == 0 else None
    sharded_run = args.shard_patterns and world > 1
    want_parity = rank == 0 and not args.no_cpu_baseline and not sharded_run

    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    res, ev = measure_device(wl, args.precision, flags, args.steps, args.warmup, peaks, sampler, device=device,
                             keep_site=want_parity, shard=(rank, world, dist) if sharded_run else None)
    # headline: the whole evaluation as the ONE call a client makes (plk_evaluate_device, graph replay); the per-phase
    # times come from the pass above, in which the four steps are issued as separate calls with events between them
    separate_ms = res["ms_per_step"]
    if res["one_call"] is not None:
        res["ms_per_step"] = res["one_call"]["ms_per_step"]
        res["launches"] = int(round(res["one_call"]["launches_per_step"] * args.steps))
    ms = torch.tensor([res["ms_per_step"]], dtype=torch.float64, device=device)
    if dist is not None:
        dist.barrier()
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_step = float(ms[0])
    e2e_dt, h2d, d2h = measure_e2e(ev, ev.wl, max(2, args.steps), max(args.warmup, 10))
    e2e_t = torch.tensor([e2e_dt], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    branch_nodes = ev.branch_nodes.copy()
    ev.close()
    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    alg = algorithmic(wl.tree.n_tips, wl.n_patterns, wl.n_states, wl.n_categories, 8 if args.precision == "fp64" else 4)
    # whole job: N replicas each do the full workload (weak); N shards together do it once (strong)
    updates_all = alg["updates"] * (1 if sharded_run else world)
    evals_all = 1 if sharded_run else world
    # roofline of the dominant kernel (largest share of the step)
    ph = res["phase_ms"]
    nuc = wl.n_states == 4
    dom = "pre_order_gradient" if ph["pre_order_gradient"] >= ph["post_order"] else "post_order"
    lean = nuc and wl.n_categories == 4 and args.staging == "tma" and args.shape != "walk"
    kname = {"post_order": ("k_post4_walk" if args.shape != "level" else "k_post4_tma") if nuc
             else (("k_post_tc5" if args.precision == "fp32" and args.codon_fp32 == "tcgen05" else "k_post_tc")
                   if args.tensor else "k_post64t"),
             "pre_order_gradient": ("k_pre4_lean+k_grad4_tips" if lean else "k_pre4_tma/k_pre4/k_pre4_walk") if nuc
             else (("k_pre_tc5" if args.precision == "fp32" and args.codon_fp32 == "tcgen05" else "k_pre_tc")
                   if args.tensor else "k_pre64")}[dom]
    n_levels_note = "all launches of the kernel in one step (one per dependency level and item class)"
    traffic, traffic_src = measured_traffic(wl.name, args.precision, kname)
    mm = measure_matmul_peaks(device) if (not nuc or not args.no_extras) else None
    ralg = res["alg"]  # this rank's share when sharded
    if nuc or args.precision == "fp32":
        achieved = res["pre_gbs"] if dom == "pre_order_gradient" else res["post_gbs"]
        roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": peaks["source"] + " hbm_gbs (copy rate, burst)",
                    "frac_of_nominal_8TBs": achieved / HBM_NOMINAL_GBS,
                    "algorithmic_bytes": ralg["pre_bytes"] if dom == "pre_order_gradient" else ralg["post_bytes"],
                    "over": n_levels_note}
    else:
        # fp64 61-state: DMMA / fp64 pipe against the fp64 matmul rate measured in this run
        achieved = res["pre_tflops"] if dom == "pre_order_gradient" else res["post_tflops"]
        roofline = {"bound": "tensor", "kernel": kname, "achieved": achieved, "peak": mm["fp64_tflops"], "unit": "TFLOP/s",
                    "frac": achieved / mm["fp64_tflops"], "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": "fp64 torch.matmul 8192^3 measured in this run", "over": n_levels_note}
    for tag, gb, tf in (("post_order", "post_gbs", "post_tflops"), ("pre_order_gradient", "pre_gbs", "pre_tflops")):
        roofline[tag] = {"GB/s": res[gb], "frac_hbm": res[gb] / peaks["hbm_gbs"],
                         "frac_hbm_of_nominal_8TBs": res[gb] / HBM_NOMINAL_GBS, "alg_TFLOP/s": res[tf], "ms": ph[tag]}

    line = {
        "metric": METRIC, "value": updates_all / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong" if sharded_run else "weak",
        "vs_baseline": None, "dtype": "f64" if args.precision == "fp64" else "f32", "data": "synthetic",
        "config": workload_config(wl, args.precision, flags,
                                  {"parallelism": ("pattern shards + one all-reduce" if sharded_run else "replicas only")
                                   if world > 1 else "single GPU"}),
        "gradient_evals_per_s": evals_all * 1e3 / ms_step,
        "bls_gradients_per_s": evals_all * (2 * wl.tree.n_tips - 2) * 1e3 / ms_step,
        "post_order_updates_per_s": res["post_order_updates_per_s"] * world,
        "phase_ms": {k: round(v, 5) for k, v in ph.items()},
        "logL": res["logL"], "finite": res["finite"],
        "clocks": res["clocks"],
        "e2e": {"value": updates_all / float(e2e_t[0]), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": float(e2e_t[0]) * 1e3,
                "what": "every step: tip states uploaded from pinned host memory (plk_set_all_tip_states_u8), host branch "
                        "lengths in and host logL + gradient out through plk_evaluate"},
        "gpu_launches": res["launches"],
        "timed_path": ("plk_evaluate_device (one call per evaluation, cached CUDA graph)" if res["one_call"] is not None
                       else "four calls per evaluation"),
        "separate_calls_ms_per_step": separate_ms,
        "phase_ms_note": "phase_ms and the roofline come from a pass with the four steps issued as separate calls and "
                         "CUDA events between them (separate_calls_ms_per_step); ms_per_step / value time the one-call path",
        "roofline": roofline,
    }
    if mm is not None:
        line["matmul_peaks"] = mm
    if (args.rate_matrix_gradient or not args.no_extras) and not sharded_run and world == 1:
        try:
            line["rate_matrix_gradient"] = measure_rate_matrix_gradient(wl, args.precision, flags, args.steps, peaks, device)
        except Exception as exc:  # report, never hide
            line["rate_matrix_gradient"] = {"error": repr(exc)}
    if not nuc and args.tensor and mm is not None:
        line["roofline_codon"] = [codon_roofline("headline", wl, args.precision,
                                                 "tcgen05" if (args.precision == "fp32" and args.codon_fp32 == "tcgen05")
                                                 else "mma.sync", res, peaks, mm)]
    if not args.no_cpu_baseline:
        # (a) one process on the largest pattern prefix that fits the budget (rate probed on a small prefix)
        probe_n = min(wl.n_patterns, 4000 if nuc else 200)
        dt_probe, _, _, _ = oracle_time(wl, probe_n)
        n1 = int(min(wl.n_patterns, max(probe_n, ORACLE_1CORE_BUDGET_S / dt_probe * probe_n)))
        dt1, cores1, n1, ref1 = oracle_time(wl, n1)
        per_update = (wl.tree.n_tips - 1) * wl.n_categories
        line["cpu_baseline"] = {"value": per_update * n1 / dt1, "unit": UNIT, "cores": cores1, "kind": "oracle",
                                "seconds": dt1, "cpu": cpu_model_string(), "host_cores": os.cpu_count(),
                                "sample": f"first {n1} of {wl.n_patterns} patterns, full logL + gradient, once, one process"}
        # (b) all host cores, pattern chunks in a process pool: the full pattern set if that takes < ~60 s
        ncpu = os.cpu_count() or 1
        ref_all, n_all = ref1, n1
        if ncpu > 1:
            est_full = dt1 / n1 * wl.n_patterns / max(1, 0.7 * ncpu)
            n_all = wl.n_patterns if est_full < 60.0 else int(wl.n_patterns * 60.0 / est_full)
            dta, used, n_all, ref_all = oracle_time(wl, n_all, workers=ncpu)
            line["cpu_baseline_all_cores"] = {"value": per_update * n_all / dta, "unit": UNIT, "cores": used,
                                              "kind": "oracle", "seconds": dta,
                                              "sample": f"first {n_all} of {wl.n_patterns} patterns by chunks in {used} processes"}
        if res["site"] is not None:
            line["parity"] = parity_against_oracle(ref_all, n_all, res["site"], wl, branch_nodes)
    if not args.no_extras and world == 1:
        line["extras"], codon = run_extras(peaks, max(3, min(args.steps, 5)), 3, mm)
        line["roofline_codon"] = line.get("roofline_codon", []) + codon
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
