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
def measure_device(wl, precision, flags, steps, warmup, peaks, sampler=None, device="cuda:0"):
    """Device-resident timing: K full evaluations, CUDA events on the launching stream; per-phase events inside."""
    import torch

    from paper_2606_27607_b200 import plk
    from paper_2606_27607_b200.client import Evaluator

    ev = Evaluator(wl, precision=plk.FP64 if precision == "fp64" else plk.FP32, flags=flags, device=device)
    ev.make_device_io()
    stream = ev.inst.stream
    for _ in range(max(warmup, 3)):
        ev.step_device()
    torch.cuda.synchronize()
    l0 = ev.inst.kernel_launch_count()
    marks = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(steps)]
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
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler is not None else None
    launches = ev.inst.kernel_launch_count() - l0
    total_ms = marks[0][0].elapsed_time(marks[-1][4])
    phase = np.zeros(4)
    for s in range(steps):
        for i in range(4):
            phase[i] += marks[s][i].elapsed_time(marks[s][i + 1])
    phase /= steps
    logl = float(ev.d_logl.cpu()[0])
    grad = ev.d_grad.cpu().numpy()
    N, P, S, C = wl.tree.n_tips, wl.n_patterns, wl.n_states, wl.n_categories
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
        "phase_ms": {"matrices": phase[0], "post_order": phase[1], "root": phase[2], "pre_order_gradient": phase[3]},
        "post_gbs": alg["post_bytes"] / (phase[1] * 1e-3) / 1e9,
        "pre_gbs": alg["pre_bytes"] / (phase[3] * 1e-3) / 1e9,
        "post_tflops": alg["post_flops"] / (phase[1] * 1e-3) / 1e12,
        "pre_tflops": alg["pre_flops"] / (phase[3] * 1e-3) / 1e12,
        "launches": int(launches), "logL": logl, "grad_norm": float(np.linalg.norm(grad)),
        "finite": bool(np.isfinite(logl) and np.all(np.isfinite(grad))),
        "alg": alg, "clocks": clocks,
    }
    return res, ev


def measure_e2e(ev, wl, steps, warmup):
    """Same evaluation through the host-pointer C-ABI calls: every step uploads the tip states (pinned host memory)
    and the branch lengths, and reads logL and the gradient back to the host."""
    import torch

    N, P = wl.tree.n_tips, wl.n_patterns
    pinned = torch.empty((N, P), dtype=torch.uint8, pin_memory=True)  # one byte per pattern: what the kernels read
    pinned.copy_(torch.from_numpy(np.minimum(wl.tip_states, 255).astype(np.uint8)))
    tips = pinned.numpy()
    t = np.ascontiguousarray(np.asarray(wl.tree.branch_length)[ev.matrix_idx])

    def one():
        for k in range(N):
            ev.inst.set_tip_states_u8(k, tips[k])
        ev.inst.update_transition_matrices(0, ev.matrix_idx, t)
        ev.inst.update_partials(ev.ops)
        logl, _ = ev.inst.root_log_likelihoods(wl.tree.root, ev.scale_idx, want_site=False)
        g, _ = ev.inst.pre_order_gradient(0, wl.tree.root, ev.pre_ops)
        return logl, g

    for _ in range(max(1, min(warmup, 3))):
        one()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        logl, g = one()
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / steps
    return dt, N * P + t.size * 8, 8 + g.size * 8


# ---- the oracle on the host cores ------------------------------------------------------------------------------------
def oracle_time(wl, n_sample, repeats=1):
    """The fp64 CPU oracle as it stands on the first `n_sample` patterns of the workload (full evaluation incl. the
    gradient).  Returns (seconds per evaluation, threads actually used = CPU time / wall time)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle_runner as orc

    n_sample = min(n_sample, wl.n_patterns)
    best = None
    cores = 1.0
    for _ in range(repeats):
        c0, t0 = os.times(), time.perf_counter()
        orc.evaluate(wl, lo=0, hi=n_sample)
        dt = time.perf_counter() - t0
        c1 = os.times()
        cpu = (c1.user - c0.user) + (c1.system - c0.system)
        if best is None or dt < best:
            best, cores = dt, max(1.0, cpu / dt)
    return best, int(round(cores)), n_sample


# measured DRAM traffic per step (bytes) of the dominant kernel's launches, keyed by (workload, precision, kernel)
# (profiles/r01_launches_cfg1_fp64.md: dram__bytes_read.sum + dram__bytes_write.sum summed over the launches of one step)
NCU_DRAM_BYTES = {("cfg1_gtr_128x100000", "fp64", "k_pre4_lean+k_grad4_tips"): 4194.4e6,
                  ("cfg1_gtr_128x100000", "fp32", "k_pre4_lean+k_grad4_tips"): 1871.9e6,
                  ("cfg3_gy94_256x20000", "fp32", "k_pre_tc5"): 17075.1e6}

ORACLE_SAMPLE = {4: 40000, 61: 4000}  # cpu_baseline leg: patterns per oracle evaluation, ~10-30 s of CPU work
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
    """--impl reference: the CPU oracle as it stands, each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args)
    n_sample = REFERENCE_SAMPLE[4 if wl.n_states == 4 else 61]
    N, C = wl.tree.n_tips, wl.n_categories
    for _ in range(min(args.warmup, 1)):
        oracle_time(wl, min(n_sample, 2000 if wl.n_states == 4 else 50))
    times, cores = [], 1
    for _ in range(args.steps):
        dt, cores, n_used = oracle_time(wl, n_sample)
        times.append(dt)
    dt = float(np.mean(times))
    value = (N - 1) * n_used * C / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, "fp64", 0, {"sample": f"first {n_used} of {wl.n_patterns} patterns per step"}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {n_used} of {wl.n_patterns} patterns, full logL + gradient, per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_extras(peaks, steps, warmup):
    """The other BASELINE configs / precisions, a few steps each (context for the headline line)."""
    from paper_2606_27607_b200 import workloads

    have_tc = os.path.exists(os.path.join(ROOT, "paper_2606_27607_b200", "csrc", "plk_tc.cuh"))
    plan = [("cfg1_fp32", 1, None, None, "fp32", 0), ("cfg0_fp64", 0, None, None, "fp64", 0),
            ("cfg2_fp64_cuda", 2, None, None, "fp64", 0), ("cfg2_fp32_cuda", 2, None, None, "fp32", 0)]
    if have_tc:
        plan += [("cfg2_fp64_tensor", 2, None, None, "fp64", 1), ("cfg2_fp32_tensor", 2, None, None, "fp32", 1),
                 ("cfg3_fp32_tensor", 3, None, None, "fp32", 1),
                 ("cfg3_fp32_tensor_mma_sync", 3, None, None, "fp32", 1 | 64)]
    else:
        plan += [("cfg3_fp32_cuda", 3, None, None, "fp32", 0)]
    plan += [("cfg4_hky_fp32_512x100000", 4, 512, 100_000, "fp32", 0), ("cfg4_hky_fp32_8x100", 4, 8, 100, "fp32", 0)]
    out = {}
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
            "post_alg_tflops": res["post_tflops"], "pre_alg_tflops": res["pre_tflops"],
            "launches_per_step": res["launches"] / steps, "finite": res["finite"],
        }
    return out


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
                "launches_per_step": res["launches"] / steps, "finite": res["finite"]})
            del wl
    print(json.dumps({"sweep": "configs[4] HKY fp32", "unit": UNIT, "steps": steps, "points": points}))


def main():
    args = parse_args()
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
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank == 0:
        build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback "
                         "(use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
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

    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    res, ev = measure_device(wl, args.precision, flags, args.steps, args.warmup, peaks, sampler,
                             device=f"cuda:{local_rank}")
    ms = torch.tensor([res["ms_per_step"]], dtype=torch.float64, device=f"cuda:{local_rank}")
    if dist is not None:
        dist.barrier()
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    ms_step = float(ms[0])
    e2e_dt, h2d, d2h = measure_e2e(ev, wl, max(2, min(args.steps, 5)), args.warmup)
    e2e_t = torch.tensor([e2e_dt], dtype=torch.float64, device=f"cuda:{local_rank}")
    if dist is not None:
        dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
    ev.close()
    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return

    alg = res["alg"]
    updates_all = alg["updates"] * world
    # roofline of the dominant kernel (largest share of the step)
    ph = res["phase_ms"]
    nuc = wl.n_states == 4
    dom = "pre_order_gradient" if ph["pre_order_gradient"] >= ph["post_order"] else "post_order"
    lean = nuc and wl.n_categories == 4 and args.staging == "tma" and args.shape != "walk"
    kname = {"post_order": ("k_post4_walk" if args.shape != "level" else "k_post4_tma") if nuc
             else (("k_post_tc5" if args.precision == "fp32" and args.codon_fp32 == "tcgen05" else "k_post_tc")
                   if args.tensor else "k_post64"),
             "pre_order_gradient": ("k_pre4_lean+k_grad4_tips" if lean else "k_pre4_tma/k_pre4/k_pre4_walk") if nuc
             else (("k_pre_tc5" if args.precision == "fp32" and args.codon_fp32 == "tcgen05" else "k_pre_tc")
                   if args.tensor else "k_pre64")}[dom]
    n_levels_note = "all launches of the kernel in one step (one per dependency level and item class)"
    # DRAM bytes (read + write) of those launches from ncu, per step: profiles/r01_launches_cfg1_fp64.md
    traffic = NCU_DRAM_BYTES.get((wl.name, args.precision, kname))
    if nuc or args.precision == "fp32":
        achieved = res["pre_gbs"] if dom == "pre_order_gradient" else res["post_gbs"]
        roofline = {"bound": "hbm", "kernel": kname, "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "peak_source": peaks["source"] + " hbm_gbs",
                    "algorithmic_bytes": alg["pre_bytes"] if dom == "pre_order_gradient" else alg["post_bytes"],
                    "over": n_levels_note}
    else:
        # fp64 61-state: tensor (DMMA) / fp64 pipe; nominal B200 fp64 ~ 40 TFLOP/s
        achieved = res["pre_tflops"] if dom == "pre_order_gradient" else res["post_tflops"]
        roofline = {"bound": "tensor", "kernel": kname, "achieved": achieved, "peak": 40.0, "unit": "TFLOP/s",
                    "frac": achieved / 40.0, "traffic": None, "peak_source": "nominal fp64 (DESIGN.md)",
                    "over": n_levels_note}
    roofline["post_order"] = {"GB/s": res["post_gbs"], "frac_hbm": res["post_gbs"] / peaks["hbm_gbs"],
                              "alg_TFLOP/s": res["post_tflops"], "ms": ph["post_order"]}
    roofline["pre_order_gradient"] = {"GB/s": res["pre_gbs"], "frac_hbm": res["pre_gbs"] / peaks["hbm_gbs"],
                                      "alg_TFLOP/s": res["pre_tflops"], "ms": ph["pre_order_gradient"]}

    line = {
        "metric": METRIC, "value": updates_all / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64" if args.precision == "fp64" else "f32", "data": "synthetic",
        "config": workload_config(wl, args.precision, flags,
                                  {"parallelism": "replicas only" if world > 1 else "single GPU"}),
        "gradient_evals_per_s": world * 1e3 / ms_step,
        "bls_gradients_per_s": world * (2 * wl.tree.n_tips - 2) * 1e3 / ms_step,
        "post_order_updates_per_s": res["post_order_updates_per_s"] * world,
        "phase_ms": {k: round(v, 5) for k, v in ph.items()},
        "logL": res["logL"], "finite": res["finite"],
        "clocks": res["clocks"],
        "e2e": {"value": updates_all / float(e2e_t[0]), "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "ms_per_step": float(e2e_t[0]) * 1e3,
                "what": "tip states (pinned uint8, plk_set_tip_states_u8) + branch lengths uploaded, logL + gradient downloaded, every step"},
        "gpu_launches": res["launches"],
        "roofline": roofline,
    }
    if not args.no_cpu_baseline:
        n_sample = ORACLE_SAMPLE[4 if nuc else 61]
        dt, cores, n_used = oracle_time(wl, n_sample)
        line["cpu_baseline"] = {"value": (wl.tree.n_tips - 1) * n_used * wl.n_categories / dt, "unit": UNIT,
                                "cores": cores, "kind": "oracle", "seconds": dt,
                                "sample": f"first {n_used} of {wl.n_patterns} patterns, full logL + gradient, once"}
    if not args.no_extras and world == 1:
        line["extras"] = run_extras(peaks, max(3, min(args.steps, 5)), 3)
    print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
