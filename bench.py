#!/usr/bin/env python
"""bench.py -- one JSON line per run (contract in the task prompt; details in DESIGN.md section 7).

A "step" is one application of the split-preconditioned operator y = L^-1 A L^-T x (bj_op_apply:
backward block solve -> CSR SpMV -> forward block solve) on BASELINE.json configs[1]
(3D 7-point variable-coefficient diffusion on 128^3, block-Jacobi b = 8, fp64), inputs resident in HBM,
ROTATING over eight distinct x / y pairs so that no vector of a step is left in L2 by the previous one.
The same run also reports: the roofline of the dominant kernel (CUDA events bracketed around each kernel by the
library's profiling hooks; algorithmic AND ncu-measured DRAM bytes), an A/B of the serpentine factor walk, setup
(wall clock, kernel-only, its own roofline), bj_apply, the Lanczos kappa estimates kappa(A) -> kappa(A^), PCG,
the end-to-end rate through the host-buffer entry point, the CPU oracle timed on the host cores, and a `configs`
section with the operator apply on the other four BASELINE.json configs.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--block B] [--impl reference]

N > 1: replicas only -- every rank runs the same problem independently; the
value is the aggregate applies/s over all ranks with max-over-ranks timing.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2410_02408_b200 import workloads as W  # noqa: E402

METRIC = "precond_operator_applies_per_s"
UNIT = "applies/s"
NOMINAL_HBM_GBS = 8000.0  # BASELINE.json north_star "~8 TB/s"
L2_MB = 126.0
PAIRS = 8                 # distinct x / y pairs the timed loops rotate over
OTHER_CONFIGS = ((1, 4), (3, 32), (4, 16), (5, 3), (5, 24))


def algorithmic_bytes(n: int, nnz: int, b: int, band: int = -1) -> dict:
    """SURVEY.md 8(d) / DESIGN.md section 6: bytes the method itself must move, per launch.  band >= 0 (banded block
    factors, opt-in): a solve pass reads (band + 1) b doubles per block instead of b(b+1)/2."""
    spmv = 12 * nnz + 4 * (n + 1) + 16 * n
    solve = (4 * n * (b + 1) + 16 * n) if b > 0 else 0
    if band >= 0:
        solve = 8 * n * (band + 1) + 16 * n
    return {"spmv": spmv, "solve_L": solve, "solve_Lt": solve, "apply": solve,
            "spmv_solve_L": spmv + solve, "op_apply": spmv + 2 * solve}


def setup_bytes(n: int, nnz: int, factor_bytes: int) -> int:
    """read the CSR once, write the factors."""
    return 12 * nnz + 4 * (n + 1) + factor_bytes


def ncu_traffic(cfg: int, b: int, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the kernel kind, from profiles/traffic.txt (JSON text
    written by `python -m paper_2410_02408_b200.ncu_traffic` from the committed ncu raw exports); None if not captured."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.txt")) as fh:
            return json.load(fh).get(f"cfg{cfg}_b{b}", {}).get(kernel)
    except Exception:
        return None


def measured_peaks() -> tuple[float, str]:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md, 6.65 TB/s)"


def workload_config(A, cfg: int, b: int, world: int) -> dict:
    """The `config` object: identical keys and values in both arms (ours and --impl reference)."""
    ab = algorithmic_bytes(A.n, A.nnz, b)
    return {"workload": A.meta.get("name"), "baseline_config": cfg, "n": A.n, "nnz": A.nnz, "block": b,
            "l2": "working set %.0f MB per apply vs %.0f MB of L2" % (ab["op_apply"] / 1e6, L2_MB),
            "parallelism": "replicas" if world > 1 else "single"}


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._t = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake_slowdown": 0x80}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.005)

    def start(self):
        if self.nv is not None:
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._t:
            self._t.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def time_oracle(A, b: int, budget_s: float, min_reps: int = 3):
    import oracle
    P = oracle.Precond(A, b)
    x = W.seeded_vector(31, A.n)
    P.op_apply(x)  # touch
    reps, t0 = 0, time.perf_counter()
    while True:
        P.op_apply(x)
        reps += 1
        el = time.perf_counter() - t0
        if reps >= min_reps and el >= budget_s:
            break
        if el > 4 * budget_s:
            break
    return reps / el, reps, oracle.num_threads()


def run_reference(args, A, b: int):
    """--impl reference: the CPU oracle, as it stands, on the host cores.  One step = one full operator apply."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    P = oracle.Precond(A, b)
    x = W.seeded_vector(31, A.n)
    for _ in range(max(1, min(args.warmup, 3))):
        P.op_apply(x)
    steps = min(args.steps, 200)  # bounded so the run ends within minutes
    t0 = time.perf_counter()
    for _ in range(steps):
        P.op_apply(x)
    el = time.perf_counter() - t0
    v = steps / el
    cores = oracle.num_threads()
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * el / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(A, args.config, b, int(os.environ.get("WORLD_SIZE", "1"))),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{steps} full operator applies (whole vector, N={A.n})"},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_batch(args):
    """Second workload (NEXT-4): many small systems per launch.  Metric: systems/s for the per-system kappa estimate
    (m Lanczos steps each) and for the per-system PCG to the paper's bar 1e-3; plus the CPU oracle on a sample."""
    import torch
    from paper_2410_02408_b200 import binding as B
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    nsys, m = args.batch, args.lanczos_iters
    b = args.block if args.block is not None else 4
    A = W.batch_poisson(nsys, 32)
    rp, ci, val = (torch.from_numpy(a).cuda() for a in (A.row_ptr, A.col_idx, A.val))
    h = B.bj_setup(rp, ci, val, b)
    x = B.bj_seeded_vector(h, 31)
    y = torch.empty_like(x)
    for _ in range(max(args.warmup, 3)):
        B.bj_op_apply(h, x, y)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        B.bj_op_apply(h, x, y)
    e1.record()
    torch.cuda.synchronize()
    us = 1e3 * e0.elapsed_time(e1) / args.steps
    B.bj_cond_estimate_batch(h, nsys, m)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    g = B.bj_cond_estimate_batch(h, nsys, m)
    t_k = time.perf_counter() - t0
    rhs = B.bj_seeded_vector(h, 17)
    B.bj_pcg_solve_batch(h, nsys, rhs, max_iters=4, rtol=0.0)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    pr = B.bj_pcg_solve_batch(h, nsys, rhs, max_iters=500, rtol=1e-3)
    t_p = time.perf_counter() - t0
    # CPU oracle on a sample of the systems (reported baseline)
    import oracle
    v0 = W.seeded_vector(B.BJ_DEFAULT_SEED, A.n)
    seg, ns = A.meta["seg"], min(nsys, 64)
    t0 = time.perf_counter()
    worst = 0.0
    for s in range(ns):
        c = oracle.Precond(W.batch_system(A, s), b).cond_estimate(m, v0=v0[s * seg:(s + 1) * seg], reorth=False)
        worst = max(worst, abs(g["kappa"][s] / c["kappa"] - 1))
    t_o = time.perf_counter() - t0
    n, nnz = A.n, A.nnz
    ab = algorithmic_bytes(n, nnz, b)
    line = {"metric": "batched_systems_kappa_per_s", "value": nsys / t_k, "unit": "systems/s", "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * t_k, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": A.meta["name"], "systems": nsys, "system_size": seg, "n": n, "nnz": nnz, "block": b,
                       "lanczos_iters": m, "paper_size": "N = 2^10 (PAPER.md:365)"},
            "op_apply": {"us": us, "applies_per_s": 1e6 / us, "alg_bytes": ab["op_apply"], "gbs": ab["op_apply"] / us / 1e3},
            "kappa": {"seconds": t_k, "min": float(g["kappa"].min()), "median": float(np.median(g["kappa"])),
                      "max": float(g["kappa"].max()), "max_rel_dev_vs_oracle_sample": worst},
            "pcg": {"rtol": 1e-3, "seconds": t_p, "systems_per_s": nsys / t_p, "iters_min": int(pr["iters"].min()),
                    "iters_max": int(pr["iters"].max()), "true_relres_max": float(pr["true_relres"].max())},
            "cpu_baseline": {"value": ns / t_o, "unit": "systems/s", "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": f"kappa estimate ({m} Lanczos steps) of {ns} of the {nsys} systems"},
            "gpu_launches": B.bj_get_info(h)["kernel_launches"]}
    B.bj_destroy(h)
    print(json.dumps(line))


def aggregate_max(ms_local: float, world: int) -> float:
    """max over ranks of the device-timed milliseconds (all_reduce MAX; identity for world == 1)."""
    if world == 1:
        return ms_local
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms_local], dtype=torch.float64, device="cuda" if dist.get_backend() == "nccl" else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def byte_model(n: int, nnz: int, b: int, info: dict) -> dict:
    """Algorithmic bytes of the layout this handle really uses (the opt-in variants have their own, smaller, models)."""
    ab = algorithmic_bytes(n, nnz, b, info.get("band_width", -1))
    if info.get("col16") and info["spmv_kernel"] == 1:  # 16-bit column deltas: 10 bytes per entry
        spmv16 = ab["spmv"] - 2 * nnz
        ab = dict(ab, spmv=spmv16, spmv_solve_L=spmv16 + ab["solve_L"], op_apply=spmv16 + 2 * ab["solve_L"])
    if info["spmv_kernel"] == 2:  # BSR(3) copy: values + one block column per nine entries + block row pointers
        spmv_bsr = 8 * nnz + 4 * (nnz // 9) + 4 * (n // 3 + 1) + 16 * n
        ab = dict(ab, spmv=spmv_bsr, spmv_solve_L=spmv_bsr + ab["solve_L"], op_apply=spmv_bsr + 2 * ab["solve_L"])
    return ab


class Rotation:
    """Eight distinct input / output pairs: consecutive timed calls never share a vector."""

    def __init__(self, B, torch, h, n: int, pairs: int = PAIRS):
        self.x = [B.bj_seeded_vector(h, 31 + k) for k in range(pairs)]
        self.y = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(pairs)]
        self.i = 0

    def next(self):
        k = self.i % len(self.x)
        self.i += 1
        return self.x[k], self.y[k]


def time_calls(torch, fn, rot: Rotation, steps: int) -> float:
    """milliseconds of `steps` back-to-back calls fn(x, y), CUDA events on the current stream."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        x, y = rot.next()
        fn(x, y)
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def kernel_profile(B, h, rot: Rotation, ab: dict, steps: int) -> dict:
    """Per-kernel durations from the library's profiling hooks (CUDA events around every kernel on the launching stream)."""
    B.bj_profile_enable(h, True)
    for _ in range(steps):
        x, y = rot.next()
        B.bj_op_apply(h, x, y)
    kinds = {B.KERNEL_KIND_NAMES[k]: B.bj_profile_get(h, k) for k in range(B.BJ_K_COUNT)}
    B.bj_profile_enable(h, False)
    return {k: {"avg_us": 1e3 * v[0] / v[1], "launches": v[1], "alg_bytes": ab[k],
                "gbs": ab[k] / (1e-3 * v[0] / v[1]) / 1e9} for k, v in kinds.items() if v[1] > 0}


def roofline_of(kern: dict, cfg: int, b: int, peak: float, peak_src: str) -> dict:
    dom = max(kern, key=lambda k: kern[k]["avg_us"])
    total_us = sum(v["avg_us"] for v in kern.values())
    traffic = ncu_traffic(cfg, b, dom)
    r = {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["gbs"], "peak": peak, "unit": "GB/s",
         "frac": kern[dom]["gbs"] / peak, "traffic": traffic, "peak_source": peak_src,
         "algorithmic_bytes": kern[dom]["alg_bytes"], "avg_us": kern[dom]["avg_us"],
         "share_of_step": kern[dom]["avg_us"] / total_us,
         "frac_of_nominal_8TBs": kern[dom]["gbs"] / NOMINAL_HBM_GBS}
    if traffic:
        # the HBM roofline fraction proper: DRAM bytes of the ncu capture over the live kernel time.  `frac` is quoted on
        # the ALGORITHMIC bytes and exceeds it when part of them is served by L2 (vectors, the serpentine factor slice)
        r["achieved_dram"] = traffic / (kern[dom]["avg_us"] * 1e-6) / 1e9
        r["frac_dram"] = r["achieved_dram"] / peak
        r["l2_assisted"] = bool(traffic < 0.98 * kern[dom]["alg_bytes"])
    return r


def var_block_bytes(n: int, nnz: int, info: dict, perm: bool) -> dict:
    """Byte model of the warp-per-block kernels of bj_setup_blocks / bj_setup_perm (their own accounting): a solve pass
    reads the packed factors with the block pointers and factor offsets (info.factor_bytes holds all three), the right-hand
    side and, with a permutation, 4 N bytes of perm; it writes the result."""
    spmv = 12 * nnz + 4 * (n + 1) + 16 * n
    solve = info["factor_bytes"] + 16 * n + (4 * n if perm else 0)
    return {"spmv": spmv, "solve_L": solve, "solve_Lt": solve, "apply": solve, "spmv_solve_L": spmv + solve,
            "op_apply": spmv + 2 * solve}


def measure_operator(B, torch, h, cfg: int, n: int, nnz: int, b: int, steps: int, warmup: int, local: int,
                     peak: float, peak_src: str, ab: dict | None = None) -> dict:
    """The operator apply on one handle: rotating inputs, clocks sampled during the timed region, per-kernel profile."""
    info = B.bj_get_info(h)
    ab = ab or byte_model(n, nnz, b, info)
    rot = Rotation(B, torch, h, n)
    fn = lambda x, y: B.bj_op_apply(h, x, y)  # noqa: E731
    for _ in range(warmup):
        fn(*rot.next())
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = B.bj_get_info(h)["kernel_launches"]
    ms = time_calls(torch, fn, rot, steps)
    launches = B.bj_get_info(h)["kernel_launches"] - l0
    clocks = sampler.stop()
    us = 1e3 * ms / steps
    kern = kernel_profile(B, h, rot, ab, min(steps, 500))
    gbs = ab["op_apply"] / us / 1e3
    out = {"us_per_apply": us, "applies_per_s": 1e6 / us, "steps": steps, "alg_bytes": ab["op_apply"], "gbs": gbs,
           "frac_of_measured": gbs / peak, "frac_of_nominal_8TBs": gbs / NOMINAL_HBM_GBS,
           "kernels": kern, "roofline": roofline_of(kern, cfg, b, peak, peak_src), "clocks": clocks,
           "gpu_launches": launches, "spmv_kernel": info["spmv_kernel"], "fused_forward": info["fused_forward"],
           "solve_kernel": info["solve_kernel"]}
    if ab["op_apply"] < 0.5 * L2_MB * 1e6:
        out["note"] = "working set fits L2: launch-bound, the GB/s figures are not HBM figures"
    return out


def measure_setup(B, torch, rp, ci, val, b: int, peak: float, **opts):
    """bj_setup: first call of the process (cold pool), wall-clock median of 3 warm calls (allocation included), device
    time of the setup kernels alone and their roofline (CSR read once + factors written)."""
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    h = B.bj_setup(rp, ci, val, b, **opts)
    torch.cuda.synchronize()
    first = 1e3 * (time.perf_counter() - t0)
    wall, kms = [], []
    for _ in range(3):
        B.bj_destroy(h)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h = B.bj_setup(rp, ci, val, b, **opts)
        torch.cuda.synchronize()
        wall.append(1e3 * (time.perf_counter() - t0))
        kms.append(B.bj_get_setup_time(h)["kernel_ms"])
    nb = B.bj_get_setup_time(h)["algorithmic_bytes"]
    k = float(np.median(kms))
    return h, {"first_call_ms": first, "wall_ms": float(np.median(wall)), "kernel_ms": k, "alg_bytes": nb,
               "gbs": nb / (k * 1e-3) / 1e9 if k > 0 else None, "frac_of_measured": nb / (k * 1e-3) / 1e9 / peak if k > 0 else None}


def graph_replay_us(B, torch, h, x, y, steps: int) -> dict:
    """Launch-bound sizes: capture G back-to-back applies in a CUDA graph on a side stream and replay it -- the kernels,
    their PDL chaining and their arguments are the library's own launches."""
    G = 64
    side = torch.cuda.Stream()
    B.bj_set_stream(h, side)
    with torch.cuda.stream(side):
        for _ in range(3):
            B.bj_op_apply(h, x, y)
        side.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            for _ in range(G):
                B.bj_op_apply(h, x, y)
        graph.replay()
        side.synchronize()
        reps = max(1, steps // G)
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record(side)
        for _ in range(reps):
            graph.replay()
        g1.record(side)
        side.synchronize()
        gus = 1e3 * g0.elapsed_time(g1) / (reps * G)
    B.bj_set_stream(h, torch.cuda.current_stream())
    del graph
    return {"applies_per_graph": G, "replays": reps, "us_per_apply": gus, "applies_per_s": 1e6 / gus}


def permutation_section(B, torch, args, local: int, peak: float, peak_src: str) -> dict:
    """config 4 numbered along the WEAK direction (x fastest).  Natural blocks of 16 are nearly useless;
    bj_setup_perm with the line permutation gives back the y-fastest preconditioner without a permuted copy of A.  Reports
    the kappa estimates (m steps, parity mode) and the operator apply of the warp-per-block kernels with their byte model."""
    t0 = time.perf_counter()
    A = W.config4(x_fastest=True)
    n, nnz, b, m = A.n, A.nnz, 16, args.lanczos_iters
    rp, ci, val = (torch.from_numpy(a).cuda() for a in (A.row_ptr, A.col_idx, A.val))
    perm = torch.from_numpy(W.config4_line_permutation(A.meta["n"])).cuda()
    out = {"workload": A.meta.get("name"), "n": n, "nnz": nnz, "block": b, "lanczos_iters": m}
    hn = B.bj_setup(rp, ci, val, b)
    r = B.bj_cond_estimate_ex(hn, m, reorth=True)
    out["natural_blocks"] = {"kappa_est": r["kappa"], "res_min": r["res_min"], "res_max": r["res_max"]}
    if args.long_iters > 0:  # m = 50 is far from converged on this operator: a long fast-mode run beside it
        rl = B.bj_cond_estimate_ex(hn, args.long_iters, reorth=False)
        out["natural_blocks"].update({"kappa_est_long": rl["kappa"], "long_iters": rl["iters_done"], "long_res_min": rl["res_min"]})
    rhs = B.bj_seeded_vector(hn, 17)
    pr = B.bj_pcg_solve(hn, rhs, max_iters=3000, rtol=1e-3)
    out["natural_blocks"]["pcg_iters_to_1e-3"] = pr["iters"] if pr["converged"] else None
    B.bj_destroy(hn)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    hp = B.bj_setup_perm(rp, ci, val, b, perm)
    torch.cuda.synchronize()
    setup_ms = 1e3 * (time.perf_counter() - t1)
    r = B.bj_cond_estimate_ex(hp, m, reorth=True)
    info = B.bj_get_info(hp)
    ab = algorithmic_bytes(n, nnz, b)   # the uniform-block kernels; each solve pass also reads 4 N bytes of perm
    solve = ab["solve_L"] + 4 * n
    ab = dict(ab, solve_L=solve, solve_Lt=solve, apply=solve, spmv_solve_L=ab["spmv"] + solve, op_apply=ab["spmv"] + 2 * solve)
    op = measure_operator(B, torch, hp, 4, n, nnz, b, max(50, args.steps), max(args.warmup, 10), local, peak, peak_src, ab=ab)
    pr = B.bj_pcg_solve(hp, rhs, max_iters=3000, rtol=1e-3)
    long_p = {}
    if args.long_iters > 0:
        rl = B.bj_cond_estimate_ex(hp, args.long_iters, reorth=False)
        long_p = {"kappa_est_long": rl["kappa"], "long_iters": rl["iters_done"], "long_res_min": rl["res_min"]}
    out["line_permutation"] = {**long_p, "kappa_est": r["kappa"], "res_min": r["res_min"], "res_max": r["res_max"],
                               "pcg_iters_to_1e-3": pr["iters"] if pr["converged"] else None, "setup_wall_ms": setup_ms,
                               "us_per_apply": op["us_per_apply"], "alg_bytes": op["alg_bytes"], "gbs": op["gbs"],
                               "frac_of_measured": op["frac_of_measured"], "kernels": op["kernels"],
                               "byte_model": "SURVEY 8(d) count + 4 N bytes of perm per solve pass"}
    B.bj_destroy(hp)
    out["section_seconds"] = time.perf_counter() - t0
    return out


def variable_blocks_section(B, torch, args, A, rp, ci, val, local: int, peak: float, peak_src: str) -> dict:
    """variable-size blocks (bj_setup_blocks) on the headline matrix with seeded sizes 1..32: the
    warp-per-block kernels against their own byte model (packed factors + block pointers + factor offsets per pass)."""
    ptr = W.random_block_ptr(A.n, seed=41, smin=1, smax=32)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    h = B.bj_setup_blocks(rp, ci, val, ptr)
    torch.cuda.synchronize()
    setup_ms = 1e3 * (time.perf_counter() - t0)
    info = B.bj_get_info(h)
    ab = var_block_bytes(A.n, A.nnz, info, False)
    op = measure_operator(B, torch, h, 2, A.n, A.nnz, -1, max(50, args.steps), max(args.warmup, 10), local, peak, peak_src, ab=ab)
    B.bj_destroy(h)
    return {"nblocks": info["nblocks"], "mean_block": A.n / info["nblocks"], "factor_bytes": info["factor_bytes"],
            "setup_wall_ms": setup_ms, "us_per_apply": op["us_per_apply"], "alg_bytes": op["alg_bytes"], "gbs": op["gbs"],
            "frac_of_measured": op["frac_of_measured"], "kernels": op["kernels"],
            "byte_model": "12 nnz + 4 (N + 1) + 16 N + 2 x (factor_bytes + 16 N), factor_bytes = packed factors + block pointers + offsets"}


def other_configs(B, torch, args, local: int, peak: float, peak_src: str) -> dict:
    """The operator apply on the other BASELINE.json configs (1, 3, 4, 5 with b = 3 and 24) in the same run, so that every
    rate quoted in profiles/ and DESIGN.md has a driver-run counterpart."""
    out = {}
    steps = max(50, args.steps)
    mats = {}
    for cfg, b in OTHER_CONFIGS:
        t0 = time.perf_counter()
        if cfg not in mats:
            mats.clear()
            torch.cuda.empty_cache()
            A = W.build(cfg, "full")
            mats[cfg] = (A, tuple(torch.from_numpy(a).cuda() for a in (A.row_ptr, A.col_idx, A.val)))
        A, (rp, ci, val) = mats[cfg]
        h, setup = measure_setup(B, torch, rp, ci, val, b, peak)
        r = measure_operator(B, torch, h, cfg, A.n, A.nnz, b, steps if cfg != 1 else max(steps, 2000), max(args.warmup, 10),
                             local, peak, peak_src)
        r["workload"] = A.meta.get("name")
        r["n"], r["nnz"], r["block"] = A.n, A.nnz, b
        r["setup"] = setup
        if cfg == 1:
            # launch-bound: graph replay, and the whole 50-step kappa estimate beside the oracle's
            x = B.bj_seeded_vector(h, 31)
            r["graph"] = graph_replay_us(B, torch, h, x, torch.empty_like(x), 2000)
            m = args.lanczos_iters
            lz = {}
            for name, fn in (("parity_mode", lambda: B.bj_cond_estimate(h, m)),
                             ("fast_mode", lambda: B.bj_cond_estimate_ex(h, m, reorth=False))):
                fn()
                ts = []
                for _ in range(5):
                    torch.cuda.synchronize()
                    t1 = time.perf_counter()
                    res = fn()
                    ts.append(time.perf_counter() - t1)
                lz[name] = {"seconds": float(np.median(ts)),
                            "kappa_est": (res[1] / res[0]) if isinstance(res, tuple) else res["kappa"]}
            import oracle
            P = oracle.Precond(A, b)
            P.cond_estimate(m)
            ts = []
            for _ in range(5):
                t1 = time.perf_counter()
                c = P.cond_estimate(m)
                ts.append(time.perf_counter() - t1)
            lz["oracle_parity_mode"] = {"seconds": float(np.median(ts)), "kappa_est": c["kappa"], "cores": oracle.num_threads()}
            lz["iters"] = m
            r["lanczos"] = lz
            # the solve-stage stand-in on the paper's size: PCG to the paper's bar, one launch of one cluster
            rhs = B.bj_seeded_vector(h, 17)
            B.bj_pcg_solve(h, rhs, max_iters=200, rtol=1e-3)
            ts = []
            for _ in range(5):
                torch.cuda.synchronize()
                t1 = time.perf_counter()
                pr = B.bj_pcg_solve(h, rhs, max_iters=200, rtol=1e-3)
                ts.append(time.perf_counter() - t1)
            r["pcg"] = {"rtol": 1e-3, "seconds": float(np.median(ts)), "iters": int(pr["iters"]), "converged": bool(pr["converged"]),
                        "true_relres": float(pr["true_relres"])}
        r["section_seconds"] = time.perf_counter() - t0
        B.bj_destroy(h)
        del h
        out[f"cfg{cfg}_b{b}"] = r
    mats.clear()
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number 1..5 (default 2 = configs[1])")
    ap.add_argument("--block", type=int, default=None)
    ap.add_argument("--scale", default="full", choices=["full", "small", "tiny"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--lanczos-iters", type=int, default=50)
    ap.add_argument("--long-iters", type=int, default=2000, help="iterations of the long fast-mode kappa runs (0: skip)")
    ap.add_argument("--cpu-budget-s", type=float, default=10.0)
    ap.add_argument("--spmv-kernel", type=int, default=-1)
    ap.add_argument("--fuse", type=int, default=-1)
    ap.add_argument("--no-extras", action="store_true", help="skip kappa / cpu_baseline / e2e / configs (profiling runs)")
    ap.add_argument("--no-configs", action="store_true", help="skip the section that runs the other four configs")
    ap.add_argument("--batch", type=int, default=0,
                    help="N > 0: second workload (SURVEY 8(f) NEXT-4): N independent 32x32 Poisson systems (the paper's N = 2^10) "
                         "in one block-diagonal CSR; prints one JSON line for it and exits")
    ap.add_argument("--band", type=int, default=0,
                    help="1: banded block factors where the diagonal blocks are banded (SURVEY 8(f) NEXT-2); "
                         "the byte model of the roofline then counts the band, the dense-packed count is given beside it")
    ap.add_argument("--col16", type=int, default=0,
                    help="1: 16-bit column deltas in the tile SpMV when the bandwidth allows (SURVEY 8(f) NEXT-2): 10 bytes per entry")
    ap.add_argument("--bsr", type=int, default=0,
                    help="1: keep a 3x3-blocked (BSR) copy of the matrix when its structure allows (config 5; SURVEY 8(f) NEXT-2); "
                         "the SpMV byte model then counts 8 nnz + 4 nnz/9, the CSR count is given beside it")
    ap.add_argument("--serp-keep-mb", type=int, default=0, help="bj_setup_opts_t.serp_keep_mb: 0 default (48), < 0 off")
    ap.add_argument("--graph", type=int, default=-1,
                    help="1: also time the operator apply replayed from a CUDA graph (default: only config 1, launch-bound)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)

    if args.impl == "reference" and int(os.environ.get("RANK", "0")) != 0:
        return  # under torchrun only rank 0 runs the CPU reference arm
    if args.batch > 0 and args.impl != "reference":
        run_batch(args)
        return
    A = W.build(args.config, args.scale)
    b = args.block if args.block is not None else W.BLOCK_SIZES[args.config][0]
    if args.impl == "reference":
        run_reference(args, A, b)
        return

    import torch
    import torch.distributed as dist
    from paper_2410_02408_b200 import binding as B

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    B.lib()  # fail loudly if the CUDA library is missing
    opts = {"band": args.band, "col16": args.col16, "bsr": args.bsr, "serp_keep_mb": args.serp_keep_mb}
    peak, peak_src = measured_peaks()

    n, nnz = A.n, A.nnz
    rp = torch.from_numpy(A.row_ptr).cuda()
    ci = torch.from_numpy(A.col_idx).cuda()
    val = torch.from_numpy(A.val).cuda()

    # ---- setup (a1-a4): wall clock including allocation, kernel-only device time, roofline ---------------
    if b < 0:
        # --block -1 (profiling aid): seeded variable-size blocks 1..32 on the warp-per-block kernels, their own byte model
        h = B.bj_setup_blocks(rp, ci, val, W.random_block_ptr(n, seed=41, smin=1, smax=32))
        info = B.bj_get_info(h)
        op = measure_operator(B, torch, h, args.config, n, nnz, -1, args.steps, args.warmup, local, peak, peak_src,
                              ab=var_block_bytes(n, nnz, info, False))
        B.bj_destroy(h)
        print(json.dumps({"metric": METRIC, "value": op["applies_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": 1e-3 * op["us_per_apply"], "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                          "config": dict(workload_config(A, args.config, 0, world), block="variable 1..32 (seed 41)"),
                          "variable_blocks": {k: v for k, v in op.items() if k != "roofline"}, "roofline": op["roofline"],
                          "gpu_launches": op["gpu_launches"], "clocks": op["clocks"]}))
        return
    h, setup = measure_setup(B, torch, rp, ci, val, b, peak, **opts)
    if args.spmv_kernel >= 0:
        B.bj_set_option(h, B.BJ_OPT_SPMV_KERNEL, args.spmv_kernel)
    if args.fuse >= 0:
        B.bj_set_option(h, B.BJ_OPT_FUSE_FORWARD, args.fuse)
    info = B.bj_get_info(h)
    ab = byte_model(n, nnz, b, info)
    ab_dense = algorithmic_bytes(n, nnz, b)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: K operator applies, inputs resident in HBM, rotating over PAIRS x / y pairs ------------
    rot = Rotation(B, torch, h, n)
    for _ in range(args.warmup):
        B.bj_op_apply(h, *rot.next())
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = B.bj_get_info(h)["kernel_launches"]
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        B.bj_op_apply(h, *rot.next())
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = B.bj_get_info(h)["kernel_launches"] - launches0
    ms = aggregate_max(e0.elapsed_time(e1), world)
    value = world * args.steps / (ms * 1e-3)
    ms_per_step = ms / args.steps

    # ---- repeatability: five more timed regions (median of >= 5 repeats) ----------------------
    kr = max(20, args.steps // 5)
    rep_us = [1e3 * time_calls(torch, lambda x, y: B.bj_op_apply(h, x, y), rot, kr) / kr for _ in range(5)]
    repeats = {"steps_each": kr, "us_median": float(np.median(rep_us)), "us_min": float(min(rep_us)), "us_max": float(max(rep_us))}

    # ---- per-kernel durations and the roofline of the dominant kernel ------------------------------------
    kern = kernel_profile(B, h, rot, ab, min(max(args.steps, 50), 500))
    roofline = roofline_of(kern, args.config, b, peak, peak_src)
    op_gbs = ab["op_apply"] / (ms_per_step * 1e-3) / 1e9

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": workload_config(A, args.config, b, world),
            "impl_config": {"spmv_kernel": info["spmv_kernel"], "fused_forward": info["fused_forward"],
                            "solve_kernel": info["solve_kernel"], "spmv_lanes": info["spmv_lanes"],
                            "serpentine_keep_mb": 48 if args.serp_keep_mb == 0 else max(args.serp_keep_mb, 0),
                            "band_width": info.get("band_width", -1), "col16": bool(info.get("col16")),
                            "bsr3": info["spmv_kernel"] == 2, "input_pairs": PAIRS},
            "clocks": clocks, "gpu_launches": launches, "repeats": repeats, "roofline": roofline,
            "op_apply": {"alg_bytes": ab["op_apply"], "gbs": op_gbs, "frac_of_measured": op_gbs / peak,
                         "frac_of_nominal_8TBs": op_gbs / NOMINAL_HBM_GBS,
                         "bytes_dense_packed_csr_model": ab_dense["op_apply"],
                         "note": "algorithmic bytes / time; part of them is served by L2 when frac_of_measured > 1 "
                                 "(roofline.frac_dram is the HBM fraction proper)"},
            "kernels": kern, "setup": setup, "setup_ms": setup["wall_ms"], "factor_bytes": info["factor_bytes"]}

    if args.graph == 1 or (args.graph < 0 and args.config == 1):
        x0, y0 = rot.next()
        line["graph"] = dict(graph_replay_us(B, torch, h, x0, y0, max(args.steps, 640)), eager_us_per_apply=1e3 * ms_per_step)

    if not args.no_extras:
        # ---- A/B: the serpentine factor walk off (what a consumer that evicts L2 between applies would see) -------
        if b > 0 and not args.serp_keep_mb:
            hb = B.bj_setup(rp, ci, val, b, **dict(opts, serp_keep_mb=-1))
            for _ in range(args.warmup):
                B.bj_op_apply(hb, *rot.next())
            k_ab = max(50, min(args.steps, 1000))
            us_off = 1e3 * time_calls(torch, lambda x, y: B.bj_op_apply(hb, x, y), rot, k_ab) / k_ab
            us_on = 1e3 * time_calls(torch, lambda x, y: B.bj_op_apply(h, x, y), rot, k_ab) / k_ab
            line["serpentine_ab"] = {"steps": k_ab, "keep48_us": us_on, "keep0_us": us_off,
                                     "keep0_gbs": ab["op_apply"] / us_off / 1e3, "keep0_frac_of_measured": ab["op_apply"] / us_off / 1e3 / peak}
            B.bj_destroy(hb)

        # ---- bj_apply (a5), rotating inputs ------------------------------------------------------------------
        if b > 0:
            fn = lambda x, y: B.bj_apply(h, x, y)  # noqa: E731
            for _ in range(10):
                fn(*rot.next())
            k_apply = max(50, args.steps // 10)
            ams = time_calls(torch, fn, rot, k_apply) / k_apply
            a_gbs = ab["apply"] / (ams * 1e-3) / 1e9
            line["apply"] = {"applies_per_s": 1e3 / ams, "us": 1e3 * ams, "alg_bytes": ab["apply"], "gbs": a_gbs,
                             "frac_of_measured": a_gbs / peak, "input_pairs": PAIRS,
                             "note": "eight distinct r / z pairs (268 MB of vectors on config 2): vectors come from HBM"}

        # ---- end to end through the host-buffer entry point (pinned host memory) -----------------------
        xh = torch.from_numpy(W.seeded_vector(31, n)).pin_memory()
        yh = torch.empty(n, dtype=torch.float64).pin_memory()
        for _ in range(3):
            B.bj_op_apply_host(h, xh, yh)
        k_e2e = max(10, min(args.steps, 200))
        barrier()
        e0.record()
        for _ in range(k_e2e):
            B.bj_op_apply_host(h, xh, yh)
        e1.record()
        barrier()
        e2e_ms = aggregate_max(e0.elapsed_time(e1), world)
        line["e2e"] = {"value": world * k_e2e / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 8 * n,
                       "d2h_bytes_per_step": 8 * n, "steps": k_e2e}

        if rank == 0:
            # ---- kappa(A) -> kappa(A^) (a8-a10), parity mode (full reorthogonalisation) ------------------
            m = args.lanczos_iters
            kap = {}
            h0 = B.bj_setup(rp, ci, val, 0)
            for name, hh in (("A", h0), (f"bj{b}", h)):
                B.bj_cond_estimate_ex(hh, m, reorth=True)  # workspace allocation outside the timed call
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                r = B.bj_cond_estimate_ex(hh, m, reorth=True)
                dt = time.perf_counter() - t0
                kap[name] = {"kappa_est": r["kappa"], "lmin": r["lmin"], "lmax": r["lmax"], "iters": r["iters_done"],
                             "res_min": r["res_min"], "res_max": r["res_max"], "seconds": dt}
            mf = max(m, 200)  # long enough that the one host synchronisation at the end does not matter
            r = B.bj_cond_estimate_ex(h, mf, reorth=False)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            r = B.bj_cond_estimate_ex(h, mf, reorth=False)
            dt = time.perf_counter() - t0
            kap["fast_mode"] = {"kappa_est": r["kappa"], "iters": r["iters_done"], "seconds": dt,
                                "lanczos_iters_per_s": r["iters_done"] / dt}
            # the same spectrum from Lanczos on M^-1 A in the M inner product: one factor pass per step
            r = B.bj_cond_estimate_minv(h, mf)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            r = B.bj_cond_estimate_minv(h, mf)
            dt = time.perf_counter() - t0
            kap["minv_mode"] = {"kappa_est": r["kappa"], "iters": r["iters_done"], "seconds": dt,
                                "lanczos_iters_per_s": r["iters_done"] / dt,
                                "note": "start vector r_0 = seeded vector, i.e. v_0 = L^-1 r_0 in fast_mode's terms: same operator, another Krylov space"}
            # long runs (fast mode: the extreme Ritz values keep converging, ghosts only repeat them) so that
            # kappa(A) -> kappa(A^) is meaningful beyond the m-step lower bounds above (SURVEY 8(c) reading 13)
            ml = args.long_iters
            if ml > 0:
                h0l = B.bj_setup(rp, ci, val, 0)
                long_run = {"iters": ml}
                for name, hh in (("A", h0l), (f"bj{b}", h)):
                    t0 = time.perf_counter()
                    r = B.bj_cond_estimate_ex(hh, ml, reorth=False)
                    long_run[name] = {"kappa_est": r["kappa"], "lmin": r["lmin"], "lmax": r["lmax"], "res_min": r["res_min"],
                                      "res_max": r["res_max"], "iters": r["iters_done"], "seconds": time.perf_counter() - t0}
                t0 = time.perf_counter()
                r = B.bj_cond_estimate_minv(h, ml)
                long_run[f"bj{b}_minv"] = {"kappa_est": r["kappa"], "lmin": r["lmin"], "lmax": r["lmax"], "res_min": r["res_min"],
                                           "res_max": r["res_max"], "iters": r["iters_done"], "seconds": time.perf_counter() - t0}
                long_run["predicted_hhl_gain_kappa_sq"] = (long_run["A"]["kappa_est"] / long_run[f"bj{b}"]["kappa_est"]) ** 2
                kap["long_run"] = long_run
                B.bj_destroy(h0l)
            kap["predicted_hhl_gain_kappa_sq"] = (kap["A"]["kappa_est"] / kap[f"bj{b}"]["kappa_est"]) ** 2
            line["kappa"] = kap
            B.bj_destroy(h0)

            # ---- PCG to the paper's residual bar 1e-3 --------------
            rhs = B.bj_seeded_vector(h, 17)
            pcg = {"rtol": 1e-3}
            h0 = B.bj_setup(rp, ci, val, 0)
            for name, hh, cap in ((f"bj{b}", h, 3000), ("A", h0, 1000)):
                B.bj_pcg_solve(hh, rhs, max_iters=4, rtol=0.0)  # workspace allocation outside the timed call
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                pr = B.bj_pcg_solve(hh, rhs, max_iters=cap, rtol=1e-3)
                torch.cuda.synchronize()
                dt = time.perf_counter() - t0
                pcg[name] = {"iters": pr["iters"], "converged": pr["converged"], "ms": 1e3 * dt,
                             "us_per_iter": 1e6 * dt / max(pr["iters"], 1), "true_relres": pr["true_relres"],
                             "relres": pr["relres"], "max_iters": cap,
                             "kappa_cg": (pr["lmax"] / pr["lmin"]) if pr["lmin"] > 0 else None}
            B.bj_destroy(h0)
            line["pcg"] = pcg

            # ---- NEXT-2 variant beside the headline: banded / compact factors (own byte model), same matrix and b ----
            if not args.band and b >= 4:
                hb = B.bj_setup(rp, ci, val, b, band=1, col16=1)
                ib = B.bj_get_info(hb)
                if ib.get("band_width", -1) >= 0 or ib.get("col16"):
                    for _ in range(10):
                        B.bj_op_apply(hb, *rot.next())
                    kb = max(100, args.steps // 10)
                    bus = 1e3 * time_calls(torch, lambda x, y: B.bj_op_apply(hb, x, y), rot, kb) / kb
                    red_bytes = byte_model(n, nnz, b, ib)["op_apply"]
                    line["banded_variant"] = {"band_width": ib["band_width"], "col16": bool(ib.get("col16")), "us_per_apply": bus,
                                              "applies_per_s": 1e6 / bus, "band_model_bytes": red_bytes,
                                              "gbs_band_model": red_bytes / bus / 1e3, "factor_bytes": ib["factor_bytes"],
                                              "note": "opt-in (bj_setup_opts_t.band / .col16; --band 1 --col16 1): banded or compact "
                                                      "factors and 16-bit column deltas; fewer bytes than the counts of SURVEY 8(d), "
                                                      "own accounting"}
                B.bj_destroy(hb)

            # ---- NEXT-3: variable-size blocks on the same matrix (warp-per-block kernels, own byte model) ------------
            line["variable_blocks"] = variable_blocks_section(B, torch, args, A, rp, ci, val, local, peak, peak_src)

            # ---- CPU oracle on the host cores (reported baseline, not the target) -------------------------
            v, reps, cores = time_oracle(A, b, args.cpu_budget_s)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{reps} full operator applies (whole vector, N={n}) in ~{args.cpu_budget_s:.0f} s"}
            # the other rows of the path on the same cores (SURVEY 8(d) "oracle timing beside it"): setup, bj_apply, one
            # Lanczos step with full reorthogonalisation (median of 3 each; a few seconds in all)
            import oracle
            xs = W.seeded_vector(31, n)

            def med3(fn):
                ts = []
                for _ in range(3):
                    t0 = time.perf_counter()
                    fn()
                    ts.append(time.perf_counter() - t0)
                return float(np.median(ts))
            P = oracle.Precond(A, b)
            extras = {"setup_ms": 1e3 * med3(lambda: oracle.Precond(A, b)), "op_apply_ms": 1e3 / v}
            if b > 0:
                extras["apply_ms"] = 1e3 * med3(lambda: P.apply(xs))
            t8 = med3(lambda: P.cond_estimate(8, reorth=True))
            t4 = med3(lambda: P.cond_estimate(4, reorth=True))
            extras["lanczos_step_ms_reorth"] = 1e3 * max(t8 - t4, 0.0) / 4.0
            line["cpu_baseline"]["other_rows"] = extras

    B.bj_destroy(h)
    del h, rot, rp, ci, val
    if rank == 0 and world == 1 and not args.no_extras and not args.no_configs and args.config == 2 and args.scale == "full":
        torch.cuda.empty_cache()
        line["configs"] = other_configs(B, torch, args, local, peak, peak_src)
        line["permutation"] = permutation_section(B, torch, args, local, peak, peak_src)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
