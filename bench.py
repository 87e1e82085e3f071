#!/usr/bin/env python
"""bench.py -- one JSON line per run (contract in the task prompt; details in DESIGN.md section 7).

A "step" is one application of the split-preconditioned operator y = L^-1 A L^-T x (bj_op_apply:
backward block solve -> CSR SpMV -> forward block solve) on BASELINE.json configs[1]
(3D 7-point variable-coefficient diffusion on 128^3, block-Jacobi b = 8, fp64), inputs resident in HBM.
The same run also reports setup ms (extraction + batched Cholesky), bj_apply, the Lanczos kappa
estimates kappa(A) -> kappa(A^), the roofline of the dominant kernel (CUDA events bracketed around
each kernel by the library's profiling hooks), the end-to-end rate through the host-buffer entry
point, and the CPU oracle timed on the host cores as a reported baseline.

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


def algorithmic_bytes(n: int, nnz: int, b: int, band: int = -1) -> dict:
    """SURVEY.md 8(d) / DESIGN.md section 6: bytes the method itself must move, per launch.  band >= 0 (banded block
    factors, opt-in): a solve pass reads (band + 1) b doubles per block instead of b(b+1)/2."""
    spmv = 12 * nnz + 4 * (n + 1) + 16 * n
    solve = (4 * n * (b + 1) + 16 * n) if b > 0 else 0
    if band >= 0:
        solve = 8 * n * (band + 1) + 16 * n
    return {"spmv": spmv, "solve_L": solve, "solve_Lt": solve, "apply": solve,
            "spmv_solve_L": spmv + solve, "op_apply": spmv + 2 * solve}


def ncu_traffic(cfg: int, b: int, kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full summary
    (profiles/traffic.txt: JSON text, written by hand from profiles/*.md); None if that kernel was not captured."""
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
            "config": {"workload": A.meta.get("name"), "n": A.n, "nnz": A.nnz, "block": b},
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
    ap.add_argument("--no-extras", action="store_true", help="skip kappa / cpu_baseline / e2e (profiling runs)")
    ap.add_argument("--batch", type=int, default=0,
                    help="N > 0: second workload (SURVEY 8(f) NEXT-4): N independent 32x32 Poisson systems (the paper's N = 2^10) "
                         "in one block-diagonal CSR; prints one JSON line for it and exits")
    ap.add_argument("--band", type=int, default=0,
                    help="1: banded block factors where the diagonal blocks are banded (b > 8; SURVEY 8(f) NEXT-2); "
                         "the byte model of the roofline then counts the band, the dense-packed count is given beside it")
    ap.add_argument("--col16", type=int, default=0,
                    help="1: 16-bit column deltas in the tile SpMV when the bandwidth allows (SURVEY 8(f) NEXT-2): 10 bytes per entry")
    ap.add_argument("--bsr", type=int, default=0,
                    help="1: keep a 3x3-blocked (BSR) copy of the matrix when its structure allows (config 5; SURVEY 8(f) NEXT-2); "
                         "the SpMV byte model then counts 8 nnz + 4 nnz/9, the CSR count is given beside it")
    ap.add_argument("--graph", type=int, default=-1,
                    help="1: also time the operator apply replayed from a CUDA graph (default: only config 1, launch-bound)")
    ap.add_argument("--gather-envelope", type=int, default=-1,
                    help="1: also measure the machine's gather+stream envelope for this matrix (default: only config 3)")
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
    if args.band:
        os.environ["BJ_BAND"] = "1"  # read by bj_setup
    if args.bsr:
        os.environ["BJ_BSR"] = "1"   # read by bj_setup
    if args.col16:
        os.environ["BJ_COL16"] = "1"

    n, nnz = A.n, A.nnz
    rp = torch.from_numpy(A.row_ptr).cuda()
    ci = torch.from_numpy(A.col_idx).cuda()
    val = torch.from_numpy(A.val).cuda()

    # ---- setup (a1-a4): wall-clock ms including allocation, median of 3 -----------------------------
    setup_ms = []
    h = None
    for _ in range(3):
        if h is not None:
            B.bj_destroy(h)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        h = B.bj_setup(rp, ci, val, b)
        torch.cuda.synchronize()
        setup_ms.append(1e3 * (time.perf_counter() - t0))
    if args.spmv_kernel >= 0:
        B.bj_set_option(h, B.BJ_OPT_SPMV_KERNEL, args.spmv_kernel)
    if args.fuse >= 0:
        B.bj_set_option(h, B.BJ_OPT_FUSE_FORWARD, args.fuse)
    info = B.bj_get_info(h)

    x = B.bj_seeded_vector(h, 31)
    y = torch.empty_like(x)
    ab = algorithmic_bytes(n, nnz, b, info.get("band_width", -1))
    ab_dense = algorithmic_bytes(n, nnz, b)
    if info.get("col16") and info["spmv_kernel"] == 1:  # 16-bit column deltas: 10 bytes per entry
        spmv16 = ab["spmv"] - 2 * nnz
        ab = dict(ab, spmv=spmv16, spmv_solve_L=spmv16 + ab["solve_L"], op_apply=spmv16 + 2 * ab["solve_L"])
    if info["spmv_kernel"] == 2:  # BSR(3) copy: values + one block column per nine entries + block row pointers
        spmv_bsr = 8 * nnz + 4 * (nnz // 9) + 4 * (n // 3 + 1) + 16 * n
        ab = dict(ab, spmv=spmv_bsr, spmv_solve_L=spmv_bsr + ab["solve_L"], op_apply=spmv_bsr + 2 * ab["solve_L"])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: K operator applies, inputs resident in HBM ------------------------------------
    for _ in range(args.warmup):
        B.bj_op_apply(h, x, y)
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = B.bj_get_info(h)["kernel_launches"]
    sampler.start()
    e0.record()
    for _ in range(args.steps):
        B.bj_op_apply(h, x, y)
    e1.record()
    barrier()
    clocks = sampler.stop()
    launches = B.bj_get_info(h)["kernel_launches"] - launches0
    ms = aggregate_max(e0.elapsed_time(e1), world)
    value = world * args.steps / (ms * 1e-3)
    ms_per_step = ms / args.steps

    # ---- repeatability: five more timed regions of K/5 steps each (median of >= 5 repeats) ----
    rep_us = []
    kr = max(20, args.steps // 5)
    for _ in range(5):
        e0.record()
        for _ in range(kr):
            B.bj_op_apply(h, x, y)
        e1.record()
        torch.cuda.synchronize()
        rep_us.append(1e3 * e0.elapsed_time(e1) / kr)
    repeats = {"steps_each": kr, "us_median": float(np.median(rep_us)), "us_min": float(min(rep_us)), "us_max": float(max(rep_us))}

    # ---- per-kernel durations (CUDA events around every kernel, on the launching stream) --------------
    B.bj_profile_enable(h, True)
    prof_steps = min(args.steps, 500)
    for _ in range(prof_steps):
        B.bj_op_apply(h, x, y)
    kinds = {B.KERNEL_KIND_NAMES[k]: B.bj_profile_get(h, k) for k in range(B.BJ_K_COUNT)}
    B.bj_profile_enable(h, False)
    kern = {k: {"avg_us": 1e3 * v[0] / v[1], "launches": v[1], "alg_bytes": ab[k],
                "gbs": ab[k] / (1e-3 * v[0] / v[1]) / 1e9} for k, v in kinds.items() if v[1] > 0}
    peak, peak_src = measured_peaks()
    dom = max(kern, key=lambda k: kern[k]["avg_us"])
    total_us = sum(v["avg_us"] for v in kern.values())
    roofline = {"bound": "hbm", "kernel": dom, "achieved": kern[dom]["gbs"], "peak": peak, "unit": "GB/s",
                "frac": kern[dom]["gbs"] / peak, "traffic": ncu_traffic(args.config, b, dom), "peak_source": peak_src,
                "algorithmic_bytes": kern[dom]["alg_bytes"],
                "share_of_step": kern[dom]["avg_us"] / total_us,
                "frac_of_nominal_8TBs": kern[dom]["gbs"] / NOMINAL_HBM_GBS}
    op_gbs = ab["op_apply"] / (ms_per_step * 1e-3) / 1e9

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": A.meta.get("name"), "baseline_config": args.config, "n": n, "nnz": nnz, "block": b,
                       "l2": "inputs larger than L2 (%.0f MB per apply)" % (ab["op_apply"] / 1e6),
                       # library default 48 (bj_internal.cuh Tuning::serp_keep_mb): consecutive applies may share up to
                       # 2 x this many MB of factor lines in L2; the rate stays quoted on the full algorithmic bytes
                       "serpentine_keep_mb": int(os.environ.get("BJ_SERP_KEEP_MB", "48")),
                       "parallelism": "replicas" if world > 1 else "single",
                       "spmv_kernel": info["spmv_kernel"], "fused_forward": info["fused_forward"],
                       "spmv_lanes": info["spmv_lanes"]},
            "clocks": clocks, "gpu_launches": launches, "repeats": repeats, "roofline": roofline,
            "op_apply": {"alg_bytes": ab["op_apply"], "gbs": op_gbs, "frac_of_measured": op_gbs / peak,
                         "frac_of_nominal_8TBs": op_gbs / NOMINAL_HBM_GBS},
            "band": {"width": info.get("band_width", -1), "bsr3": info["spmv_kernel"] == 2, "col16": bool(info.get("col16")), "op_apply_bytes_dense_packed": ab_dense["op_apply"],
                     "gbs_vs_dense_packed_count": ab_dense["op_apply"] / (ms_per_step * 1e-3) / 1e9},
            "kernels": kern, "setup_ms": float(np.median(setup_ms)),
            "factor_bytes": info["factor_bytes"]}

    if args.graph == 1 or (args.graph < 0 and args.config == 1):
        # Launch-bound sizes (config 1: 0.15 MB per apply): capture G back-to-back applies in a CUDA graph on a side
        # stream and replay it -- the kernels, their PDL chaining and their arguments are the library's own launches.
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
            reps = max(1, args.steps // G)
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(side)
            for _ in range(reps):
                graph.replay()
            g1.record(side)
            side.synchronize()
            gus = 1e3 * g0.elapsed_time(g1) / (reps * G)
        B.bj_set_stream(h, torch.cuda.current_stream())
        line["graph"] = {"applies_per_graph": G, "replays": reps, "us_per_apply": gus, "applies_per_s": 1e6 / gus,
                         "eager_us_per_apply": 1e3 * ms_per_step}
        del graph

    if args.gather_envelope == 1 or (args.gather_envelope < 0 and args.config == 3):
        # The SpMV of a matrix with random column structure is bound by one L1 wavefront per 8-byte gather plus the
        # matrix stream sharing the SM <-> L2 path, not by HBM: measure that envelope on this device for this mix.
        env = B.bj_probe_gather_stream(n, nnz, 12 * nnz + 4 * (n + 1))
        sp_us = kern.get("spmv", kern.get("spmv_solve_L", {})).get("avg_us")
        env.update({"gathers": nnz, "stream_bytes": 12 * nnz + 4 * (n + 1), "vec_len": n, "spmv_us": sp_us,
                    "spmv_frac_of_envelope": (env["us_both"] / sp_us) if sp_us else None,
                    "gathers_per_clk_per_sm": nnz / (env["us_gather"] * 1e-6) / (clocks["sm_mhz"] * 1e6) / 148
                    if clocks.get("sm_mhz") else None})
        line["gather_envelope"] = env

    if not args.no_extras:
        # ---- bj_apply (a5) -----------------------------------------------------------------------------
        if b > 0:
            for _ in range(10):
                B.bj_apply(h, x, y)
            k_apply = max(50, args.steps // 10)
            e0.record()
            for _ in range(k_apply):
                B.bj_apply(h, x, y)
            e1.record()
            torch.cuda.synchronize()
            ams = e0.elapsed_time(e1) / k_apply
            line["apply"] = {"applies_per_s": 1e3 / ams, "gbs": ab["apply"] / (ams * 1e-3) / 1e9}

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
                os.environ["BJ_BAND"] = "1"
                os.environ["BJ_COL16"] = "1"
                hb = B.bj_setup(rp, ci, val, b)
                os.environ.pop("BJ_BAND", None)
                os.environ.pop("BJ_COL16", None)
                ib = B.bj_get_info(hb)
                if ib.get("band_width", -1) >= 0 or ib.get("col16"):
                    for _ in range(10):
                        B.bj_op_apply(hb, x, y)
                    kb = max(100, args.steps // 10)
                    e0.record()
                    for _ in range(kb):
                        B.bj_op_apply(hb, x, y)
                    e1.record()
                    torch.cuda.synchronize()
                    bus = 1e3 * e0.elapsed_time(e1) / kb
                    abb = algorithmic_bytes(n, nnz, b, ib["band_width"])
                    red_bytes = abb["op_apply"] - (2 * nnz if ib.get("col16") and ib["spmv_kernel"] == 1 else 0)
                    line["banded_variant"] = {"band_width": ib["band_width"], "col16": bool(ib.get("col16")), "us_per_apply": bus,
                                              "applies_per_s": 1e6 / bus, "band_model_bytes": red_bytes,
                                              "gbs_band_model": red_bytes / bus / 1e3, "factor_bytes": ib["factor_bytes"],
                                              "note": "opt-in (--band 1 --col16 1 / BJ_BAND=1 BJ_COL16=1): banded or compact "
                                                      "factors and 16-bit column deltas; fewer bytes than the counts of SURVEY 8(d), "
                                                      "own accounting"}
                B.bj_destroy(hb)

            # ---- CPU oracle on the host cores (reported baseline, not the target) -------------------------
            v, reps, cores = time_oracle(A, b, args.cpu_budget_s)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"{reps} full operator applies (whole vector, N={n}) in ~{args.cpu_budget_s:.0f} s"}

    B.bj_destroy(h)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
