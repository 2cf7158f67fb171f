#!/usr/bin/env python
"""bench.py -- FP64 TFLOP/s of the Cholesky vvvv ladder on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--split 0|1] [--impl ours|reference]

One "step" is one pass of the whole hot path (schedule -> GEMM-1 -> regroup -> GEMM-2 -> accumulate, SURVEY.md
8(a)) = one `cc_ladder` call over one synthetic problem.  Default workload: BASELINE.json configs[2]
(nocc=40, nvirt=300, nchol=1000; the smallest of "the three largest configs" the metric is quoted on, so the
default run ends within minutes); `--config 3|4` run the larger ones, `--config 1|0` the parity-sized ones.

value      = effective TFLOP/s = 2 v^4 (x + o^2) / device time, operands resident in HBM (CUDA events on the
             launching stream, max over ranks).  Split mode executes about half of these flops; the effective rate
             still divides the full count so that modes are comparable.
e2e        = same metric through cc_ladder_host(): pinned HOST buffers, H2D of L, t, R and D2H of R inside the
             timed region.
roofline   = FP64 tensor pipe: algorithmic flops per launch / mean launch duration vs the DMMA peak
             148 SM x 128 flop/clk/SM x 1.965 GHz = 37.2 TFLOP/s (measured: 37.0, profiles/r01_microbench.md).
split_mode = the same workload with CC_LADDER_OPT_SPLIT = 1 (t+/t-), an extra key; `value` stays the mode asked for.
cpu_baseline = the oracle (oracle/ladder_oracle.c, as it stands) on the box's host cores, bounded sample.
N > 1      = the path does not shard (north_star: one GPU, no collectives): N independent replicas, "weak".
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "FP64 TFLOP/s of Cholesky vvvv ladder (1 B200) and fraction of FP64 peak"
UNIT = "TFLOP/s"
FP64_PEAK_TFLOPS = 148 * 128 * 1.965e9 / 1e12          # 37.2; DESIGN.md section 6
PEAK_SOURCE = ("148 SMs x 128 FP64 flop/clk/SM (DMMA.8x8x4, measured 128.0) x 1.965 GHz (MEASURED_PEAKS.json "
               "sm_max_mhz); DMMA microbenchmark on this pool: 37.0 TFLOP/s sustained, cuBLAS DGEMM 35.4-36.2")
# dram__bytes_read.sum + dram__bytes_write.sum per launch of ladder_ws_kernel from `ncu --set full`
# (profiles/): config -> bytes.  None where no capture exists.
NCU_TRAFFIC_BYTES = {2: 763.8e9 + 63.6e9}    # profiles/r02_ncu_c2.md (full mode, tile <8,12,20,8>)


# --------------------------------------------------------------------------------------------- helpers
def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def reduce_max_over_ranks(value: float, world: int, device=None) -> float:
    """max over ranks of a local scalar (device time); identity for world == 1.  Works with gloo (CPU tests)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_tflops(flops_per_rank: float, world: int, ms: float) -> float:
    """Whole-job aggregate: N replicas each doing flops_per_rank in (max over ranks) ms."""
    return world * flops_per_rank / (ms * 1e-3) / 1e12


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for ln in self.lines:
            f = [s.strip() for s in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val == "Active":
                    reasons.add(name)
        # "under load": samples drawing more than 60 % of the highest power seen
        load = [s for s, p in zip(sm, pw) if pw and p >= 0.6 * max(pw)]
        return {"sm_mhz": statistics.median(load) if load else (statistics.median(sm) if sm else None),
                "sm_max_mhz": max(mx) if mx else None, "power_w_max": max(pw) if pw else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def ab_ij_sample(v: int, o: int, n_ab: int, n_ij: int, seed: int):
    """Structured + seeded random sample of (a,b) and (i,j) pairs."""
    import numpy as np
    rng = np.random.default_rng(1000 + seed)
    ab = [(0, 0), (v - 1, v - 1), (0, v - 1), (v - 1, 0), (v // 2, v // 2)]
    for e in (8, 16, 32, 64, 128):                     # both sides of tile boundaries
        for a in (e - 1, e):
            if 0 <= a < v:
                ab += [(a, (a * 7 + 3) % v), ((a * 5 + 1) % v, a)]
    ab = ab[:n_ab]
    while len(ab) < n_ab:
        ab.append(tuple(int(z) for z in rng.integers(0, v, 2)))
    ij = [(0, 0), (o - 1, o - 1), (0, o - 1), (o - 1, 0)][:n_ij]
    while len(ij) < n_ij:
        ij.append(tuple(int(z) for z in rng.integers(0, o, 2)))
    return np.array(ab, dtype=np.int32), np.array(ij, dtype=np.int32)


def oracle_sample_flops(v, x, n_ab, n_ij):
    return n_ab * (2.0 * x * v * v + n_ij * 2.0 * v * v)


def time_oracle_sample(L, t, n_ab, n_ij, seed):
    import oracle
    o, v, x = t.shape[0], t.shape[2], L.shape[0]
    ab, ij = ab_ij_sample(v, o, n_ab, n_ij, seed)
    t0 = time.perf_counter()
    oracle.ladder_sampled(L, t, ab, ij)
    return time.perf_counter() - t0


def calibrate_oracle(L, t, seed, target_s):
    """Pick n_ab so that one sampled oracle evaluation takes about target_s seconds."""
    import oracle
    cores = oracle.num_threads()
    v, x = t.shape[2], L.shape[0]
    n_ij = 64
    pilot = max(cores, 8)
    dt = time_oracle_sample(L, t, pilot, n_ij, seed)
    n_ab = int(max(pilot, min(v * v, pilot * target_s / max(dt, 1e-3))))
    n_ab = (n_ab // cores) * cores or cores
    return n_ab, n_ij, cores


def dgemm_ceiling(o, v, x, dev):
    """cuBLAS DGEMM (torch.matmul, float64) with the path's own aspect ratios, as a measured ceiling reference
    (north_star): GEMM-1-like M = N = n, K = x (both operands K-major) and GEMM-2-like M = o^2, N = K = n, plus a
    large square.  'ladder_equivalent' weights the two by the ladder's own flop split x : o^2."""
    import torch
    n = 16384
    res = {}

    def t_ms(fn, reps=3):
        fn(); torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    g = torch.Generator(device=dev); g.manual_seed(1)
    A = torch.randn(x, n, dtype=torch.float64, device=dev, generator=g)
    B = torch.randn(x, n, dtype=torch.float64, device=dev, generator=g)
    C = torch.empty(n, n, dtype=torch.float64, device=dev)
    ms = t_ms(lambda: torch.matmul(A.t(), B, out=C))
    r1 = 2.0 * n * n * x / ms * 1e-9
    res["gemm1_like"] = {"M": n, "N": n, "K": x, "tflops": r1}
    del A, B, C
    oo = o * o
    T = torch.randn(oo, n, dtype=torch.float64, device=dev, generator=g)
    V = torch.randn(n, n, dtype=torch.float64, device=dev, generator=g)
    Rr = torch.empty(oo, n, dtype=torch.float64, device=dev)
    ms = t_ms(lambda: torch.matmul(T, V, out=Rr))
    r2 = 2.0 * oo * n * n / ms * 1e-9
    res["gemm2_like"] = {"M": oo, "N": n, "K": n, "tflops": r2}
    del T, Rr
    S = torch.empty(n, n, dtype=torch.float64, device=dev)
    ms = t_ms(lambda: torch.matmul(V, V, out=S))
    res["square"] = {"M": n, "N": n, "K": n, "tflops": 2.0 * n ** 3 / ms * 1e-9}
    res["ladder_equivalent_tflops"] = (x + oo) / (x / r1 + oo / r2)
    res["kind"] = "cuBLAS DGEMM via torch.matmul(float64), best of 3"
    return res


# --------------------------------------------------------------------------------------------- reference arm
def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if rank != 0:
        return
    import ladder_inputs as gen
    o, v, x = gen.CONFIGS[args.config]
    L, t, _ = gen.make_inputs(o, v, x, seed=args.config)
    n_ab, n_ij, cores = calibrate_oracle(L, t, args.config, target_s=6.0)
    fl = oracle_sample_flops(v, x, n_ab, n_ij)
    for _ in range(args.warmup):
        time_oracle_sample(L, t, n_ab, n_ij, args.config)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        time_oracle_sample(L, t, n_ab, n_ij, args.config)
    dt = (time.perf_counter() - t0) / args.steps
    val = fl / dt / 1e12
    sample = (f"{n_ab} (a,b) pairs x {n_ij} (i,j) pairs of config {args.config} per step "
              f"({fl:.3e} flop of the {gen.ladder_flops(o, v, x):.3e} flop evaluation)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]: nocc={o} nvirt={v} nchol={x}, seed {args.config}",
                   "nocc": o, "nvirt": v, "nchol": x, "split": 0},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# --------------------------------------------------------------------------------------------- our arm
def run_ours(args, rank, local_rank, world):
    import numpy as np
    import torch

    import ladder_inputs as gen
    import paper_2310_04559_b200 as cl

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the ladder has no CPU path")
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    o, v, x = gen.CONFIGS[args.config]
    flops = float(gen.ladder_flops(o, v, x))
    L, t, R0 = gen.make_inputs(o, v, x, seed=args.config)
    t_dev_layout = np.ascontiguousarray(t.transpose(0, 2, 1, 3)) if args.layout else t    # the paper's [i,c,j,d]
    hL, ht = torch.from_numpy(L).pin_memory(), torch.from_numpy(t_dev_layout).pin_memory()
    hR = torch.from_numpy(R0).pin_memory()
    dL, dt_ = hL.to(dev, non_blocking=True), ht.to(dev, non_blocking=True)
    dR = torch.zeros_like(hR, device=dev)
    torch.cuda.synchronize()

    plan = cl.cc_ladder_plan(o, v, x)
    cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, args.split)
    if args.tile:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_TILE, args.tile)
    if args.supertile:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SUPERTILE, args.supertile)
    if args.exchange:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, 1)
    if args.layout:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_LAYOUT, cl.CC_LADDER_LAYOUT_IAJB)
    ws = None
    nws = cl.cc_ladder_workspace_bytes(plan)
    if nws:
        ws = torch.empty(nws, dtype=torch.uint8, device=dev)
        cl.cc_ladder_set_workspace(plan, ws, nws)
    launches_per_step = cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_KERNEL_LAUNCHES)
    shp = cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_TILE_SHAPE)
    tile_shape = [(shp >> 24) & 255, (shp >> 16) & 255, (shp >> 8) & 255, shp & 255]
    flops_exec = float(cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_FLOPS_EXECUTED))
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up, then exactly K steps, CUDA events on the launching stream
    for _ in range(args.warmup):
        cl.cc_ladder(plan, dL, dt_, dR, stream)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e_begin.record(stream)
    for k in range(args.steps):
        evs[k][0].record(stream)
        cl.cc_ladder(plan, dL, dt_, dR, stream)
        evs[k][1].record(stream)
    e_end.record(stream)
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    total_ms = e_begin.elapsed_time(e_end)
    kernel_ms = [a.elapsed_time(b) for a, b in evs]
    ms_per_step = reduce_max_over_ranks(total_ms / args.steps, world, dev)
    kernel_ms_mean = reduce_max_over_ranks(sum(kernel_ms) / len(kernel_ms), world, dev)
    value = whole_job_tflops(flops, world, ms_per_step)

    # parity spot check on the timed output (dR = (W+K) x ladder since R0 = 0): sampled oracle, rank 0 only
    parity = None
    if rank == 0 and not args.no_check:
        import oracle
        ab, ij = ab_ij_sample(v, o, 16, 8, args.config)
        ref = oracle.ladder_sampled(L, t, ab, ij) * float(args.warmup + args.steps)
        ij_t, ab_t = torch.from_numpy(ij).long().to(dev), torch.from_numpy(ab).long().to(dev)
        ka, kb = (1, 0) if args.exchange else (0, 1)   # E[i,j,a,b] == ladder[i,j,b,a] (tests/test_oracle_pins.py)
        if args.layout:         # R is stored [i,a,j,b]
            got = dR.view(o, v, o, v)[ij_t[None, :, 0], ab_t[:, None, ka], ij_t[None, :, 1], ab_t[:, None, kb]].cpu().numpy()
        else:
            got = dR[ij_t[None, :, 0], ij_t[None, :, 1], ab_t[:, None, ka], ab_t[:, None, kb]].cpu().numpy()
        scale = float(dR.abs().max().item())
        parity = float(np.max(np.abs(got - ref)) / scale)

    # ---- the optional t+/t- split mode on the same workload (an extra key; `value` stays the mode asked for)
    split_leg = None
    if not args.split and not args.exchange and not args.layout and args.split_leg and world == 1:
        plan_s = cl.cc_ladder_plan(o, v, x)
        cl.cc_ladder_set_option(plan_s, cl.CC_LADDER_OPT_SPLIT, 1)
        nws_s = cl.cc_ladder_workspace_bytes(plan_s)
        ws_s = torch.empty(nws_s, dtype=torch.uint8, device=dev)
        cl.cc_ladder_set_workspace(plan_s, ws_s, nws_s)
        dR.zero_()
        for _ in range(args.warmup):
            cl.cc_ladder(plan_s, dL, dt_, dR, stream)
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        for _ in range(args.steps):
            cl.cc_ladder(plan_s, dL, dt_, dR, stream)
        s1.record(stream)
        torch.cuda.synchronize()
        ms_s = s0.elapsed_time(s1) / args.steps
        par_s = None
        if not args.no_check:
            got = dR[ij_t[None, :, 0], ij_t[None, :, 1], ab_t[:, None, 0], ab_t[:, None, 1]].cpu().numpy()
            par_s = float(np.max(np.abs(got - ref)) / float(dR.abs().max().item()))
        fx = float(cl.cc_ladder_get_info(plan_s, cl.CC_LADDER_INFO_FLOPS_EXECUTED))
        split_leg = {"value": flops / (ms_s * 1e-3) / 1e12, "unit": UNIT + " effective (2 v^4 (x + o^2) / time)",
                     "ms_per_step": ms_s, "executed_tflops": fx / (ms_s * 1e-3) / 1e12,
                     "executed_fraction_of_fp64_peak": fx / (ms_s * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                     "gpu_launches": int(cl.cc_ladder_get_info(plan_s, cl.CC_LADDER_INFO_KERNEL_LAUNCHES)) * args.steps,
                     "workspace_bytes": int(nws_s), "parity_max_rel_err": par_s}
        cl.cc_ladder_destroy(plan_s)
        del ws_s

    # ---- end to end through the host-pointer entry point (H2D of L, t, R and D2H of R inside the timed region)
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    del dR
    torch.cuda.empty_cache()
    e2e_ms = None
    if not args.no_e2e:
        hR.zero_()
        cl.cc_ladder_host(plan, hL, ht, hR)          # warm-up (allocations, page faults)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            cl.cc_ladder_host(plan, hL, ht, hR)
        torch.cuda.synchronize()
        e2e_ms = reduce_max_over_ranks((time.perf_counter() - t0) * 1e3 / e2e_steps, world, dev)
    h2d = (L.nbytes + t.nbytes + R0.nbytes)
    d2h = R0.nbytes
    cl.cc_ladder_destroy(plan)

    ceiling = None
    if rank == 0 and world == 1 and not args.no_ceiling:
        torch.cuda.empty_cache()
        ceiling = dgemm_ceiling(o, v, x, dev)

    if rank != 0:
        return

    # ---- CPU baseline: the oracle on a bounded sample of the same workload (N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_ab, n_ij, cores = calibrate_oracle(L, t, args.config, target_s=12.0)
        dt_s = time_oracle_sample(L, t, n_ab, n_ij, args.config)
        fl = oracle_sample_flops(v, x, n_ab, n_ij)
        cpu = {"value": fl / dt_s / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{n_ab} (a,b) pairs x {n_ij} (i,j) pairs of the same workload, {fl:.3e} flop in {dt_s:.1f} s "
                         f"(long-double scalar C, OpenMP over (a,b))"}

    # algorithmic flops of one launch: F = 2 v^4 (x + o^2); split mode F_split = [v(v+1)/2]^2 4 (x + o^2)
    flops_alg = float((v * (v + 1) // 2) ** 2 * 4 * (x + o * o)) if args.split else flops
    achieved = flops_alg / (kernel_ms_mean * 1e-3) / 1e12
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]: nocc={o} nvirt={v} nchol={x}, seed {args.config}",
                   "nocc": o, "nvirt": v, "nchol": x, "split": args.split, "exchange": args.exchange,
                   "layout": "t[i,c,j,d], R[i,a,j,b] (the paper's)" if args.layout else "t[i,j,c,d], R[i,j,a,b]",
                   "tile_shape_TA_TB_TC_TD": tile_shape,
                   "l2": "operands (L+t+R = %.2f GB) are larger than the 126 MB L2; no flush needed" %
                         ((L.nbytes + 2 * t.nbytes) / 1e9),
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "fraction_of_fp64_peak": value / (world * FP64_PEAK_TFLOPS),
        "executed_tflops": flops_exec * world / (ms_per_step * 1e-3) / 1e12,
        "e2e": None if e2e_ms is None else
               {"value": whole_job_tflops(flops, world, e2e_ms), "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "api": "cc_ladder_host (pinned host buffers)"},
        "gpu_launches": int(launches_per_step * args.steps),
        "roofline": {"bound": "tensor", "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": UNIT,
                     "frac": achieved / FP64_PEAK_TFLOPS, "traffic": NCU_TRAFFIC_BYTES.get(args.config),
                     "kernel": "ladder_ws_kernel", "kernel_ms": kernel_ms_mean, "flops_per_launch": flops_alg,
                     "peak_source": PEAK_SOURCE},
        "cpu_baseline": cpu,
        "dgemm_ceiling": ceiling,
        "fraction_of_dgemm_ceiling": (value / ceiling["ladder_equivalent_tflops"]) if ceiling else None,
        "clocks": clocks,
        "parity_max_rel_err": parity,
        "split_mode": split_leg,
    }
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--split", type=int, default=0, choices=[0, 1])
    ap.add_argument("--tile", type=int, default=0, help="CC_LADDER_OPT_TILE (0 = auto)")
    ap.add_argument("--supertile", type=int, default=0, help="CC_LADDER_OPT_SUPERTILE (0 = auto)")
    ap.add_argument("--layout", type=int, default=0, choices=[0, 1],
                    help="1: t and R in the paper's own [i,a,j,b] storage (CC_LADDER_LAYOUT_IAJB)")
    ap.add_argument("--exchange", type=int, default=0, choices=[0, 1],
                    help="time the exchange variant (PAPER.md Eq. 7) instead of the ladder (same flop count)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-check", action="store_true")
    ap.add_argument("--split-leg", type=int, default=1, choices=[0, 1],
                    help="also time the t+/t- split mode on the same workload (reported under 'split_mode')")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-pointer leg (kernel sweeps only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-ceiling", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank, local_rank, world = env_int("RANK", 0), env_int("LOCAL_RANK", 0), env_int("WORLD_SIZE", 1)
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_ours(args, rank, local_rank, world)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
