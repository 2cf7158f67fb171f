#!/usr/bin/env python
"""bench.py -- FP64 TFLOP/s of the Cholesky vvvv ladder on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--split 0|1] [--impl ours|reference]
                    [--family ladder|ov]

One "step" is one pass of the whole hot path (schedule -> GEMM-1 -> regroup -> GEMM-2 -> accumulate, SURVEY.md
8(a)) = one `cc_ladder` call over one synthetic problem.  Default workload: BASELINE.json configs[4]
(nocc=64, nvirt=520, nchol=1800), the largest single-GPU configuration and the one the metric's "with and without
split" is quoted on; the other two of "the three largest configs" (2 and 3) are timed in the same run with the same
CUDA-event protocol and reported under `other_configs`.  `--config k` times another one as the headline.

value      = effective TFLOP/s = 2 v^4 (x + o^2) / device time, operands resident in HBM (CUDA events on the
             launching stream, max over ranks).  Split mode executes about half of these flops; the effective rate
             still divides the full count so that modes are comparable.
e2e        = same metric through cc_ladder_host(): pinned HOST buffers, H2D of L, t, R and D2H of R inside the
             timed region.
roofline   = FP64 tensor pipe: algorithmic flops per launch / mean launch duration vs the DMMA peak
             148 SM x 128 flop/clk/SM x 1.965 GHz = 37.2 TFLOP/s; `measured_dmma_peak` is the same pipe measured in
             this run on this box by cc_ladder_fp64_peak (a register-only DMMA loop).
split_mode = the same workload with CC_LADDER_OPT_SPLIT = 1 (t+/t-), an extra key; `value` stays the mode asked for.
ov_family  = PAPER.md Eq. 9 (recipe "abcd,ecfd->efab", cc_ladder_xy with X = L_ov, Y = L_vv) at configs[2] sizes;
             `--family ov` makes it the headline instead (roofline on its own count 2 nr ns v^2 (x + o^2)).
cpu_baseline = the oracle (oracle/ladder_oracle.c, as it stands) on the box's host cores, bounded sample.
N > 1      = the path does not shard (north_star: one GPU, no collectives): N independent replicas, "weak".
             `python bench.py --gpus N` without a torchrun environment re-launches itself under torchrun.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
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
               "sm_max_mhz); the same pipe measured in this run: measured_dmma_peak")
# dram__bytes_read.sum + dram__bytes_write.sum per launch of ladder_ws_kernel (full mode, dynamic schedule), from ncu
# captures of the final kernel of this round (profiles/round2_ncu.md, round2_final_*): config 2 from the `--set full`
# capture; configs 3 and 4 from a single-pass capture of these two counters (one launch under `--set full`'s ~40 replays
# would take 5 / 20 minutes) -- at config 2 the single pass reads 314.0 GB, the full capture 306.6 GB.
NCU_TRAFFIC_BYTES = {2: 275.16e9 + 31.40e9, 3: 2109.7e9 + 385.7e9, 4: 9951.3e9 + 3339.0e9}
NCU_TRAFFIC_KIND = {2: "ncu --set full", 3: "ncu, single pass over the two DRAM counters",
                    4: "ncu, single pass over the two DRAM counters"}


# --------------------------------------------------------------------------------------------- helpers
def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def log(*a):
    print("[bench]", *a, file=sys.stderr, flush=True)


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
        return self

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
        sm, mx, pw, reasons, capped = [], [], [], set(), 0
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
                    capped += name == "sw_power_cap"
        # "under load": samples drawing more than 60 % of the highest power seen
        load = [s for s, p in zip(sm, pw) if pw and p >= 0.6 * max(pw)]
        return {"sm_mhz": statistics.median(load) if load else (statistics.median(sm) if sm else None),
                "sm_mhz_min_under_load": min(load) if load else None,
                "sm_max_mhz": max(mx) if mx else None, "power_w_max": max(pw) if pw else None,
                "reasons": sorted(reasons), "sw_power_cap_samples": capped, "samples": len(sm)}


def ab_ij_sample(v: int, o: int, n_ab: int, n_ij: int, seed: int, tile_shape=None, supertile_shape=None, ns=None):
    """Structured + seeded random sample of (a,b) and (i,j) pairs.  The structured part sits on
    both sides of the edges the kernel actually has: block edges (multiples of TA along a, of TB along b, taken from
    CC_LADDER_INFO_TILE_SHAPE), super-tile edges (SA*TA, SB*TB) and the 64-row chunk edges of the (ij) dimension.
    `v` bounds a, `ns` (default v) bounds b (cc_ladder_xy outputs are rectangular)."""
    import numpy as np
    ns = v if ns is None else ns
    rng = np.random.default_rng(1000 + seed)
    TA, TB = (tile_shape[0], tile_shape[1]) if tile_shape else (8, 12)
    SA, SB = (supertile_shape[0], supertile_shape[1]) if supertile_shape else (3, 4)
    ab = [(0, 0), (v - 1, ns - 1), (0, ns - 1), (v - 1, 0), (v // 2, ns // 2)]

    def edges(n, T, S):
        last = ((n - 1) // T) * T                       # first index of the last (possibly ragged) block
        return [e for e in (T, 2 * T, S * T, 2 * S * T, (n // (2 * T)) * T, last) if 0 < e < n]
    for e in edges(v, TA, SA):
        for a in (e - 1, e):
            ab.append((a, int(rng.integers(0, ns))))
    for e in edges(ns, TB, SB):
        for b in (e - 1, e):
            ab.append((int(rng.integers(0, v)), b))
    ab = ab[:n_ab]
    while len(ab) < n_ab:
        ab.append((int(rng.integers(0, v)), int(rng.integers(0, ns))))
    ij = [(0, 0), (o - 1, o - 1), (0, o - 1), (o - 1, 0)]
    for r in (63, 64, ((o * o - 1) // 64) * 64 - 1, ((o * o - 1) // 64) * 64):      # chunk edges: row = i*o + j
        if 0 <= r < o * o:
            ij.append((r // o, r % o))
    ij = ij[:n_ij]
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


def workload_name(k, o, v, x):
    return f"BASELINE.json configs[{k}]: nocc={o} nvirt={v} nchol={x}, seed {k}"


def config_dict(k, o, v, x, *, split=0, exchange=0, layout=0, symm=0, tile_shape=None, family="ladder", world=1, gb=None):
    """The `config` object of the JSON line; the reference arm prints the same keys (nulls where the oracle has no such
    notion) so that the two lines describe the same workload."""
    return {"workload": workload_name(k, o, v, x), "nocc": o, "nvirt": v, "nchol": x, "family": family,
            "split": split, "exchange": exchange, "symm_l": symm,
            "layout": "t[i,c,j,d], R[i,a,j,b] (the paper's)" if layout else "t[i,j,c,d], R[i,j,a,b]",
            "tile_shape_TA_TB_TC_TD": tile_shape,
            "l2": None if gb is None else
                  "operands (L+t+R = %.2f GB) are larger than the 126 MB L2; no flush needed" % gb,
            "parallelism": "replicas only" if world > 1 else "1 GPU"}


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
        "config": config_dict(args.config, o, v, x, split=args.split, exchange=args.exchange, layout=args.layout,
                              symm=args.symm, tile_shape=None, gb=(L.nbytes + 2 * t.nbytes) / 1e9),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


# --------------------------------------------------------------------------------------------- our arm
class Leg:
    """One workload resident on the device: inputs, plan, timed calls, parity against oracle samples."""

    def __init__(self, cl, dev, k, *, split=0, tile=0, supertile=0, exchange=0, layout=0, symm=0, schedule=0, pin=False,
                 paper=0):
        import numpy as np
        import torch
        import ladder_inputs as gen
        self.cl, self.dev, self.k = cl, dev, k
        # paper = K: the paper's own timing shapes (Table 1: nocc = K/4, nvirt = 3K/4, nchol = 5K), iid
        # N(0,1) operands without any symmetry, seed K -- context runs, not BASELINE.json configs
        self.o, self.v, self.x = gen.PAPER_SHAPES[paper] if paper else gen.CONFIGS[k]
        o, v, x = self.o, self.v, self.x
        self.flops = float(gen.ladder_flops(o, v, x))
        t0 = time.perf_counter()
        if paper:
            self.L, self.t = gen.paper_shaped(paper, seed=paper)
            self.R0 = np.zeros((o, o, v, v), dtype=np.float64)
        else:
            self.L, self.t, self.R0 = gen.make_inputs(o, v, x, seed=k)
        self.layout, self.exchange, self.split, self.schedule = layout, exchange, split, schedule
        t_dev_layout = np.ascontiguousarray(self.t.transpose(0, 2, 1, 3)) if layout else self.t    # the paper's [i,c,j,d]
        self.hL, self.ht, self.hR = torch.from_numpy(self.L), torch.from_numpy(t_dev_layout), torch.from_numpy(self.R0)
        if pin:
            self.hL, self.ht, self.hR = self.hL.pin_memory(), self.ht.pin_memory(), self.hR.pin_memory()
        self.dL, self.dt = self.hL.to(dev, non_blocking=True), self.ht.to(dev, non_blocking=True)
        self.dR = torch.zeros_like(self.hR, device=dev)
        torch.cuda.synchronize()
        log(f"{'paper shape K = %d' % paper if paper else 'config %d' % k}: inputs generated and resident after "
            f"{time.perf_counter() - t0:.1f} s")
        self.plan = self.make_plan(split=split, tile=tile, supertile=supertile, exchange=exchange, layout=layout, symm=symm)
        self.calls = 0

    def make_plan(self, *, split=0, tile=0, supertile=0, exchange=0, layout=0, symm=0):
        import torch
        cl = self.cl
        plan = cl.cc_ladder_plan(self.o, self.v, self.x)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, split)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_TILE, tile)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SUPERTILE, supertile)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, exchange)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_LAYOUT, cl.CC_LADDER_LAYOUT_IAJB if layout else 0)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SYMM_L, symm)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SCHEDULE, self.schedule)
        nws = cl.cc_ladder_workspace_bytes(plan)
        ws = None
        if nws:
            ws = torch.empty(nws, dtype=torch.uint8, device=self.dev)
            cl.cc_ladder_set_workspace(plan, ws, nws)
        return {"h": plan, "ws": ws, "ws_bytes": int(nws)}

    def info(self, plan):
        cl, h = self.cl, plan["h"]
        unpack = lambda s: [(s >> 24) & 255, (s >> 16) & 255, (s >> 8) & 255, s & 255]
        return {"tile_shape": unpack(cl.cc_ladder_get_info(h, cl.CC_LADDER_INFO_TILE_SHAPE)),
                "supertile_shape": unpack(cl.cc_ladder_get_info(h, cl.CC_LADDER_INFO_SUPERTILE_SHAPE)),
                "flops_exec": float(cl.cc_ladder_get_info(h, cl.CC_LADDER_INFO_FLOPS_EXECUTED)),
                "launches": int(cl.cc_ladder_get_info(h, cl.CC_LADDER_INFO_KERNEL_LAUNCHES))}

    def timed(self, plan, steps, warmup, barrier, sample_clocks, local_rank=0):
        """W warm-up calls, then exactly K calls bracketed by barrier + synchronize, CUDA events on the launching stream
        around the region and around every call.  -> (total ms / K, mean per-call ms, clocks)."""
        import torch
        cl, stream = self.cl, torch.cuda.current_stream()
        self.dR.zero_()
        self.calls = 0
        for _ in range(warmup):
            cl.cc_ladder(plan["h"], self.dL, self.dt, self.dR, stream)
        barrier()
        sampler = ClockSampler(local_rank).start() if sample_clocks else None
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        e_begin, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e_begin.record(stream)
        for k in range(steps):
            evs[k][0].record(stream)
            cl.cc_ladder(plan["h"], self.dL, self.dt, self.dR, stream)
            evs[k][1].record(stream)
        e_end.record(stream)
        barrier()
        clocks = sampler.stop() if sampler else None
        self.calls = warmup + steps
        per_call = [a.elapsed_time(b) for a, b in evs]
        return e_begin.elapsed_time(e_end) / steps, sum(per_call) / len(per_call), clocks

    def parity(self, plan, n_ab=16, n_ij=8):
        """Sampled oracle values against the timed output (dR = calls x ladder since R0 = 0)."""
        import numpy as np
        import torch
        import oracle
        inf = self.info(plan)
        ab, ij = ab_ij_sample(self.v, self.o, n_ab, n_ij, self.k, inf["tile_shape"], inf["supertile_shape"])
        ref = oracle.ladder_sampled(self.L, self.t, ab, ij) * float(self.calls)
        ij_t, ab_t = torch.from_numpy(ij).long().to(self.dev), torch.from_numpy(ab).long().to(self.dev)
        ka, kb = (1, 0) if self.exchange else (0, 1)   # E[i,j,a,b] == ladder[i,j,b,a] (tests/test_oracle_pins.py)
        o, v = self.o, self.v
        if self.layout:         # R is stored [i,a,j,b]
            got = self.dR.view(o, v, o, v)[ij_t[None, :, 0], ab_t[:, None, ka], ij_t[None, :, 1], ab_t[:, None, kb]]
        else:
            got = self.dR[ij_t[None, :, 0], ij_t[None, :, 1], ab_t[:, None, ka], ab_t[:, None, kb]]
        scale = float(self.dR.abs().max().item())
        return float(np.max(np.abs(got.cpu().numpy() - ref)) / scale)

    def destroy(self, plan):
        self.cl.cc_ladder_destroy(plan["h"])
        plan["ws"] = None


def headline_traffic(args):
    """(bytes, where they come from) of the headline kernel's ncu DRAM counters, or (None, why not)."""
    single = "ncu, single pass over the two DRAM counters"
    if args.exchange or args.layout or args.schedule or args.family != "ladder":
        return None, "no ncu capture in this mode"
    if args.split:
        return (481.5e9 + 56.7e9, single) if args.config == 2 else (None, "split mode captured at config 2 only")
    if args.symm:
        return (423.9e9 + 121.1e9, single) if args.config == 2 else (None, "symmetry mode captured at config 2 only")
    if args.config in NCU_TRAFFIC_BYTES:
        return NCU_TRAFFIC_BYTES[args.config], NCU_TRAFFIC_KIND[args.config]
    return None, "no ncu capture at this size"


def leg_summary(leg, plan, ms_per_step, kernel_ms, clocks, parity, steps, warmup):
    inf = leg.info(plan)
    val = leg.flops / (ms_per_step * 1e-3) / 1e12
    return {"workload": workload_name(leg.k, leg.o, leg.v, leg.x), "value": val, "unit": UNIT, "steps": steps,
            "warmup": warmup, "ms_per_step": ms_per_step, "kernel_ms": kernel_ms,
            "frac": leg.flops / (kernel_ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
            "executed_tflops": inf["flops_exec"] / (ms_per_step * 1e-3) / 1e12,
            "tile_shape_TA_TB_TC_TD": inf["tile_shape"], "parity_max_rel_err": parity, "clocks": clocks,
            "traffic": NCU_TRAFFIC_BYTES.get(leg.k)}


def run_ov_family(cl, dev, k, steps, warmup, check=True):
    """PAPER.md Eq. 9 through cc_ladder_xy at configs[k] sizes: X = L_ov (nocc rows), Y = L_vv, out[i,j,k,b]."""
    import numpy as np
    import torch
    import ladder_inputs as gen
    o, v, x = gen.CONFIGS[k]
    X = gen.cholesky_block(k, o, v, x)
    Y, t, _ = gen.make_inputs(o, v, x, seed=k)
    dX, dY, dt = (torch.from_numpy(a).to(dev) for a in (X, Y, t))
    dout = torch.zeros(o, o, o, v, dtype=torch.float64, device=dev)
    plan = cl.cc_ladder_plan(o, v, x)
    stream = torch.cuda.current_stream()
    call = lambda: cl.cc_ladder_xy(plan, dX, o * v, v, o, dY, v * v, v, v, dt, dout, stream)
    for _ in range(warmup):
        call()
    torch.cuda.synchronize()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in evs:
        e0.record(stream); call(); e1.record(stream)
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in evs) / steps
    flops = 2.0 * o * v * v * v * (x + o * o)
    shp = cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_TILE_SHAPE)
    tile_shape = [(shp >> 24) & 255, (shp >> 16) & 255, (shp >> 8) & 255, shp & 255]
    fx = float(cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_FLOPS_EXECUTED))
    par = None
    if check:
        import oracle
        rs, ij = ab_ij_sample(o, o, 16, 8, k, tile_shape, None, ns=v)
        ref = oracle.ladder_xy_sampled(X, Y, t, rs, ij) * float(warmup + steps)
        ij_t, rs_t = torch.from_numpy(ij).long().to(dev), torch.from_numpy(rs).long().to(dev)
        got = dout[ij_t[None, :, 0], ij_t[None, :, 1], rs_t[:, None, 0], rs_t[:, None, 1]].cpu().numpy()
        par = float(np.max(np.abs(got - ref)) / float(dout.abs().max().item()))
    cl.cc_ladder_destroy(plan)
    return {"contraction": "PAPER.md Eq. 9 / recipe abcd,ecfd->efab: out[i,j,k,b] += sum_cd (sum_P L_ov[P,k,c] L_vv[P,b,d]) "
                           "t[i,j,c,d] (cc_ladder_xy)",
            "workload": f"configs[{k}] sizes: nocc={o} nvirt={v} nchol={x}, X = {o} x {v} rows, Y = {v} x {v}",
            "value": flops / (ms * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": ms, "steps": steps, "warmup": warmup,
            "flops_per_launch": flops, "frac": flops / (ms * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
            "executed_tflops": fx / (ms * 1e-3) / 1e12, "tile_shape_TA_TB_TC_TD": tile_shape,
            "parity_max_rel_err": par, "gpu_launches": steps}


def run_ours(args, rank, local_rank, world):
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

    def barrier():
        if world > 1:
            import torch.distributed as dist
            dist.barrier()
        torch.cuda.synchronize()

    t_start = time.perf_counter()
    solo = world == 1
    measured_peak = None
    if rank == 0:
        tf, fpc = cl.cc_ladder_fp64_peak(torch.cuda.current_stream())
        measured_peak = {"tflops": tf, "flop_per_clk_per_sm": fpc,
                         "kind": "cc_ladder_fp64_peak: register-only DMMA.8x8x4 loop on this device, this run"}
    check = not args.no_check

    # ---- the other target configs, same protocol, a few steps each (N = 1 only)
    other = []
    if solo and args.family == "ladder":
        for k in [int(s) for s in args.other_configs.split(",") if s.strip() != ""]:
            if k == args.config:
                continue
            leg = Leg(cl, dev, k)
            ms, kms, clocks = leg.timed(leg.plan, args.other_steps, 1, barrier, True, local_rank)
            par = leg.parity(leg.plan) if check else None
            other.append(leg_summary(leg, leg.plan, ms, kms, clocks, par, args.other_steps, 1))
            leg.destroy(leg.plan)
            del leg
            torch.cuda.empty_cache()
            log(f"other config {k} done at {time.perf_counter() - t_start:.0f} s")

    # ---- context: the paper's own benchmark shapes (Table 1), iid operands, same protocol
    paper_legs = []
    if solo and args.family == "ladder" and not args.lean:
        for K in [int(s) for s in args.paper_shapes.split(",") if s.strip() != ""]:
            leg = Leg(cl, dev, 0, paper=K)
            ms, kms, clocks = leg.timed(leg.plan, 2, 1, barrier, True, local_rank)
            par = leg.parity(leg.plan) if check else None
            summ = leg_summary(leg, leg.plan, ms, kms, clocks, par, 2, 1)
            summ["workload"] = (f"paper-shaped (PAPER.md Table 1, K = {K}): nocc={leg.o} nvirt={leg.v} nchol={leg.x}, "
                                f"iid N(0,1) L and t without symmetry, seed {K}")
            summ["traffic"] = None
            paper_legs.append(summ)
            leg.destroy(leg.plan)
            del leg
            torch.cuda.empty_cache()
            log(f"paper shape K = {K} done at {time.perf_counter() - t_start:.0f} s")

    # ---- the occupied-virtual family (Eqs. 8-9) at configs[2] sizes
    ov = None
    if solo and (args.ov_leg or args.family == "ov"):
        ov = run_ov_family(cl, dev, args.ov_config, max(args.steps, 3) if args.family == "ov" else 3, 3, check)
        torch.cuda.empty_cache()
    if args.family == "ov":
        if rank == 0:
            o, v, x = gen.CONFIGS[args.ov_config]
            print(json.dumps({
                "metric": METRIC, "value": ov["value"], "unit": UNIT, "n_gpus": 1, "steps": ov["steps"],
                "warmup": ov["warmup"], "ms_per_step": ov["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": config_dict(args.ov_config, o, v, x, tile_shape=ov["tile_shape_TA_TB_TC_TD"], family="ov (Eq. 9)"),
                "gpu_launches": ov["gpu_launches"],
                "roofline": {"bound": "tensor", "achieved": ov["value"], "peak": FP64_PEAK_TFLOPS, "unit": UNIT,
                             "frac": ov["frac"], "traffic": None, "kernel": "ladder_ws_kernel",
                             "kernel_ms": ov["ms_per_step"], "flops_per_launch": ov["flops_per_launch"],
                             "peak_source": PEAK_SOURCE},
                "measured_dmma_peak": measured_peak, "ov_family": ov, "parity_max_rel_err": ov["parity_max_rel_err"]}))
        return

    # ---- the headline workload: W warm-up, then exactly K steps
    leg = Leg(cl, dev, args.config, split=args.split, tile=args.tile, supertile=args.supertile,
              exchange=args.exchange, layout=args.layout, symm=args.symm, schedule=args.schedule, pin=not args.no_e2e)
    o, v, x, flops = leg.o, leg.v, leg.x, leg.flops
    inf = leg.info(leg.plan)
    total_ms, kernel_ms, clocks = leg.timed(leg.plan, args.steps, args.warmup, barrier, rank == 0, local_rank)
    ms_per_step = reduce_max_over_ranks(total_ms, world, dev)
    kernel_ms_mean = reduce_max_over_ranks(kernel_ms, world, dev)
    value = whole_job_tflops(flops, world, ms_per_step)
    log(f"headline config {args.config}: {ms_per_step:.1f} ms/step at {time.perf_counter() - t_start:.0f} s")
    parity = leg.parity(leg.plan) if (rank == 0 and check) else None

    # ---- the optional t+/t- split mode on the same workload (an extra key; `value` stays the mode asked for)
    split_leg = None
    if not args.split and not args.exchange and not args.layout and args.split_leg and solo:
        plan_s = leg.make_plan(split=1)
        ssteps = max(1, min(args.steps, args.aux_steps))
        ms_s, _, clocks_s = leg.timed(plan_s, ssteps, 1, barrier, True, local_rank)
        par_s = leg.parity(plan_s) if check else None
        inf_s = leg.info(plan_s)
        fx = inf_s["flops_exec"]
        f_split = float((v * (v + 1) // 2) ** 2 * 4 * (x + o * o))
        split_leg = {"value": flops / (ms_s * 1e-3) / 1e12, "unit": UNIT + " effective (2 v^4 (x + o^2) / time)",
                     "ms_per_step": ms_s, "steps": ssteps, "warmup": 1,
                     "executed_tflops": fx / (ms_s * 1e-3) / 1e12,
                     "executed_fraction_of_fp64_peak": fx / (ms_s * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                     "algorithmic_flops": f_split, "executed_over_algorithmic": fx / f_split,
                     "algorithmic_fraction_of_fp64_peak": f_split / (ms_s * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                     "gpu_launches": inf_s["launches"] * ssteps, "tile_shape_TA_TB_TC_TD": inf_s["tile_shape"],
                     "workspace_bytes": plan_s["ws_bytes"], "parity_max_rel_err": par_s, "clocks": clocks_s}
        leg.destroy(plan_s)
        torch.cuda.empty_cache()
        log(f"split leg done at {time.perf_counter() - t_start:.0f} s")

    # ---- the 8-fold-symmetry mode (CC_LADDER_OPT_SYMM_L; the BASELINE.json generator's L is symmetric) on the same workload
    symm_leg = None
    if not args.split and not args.exchange and not args.layout and not args.symm and args.symm_leg and solo:
        plan_y = leg.make_plan(symm=1)
        ysteps = max(1, min(args.steps, args.aux_steps))
        n_bad = cl.cc_ladder_check_symmetric(plan_y["h"], leg.dL, torch.cuda.current_stream())
        ms_y, _, clocks_y = leg.timed(plan_y, ysteps, 1, barrier, True, local_rank)
        par_y = leg.parity(plan_y) if check else None
        inf_y = leg.info(plan_y)
        symm_leg = {"value": flops / (ms_y * 1e-3) / 1e12, "unit": UNIT + " effective (2 v^4 (x + o^2) / time)",
                    "ms_per_step": ms_y, "steps": ysteps, "warmup": 1,
                    "executed_tflops": inf_y["flops_exec"] / (ms_y * 1e-3) / 1e12,
                    "executed_fraction_of_fp64_peak": inf_y["flops_exec"] / (ms_y * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
                    "executed_over_full_mode": inf_y["flops_exec"] / inf["flops_exec"],
                    "tile_shape_TA_TB_TC_TD": inf_y["tile_shape"], "L_symmetry_mismatches": n_bad,
                    "gpu_launches": inf_y["launches"] * ysteps, "parity_max_rel_err": par_y, "clocks": clocks_y}
        leg.destroy(plan_y)
        log(f"symm leg done at {time.perf_counter() - t_start:.0f} s")

    # ---- end to end through the host-pointer entry point (H2D of L, t, R and D2H of R inside the timed region)
    e2e_steps = max(1, min(args.steps, args.aux_steps))
    leg.dR = None
    torch.cuda.empty_cache()
    e2e_ms, e2e_blocks = None, 1
    if not args.no_e2e:
        leg.hR.zero_()
        if args.e2e_warmup:
            cl.cc_ladder_host(leg.plan["h"], leg.hL, leg.ht, leg.hR)      # allocations, page faults
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            cl.cc_ladder_host(leg.plan["h"], leg.hL, leg.ht, leg.hR)
        torch.cuda.synchronize()
        e2e_ms = reduce_max_over_ranks((time.perf_counter() - t0) * 1e3 / e2e_steps, world, dev)
        e2e_blocks = int(cl.cc_ladder_get_info(leg.plan["h"], cl.CC_LADDER_INFO_HOST_CHUNKS))
        log(f"e2e leg done at {time.perf_counter() - t_start:.0f} s")
    h2d = (leg.L.nbytes + leg.t.nbytes + leg.R0.nbytes)
    d2h = leg.R0.nbytes
    leg.destroy(leg.plan)
    L, t = leg.L, leg.t
    leg.dL = leg.dt = None
    torch.cuda.empty_cache()

    ceiling = None
    if rank == 0 and solo and not args.no_ceiling:
        ceiling = dgemm_ceiling(o, v, x, dev)

    if rank != 0:
        return

    # ---- CPU baseline: the oracle on a bounded sample of the same workload (N = 1 only)
    cpu = None
    if solo and not args.no_cpu_baseline:
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
        "config": config_dict(args.config, o, v, x, split=args.split, exchange=args.exchange, layout=args.layout,
                              symm=args.symm, tile_shape=inf["tile_shape"], world=world, gb=(L.nbytes + 2 * t.nbytes) / 1e9),
        "fraction_of_fp64_peak": value / (world * FP64_PEAK_TFLOPS),
        "executed_tflops": inf["flops_exec"] * world / (ms_per_step * 1e-3) / 1e12,
        "e2e": None if e2e_ms is None else
               {"value": whole_job_tflops(flops, world, e2e_ms), "unit": UNIT, "ms_per_step": e2e_ms,
                "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "api": "cc_ladder_host (pinned host buffers)", "r_column_blocks": e2e_blocks,
                "note": "R streamed in column blocks: its H2D / D2H copies overlap the kernels" if e2e_blocks > 1 else None},
        "gpu_launches": int(inf["launches"] * args.steps),
        "roofline": {"bound": "tensor", "achieved": achieved, "peak": FP64_PEAK_TFLOPS, "unit": UNIT,
                     "frac": achieved / FP64_PEAK_TFLOPS, "traffic": headline_traffic(args)[0],
                     "traffic_note": headline_traffic(args)[1],
                     "kernel": "ladder_ws_kernel", "kernel_ms": kernel_ms_mean, "flops_per_launch": flops_alg,
                     "peak_source": PEAK_SOURCE,
                     "frac_of_measured_dmma_peak": (achieved / measured_peak["tflops"]) if measured_peak else None},
        "measured_dmma_peak": measured_peak,
        "cpu_baseline": cpu,
        "dgemm_ceiling": ceiling,
        "fraction_of_dgemm_ceiling": (value / ceiling["ladder_equivalent_tflops"]) if ceiling else None,
        "clocks": clocks,
        "parity_max_rel_err": parity,
        "other_configs": other,
        "paper_shapes": paper_legs,
        "split_mode": split_leg,
        "symm_mode": symm_leg,
        "ov_family": ov,
        "bench_wall_s": time.perf_counter() - t_start,
    }
    print(json.dumps(out))


def relaunch_under_torchrun(args):
    """`python bench.py --gpus N` (N > 1) outside torchrun: start N replicas, one per GPU, the way the driver does."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--family", default="ladder", choices=["ladder", "ov"],
                    help="ov: time PAPER.md Eq. 9 (cc_ladder_xy) at --ov-config sizes as the headline")
    ap.add_argument("--split", type=int, default=0, choices=[0, 1])
    ap.add_argument("--tile", type=int, default=0, help="CC_LADDER_OPT_TILE (0 = auto)")
    ap.add_argument("--supertile", type=int, default=0, help="CC_LADDER_OPT_SUPERTILE (0 = auto)")
    ap.add_argument("--layout", type=int, default=0, choices=[0, 1],
                    help="1: t and R in the paper's own [i,a,j,b] storage (CC_LADDER_LAYOUT_IAJB)")
    ap.add_argument("--exchange", type=int, default=0, choices=[0, 1],
                    help="time the exchange variant (PAPER.md Eq. 7) instead of the ladder (same flop count)")
    ap.add_argument("--other-configs", default=None,
                    help="comma list of further configs timed in the same run (default: 2,3 when --config 4, else none)")
    ap.add_argument("--other-steps", type=int, default=3)
    ap.add_argument("--paper-shapes", default=None,
                    help="comma-separated K of the paper's Table-1 shapes (300, 400, 500) timed as context legs; '' = none "
                         "(default: 300,400 beside the configs[4] headline, none otherwise)")
    ap.add_argument("--aux-steps", type=int, default=2, help="cap on the steps of the split_mode and e2e legs")
    ap.add_argument("--schedule", type=int, default=0, choices=[0, 1],
                    help="CC_LADDER_OPT_SCHEDULE: 0 = dynamic tile scheduler (default), 1 = static round-robin")
    ap.add_argument("--symm", type=int, default=0, choices=[0, 1],
                    help="CC_LADDER_OPT_SYMM_L: 8-fold-symmetry mode (L symmetric) as the headline mode")
    ap.add_argument("--symm-leg", type=int, default=1, choices=[0, 1],
                    help="also time the 8-fold-symmetry mode on the same workload (reported under 'symm_mode')")
    ap.add_argument("--e2e-warmup", type=int, default=0, choices=[0, 1])
    ap.add_argument("--ov-leg", type=int, default=1, choices=[0, 1])
    ap.add_argument("--ov-config", type=int, default=2, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--no-check", action="store_true")
    ap.add_argument("--split-leg", type=int, default=1, choices=[0, 1],
                    help="also time the t+/t- split mode on the same workload (reported under 'split_mode')")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-pointer leg (kernel sweeps only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-ceiling", action="store_true")
    ap.add_argument("--lean", action="store_true", help="headline leg only (kernel sweeps, ncu captures)")
    args = ap.parse_args()
    if args.lean:
        args.no_e2e = args.no_cpu_baseline = args.no_ceiling = True
        args.split_leg = args.ov_leg = args.symm_leg = 0
        args.other_configs = ""
    if args.other_configs is None:
        args.other_configs = "2,3" if args.config == 4 else ""
    if args.paper_shapes is None:
        args.paper_shapes = "300,400" if (args.config == 4 and not args.lean) else ""
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank, local_rank, world = env_int("RANK", 0), env_int("LOCAL_RANK", 0), env_int("WORLD_SIZE", 1)
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        relaunch_under_torchrun(args)
    if args.gpus != world:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with torchrun --nproc-per-node {args.gpus}")
    run_ours(args, rank, local_rank, world)
    if world > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
