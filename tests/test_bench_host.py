"""Host-side logic of bench.py that needs no GPU: the max-over-ranks reduction (gloo, world_size 2), the whole-job
aggregation for N replicas, the sampling helpers, and the reference arm's JSON contract on a tiny config."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    local_ms = 10.0 + 5.0 * rank            # rank 1 is the slow one
    mx = bench.reduce_max_over_ranks(local_ms, world)
    q.put((rank, mx, bench.whole_job_tflops(1e12, world, mx)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, tf in got:
        assert mx == 15.0                           # every rank sees the slowest rank's time
        assert abs(tf - 2 * 1e12 / 15e-3 / 1e12) < 1e-9   # N replicas / max time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_max_over_ranks(3.5, 1) == 3.5
    assert bench.whole_job_tflops(2e12, 1, 1000.0) == 2.0


def test_sampling_helpers():
    sys.path.insert(0, ROOT)
    import bench
    ab, ij = bench.ab_ij_sample(20, 5, 40, 12, 0)
    assert ab.shape == (40, 2) and ij.shape == (12, 2)
    assert ab.min() >= 0 and ab.max() < 20 and ij.min() >= 0 and ij.max() < 5
    assert (0, 0) in map(tuple, ab) and (19, 19) in map(tuple, ab)
    assert bench.oracle_sample_flops(20, 60, 2, 3) == 2 * (2 * 60 * 400 + 3 * 2 * 400)


def test_reference_arm_json_contract():
    """`bench.py --impl reference` (the oracle on host cores) prints the contract's line; tiny config here."""
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, check=True)
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "TFLOP/s" and line["higher_is_better"] is True
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["value"] == line["value"]
    assert line["value"] > 0
