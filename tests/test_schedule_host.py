"""Step a1 (tile schedule) on the host: the decode functions of csrc/ladder_ws.cuh are __host__ __device__, so their
bijectivity (32- and 64-bit index arithmetic, ragged super-tiles, banded block-pair enumeration of the split mode) is
checked without a GPU by a small nvcc-built harness (tests/host_schedule_check.cu)."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(shutil.which(os.environ.get("NVCC", "nvcc")) is None, reason="nvcc not on PATH")
def test_tile_decodes_are_bijections(tmp_path):
    exe = str(tmp_path / "host_schedule_check")
    src = os.path.join(ROOT, "tests", "host_schedule_check.cu")
    subprocess.run([os.environ.get("NVCC", "nvcc"), "-std=c++17", "-O1", "-arch=sm_100a", "-o", exe, src], check=True)
    out = subprocess.run([exe], capture_output=True, text=True)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "bad=0" in out.stdout
