"""CPU-side checks of the boundary: the library builds, loads and exports what include/cc_ladder.h declares.

No compute call is made here (no GPU in the CPU suite); error paths that need no device are exercised.
"""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "cc_ladder.h")


@pytest.fixture(scope="module")
def cl():
    from paper_2310_04559_b200 import build as _build
    _build.build()
    import paper_2310_04559_b200 as _cl
    return _cl


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(cc_ladder\w*)\s*\(", src)))


def test_header_symbols_exported(cl):
    lib = ctypes.CDLL(cl.library_path())
    names = _declared_functions()
    assert "cc_ladder_plan" in names and "cc_ladder" in names and "cc_ladder_destroy" in names
    for n in names:
        assert hasattr(lib, n), f"{n} declared in cc_ladder.h but not exported"
    assert set(names) == set(cl.binding.EXPORTS)


def test_header_constants_match_binding(cl):
    src = open(HEADER).read()
    for name, val in re.findall(r"#define\s+(CC_LADDER_[A-Z_0-9]+)\s+\(?(-?\d+)\)?", src):
        assert getattr(cl.binding, name) == int(val), name


def test_status_strings(cl):
    assert cl.status_string(0) == "ok"
    for s in (-1, -2, -3, -4, -5, -6):
        assert cl.status_string(s) and cl.status_string(s) != "unknown status"
    assert cl.status_string(-99) == "unknown status"


def test_plan_rejects_bad_sizes_without_a_device(cl):
    for args in [(0, 4, 4), (4, 0, 4), (4, 4, 0), (-1, 4, 4)]:
        with pytest.raises(cl.CCLadderError) as e:
            cl.cc_ladder_plan(*args)
        assert e.value.status == cl.binding.CC_LADDER_EINVAL


def test_no_cpu_fallback(cl):
    """Without a CUDA device the product fails loudly instead of computing anything on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(cl.CCLadderError) as e:
        cl.cc_ladder_plan(5, 20, 60)
    assert e.value.status in (cl.binding.CC_LADDER_ECUDA, cl.binding.CC_LADDER_EARCH)


def test_null_plan_calls(cl):
    b = cl.binding
    assert b._lib.cc_ladder_destroy(None) == 0
    assert b._lib.cc_ladder(None, None, None, None, None) == b.CC_LADDER_EINVAL
    assert b._lib.cc_ladder_set_option(None, 1, 0) == b.CC_LADDER_EINVAL
    assert b._lib.cc_ladder_workspace_bytes(None) == 0


def test_static_entry_size_checks_need_no_device(cl):
    """cc_ladder_split_static rejects bad sizes and problems beyond its static scratch before any CUDA call."""
    b = cl.binding
    assert b._lib.cc_ladder_static_scratch_bytes() == b.CC_LADDER_STATIC_SCRATCH_BYTES
    assert b._lib.cc_ladder_split_static_bytes(0, 5) == 0
    # 8 o^2 (4 tri(v) + 16) with tri(96) = 4800 slots (rows of the packed triangle start on multiples of 4)
    assert b._lib.cc_ladder_split_static_bytes(12, 96) == 8 * 144 * (4 * 4800 + 16)
    assert b._lib.cc_ladder_split_static(0, 4, 4, 16, 16, 16, None) == b.CC_LADDER_EINVAL
    assert b._lib.cc_ladder_split_static(4, 4, 4, None, 16, 16, None) == b.CC_LADDER_EINVAL
    assert b._lib.cc_ladder_split_static(40, 300, 1000, 16, 32, 48, None) == b.CC_LADDER_ESCRATCH


def test_product_does_not_import_oracle():
    """The product package and the oracle share nothing (neither imports the other)."""
    pkg = os.path.join(ROOT, "paper_2310_04559_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "ladder_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2310_04559_b200 import" not in txt and "import paper_2310_04559_b200" not in txt, f
            assert "cc_ladder.h" not in txt, f
