"""cc_ladder_split_static: the allocation-free entry point (scratch in the library's static device array).

Collected last on purpose (the suite runs with `pytest -x`).  Checks, on two calls in a row, that the entry point
gives what the existing split-mode path (plan + caller workspace) gives, within the parity bar of the other GPU tests
(1e-11 of max|R|), and what the oracle gives; that a second problem of another size is not disturbed by what the first
left in the shared array; that sizes beyond the array are rejected without touching R.
"""
import numpy as np
import pytest

import ladder_inputs as gen

pytestmark = pytest.mark.gpu

TOL = 1e-11


@pytest.fixture(scope="module")
def cl():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2310_04559_b200 as _cl
    return _cl


def rel(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def existing_split_path(cl, L, t, R0, calls):
    """cc_ladder with CC_LADDER_OPT_SPLIT = 1 and a torch-allocated workspace (the path the other GPU tests cover)."""
    import torch
    x, v, _ = L.shape
    o = t.shape[0]
    dL, dt, dR = torch.from_numpy(L).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(R0).cuda()
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
        nb = cl.cc_ladder_workspace_bytes(plan)
        assert nb == cl.cc_ladder_split_static_bytes(o, v)
        ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
        cl.cc_ladder_set_workspace(plan, ws, nb)
        for _ in range(calls):
            cl.cc_ladder(plan, dL, dt, dR, torch.cuda.current_stream())
        torch.cuda.synchronize()
    finally:
        cl.cc_ladder_destroy(plan)
    return dR.cpu().numpy()


def static_path(cl, L, t, R0, calls):
    import torch
    x, v, _ = L.shape
    o = t.shape[0]
    dL, dt, dR = torch.from_numpy(L).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(R0).cuda()
    for _ in range(calls):
        cl.cc_ladder_split_static(o, v, x, dL, dt, dR, torch.cuda.current_stream())
    torch.cuda.synchronize()
    return dR.cpu().numpy()


@pytest.mark.parametrize("o,v,x", [(6, 44, 60), (5, 37, 23), (12, 96, 40)])
def test_static_entry_two_calls_in_a_row(cl, o, v, x):
    import oracle
    assert cl.cc_ladder_split_static_bytes(o, v) <= cl.cc_ladder_static_scratch_bytes()
    L, t, R0 = gen.make_inputs(o, v, x, seed=900 + o + v + x, symmetric=False, r0=True)
    got = static_path(cl, L, t, R0, calls=2)
    ref = existing_split_path(cl, L, t, R0, calls=2)
    assert rel(got, ref) <= TOL
    want = R0 + 2.0 * oracle.ladder_full(L, t)          # two accumulating calls (reading 1)
    assert rel(got, want) <= TOL


def test_static_entry_shared_array_keeps_no_state_between_problems(cl):
    """A large problem, then a small one of another shape, then the large one again: every call rewrites what it reads."""
    big = gen.make_inputs(10, 120, 30, seed=931, symmetric=False, r0=True)
    small = gen.make_inputs(3, 18, 11, seed=932, symmetric=False, r0=True)
    for L, t, R0 in (big, small, big):
        assert rel(static_path(cl, L, t, R0, calls=1), existing_split_path(cl, L, t, R0, calls=1)) <= TOL


def test_static_entry_allocates_nothing(cl):
    """Free device memory as the driver reports it is the same before and after a burst of calls (after one warm-up
    call, which loads the kernels)."""
    import torch
    o, v, x = 6, 44, 60
    L, t, R0 = gen.make_inputs(o, v, x, seed=941, symmetric=False, r0=False)
    dL, dt, dR = torch.from_numpy(L).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(R0).cuda()
    s = torch.cuda.current_stream()
    cl.cc_ladder_split_static(o, v, x, dL, dt, dR, s)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(20):
        cl.cc_ladder_split_static(o, v, x, dL, dt, dR, s)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0


def test_static_entry_rejects_what_does_not_fit(cl):
    import torch
    limit = cl.cc_ladder_static_scratch_bytes()
    assert limit == cl.CC_LADDER_STATIC_SCRATCH_BYTES == 32 << 20
    o, v, x = 16, 96, 4                                  # needs 37.5 MiB
    assert cl.cc_ladder_split_static_bytes(o, v) > limit
    dL = torch.zeros(x * v * v, dtype=torch.float64, device="cuda")
    dt = torch.zeros(o * o * v * v, dtype=torch.float64, device="cuda")
    dR = torch.full((o * o * v * v,), 3.0, dtype=torch.float64, device="cuda")
    with pytest.raises(cl.CCLadderError) as e:
        cl.cc_ladder_split_static(o, v, x, dL, dt, dR)
    assert e.value.status == cl.CC_LADDER_ESCRATCH
    assert "static" in cl.status_string(cl.CC_LADDER_ESCRATCH)
    torch.cuda.synchronize()
    assert bool((dR == 3.0).all())
    for bad in [(0, 4, 4), (4, 0, 4), (4, 4, 0)]:
        with pytest.raises(cl.CCLadderError) as e:
            cl.cc_ladder_split_static(*bad, dL, dt, dR)
        assert e.value.status == cl.CC_LADDER_EINVAL
    with pytest.raises(cl.CCLadderError) as e:
        cl.cc_ladder_split_static(4, 8, 4, 0, dt, dR)
    assert e.value.status == cl.CC_LADDER_EINVAL
