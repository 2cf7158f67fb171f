"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, same seeded inputs.

Bar (BASELINE.json north_star): max |R_gpu - R_oracle| / max |R_oracle| <= 1e-11.  With ~v^2 <= 2.7e5-term FP64
sums the expected difference is 1e-16..1e-13, so 1e-11 leaves two orders of margin.
The result is unique up to rounding; the L2 reductions make it reproducible to ~1e-15, not bitwise.
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


def run_gpu(cl, L, t, R0, *, tile=0, algo=0, split=0, num_ctas=0, supertile=0, stream=None, calls=1, exchange=0, layout=0):
    import torch
    x, v, _ = L.shape
    o = t.shape[0]
    if layout:      # the paper's own storage t_old[i,c,j,d], t_new[i,a,j,b]; results are mapped back
        t, R0 = np.ascontiguousarray(t.transpose(0, 2, 1, 3)), np.ascontiguousarray(R0.transpose(0, 2, 1, 3))
    dL, dt, dR = torch.from_numpy(L).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(R0).cuda()
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_TILE, tile)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_ALGO, algo)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, split)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_NUM_CTAS, num_ctas)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SUPERTILE, supertile)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, exchange)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_LAYOUT, layout)
        nb = cl.cc_ladder_workspace_bytes(plan)
        ws = None
        if nb:
            ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
            cl.cc_ladder_set_workspace(plan, ws, nb)
        s = stream if stream is not None else torch.cuda.current_stream()
        for _ in range(calls):
            cl.cc_ladder(plan, dL, dt, dR, s)
        s.synchronize()
        torch.cuda.synchronize()
    finally:
        cl.cc_ladder_destroy(plan)
    out = dR.cpu().numpy()
    return np.ascontiguousarray(out.transpose(0, 2, 1, 3)) if layout else out


def rel(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def structured_sample(v, o, n_ab, n_ij, seed):
    rng = np.random.default_rng(seed)
    ab = [(0, 0), (v - 1, v - 1), (0, v - 1), (v - 1, 0), (v // 2, v // 2), (1, 0), (0, 1)]
    for e in (4, 8, 16, 32, 64, 128, 256, 512):          # both sides of every tile edge of both tile shapes
        for a in (e - 1, e):
            if 0 < a < v:
                ab += [(a, int(rng.integers(0, v))), (int(rng.integers(0, v)), a), (a, a)]
    ab = [p for p in ab if 0 <= p[0] < v and 0 <= p[1] < v]
    while len(ab) < n_ab:
        ab.append((int(rng.integers(0, v)), int(rng.integers(0, v))))
    ij = [(0, 0), (o - 1, o - 1), (0, o - 1), (o - 1, 0), (o // 2, o // 2)]
    for e in (8, 16, 32, 64):                           # chunk edges of the (ij) dimension: ij = i*o + j
        for r in (e - 1, e):
            if r < o * o:
                ij.append((r // o, r % o))
    while len(ij) < n_ij:
        ij.append((int(rng.integers(0, o)), int(rng.integers(0, o))))
    return np.array(ab, dtype=np.int32), np.array(ij, dtype=np.int32)


# ------------------------------------------------------------------------------------------ full-tensor parity
SMALL = [
    # o, v, x, symmetric operands?
    (5, 20, 60, True),       # BASELINE.json configs[0]
    (1, 1, 1, False),        # every dimension degenerate
    (1, 3, 2, False),
    (3, 7, 5, False),        # all odd
    (2, 9, 11, False),
    (4, 33, 37, False),      # odd v: 8-byte copy path, ragged tiles in a, b, c, d
    (6, 40, 50, False),      # several tiles per dimension, x not a multiple of 16
    (9, 24, 16, True),       # o^2 = 81: ragged last 64-row chunk
    (12, 18, 3, False),      # o^2 = 144: three row chunks, x < 4
    (2, 66, 9, False),       # 5 b-blocks / 9 a-blocks, many (cd) tiles
]


MODES = {"tile_8_12_16_8": dict(tile=1), "tile_12_8_12_12": dict(tile=2), "tile_8_12_20_8": dict(tile=3),
         "split": dict(split=1)}


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("o,v,x,sym", SMALL)
def test_full_parity_small(cl, oracle, o, v, x, sym, mode):
    L, t, R0 = gen.make_inputs(o, v, x, seed=o + v + x, symmetric=sym, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    got = run_gpu(cl, L, t, R0, **MODES[mode])
    assert rel(got, ref) <= TOL


# ------------------------------------------------------------------------------------------ exchange variant (Eq. 7)
@pytest.mark.parametrize("o,v,x,sym", SMALL)
def test_exchange_parity_small(cl, oracle, o, v, x, sym):
    """CC_LADDER_OPT_EXCHANGE: R += sum_cd (ad|bc) t_ij^cd, element by element against the oracle."""
    L, t, R0 = gen.make_inputs(o, v, x, seed=7 + o + v + x, symmetric=sym, r0=True)
    ref = oracle.ladder_exchange(L, t, R0)
    got = run_gpu(cl, L, t, R0, exchange=1)
    assert rel(got, ref) <= TOL


def test_exchange_many_tiles_and_options(cl, oracle):
    L, t, R0 = gen.make_inputs(12, 26, 35, seed=22, symmetric=False, r0=True)
    ref = oracle.ladder_exchange(L, t, R0)
    for kw in (dict(num_ctas=3), dict(num_ctas=148, supertile=5), dict(calls=1, stream=None)):
        assert rel(run_gpu(cl, L, t, R0, exchange=1, **kw), ref) <= TOL, kw
    b = cl.binding
    plan = cl.cc_ladder_plan(2, 4, 3)
    try:                                               # exchange is a full-mode option
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, 1)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
        import torch
        z = torch.zeros(64, dtype=torch.float64, device="cuda")
        Lz = torch.zeros(48, dtype=torch.float64, device="cuda")
        ws = torch.zeros(4 * 64, dtype=torch.float64, device="cuda")
        cl.cc_ladder_set_workspace(plan, ws, ws.numel() * 8)
        s = torch.cuda.current_stream().cuda_stream
        assert b._lib.cc_ladder(plan, Lz.data_ptr(), z.data_ptr(), z.clone().data_ptr(), s) == b.CC_LADDER_EINVAL
    finally:
        cl.cc_ladder_destroy(plan)


def test_exchange_config1_is_the_transposed_ladder(cl, oracle):
    """configs[1] at full size: E[i,j,a,b] == ladder[i,j,b,a] (both from the GPU, different tile shapes), plus oracle
    samples of the ladder at the swapped pairs."""
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1)
    E = run_gpu(cl, L, t, R0, exchange=1)
    lad = run_gpu(cl, L, t, R0)
    assert rel(E, lad.transpose(0, 1, 3, 2)) <= 1e-12
    ab, ij = structured_sample(v, o, 48, 40, 5)
    ref = oracle.ladder_sampled(L, t, ab, ij)                     # ladder at (a,b) == exchange at (b,a)
    smp = E[ij[None, :, 0], ij[None, :, 1], ab[:, None, 1], ab[:, None, 0]]
    assert float(np.max(np.abs(smp - ref)) / np.max(np.abs(E))) <= TOL


# ------------------------------------------------------------------------------------------ the paper's [i,a,j,b] storage
@pytest.mark.parametrize("tile", [1, 2, 3])
@pytest.mark.parametrize("o,v,x,sym", SMALL)
def test_iajb_layout_parity_small(cl, oracle, o, v, x, sym, tile):
    """CC_LADDER_OPT_LAYOUT = IAJB: t_old[i,c,j,d] in, t_new[i,a,j,b] += out, element by element."""
    L, t, R0 = gen.make_inputs(o, v, x, seed=3 + o + v + x, symmetric=sym, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    assert rel(run_gpu(cl, L, t, R0, layout=1, tile=tile), ref) <= TOL


def test_iajb_layout_many_tiles_exchange_and_einsum(cl, oracle):
    L, t, R0 = gen.make_inputs(12, 26, 35, seed=23, symmetric=False, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    for kw in (dict(num_ctas=3, tile=1), dict(num_ctas=5, tile=3, supertile=3), dict(num_ctas=148)):
        assert rel(run_gpu(cl, L, t, R0, layout=1, **kw), ref) <= TOL, kw
    assert rel(run_gpu(cl, L, t, R0, layout=1, exchange=1, num_ctas=4), oracle.ladder_exchange(L, t, R0)) <= TOL
    # the paper's one-liner on its own storage: t_new += einsum("xac,xbd,icjd->iajb", L, L, t_old)
    Ls, ts, _ = gen.make_inputs(3, 10, 6, seed=2, symmetric=False)
    t_old = np.ascontiguousarray(ts.transpose(0, 2, 1, 3))
    t_new = np.einsum("xac,xbd,icjd->iajb", Ls, Ls, t_old)
    got = run_gpu(cl, Ls, ts, np.zeros_like(ts), layout=1)            # run_gpu maps [i,a,j,b] back to [i,j,a,b]
    assert rel(got.transpose(0, 2, 1, 3), t_new) <= 1e-12


def test_iajb_layout_config1(cl, oracle):
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1)
    a = run_gpu(cl, L, t, R0, layout=1)
    b = run_gpu(cl, L, t, R0)
    assert rel(a, b) <= 1e-12
    ab, ij = structured_sample(v, o, 32, 40, 6)
    ref = oracle.ladder_sampled(L, t, ab, ij)
    smp = a[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
    assert float(np.max(np.abs(smp - ref)) / np.max(np.abs(a))) <= TOL


def test_split_pack_step_against_oracle(cl, oracle):
    """Step a0 alone: T+ / T- written by the pack kernel equal the oracle's packing (reading 10), bit for bit."""
    import torch
    o, v, x = 3, 37, 4
    L, t, R0 = gen.make_inputs(o, v, x, seed=11, symmetric=False)
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
        nb = cl.cc_ladder_workspace_bytes(plan)
        assert nb == 4 * o * o * v * v * 8
        ws = torch.zeros(nb // 8, dtype=torch.float64, device="cuda")
        cl.cc_ladder_set_workspace(plan, ws, nb)
        dL, dt, dR = torch.from_numpy(L).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(R0).cuda()
        cl.cc_ladder(plan, dL, dt, dR, torch.cuda.current_stream())
        torch.cuda.synchronize()
    finally:
        cl.cc_ladder_destroy(plan)
    n = o * o * v * v
    Tp = ws[:n].cpu().numpy().reshape(o * o, v, v)
    Tm = ws[n:2 * n].cpu().numpy().reshape(o * o, v, v)
    tp, tm = oracle.pack_tpm(t)                      # packed (c<=d) / (c<d), row-major
    iu, il = np.triu_indices(v), np.triu_indices(v, 1)
    assert np.array_equal(Tp[:, il[0], il[1]], tp[:, iu[0] != iu[1]])          # c < d: t_cd + t_dc
    assert np.array_equal(Tp[:, np.arange(v), np.arange(v)], 2.0 * tp[:, iu[0] == iu[1]])   # c == d: full square holds 2 t_cc
    assert np.array_equal(Tm[:, il[0], il[1]], tm)
    assert np.array_equal(Tm, -Tm.transpose(0, 2, 1)) and np.array_equal(Tp, Tp.transpose(0, 2, 1))


def test_split_needs_workspace(cl):
    import torch
    b = cl.binding
    plan = cl.cc_ladder_plan(2, 4, 3)
    try:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
        L = torch.zeros(48, dtype=torch.float64, device="cuda")
        t = torch.zeros(64, dtype=torch.float64, device="cuda")
        R = torch.zeros(64, dtype=torch.float64, device="cuda")
        s = torch.cuda.current_stream().cuda_stream
        assert b._lib.cc_ladder(plan, L.data_ptr(), t.data_ptr(), R.data_ptr(), s) == b.CC_LADDER_EWORKSPACE
        assert cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_KERNEL_LAUNCHES) == 3
    finally:
        cl.cc_ladder_destroy(plan)


@pytest.mark.parametrize("o,v,x,sym", SMALL[:7])
def test_simple_path_parity(cl, oracle, o, v, x, sym):
    L, t, R0 = gen.make_inputs(o, v, x, seed=3, symmetric=sym, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    got = run_gpu(cl, L, t, R0, algo=cl.CC_LADDER_ALGO_SIMPLE)
    assert rel(got, ref) <= TOL


def test_accumulates_and_repeats(cl, oracle):
    """Reading 1 ('+='): two calls on a non-zero R0 give R0 + 2 ladder."""
    L, t, R0 = gen.make_inputs(4, 21, 13, seed=5, symmetric=False, r0=True)
    lad = oracle.ladder_full(L, t)
    got = run_gpu(cl, L, t, R0, calls=2)
    assert rel(got, R0 + 2.0 * lad) <= TOL


def test_scheduler_options_do_not_change_the_result(cl, oracle):
    """Few CTAs (many tiles per CTA), odd super-tile edges (ragged super-rows/columns), non-default stream."""
    import torch
    L, t, R0 = gen.make_inputs(3, 42, 10, seed=9, symmetric=False, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    for kw in (dict(num_ctas=1), dict(num_ctas=7, supertile=1), dict(supertile=5), dict(supertile=4096),
               dict(num_ctas=1000, tile=1), dict(num_ctas=5, tile=2, supertile=2), dict(tile=3, supertile=7),
               dict(stream=torch.cuda.Stream()),
               dict(split=1, num_ctas=2), dict(split=1, num_ctas=7, supertile=3), dict(split=1, num_ctas=1),
               dict(split=1, supertile=4096)):      # the last one decodes tile indices in 64-bit arithmetic
        assert rel(run_gpu(cl, L, t, R0, **kw), ref) <= TOL, kw


def test_many_tiles_per_cta_three_row_chunks(cl, oracle):
    """Few CTAs on a problem with 3 row chunks (the last ragged), 3 GEMM-1 stages per tile and tiles on the edge of R:
    the stage ring, the head slot, the Vs hand-over and the parked reductions all wrap many times per CTA."""
    L, t, R0 = gen.make_inputs(12, 26, 35, seed=21, symmetric=False, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    for kw in (dict(num_ctas=3, tile=1), dict(num_ctas=2, tile=2), dict(num_ctas=5, tile=3, supertile=3),
               dict(num_ctas=4, split=1), dict(num_ctas=148)):
        assert rel(run_gpu(cl, L, t, R0, **kw), ref) <= TOL, kw


def test_run_to_run_reproducible_to_rounding(cl):
    L, t, R0 = gen.make_inputs(6, 40, 50, seed=2, symmetric=True)
    a = run_gpu(cl, L, t, R0)
    b = run_gpu(cl, L, t, R0)
    assert rel(a, b) <= 1e-13


def test_host_entry_point(cl, oracle):
    L, t, R0 = gen.make_inputs(5, 20, 60, seed=0, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    R = R0.copy()
    plan = cl.cc_ladder_plan(5, 20, 60)
    try:
        cl.cc_ladder_host(plan, L, t, R)
    finally:
        cl.cc_ladder_destroy(plan)
    assert rel(R, ref) <= TOL


def test_plan_picks_the_least_padded_tile_shape(cl):
    """Step a1 at plan time: block edges <TA,TB,TC,TD> that minimise the padded (a,b,c,d) volume."""
    def shape(v, split=0):
        plan = cl.cc_ladder_plan(3, v, 7)
        try:
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, split)
            s = cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_TILE_SHAPE)
            tiles = cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_NUM_TILES)
        finally:
            cl.cc_ladder_destroy(plan)
        return ((s >> 24) & 255, (s >> 16) & 255, (s >> 8) & 255, s & 255), tiles
    # (nocc, nchol) = (3, 7): every footprint fits L2, so the choice is padded volume / relative efficiency
    assert shape(300) == ((12, 8, 12, 12), 25 * 38 * 25 * 25) or shape(300)[0] == (8, 12, 20, 8)
    assert shape(420)[0] in ((12, 8, 12, 12), (8, 12, 20, 8))
    assert shape(520) == ((8, 12, 20, 8), 65 * 44 * 26 * 65)        # b padded to 528
    assert shape(128)[0] == (8, 12, 16, 8)                          # generic shape wins ties
    assert shape(300, split=1) == ((8, 8, 16, 16), (38 * 39 // 2) * (19 * 20 // 2))


# ------------------------------------------------------------------------------------------ error paths
def test_error_paths(cl):
    import torch
    b = cl.binding
    plan = cl.cc_ladder_plan(2, 4, 3)
    try:
        L = torch.zeros(3 * 16 + 2, dtype=torch.float64, device="cuda")
        t = torch.zeros(4 * 16, dtype=torch.float64, device="cuda")
        R = torch.zeros(4 * 16, dtype=torch.float64, device="cuda")
        s = torch.cuda.current_stream().cuda_stream
        assert b._lib.cc_ladder(plan, None, t.data_ptr(), R.data_ptr(), s) == b.CC_LADDER_EINVAL
        assert b._lib.cc_ladder(plan, L.data_ptr() + 8, t.data_ptr(), R.data_ptr(), s) == b.CC_LADDER_EINVAL   # misaligned
        assert b._lib.cc_ladder(plan, L.data_ptr(), t.data_ptr(), t.data_ptr(), s) == b.CC_LADDER_EINVAL      # R aliases t
        assert b._lib.cc_ladder(plan, L.data_ptr(), t.data_ptr(), L.data_ptr(), s) == b.CC_LADDER_EINVAL      # R aliases L
        with pytest.raises(cl.CCLadderError):
            cl.cc_ladder_set_option(plan, 999, 0)
        with pytest.raises(cl.CCLadderError):
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 2)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_ALGO, cl.CC_LADDER_ALGO_SIMPLE)
        assert cl.cc_ladder_workspace_bytes(plan) > 0
        assert b._lib.cc_ladder(plan, L.data_ptr(), t.data_ptr(), R.data_ptr(), s) == b.CC_LADDER_EWORKSPACE
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_ALGO, cl.CC_LADDER_ALGO_FUSED)
        assert cl.cc_ladder_workspace_bytes(plan) == 0
        assert b._lib.cc_ladder(plan, L.data_ptr(), t.data_ptr(), R.data_ptr(), s) == b.CC_LADDER_OK
        torch.cuda.synchronize()
        assert cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_NUM_SMS) == torch.cuda.get_device_properties(0).multi_processor_count
        assert cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_FLOPS_FULL) == gen.ladder_flops(2, 4, 3)
    finally:
        cl.cc_ladder_destroy(plan)


# ------------------------------------------------------------------------------------------ BASELINE sizes
def _sampled_and_projected(cl, oracle, k, n_ab, n_ij, proj_occ, **kw):
    import torch
    o, v, x = gen.CONFIGS[k]
    L, t, R0 = gen.make_inputs(o, v, x, seed=k)
    got = run_gpu(cl, L, t, R0, **kw)
    scale = float(np.max(np.abs(got)))
    # (1) sampled outputs, one by one
    ab, ij = structured_sample(v, o, n_ab, n_ij, k)
    ref = oracle.ladder_sampled(L, t, ab, ij)
    smp = got[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
    err_s = float(np.max(np.abs(smp - ref)) / scale)
    # (2) whole-tensor projection over the virtual pair: touches every (a,b) of every (i,j)   (pin P7b)
    rng = np.random.default_rng(77 + k)
    p, q = rng.standard_normal(v), rng.standard_normal(v)
    proj_ref = oracle.project_virt(L, t, p, q)
    G = torch.from_numpy(got)
    proj = torch.einsum("a,b,ijab->ij", torch.from_numpy(p), torch.from_numpy(q), G).numpy()
    err_v = float(np.max(np.abs(proj - proj_ref)) / np.max(np.abs(proj_ref)))
    err_o = 0.0
    if proj_occ:                                     # (3) projection over the occupied pair (pin P7a)
        u, w = rng.standard_normal(o), rng.standard_normal(o)
        po_ref = oracle.project_occ(L, t, u, w)
        po = torch.einsum("i,j,ijab->ab", torch.from_numpy(u), torch.from_numpy(w), G).numpy()
        err_o = float(np.max(np.abs(po - po_ref)) / np.max(np.abs(po_ref)))
    return err_s, err_v, err_o


def test_config1_full_size(cl, oracle):
    """configs[1] (20, 120, 400): all (i,j) for 160 sampled (a,b) + both whole-tensor projections."""
    err = _sampled_and_projected(cl, oracle, 1, 160, 400, True)
    assert max(err) <= TOL, err


def test_config1_all_tile_shapes_agree_everywhere(cl):
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1)
    a = run_gpu(cl, L, t, R0, tile=1)
    for tile in (2, 3):
        assert rel(a, run_gpu(cl, L, t, R0, tile=tile)) <= 1e-12, tile


def test_config1_split(cl, oracle):
    err = _sampled_and_projected(cl, oracle, 1, 160, 400, True, split=1)
    assert max(err) <= TOL, err


def test_config2_bench_workload(cl, oracle):
    """configs[2] (40, 300, 1000), the default bench.py workload in its launch configuration."""
    err = _sampled_and_projected(cl, oracle, 2, 96, 64, True)
    assert max(err) <= TOL, err


def test_config2_bench_workload_split(cl, oracle):
    err = _sampled_and_projected(cl, oracle, 2, 96, 64, True, split=1)
    assert max(err) <= TOL, err


def test_config3_sampled(cl, oracle):
    """configs[3] (50, 420, 1400): the v^4 tensor (250 GB) could not exist in HBM."""
    err = _sampled_and_projected(cl, oracle, 3, 64, 48, False)
    assert max(err) <= TOL, err


def test_config4_sampled_with_and_without_split(cl, oracle):
    """configs[4] (64, 520, 1800), ~1e15 flop per evaluation; both modes against the same oracle samples."""
    import torch
    o, v, x = gen.CONFIGS[4]
    L, t, R0 = gen.make_inputs(o, v, x, seed=4)
    ab, ij = structured_sample(v, o, 64, 48, 4)
    ref = oracle.ladder_sampled(L, t, ab, ij)
    rng = np.random.default_rng(81)
    p, q = rng.standard_normal(v), rng.standard_normal(v)
    proj_ref = oracle.project_virt(L, t, p, q)
    for split in (0, 1):
        got = run_gpu(cl, L, t, R0, split=split)
        scale = float(np.max(np.abs(got)))
        smp = got[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
        assert float(np.max(np.abs(smp - ref)) / scale) <= TOL, split
        proj = torch.einsum("a,b,ijab->ij", torch.from_numpy(p), torch.from_numpy(q), torch.from_numpy(got)).numpy()
        assert float(np.max(np.abs(proj - proj_ref)) / np.max(np.abs(proj_ref))) <= TOL, split
        del got
