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


def run_gpu(cl, L, t, R0, *, tile=0, algo=0, split=0, num_ctas=0, supertile=0, stream=None, calls=1, exchange=0, layout=0,
            symm=0, index_bits=0, info=None):
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
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SYMM_L, symm)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_INDEX_BITS, index_bits)
        if info is not None:
            info.update(plan_info(cl, plan))
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


def _unpack4(s):
    return ((s >> 24) & 255, (s >> 16) & 255, (s >> 8) & 255, s & 255)


def plan_info(cl, plan):
    return {"tile": _unpack4(cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_TILE_SHAPE)),
            "supertile": _unpack4(cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_SUPERTILE_SHAPE)),
            "index_bits": cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_INDEX_BITS),
            "tiles": cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_NUM_TILES),
            "flops_executed": cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_FLOPS_EXECUTED)}


def shape_of(cl, o, v, x, **opts):
    """Tile and super-tile shape the plan would use for these sizes and options (CC_LADDER_INFO_*), without running."""
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        for key, val in opts.items():
            cl.cc_ladder_set_option(plan, getattr(cl, "CC_LADDER_OPT_" + key.upper()), val)
        return plan_info(cl, plan)
    finally:
        cl.cc_ladder_destroy(plan)


def structured_sample(v, o, n_ab, n_ij, seed, tile=(8, 12, 20, 8), supertile=(3, 4, 3, 4)):
    """(a,b) and (i,j) picks on both sides of the edges the kernel really has: block edges (multiples of TA along a, of
    TB along b -- pass the plan's CC_LADDER_INFO_TILE_SHAPE), L2 super-tile edges (SA*TA, SB*TB), the first index of the
    last (ragged) block, and the 64-row chunk edges of the (ij) dimension; then seeded random pairs."""
    rng = np.random.default_rng(seed)
    ab = [(0, 0), (v - 1, v - 1), (0, v - 1), (v - 1, 0), (v // 2, v // 2), (1, 0), (0, 1)]
    for T, S, axis in ((tile[0], supertile[0], 0), (tile[1], supertile[1], 1)):
        for e in (T, 2 * T, S * T, 2 * S * T, (v // (2 * T)) * T, ((v - 1) // T) * T):
            for a in (e - 1, e):
                if 0 < a < v:
                    other = int(rng.integers(0, v))
                    ab += [(a, other) if axis == 0 else (other, a), (a, a)]
    ab = [p for p in ab if 0 <= p[0] < v and 0 <= p[1] < v]
    while len(ab) < n_ab:
        ab.append((int(rng.integers(0, v)), int(rng.integers(0, v))))
    ij = [(0, 0), (o - 1, o - 1), (0, o - 1), (o - 1, 0), (o // 2, o // 2)]
    for e in (64, 128, ((o * o - 1) // 64) * 64):       # 64-row chunk edges of the (ij) dimension: row = i*o + j
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
         "split": dict(split=1, tile=5), "split_8_8_12_12": dict(split=1, tile=4)}


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("o,v,x,sym", SMALL)
def test_full_parity_small(cl, oracle, o, v, x, sym, mode):
    L, t, R0 = gen.make_inputs(o, v, x, seed=o + v + x, symmetric=sym, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    got = run_gpu(cl, L, t, R0, **MODES[mode])
    assert rel(got, ref) <= TOL


@pytest.mark.parametrize("v", [26, 27])
@pytest.mark.parametrize("x", [8, 9, 15, 16, 17, 24, 31, 32, 33, 40, 48, 57])
def test_stage_boundaries_of_the_cholesky_loop(cl, oracle, x, v):
    """K = nchol around the 16-vector stages of GEMM-1 and their halves: the three L producer warps copy rows 0-7 and 8-15 of
    every X stage and all rows of every Y stage, full stages through the one-increment-per-copy path (16-byte copies for
    nvirt = 26, 8-byte copies for 27), the last, partial stage through the general loop with zero fill -- including tails that
    leave the upper-half warp no row at all (x mod 16 <= 8) -- in full mode (every tile shape) and in split mode."""
    o = 3
    L, t, R0 = gen.make_inputs(o, v, x, seed=1000 + 31 * x + v, symmetric=False, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    for mode in ("tile_8_12_16_8", "tile_12_8_12_12", "tile_8_12_20_8", "split"):
        got = run_gpu(cl, L, t, R0, **MODES[mode])
        assert rel(got, ref) <= TOL, mode


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
    # split mode combines with the exchange variant (same T+, negated T-) and with the paper's storage (pack / unpack addressing)
    for kw in (dict(split=1, exchange=1), dict(split=1, exchange=1, num_ctas=4, tile=4), dict(split=1, exchange=1, layout=1)):
        assert rel(run_gpu(cl, L, t, R0, **kw), ref) <= TOL, kw
    lad = oracle.ladder_full(L, t, R0)
    for kw in (dict(split=1, layout=1), dict(split=1, layout=1, num_ctas=6, tile=5)):
        assert rel(run_gpu(cl, L, t, R0, **kw), lad) <= TOL, kw
    b = cl.binding
    plan = cl.cc_ladder_plan(2, 4, 3)
    try:                                               # the simple path is a cross-check of the plain ladder only
        import torch
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, 1)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_ALGO, cl.CC_LADDER_ALGO_SIMPLE)
        z = torch.zeros(64, dtype=torch.float64, device="cuda")
        Lz = torch.zeros(48, dtype=torch.float64, device="cuda")
        ws = torch.zeros(1 << 16, dtype=torch.float64, device="cuda")
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


def _tri_layout(v):
    """The packed-triangle layout of the split workspace (csrc/ladder_common.cuh: tri_base / tri_size), restated: row c owns
    the slot d in [4*(c//4), v4) at base(c) + d, every base a multiple of 4 (128-bit copies, full-sector reductions)."""
    v4 = (v + 3) & ~3

    def base(c):
        m, r = c >> 2, c & 3
        return 4 * m * v4 - 8 * m * (m - 1) + r * (v4 - 4 * m) - 4 * m
    return v4, base, base(v) + 4 * (v >> 2)


def test_split_pack_step_against_oracle(cl, oracle):
    """Step a0 alone: the pack kernel writes T+ and T- as packed upper triangles (~v^2/2 doubles per (i,j)
    instead of v^2): the elements c <= d equal oracle_pack_tpm's arrays bit for bit (gathered through the layout's index
    map), every other slot entry is zero, and the workspace is half of the four o^2 v^2 squares of round 1."""
    import torch
    for o, v, x in ((3, 37, 4), (2, 8, 3), (1, 1, 2), (2, 33, 2), (2, 66, 3)):
        L, t, R0 = gen.make_inputs(o, v, x, seed=11, symmetric=False)
        v4, base, nt = _tri_layout(v)
        plan = cl.cc_ladder_plan(o, v, x)
        try:
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
            nb = cl.cc_ladder_workspace_bytes(plan)
            assert nb == o * o * (4 * nt + 16) * 8
            if v >= 66:
                assert nb < 0.6 * 4 * o * o * v * v * 8
            ws = torch.full((nb // 8,), 7.0, dtype=torch.float64, device="cuda")
            cl.cc_ladder_set_workspace(plan, ws, nb)
            dL, dt, dR = torch.from_numpy(L).cuda(), torch.from_numpy(t).cuda(), torch.from_numpy(R0).cuda()
            cl.cc_ladder(plan, dL, dt, dR, torch.cuda.current_stream())
            torch.cuda.synchronize()
        finally:
            cl.cc_ladder_destroy(plan)
        oo = o * o
        Tp = ws[:oo * nt].cpu().numpy().reshape(oo, nt)
        Tm = ws[oo * nt:2 * oo * nt].cpu().numpy().reshape(oo, nt)
        tp, tm = oracle.pack_tpm(t)                      # packed (c<=d) / (c<d), row-major
        kp = np.array([base(c) + d for c in range(v) for d in range(c, v)])
        km = np.array([base(c) + d for c in range(v) for d in range(c + 1, v)], dtype=np.int64)
        assert np.array_equal(Tp[:, kp], tp), (o, v)
        assert np.array_equal(Tm[:, km], tm), (o, v)
        rest_p = np.ones(nt, dtype=bool); rest_p[kp] = False
        rest_m = np.ones(nt, dtype=bool); rest_m[km] = False
        assert not Tp[:, rest_p].any() and not Tm[:, rest_m].any()      # left of the diagonal, padding, T- diagonal: zeros
        assert rel(dR.cpu().numpy(), oracle.ladder_full(L, t, R0)) <= TOL


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
               dict(split=1, tile=4, num_ctas=3), dict(split=1, tile=4, supertile=2),
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
    assert shape(300) == ((12, 8, 12, 12), 25 * 38 * 25 * 25) or shape(300)[0] == (8, 12, 20, 8)
    assert shape(420)[0] in ((12, 8, 12, 12), (8, 12, 20, 8))
    assert shape(520) == ((8, 12, 20, 8), 65 * 44 * 26 * 65)        # b padded to 528
    assert shape(128)[0] == (8, 12, 16, 8)                          # generic shape wins ties
    assert shape(300, split=1) == ((8, 8, 16, 16), (38 * 39 // 2) * (19 * 20 // 2))
    assert shape(420, split=1)[0] == (8, 8, 16, 16) and shape(520, split=1)[0] == (8, 8, 16, 16)
    assert shape(120, split=1)[0] == (8, 8, 12, 12)                 # 13.8 % fewer executed flops than with 16-wide (c,d) blocks


def test_host_entry_overlaps_R_copies_at_config2(cl, oracle):
    """cc_ladder_host with pinned buffers at configs[2] (R = 1.15 GB >= 256 MB): auto streams R in 72-row blocks (5) so
    that its copies overlap the kernels; oracle samples on both sides of the block edges and whole-tensor projections."""
    import torch
    o, v, x = gen.CONFIGS[2]
    L, t, R0 = gen.make_inputs(o, v, x, seed=2, r0=True)
    Lp, tp, Rp = (torch.from_numpy(a).pin_memory() for a in (L, t, R0.copy()))
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        cl.cc_ladder_host(plan, Lp, tp, Rp)
        assert cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_HOST_CHUNKS) == 5
    finally:
        cl.cc_ladder_destroy(plan)
    lad = Rp.numpy() - R0
    ab, ij = structured_sample(v, o, 48, 48, 31, (8, 12, 20, 8))
    edges = [(a, b) for a in (71, 72, 143, 144, 215, 216, 287, 288, 299) for b in (0, 151, 299)]
    ab = np.concatenate([ab, np.array(edges, dtype=np.int32)])
    ref = oracle.ladder_sampled(L, t, ab, ij)
    smp = lad[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
    scale = float(np.max(np.abs(lad)))
    assert float(np.max(np.abs(smp - ref))) / scale <= TOL
    rng = np.random.default_rng(77)
    u, w = rng.standard_normal(o), rng.standard_normal(o)
    proj = np.einsum("i,j,ijab->ab", u, w, lad)
    assert float(np.max(np.abs(proj - oracle.project_occ(L, t, u, w))) / np.max(np.abs(proj))) <= TOL


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
def _sampled_and_projected(cl, oracle, k, n_ab, n_ij, proj_occ, symmetric=True, r0=False, **kw):
    import torch
    o, v, x = gen.CONFIGS[k]
    L, t, R0 = gen.make_inputs(o, v, x, seed=k, symmetric=symmetric, r0=r0)
    info = {}
    got = run_gpu(cl, L, t, R0, info=info, **kw)
    if r0:
        got = got - R0              # the ladder part (R0 is O(1), the ladder O(10): the subtraction costs ~1e-16 of max|R|)
    scale = float(np.max(np.abs(got)))
    # (1) sampled outputs, one by one, on both sides of the block / super-tile / chunk edges of this plan
    ab, ij = structured_sample(v, o, n_ab, n_ij, k, info["tile"], info["supertile"])
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


def test_config1_full_size_unsymmetric_operands_and_nonzero_R0(cl, oracle):
    """configs[1] sizes with operands that have no symmetry at all and R0 = seeded noise (reading 1, reading 9)."""
    err = _sampled_and_projected(cl, oracle, 1, 120, 200, True, symmetric=False, r0=True)
    assert max(err) <= TOL, err
    err = _sampled_and_projected(cl, oracle, 1, 64, 100, False, symmetric=False, r0=True, split=1)
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
    # edges of both plans' block partitions: full mode <8,12,16,8> (or <8,12,20,8>) and split mode's square blocks
    tf, ts = shape_of(cl, o, v, x), shape_of(cl, o, v, x, split=1)
    ab1, ij = structured_sample(v, o, 40, 48, 4, tf["tile"], tf["supertile"])
    ab2, _ = structured_sample(v, o, 40, 48, 5, ts["tile"], ts["supertile"])
    ab = np.concatenate([ab1, ab2])
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


def test_paper_shaped_k300_full_and_split(cl, oracle):
    """The paper's own benchmark shape (Table 1: K = 300 -> nocc 75, nvirt 225, nchol 1500) with its iid
    operands (no symmetry in L or t; odd nvirt: 8-byte copies, ragged blocks on every axis) -- bench.py's `paper_shapes` leg."""
    import torch
    o, v, x = gen.PAPER_SHAPES[300]
    L, t = gen.paper_shaped(300, seed=300)
    R0 = np.zeros((o, o, v, v), dtype=np.float64)
    tf, ts = shape_of(cl, o, v, x), shape_of(cl, o, v, x, split=1)
    ab1, ij = structured_sample(v, o, 24, 32, 300, tf["tile"], tf["supertile"])
    ab2, _ = structured_sample(v, o, 24, 32, 301, ts["tile"], ts["supertile"])
    ab = np.concatenate([ab1, ab2])
    ref = oracle.ladder_sampled(L, t, ab, ij)
    rng = np.random.default_rng(300)
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


# ------------------------------------------------------------------------------------------ 64-bit tile decode, full mode
def test_full_mode_64bit_tile_decode(cl, oracle):
    """CC_LADDER_OPT_INDEX_BITS = 64 runs decode_tile4_t<long long> on the device (what nvirt > ~2000 would select by itself);
    the schedule is the same, so the result must be too."""
    L, t, R0 = gen.make_inputs(3, 42, 10, seed=9, symmetric=False, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    for kw in (dict(), dict(num_ctas=7, supertile=5), dict(tile=1, num_ctas=3), dict(tile=2), dict(exchange=1), dict(layout=1)):
        info = {}
        want = oracle.ladder_exchange(L, t, R0) if kw.get("exchange") else ref
        assert rel(run_gpu(cl, L, t, R0, index_bits=64, info=info, **kw), want) <= TOL, kw
        assert info["index_bits"] == 64
    info = {}
    run_gpu(cl, L, t, R0, info=info)
    assert info["index_bits"] == 32
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1)
    assert rel(run_gpu(cl, L, t, R0, index_bits=64), run_gpu(cl, L, t, R0)) <= 1e-12


def test_host_entry_point_pageable_buffers_split_mode_config1(cl, oracle):
    """cc_ladder_host with plain NumPy (pageable) buffers at configs[1] size in split mode: workspace allocated inside."""
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1, r0=True)
    R = R0.copy()
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
        cl.cc_ladder_host(plan, L, t, R)
        assert cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_HOST_CHUNKS) == 1
    finally:
        cl.cc_ladder_destroy(plan)
    lad = R - R0
    ab, ij = structured_sample(v, o, 64, 64, 12, (8, 8, 16, 16))
    ref = oracle.ladder_sampled(L, t, ab, ij)
    smp = lad[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
    assert float(np.max(np.abs(smp - ref)) / np.max(np.abs(lad))) <= TOL


# ------------------------------------------------------------------------------------------ 8-fold-symmetry mode
def symm_problem(o, v, x, seed, r0=True):
    """Symmetric Cholesky vectors (BASELINE.json generator) with amplitudes and R0 that have no symmetry at all."""
    L = gen.cholesky_vectors(seed, v, x, symmetric=True)
    t = gen.noise(seed, gen.STREAM_T_IID, (o, o, v, v), 0.05)
    R0 = gen.noise(seed, gen.STREAM_R0, (o, o, v, v), 1.0) if r0 else np.zeros((o, o, v, v))
    return L, t, R0


@pytest.mark.parametrize("o,v,x", [(5, 20, 60), (1, 1, 1), (1, 3, 2), (3, 7, 5), (2, 9, 11), (4, 33, 37), (6, 40, 50),
                                   (9, 24, 16), (12, 18, 3), (2, 66, 9)])
def test_symm_mode_parity_small(cl, oracle, o, v, x):
    """CC_LADDER_OPT_SYMM_L: only (a,b)-block <= (c,d)-block integral tiles are built and each is used twice; for a
    symmetric L the result is Eq. 6, element by element."""
    L, t, R0 = symm_problem(o, v, x, seed=o + v + x)
    ref = oracle.ladder_full(L, t, R0)
    assert rel(run_gpu(cl, L, t, R0, symm=1), ref) <= TOL
    if v <= 9:
        assert rel(oracle.ladder_symm(L, t, R0), ref) <= 1e-13          # the oracle's own statement of the mode


def test_symm_mode_scheduler_options_and_misuse(cl, oracle):
    import torch
    L, t, R0 = symm_problem(12, 26, 35, seed=41)
    ref = oracle.ladder_full(L, t, R0)
    for kw in (dict(num_ctas=1), dict(num_ctas=3, supertile=3), dict(num_ctas=5, supertile=1), dict(supertile=4096),
               dict(index_bits=64, num_ctas=7), dict(calls=1, num_ctas=148)):
        assert rel(run_gpu(cl, L, t, R0, symm=1, **kw), ref) <= TOL, kw
    lad = oracle.ladder_full(L, t)
    assert rel(run_gpu(cl, L, t, R0, symm=1, calls=2), R0 + 2.0 * lad) <= TOL
    # the precondition: an unsymmetric L is misuse (documented), detected by cc_ladder_check_symmetric
    Lu, tu, R0u = gen.make_inputs(4, 26, 9, seed=3, symmetric=False, r0=True)
    assert rel(run_gpu(cl, Lu, tu, R0u, symm=1), oracle.ladder_full(Lu, tu, R0u)) > 1e-6
    b = cl.binding
    plan = cl.cc_ladder_plan(4, 26, 9)
    try:
        dLu = torch.from_numpy(Lu).cuda()
        dLs = torch.from_numpy(gen.cholesky_vectors(3, 26, 9, symmetric=True)).cuda()
        assert cl.cc_ladder_check_symmetric(plan, dLs, torch.cuda.current_stream()) == 0
        assert cl.cc_ladder_check_symmetric(plan, dLu, torch.cuda.current_stream()) == 9 * 26 * 25 // 2
        Ls1 = dLs.clone(); Ls1[5, 3, 20] += 1.0
        assert cl.cc_ladder_check_symmetric(plan, Ls1) == 1
        # plain ladder only
        z = torch.zeros(16 * 26 * 26, dtype=torch.float64, device="cuda")
        s = torch.cuda.current_stream().cuda_stream
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SYMM_L, 1)
        assert b._lib.cc_ladder(plan, dLs.data_ptr(), z.data_ptr(), z.clone().data_ptr(), s) == b.CC_LADDER_OK
        for key in (cl.CC_LADDER_OPT_EXCHANGE, cl.CC_LADDER_OPT_LAYOUT):
            cl.cc_ladder_set_option(plan, key, 1)
            assert b._lib.cc_ladder(plan, dLs.data_ptr(), z.data_ptr(), z.clone().data_ptr(), s) == b.CC_LADDER_EINVAL
            cl.cc_ladder_set_option(plan, key, 0)
        torch.cuda.synchronize()
    finally:
        cl.cc_ladder_destroy(plan)


def test_symm_mode_config1_and_flop_count(cl, oracle):
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1)
    info = {}
    a = run_gpu(cl, L, t, R0, symm=1, info=info)
    assert rel(a, run_gpu(cl, L, t, R0)) <= 1e-12
    assert info["tile"] == (16, 8, 16, 8)
    n_blk = -(-v // 16) * (v // 8)
    assert info["tiles"] == n_blk * (n_blk + 1) // 2
    full = shape_of(cl, o, v, x)
    assert info["flops_executed"] < 0.88 * full["flops_executed"]          # GEMM-1 (50 % of the flops here) halves
    ab, ij = structured_sample(v, o, 64, 64, 13, info["tile"], info["supertile"])
    ref = oracle.ladder_sampled(L, t, ab, ij)
    smp = a[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
    assert float(np.max(np.abs(smp - ref)) / np.max(np.abs(a))) <= TOL


def test_symm_mode_config2(cl, oracle):
    err = _sampled_and_projected(cl, oracle, 2, 96, 64, True, symm=1)
    assert max(err) <= TOL, err


# ------------------------------------------------------------------------------------------ host-resident streaming
def test_host_streaming_of_R_column_blocks(cl, oracle):
    """cc_ladder_host when L + t + R exceed CC_LADDER_OPT_HOST_BUDGET (the paper's VRAM problem): R
    streams through two device buffers in blocks of `a`, L and t stay resident.  Forced at configs[1] size; pageable and
    pinned host buffers, both storages, the exchange variant; result equal to the resident path and to the oracle."""
    import torch
    o, v, x = gen.CONFIGS[1]
    L, t, R0 = gen.make_inputs(o, v, x, seed=1, symmetric=False, r0=True)
    nL, nT = L.nbytes, t.nbytes
    per_a = o * o * v * 8
    ab, ij = structured_sample(v, o, 64, 64, 14, (8, 12, 20, 8))
    ab = np.concatenate([ab, np.array([(23, 5), (24, 5), (47, 100), (48, 100), (95, 0), (96, 119)], dtype=np.int32)])
    ref = oracle.ladder_sampled(L, t, ab, ij)

    def run(budget, layout=0, exchange=0, pinned=False, block_rows=0, split=0):
        th = np.ascontiguousarray(t.transpose(0, 2, 1, 3)) if layout else t
        Rh = np.ascontiguousarray(R0.transpose(0, 2, 1, 3)) if layout else R0.copy()
        if pinned:
            Lp, tp, Rp = (torch.from_numpy(a).pin_memory() for a in (L, th, Rh))
        else:
            Lp, tp, Rp = L, th, Rh
        plan = cl.cc_ladder_plan(o, v, x)
        try:
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_HOST_BUDGET, budget)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_LAYOUT, layout)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, exchange)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_HOST_BLOCK_ROWS, block_rows)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, split)
            cl.cc_ladder_host(plan, Lp, tp, Rp)
            chunks = cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_HOST_CHUNKS)
        finally:
            cl.cc_ladder_destroy(plan)
        out = Rp.numpy() if pinned else Rp
        out = np.ascontiguousarray(out.transpose(0, 2, 1, 3)) if layout else out
        return out - R0, chunks

    resident, n1 = run(0)
    assert n1 == 1
    budget = nL + nT + 2 * 24 * per_a + 4096           # room for two blocks of 24 rows of a: 5 blocks
    for kw in (dict(), dict(pinned=True), dict(layout=1), dict(layout=1, pinned=True)):
        got, n = run(budget, **kw)
        assert n == 5, (kw, n)
        assert rel(got, resident) <= 1e-12, kw
        smp = got[ij[None, :, 0], ij[None, :, 1], ab[:, None, 0], ab[:, None, 1]]
        assert float(np.max(np.abs(smp - ref)) / np.max(np.abs(got))) <= TOL, kw
    got, n = run(nL + nT + 2 * 50 * per_a, exchange=1)            # 48 rows per block: 3 blocks (48, 48, 24)
    assert n == 3
    assert rel(got, resident.transpose(0, 1, 3, 2)) <= 1e-12      # E[i,j,a,b] == ladder[i,j,b,a]
    # everything fits: pinned buffers still stream R (overlap of its copies with the kernels) when asked for by
    # CC_LADDER_OPT_HOST_BLOCK_ROWS (auto only does so from 256 MB of R); pageable buffers, split mode and -1 stay resident
    for kw, want in ((dict(pinned=True, block_rows=40), 3), (dict(pinned=True, block_rows=24, layout=1), 5),
                     (dict(pinned=True, block_rows=0), 1), (dict(pinned=True, block_rows=-1), 1),
                     (dict(pinned=False, block_rows=24), 1), (dict(pinned=True, block_rows=24, split=1), 1),
                     (dict(pinned=True, block_rows=200), 1)):
        got, n = run(0, **kw)
        assert n == want, (kw, n)
        assert rel(got, resident) <= 1e-12, kw
    got, n = run(budget, pinned=True, block_rows=48)               # the budget's 24 rows cap the requested 48
    assert n == 5 and rel(got, resident) <= 1e-12
    # not even two minimal blocks next to L and t: ENOMEM; split mode cannot stream
    for budget, split in ((nL + nT + per_a, 0), (nL + nT + 100 * per_a, 1)):
        plan = cl.cc_ladder_plan(o, v, x)
        try:
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_HOST_BUDGET, budget)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, split)
            with pytest.raises(cl.CCLadderError) as ei:
                cl.cc_ladder_host(plan, L, t, R0.copy())
            assert ei.value.status == cl.binding.CC_LADDER_ENOMEM
        finally:
            cl.cc_ladder_destroy(plan)
