"""Parity of cc_ladder_xy (the occupied-virtual family, Eqs. 8-9, recipe "abcd,ecfd->efab") against the
CPU oracle, element by element on the same seeded inputs; bar 1e-11 of max|out| as for the ladder."""
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
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def run_xy(cl, X, Y, t, out0, *, tile=0, num_ctas=0, supertile=0, exchange=0, layout=0, calls=1, index_bits=0):
    """X, Y: numpy views (possibly strided slices of a larger array, last axis contiguous); returns out[i,j,r,s]."""
    import torch
    x, nr, v = X.shape
    ns = Y.shape[1]
    o = t.shape[0]

    def dev(a):      # upload the underlying contiguous base once, pass the view's pointer and strides
        base = a.base if a.base is not None else a
        base = np.ascontiguousarray(base) if not base.flags["C_CONTIGUOUS"] else base
        d = torch.from_numpy(base).cuda()
        off = (a.__array_interface__["data"][0] - base.__array_interface__["data"][0]) // 8
        assert a.strides[2] == 8
        return d, d.data_ptr() + 8 * off, a.strides[0] // 8, a.strides[1] // 8

    dX, pX, xps, xrs = dev(X)
    dY, pY, yps, yrs = dev(Y)
    if layout:
        t, out0 = np.ascontiguousarray(t.transpose(0, 2, 1, 3)), np.ascontiguousarray(out0.transpose(0, 2, 1, 3))
    dt, dout = torch.from_numpy(np.ascontiguousarray(t)).cuda(), torch.from_numpy(np.ascontiguousarray(out0)).cuda()
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_TILE, tile)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_NUM_CTAS, num_ctas)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SUPERTILE, supertile)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, exchange)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_LAYOUT, layout)
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_INDEX_BITS, index_bits)
        for _ in range(calls):
            cl.cc_ladder_xy(plan, pX, xps, xrs, nr, pY, yps, yrs, ns, dt, dout, torch.cuda.current_stream())
        torch.cuda.synchronize()
        assert cl.cc_ladder_get_option(plan, cl.CC_LADDER_OPT_XY_ROWS_X) == nr
        assert cl.cc_ladder_get_info(plan, cl.CC_LADDER_INFO_FLOPS_FULL) == 2 * nr * ns * v * v * (x + o * o)
    finally:
        cl.cc_ladder_destroy(plan)
    res = dout.cpu().numpy()
    return np.ascontiguousarray(res.transpose(0, 2, 1, 3)) if layout else res


def problem(o, v, x, nr, ns, seed):
    X = gen.cholesky_block(seed, nr, v, x)
    Y = gen.cholesky_block(seed + 1000, ns, v, x)
    t = gen.noise(seed, gen.STREAM_T_IID, (o, o, v, v), 0.05)
    out0 = gen.noise(seed, gen.STREAM_R0, (o, o, nr, ns), 1.0)
    return X, Y, t, out0


SMALL = [
    # o, v, x, nr, ns
    (5, 20, 60, 5, 20),       # Eq. 9 shape at BASELINE.json configs[0]: X = L_ov, Y = L_vv
    (5, 20, 60, 5, 5),        # Eq. 8 shape
    (1, 1, 1, 1, 1),
    (1, 3, 2, 1, 4),          # nr = o = 1
    (3, 7, 5, 3, 7),          # all odd: 8-byte copy path
    (2, 9, 11, 13, 2),        # nr > v, ns small
    (4, 33, 37, 4, 33),
    (6, 40, 50, 6, 41),       # several tiles, x not a multiple of 16, odd ns with even v
    (9, 24, 16, 9, 9),        # o^2 = 81: ragged last 64-row chunk
    (12, 18, 3, 12, 30),      # three row chunks, x < 4
    (2, 66, 9, 17, 66),
]


@pytest.mark.parametrize("tile", [0, 1, 2, 3])
@pytest.mark.parametrize("o,v,x,nr,ns", SMALL)
def test_xy_parity_small(cl, oracle, o, v, x, nr, ns, tile):
    X, Y, t, out0 = problem(o, v, x, nr, ns, seed=o + v + x + nr + ns)
    ref = oracle.ladder_xy(X, Y, t, out0)
    assert rel(run_xy(cl, X, Y, t, out0, tile=tile), ref) <= TOL


def test_xy_blocks_of_a_larger_cholesky_array_need_no_copy(cl, oracle):
    """X = L[:, :o, o:], Y = L[:, o:, o:] as strided views of one L[P][p][q] over all K = o + v orbitals (PAPER.md:135:
    the engine slices the Cholesky array): Eq. 9 and Eq. 8 through pointer + stride arguments; accumulation over two calls."""
    o, v, x = 4, 22, 13
    K = o + v
    Lall = gen.noise(5, gen.STREAM_L, (x, K, K), 1.0)
    Lov, Lvv = Lall[:, :o, o:], Lall[:, o:, o:]
    t = gen.noise(5, gen.STREAM_T_IID, (o, o, v, v), 0.05)
    out0 = gen.noise(5, gen.STREAM_R0, (o, o, o, v), 1.0)
    e9 = oracle.ladder_xy(np.ascontiguousarray(Lov), np.ascontiguousarray(Lvv), t)
    assert rel(run_xy(cl, Lov, Lvv, t, out0, calls=2), out0 + 2.0 * e9) <= TOL
    e8 = oracle.ladder_xy(np.ascontiguousarray(Lov), np.ascontiguousarray(Lov), t)
    assert rel(run_xy(cl, Lov, Lov, t, np.zeros((o, o, o, o))), e8) <= TOL
    # odd K: every row of the blocks is only 8-byte aligned
    Lodd = gen.noise(6, gen.STREAM_L, (x, K + 1, K + 1), 1.0)
    Xo, Yo = Lodd[:, 1:o + 1, o + 1:], Lodd[:, o + 1:, o + 1:]
    ref = oracle.ladder_xy(np.ascontiguousarray(Xo), np.ascontiguousarray(Yo), t)
    assert rel(run_xy(cl, Xo, Yo, t, np.zeros((o, o, o, v))), ref) <= TOL


def test_xy_reduces_to_the_ladder(cl, oracle):
    L, t, R0 = gen.make_inputs(6, 40, 50, seed=3, symmetric=False, r0=True)
    ref = oracle.ladder_full(L, t, R0)
    assert rel(run_xy(cl, L, L, t, R0), ref) <= TOL


def test_xy_scheduler_options_exchange_and_layout(cl, oracle):
    X, Y, t, out0 = problem(12, 26, 35, 12, 26, seed=31)
    ref = oracle.ladder_xy(X, Y, t, out0)
    for kw in (dict(num_ctas=1), dict(num_ctas=3, tile=1), dict(num_ctas=5, tile=3, supertile=3), dict(supertile=4096),
               dict(tile=2, num_ctas=7, supertile=1), dict(index_bits=64), dict(index_bits=64, num_ctas=2, tile=3),
               dict(layout=1), dict(layout=1, tile=2, num_ctas=4)):
        assert rel(run_xy(cl, X, Y, t, out0, **kw), ref) <= TOL, kw
    # exchange pairing: out[i,j,r,s] += sum_cd (sum_P X[P,r,d] Y[P,s,c]) t[i,j,c,d] == xy(X, Y, t^T_cd)
    ref_x = oracle.ladder_xy(X, Y, np.ascontiguousarray(t.transpose(0, 1, 3, 2)), out0)
    assert rel(run_xy(cl, X, Y, t, out0, exchange=1), ref_x) <= TOL
    assert rel(run_xy(cl, X, Y, t, out0, exchange=1, layout=1, num_ctas=3), ref_x) <= TOL


def test_xy_error_paths(cl):
    import torch
    b = cl.binding
    o, v, x = 2, 4, 3
    plan = cl.cc_ladder_plan(o, v, x)
    try:
        X = torch.zeros(x * 2 * v, dtype=torch.float64, device="cuda")
        Y = torch.zeros(x * v * v, dtype=torch.float64, device="cuda")
        t = torch.zeros(o * o * v * v, dtype=torch.float64, device="cuda")
        out = torch.zeros(o * o * 2 * v, dtype=torch.float64, device="cuda")
        s = torch.cuda.current_stream().cuda_stream
        args = lambda **k: (plan, k.get("X", X.data_ptr()), k.get("xps", 2 * v), k.get("xrs", v), k.get("nr", 2),
                            Y.data_ptr(), v * v, v, v, t.data_ptr(), k.get("out", out.data_ptr()), s)
        assert b._lib.cc_ladder_xy(*args()) == b.CC_LADDER_OK
        assert b._lib.cc_ladder_xy(*args(nr=0)) == b.CC_LADDER_EINVAL
        assert b._lib.cc_ladder_xy(*args(xrs=v - 1)) == b.CC_LADDER_EINVAL          # rows would overlap
        assert b._lib.cc_ladder_xy(*args(xps=v)) == b.CC_LADDER_EINVAL              # P stride smaller than the block
        assert b._lib.cc_ladder_xy(*args(X=None)) == b.CC_LADDER_EINVAL
        assert b._lib.cc_ladder_xy(*args(out=t.data_ptr())) == b.CC_LADDER_EINVAL   # out aliases t
        assert b._lib.cc_ladder_xy(*args(out=out.data_ptr() + 8)) == b.CC_LADDER_EINVAL
        cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, 1)
        assert b._lib.cc_ladder_xy(*args()) == b.CC_LADDER_EINVAL                   # full mode only
        torch.cuda.synchronize()
    finally:
        cl.cc_ladder_destroy(plan)


def test_xy_eq9_at_config2_sizes(cl, oracle):
    """Eq. 9 at BASELINE.json configs[2] sizes (o=40 rows of L_ov against v=300, x=1000) in the bench launch
    configuration: oracle samples one by one + a whole-tensor projection over (r,s) that touches every output."""
    import torch
    o, v, x = gen.CONFIGS[2]
    X = gen.cholesky_block(2, o, v, x)
    Y, t, _ = gen.make_inputs(o, v, x, seed=2)
    out0 = np.zeros((o, o, o, v))
    got = run_xy(cl, X, Y, t, out0)
    scale = float(np.max(np.abs(got)))
    rng = np.random.default_rng(5)
    rs = [(0, 0), (o - 1, v - 1), (0, v - 1), (o - 1, 0), (7, 11), (8, 12), (15, 239), (16, 240), (39, 299), (23, 19), (24, 20)]
    rs += [(int(rng.integers(0, o)), int(rng.integers(0, v))) for _ in range(37)]
    ij = [(0, 0), (o - 1, o - 1), (0, o - 1), (o - 1, 0), (1, 23), (1, 24)] + \
         [(int(rng.integers(0, o)), int(rng.integers(0, o))) for _ in range(26)]
    rs, ij = np.array(rs, dtype=np.int32), np.array(ij, dtype=np.int32)
    ref = oracle.ladder_xy_sampled(X, Y, t, rs, ij)
    smp = got[ij[None, :, 0], ij[None, :, 1], rs[:, None, 0], rs[:, None, 1]]
    assert float(np.max(np.abs(smp - ref)) / scale) <= TOL
    # projection: sum_rs p_r q_s out[i,j,r,s] = sum_cd t_ij^cd W_cd,  W = sum_P (p^T X_P)^T (q^T Y_P)   (linearity of Eq. 9)
    p, q = rng.standard_normal(o), rng.standard_normal(v)
    W = np.einsum("Pc,Pd->cd", np.einsum("r,Prc->Pc", p, X), np.einsum("s,Psd->Pd", q, Y))
    proj_ref = np.einsum("ijcd,cd->ij", t, W)
    proj = torch.einsum("r,s,ijrs->ij", torch.from_numpy(p), torch.from_numpy(q), torch.from_numpy(got)).numpy()
    assert float(np.max(np.abs(proj - proj_ref)) / np.max(np.abs(proj_ref))) <= 1e-10
