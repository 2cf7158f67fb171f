"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU, no CUDA code).

Every test here would fail for a plausible mistake in oracle/ladder_oracle.c (dropped term, wrong sign or
index, transposed operand).  Citations are PAPER.md lines.
"""
import os

import numpy as np
import pytest

import ladder_inputs as gen

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.default_rng(20231004)


def rel(a, b):
    return np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300)


def rand_problem(o, v, x, seed=0):
    r = np.random.default_rng(seed)
    return r.standard_normal((x, v, v)), r.standard_normal((o, o, v, v))


# ---------------------------------------------------------------------------------------- golden fixtures
def _records():
    out = []
    with open(os.path.join(GOLDEN, "hand_worked_2x2.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            Ls, ts, Rs = [np.array(p.split(), dtype=float).reshape(2, 2) for p in line.split("|")]
            out.append((Ls, ts, Rs))
    return out


@pytest.mark.parametrize("fn", ["ladder_full", "ladder_brute", "ladder_split", "ladder_sampled"])
def test_hand_worked_example(oracle, fn):
    """Eq. 6 worked by hand for o=1, v=2, x=1 (tests/golden/hand_worked_2x2.txt)."""
    recs = _records()
    assert len(recs) == 4
    for L2, t2, R2 in recs:
        L = L2.reshape(1, 2, 2)
        t = t2.reshape(1, 1, 2, 2)
        if fn == "ladder_sampled":
            ab = [(a, b) for a in range(2) for b in range(2)]
            got = oracle.ladder_sampled(L, t, ab, [(0, 0)]).reshape(2, 2)
        else:
            got = getattr(oracle, fn)(L, t).reshape(2, 2)
        assert np.array_equal(got, R2), (fn, got, R2)


def test_accumulates_into_R0(oracle):
    """Reading 1: '+='."""
    L, t = rand_problem(2, 3, 4, 1)
    R0 = RNG.standard_normal((2, 2, 3, 3))
    for f in (oracle.ladder_full, oracle.ladder_brute, oracle.ladder_split):
        assert rel(f(L, t, R0), R0 + f(L, t)) < 1e-15


# ---------------------------------------------------------------------------------------- P1 brute force
@pytest.mark.parametrize("o,v,x", [(3, 7, 5), (1, 4, 3), (2, 1, 3), (2, 5, 1), (1, 1, 1), (2, 9, 11)])
def test_full_equals_brute_force(oracle, o, v, x):
    """P1: the two-stage order equals the literal 7-index sum of Eq. 6."""
    L, t = rand_problem(o, v, x, seed=o * 100 + v * 10 + x)
    a = oracle.ladder_full(L, t)
    b = oracle.ladder_brute(L, t)
    assert rel(a, b) < 5e-15


def test_full_equals_brute_force_config0(oracle):
    o, v, x = gen.CONFIGS[0]
    L, t, _ = gen.make_inputs(o, v, x, 0)
    assert rel(oracle.ladder_full(L, t), oracle.ladder_brute(L, t)) < 5e-15


def test_sampled_equals_full(oracle):
    L, t = rand_problem(3, 6, 5, 7)
    full = oracle.ladder_full(L, t)
    ab = [(0, 0), (5, 5), (0, 5), (5, 0), (2, 3), (3, 2)]
    ij = [(0, 0), (2, 2), (0, 2), (2, 0), (1, 2)]
    got = oracle.ladder_sampled(L, t, ab, ij)
    for s, (a, b) in enumerate(ab):
        for r, (i, j) in enumerate(ij):
            assert got[s, r] == full[i, j, a, b]


# ---------------------------------------------------------------------------------------- P2 explicit (ac|bd)
def test_explicit_integrals(oracle):
    """P2: Eq. 5.  V[a,b,c,d] = <ab|cd>; Gram structure and its symmetries."""
    v, x = 5, 4
    L = RNG.standard_normal((x, v, v))
    V = oracle.eri(L)
    # independent construction
    ref = np.einsum("xac,xbd->abcd", L, L)
    assert rel(V, ref) < 1e-15
    # always true (any L): <ab|cd> = <ba|dc>
    assert rel(V, V.transpose(1, 0, 3, 2)) < 1e-15
    # the (ac),(bd) matrix is a Gram matrix: symmetric PSD
    G = V.transpose(0, 2, 1, 3).reshape(v * v, v * v)
    assert rel(G, G.T) < 1e-15
    assert np.linalg.eigvalsh(0.5 * (G + G.T)).min() > -1e-12 * np.abs(G).max()
    # for an unsymmetric L the a<->c swap is NOT a symmetry (guards against symmetrising by accident)
    assert rel(V, V.transpose(2, 1, 0, 3)) > 1e-3
    # 8-fold symmetry when L is symmetric in its orbital indices
    Ls = L + L.transpose(0, 2, 1)
    Vs = oracle.eri(Ls)
    for perm in [(2, 1, 0, 3), (0, 3, 2, 1), (2, 3, 0, 1), (1, 0, 3, 2)]:
        assert rel(Vs, Vs.transpose(perm)) < 1e-14


def test_dense_ladder_equals_cholesky_ladder(oracle):
    """Eq. 4 with the explicit integrals equals Eq. 6."""
    L, t = rand_problem(2, 5, 6, 3)
    V = oracle.eri(L)
    assert rel(oracle.ladder_dense(V, t), oracle.ladder_full(L, t)) < 5e-15


# ---------------------------------------------------------------------------------------- P3 closed forms
def test_nchol_one_closed_form(oracle):
    """P3: x = 1  =>  R_ij = L0 t_ij L0^T (north_star)."""
    o, v = 3, 6
    L, t = rand_problem(o, v, 1, 11)
    R = oracle.ladder_full(L, t)
    L0 = L[0]
    for i in range(o):
        for j in range(o):
            assert rel(R[i, j], L0 @ t[i, j] @ L0.T) < 1e-14


def test_separable_closed_form(oracle):
    """P6: L[P,a,c] = u_P w_a w_c  =>  R_ij^ab = (sum u^2) w_a w_b (w^T t_ij w)."""
    o, v, x = 2, 5, 7
    u, w = RNG.standard_normal(x), RNG.standard_normal(v)
    L = np.einsum("p,a,c->pac", u, w, w)
    t = RNG.standard_normal((o, o, v, v))
    R = oracle.ladder_full(L, t)
    ref = (u @ u) * np.einsum("a,b,ij->ijab", w, w, np.einsum("c,ijcd,d->ij", w, t, w))
    assert rel(R, ref) < 1e-13


def test_unit_vectors_pick_single_terms(oracle):
    """One non-zero in L and t: R has exactly the element Eq. 6 says (index placement)."""
    o, v, x = 2, 4, 3
    for (P, a, c, b, d, i, j) in [(1, 0, 3, 2, 1, 0, 1), (2, 3, 3, 0, 0, 1, 0), (0, 1, 2, 1, 3, 1, 1)]:
        L = np.zeros((x, v, v))
        L[P, a, c] = 2.0
        L[P, b, d] = 3.0 if (a, c) != (b, d) else 2.0
        t = np.zeros((o, o, v, v))
        t[i, j, c, d] = 5.0
        R = oracle.ladder_full(L, t)
        expect = np.zeros_like(R)
        # sum_{c'd'} L[a',c'] L[b',d'] t[c',d'] with only t[c,d] != 0
        LP = L[P]
        expect[i, j] = 5.0 * np.outer(LP[:, c], LP[:, d])
        assert np.array_equal(R, expect)


# ---------------------------------------------------------------------------------------- P4 symmetry
@pytest.mark.parametrize("symL", [True, False])
def test_pair_symmetry(oracle, symL):
    """P4: t_ij^ab = t_ji^ba  =>  R_ij^ab = R_ji^ba for ANY L (north_star)."""
    o, v, x = 3, 5, 4
    L = RNG.standard_normal((x, v, v))
    if symL:
        L = L + L.transpose(0, 2, 1)
    t = RNG.standard_normal((o, o, v, v))
    t = t + t.transpose(1, 0, 3, 2)
    R = oracle.ladder_full(L, t)
    assert rel(R, R.transpose(1, 0, 3, 2)) < 1e-14
    # and without the t symmetry it does not hold
    t2 = RNG.standard_normal((o, o, v, v))
    R2 = oracle.ladder_full(L, t2)
    assert rel(R2, R2.transpose(1, 0, 3, 2)) > 1e-3


def test_generated_inputs_have_the_symmetries():
    o, v, x = 4, 6, 5
    L, t, R0 = gen.make_inputs(o, v, x, 3)
    assert np.array_equal(L, L.transpose(0, 2, 1))
    assert np.array_equal(t, t.transpose(1, 0, 3, 2))
    assert not R0.any()
    L2, t2, R2 = gen.make_inputs(o, v, x, 3, symmetric=False, r0=True)
    assert not np.array_equal(L2, L2.transpose(0, 2, 1))
    assert not np.array_equal(t2, t2.transpose(1, 0, 3, 2))
    assert R2.any()
    # same seed -> same bits; other seed -> other bits
    La, ta, _ = gen.make_inputs(o, v, x, 3)
    assert np.array_equal(L, La) and np.array_equal(t, ta)
    Lb, _, _ = gen.make_inputs(o, v, x, 4)
    assert not np.array_equal(L, Lb)


# ---------------------------------------------------------------------------------------- P5 linearity
def test_linearity_bilinearity_stacking(oracle):
    o, v, x = 2, 4, 3
    L1, t1 = rand_problem(o, v, x, 21)
    L2, t2 = rand_problem(o, v, x + 2, 22)
    al, be, s = 0.7, -1.9, 1.5
    f = oracle.ladder_full
    assert rel(f(L1, al * t1 + be * t2[:, :, :, :]), al * f(L1, t1) + be * f(L1, t2)) < 1e-14
    assert rel(f(s * L1, t1), s * s * f(L1, t1)) < 1e-14
    assert rel(f(np.concatenate([L1, L2], axis=0), t1), f(L1, t1) + f(L2, t1)) < 1e-14
    # zero operands
    assert not f(np.zeros_like(L1), t1).any()
    assert not f(L1, np.zeros_like(t1)).any()


# ---------------------------------------------------------------------------------------- P7 projections
def test_projections_match_full(oracle):
    o, v, x = 3, 6, 5
    L, t = rand_problem(o, v, x, 31)
    R = oracle.ladder_full(L, t)
    u, w = RNG.standard_normal(o), RNG.standard_normal(o)
    p, q = RNG.standard_normal(v), RNG.standard_normal(v)
    assert rel(oracle.project_occ(L, t, u, w), np.einsum("i,j,ijab->ab", u, w, R)) < 1e-13
    assert rel(oracle.project_virt(L, t, p, q), np.einsum("a,b,ijab->ij", p, q, R)) < 1e-13


# ---------------------------------------------------------------------------------------- P8 library cross-check
@pytest.mark.parametrize("o,v,x", [(2, 6, 9), (3, 5, 2), (5, 20, 60)])
def test_numpy_einsum_crosscheck(oracle, o, v, x):
    """P8: NumPy einsum of the paper's string ('xac,xbd,icjd->iajb') under reading 8."""
    L, t = rand_problem(o, v, x, 41 + o)
    t_paper = np.ascontiguousarray(t.transpose(0, 2, 1, 3))                 # t_paper[i,c,j,d] = t[i,j,c,d]
    tnew_paper = np.einsum("xac,xbd,icjd->iajb", L, L, t_paper, optimize=True)
    R = oracle.ladder_full(L, t)
    assert rel(R, tnew_paper.transpose(0, 2, 1, 3)) < 1e-13


def test_paper_for_loop_tensordot_routine(oracle):
    """The paper's CPU routine restated with NumPy, against the oracle."""
    o, v, x = 3, 6, 4
    L, t = rand_problem(o, v, x, 51)
    L_0 = L_1 = L
    t_old = np.ascontiguousarray(t.transpose(0, 2, 1, 3))                  # [i,c,j,d]
    t_new = np.zeros((o, v, o, v))                                          # [i,a,j,b]
    for a in range(L_0.shape[1]):
        eri_bdc = np.tensordot(L_1, L_0[:, a, :], axes=([0, 0]))            # [b,d,c]
        t_new[:, a, :, :] += np.tensordot(t_old, eri_bdc, axes=([1, 3], [2, 1]))
    assert rel(oracle.ladder_full(L, t), t_new.transpose(0, 2, 1, 3)) < 1e-13


def test_paper_gpu_batch_routine(oracle):
    """The paper's batched GPU algorithm (reading 5: loops e > a > b) restated with NumPy."""
    o, v, x = 4, 7, 5
    L, t = rand_problem(o, v, x, 52)
    t_old = np.ascontiguousarray(t.transpose(0, 2, 1, 3))                  # [e,c,f,d]
    t_new = np.zeros((o, v, o, v))
    parts_c, parts_d = 3, 2
    e_chunks = np.array_split(np.arange(o), parts_d)
    a_chunks = np.array_split(np.arange(v), parts_c)
    for es in e_chunks:
        for as_ in a_chunks:
            for bs in a_chunks:
                chol_0, chol_1 = L[:, as_, :], L[:, bs, :]
                result_temp = np.tensordot(chol_0, chol_1, axes=(0, 0))            # acbd
                operand = t_old[es]
                result_temp_2 = np.tensordot(result_temp, operand, axes=([1, 3], [1, 3]))   # abef
                result_part = np.transpose(result_temp_2, axes=(2, 0, 3, 1))        # eafb
                t_new[np.ix_(es, as_, np.arange(o), bs)] = result_part
    assert rel(oracle.ladder_full(L, t), t_new.transpose(0, 2, 1, 3)) < 1e-13


# ---------------------------------------------------------------------------------------- split mode (reading 10)
@pytest.mark.parametrize("o,v,x", [(2, 5, 3), (3, 4, 6), (1, 1, 2), (2, 2, 1)])
def test_split_equals_full_for_unsymmetric_operands(oracle, o, v, x):
    L, t = rand_problem(o, v, x, 61 + v)
    assert rel(oracle.ladder_split(L, t), oracle.ladder_full(L, t)) < 1e-14


def test_pack_tpm(oracle):
    o, v = 2, 5
    t = RNG.standard_normal((o, o, v, v))
    tp, tm = oracle.pack_tpm(t)
    iu = np.triu_indices(v)          # row-major (c<=d) order
    il = np.triu_indices(v, 1)
    T = t.reshape(o * o, v, v)
    S = T + T.transpose(0, 2, 1)
    S[:, np.arange(v), np.arange(v)] = T[:, np.arange(v), np.arange(v)]
    A = T - T.transpose(0, 2, 1)
    assert np.array_equal(tp, S[:, iu[0], iu[1]])
    assert np.array_equal(tm, A[:, il[0], il[1]])


# ---------------------------------------------------------------------------------------- P9 Table 1
def test_table1_size_arithmetic():
    """P9: Table 1 from v = int(3K/4), o = K - v; needs 64-bit counts."""
    rows = []
    with open(os.path.join(GOLDEN, "table1_problem_sizes.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([int(s) for s in line.split()])
    assert [r[0] for r in rows] == [300, 400, 500]
    for K, n1, n2, n3 in rows:
        o, v, x = gen.PAPER_SHAPES[K]
        assert v == int(0.75 * K) and o == K - v and x == 5 * K
        assert o * o * v * v == n1 == n2
        assert o ** 3 * v == n3
    assert rows[-1][1] > 2 ** 31


def test_flop_formula():
    # totals 2 v^4 (x + o^2) at the five configs
    expect = {0: 2.72e7, 1: 3.32e11, 2: 4.21e13, 3: 2.43e14, 4: 8.62e14}
    for k, (o, v, x) in gen.CONFIGS.items():
        assert abs(gen.ladder_flops(o, v, x) / expect[k] - 1) < 5e-3


# ------------------------------------------------------------------------------------------ exchange variant (Eq. 7)
@pytest.mark.parametrize("o,v,x", [(1, 1, 1), (2, 3, 2), (3, 5, 4), (2, 7, 3)])
def test_exchange_equals_einsum_and_transposed_ladder(oracle, o, v, x):
    """PAPER.md:283-288 (Eq. 7): E_ij^ab = sum_xcd L^x_ad L^x_bc t_ij^cd, for operands with no symmetry at all.
    Three independent statements of it: the literal einsum, the ladder with (a,b) swapped on the output
    ((bd|ac) = (ac|bd)), and the ladder applied to t with c and d swapped."""
    L, t, R0 = gen.make_inputs(o, v, x, seed=40 + v, symmetric=False, r0=True)
    E = oracle.ladder_exchange(L, t, R0)
    ref = R0 + np.einsum("Pad,Pbc,ijcd->ijab", L, L, t)
    assert np.max(np.abs(E - ref)) <= 1e-13 * np.max(np.abs(ref))
    lad = oracle.ladder_full(L, t)
    assert np.max(np.abs((E - R0) - lad.transpose(0, 1, 3, 2))) <= 1e-13 * np.max(np.abs(lad))
    lad_t = oracle.ladder_full(L, np.ascontiguousarray(t.transpose(0, 1, 3, 2)))
    assert np.max(np.abs((E - R0) - lad_t)) <= 1e-13 * np.max(np.abs(lad_t))


def test_exchange_differs_from_ladder_and_has_a_closed_form(oracle):
    """A transposed or dropped index must change the answer: for unsymmetric t the exchange term is not the ladder;
    for separable L = u (x) w (x) z (unsymmetric in its orbital indices) E_ij^ab = (sum u^2) w_a w_b (z^T t_ij^T z)."""
    rng = np.random.default_rng(5)
    o, v, x = 2, 6, 3
    u, w, z = rng.standard_normal(x), rng.standard_normal(v), rng.standard_normal(v)
    L = np.einsum("P,a,c->Pac", u, w, z)
    t = rng.standard_normal((o, o, v, v))
    E = oracle.ladder_exchange(L, t)
    closed = np.sum(u * u) * np.einsum("a,b,ij->ijab", w, w, np.einsum("d,ijcd,c->ij", z, t, z))
    assert np.max(np.abs(E - closed)) <= 1e-13 * np.max(np.abs(closed))
    L2, t2, _ = gen.make_inputs(o, v, x, seed=3, symmetric=False)
    assert np.max(np.abs(oracle.ladder_exchange(L2, t2) - oracle.ladder_full(L2, t2))) > 1e-3


# ------------------------------------------------------------------------------------------ occupied-virtual family (Eqs. 8-9)
def _xy_problem(o, v, x, nr, ns, seed):
    r = np.random.default_rng(seed)
    return (r.standard_normal((x, nr, v)), r.standard_normal((x, ns, v)), r.standard_normal((o, o, v, v)))


def test_xy_hand_worked_example(oracle):
    """PAPER.md:288-298 worked by hand (tests/golden/hand_worked_xy.txt): out = X t Y^T for nchol = 1."""
    n = 0
    with open(os.path.join(GOLDEN, "hand_worked_xy.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            Xs, Ys, ts, outs = [np.array(p.split(), dtype=float) for p in line.split("|")]
            X, Y, t = Xs.reshape(1, 1, 2), Ys.reshape(1, 2, 2), ts.reshape(1, 1, 2, 2)
            assert np.array_equal(oracle.ladder_xy(X, Y, t).reshape(2), outs)
            got = oracle.ladder_xy_sampled(X, Y, t, [(0, 0), (0, 1)], [(0, 0)]).reshape(2)
            assert np.array_equal(got, outs)
            n += 1
    assert n == 3


@pytest.mark.parametrize("o,v,x,nr,ns", [(2, 5, 3, 2, 5), (3, 4, 2, 3, 3), (1, 1, 1, 1, 1), (2, 6, 4, 1, 7), (2, 3, 5, 4, 2)])
def test_xy_equals_the_papers_einsum_string(oracle, o, v, x, nr, ns):
    """The paper's recipe, literally: "abcd,ecfd->efab" with "abcd" replaced by "xac,xbd", on
    explicit integrals and on the paper's own t storage t[e,c,f,d]; plus accumulation into a non-zero out0."""
    X, Y, t = _xy_problem(o, v, x, nr, ns, 100 + nr * 7 + ns)
    out0 = np.random.default_rng(3).standard_normal((o, o, nr, ns))
    V = np.einsum("xac,xbd->abcd", X, Y)                         # <ab|cd> with a in X's rows, b in Y's rows
    t_paper = np.ascontiguousarray(t.transpose(0, 2, 1, 3))      # t[e,c,f,d]
    ref = np.einsum("abcd,ecfd->efab", V, t_paper)
    got = oracle.ladder_xy(X, Y, t, out0)
    assert rel(got - out0, ref) < 1e-13
    assert rel(oracle.ladder_xy(X, Y, t), ref) < 1e-14


def test_xy_is_eq8_and_eq9(oracle):
    """Eq. 9: t~_ijbk = sum_xcd L_bd L_kc t_ij^cd -> out[i,j,k,b] with X = L_ov, Y = L_vv;
    Eq. 8: t~_ijkl = sum_xcd L_kc L_ld t_ij^cd -> out[i,j,k,l] with X = Y = L_ov.  Literal loops."""
    o, v, x = 2, 3, 2
    r = np.random.default_rng(9)
    Lov, Lvv, t = r.standard_normal((x, o, v)), r.standard_normal((x, v, v)), r.standard_normal((o, o, v, v))
    e9 = np.zeros((o, o, o, v))
    e8 = np.zeros((o, o, o, o))
    for i in range(o):
        for j in range(o):
            for P in range(x):
                for c in range(v):
                    for d in range(v):
                        for k in range(o):
                            for b in range(v):
                                e9[i, j, k, b] += Lvv[P, b, d] * Lov[P, k, c] * t[i, j, c, d]
                            for l in range(o):
                                e8[i, j, k, l] += Lov[P, k, c] * Lov[P, l, d] * t[i, j, c, d]
    assert rel(oracle.ladder_xy(Lov, Lvv, t), e9) < 1e-14
    assert rel(oracle.ladder_xy(Lov, Lov, t), e8) < 1e-14


def test_xy_reduces_to_the_ladder_and_slices_by_rows(oracle):
    """X = Y = L gives Eq. 6; rows of X (of Y) select rows r (columns s) of the result; a transposed t or swapped
    operands change it."""
    L, t = rand_problem(2, 6, 4, 17)
    full = oracle.ladder_full(L, t)
    assert rel(oracle.ladder_xy(L, L, t), full) < 1e-15
    rows, cols = [4, 0, 3], [5, 1]
    Xs, Ys = np.ascontiguousarray(L[:, rows, :]), np.ascontiguousarray(L[:, cols, :])
    sub = oracle.ladder_xy(Xs, Ys, t)
    assert rel(sub, full[:, :, rows][:, :, :, cols]) < 1e-15
    X, Y, t2 = _xy_problem(2, 4, 3, 4, 4, 23)
    a = oracle.ladder_xy(X, Y, t2)
    assert rel(oracle.ladder_xy(Y, X, t2), a) > 1e-2                                   # operands are not interchangeable
    assert rel(oracle.ladder_xy(X, Y, np.ascontiguousarray(t2.transpose(0, 1, 3, 2))), a) > 1e-2
    assert rel(oracle.ladder_xy(Y, X, np.ascontiguousarray(t2.transpose(0, 1, 3, 2))), a.transpose(0, 1, 3, 2)) < 1e-14


def test_xy_closed_forms_and_unit_placement(oracle):
    """x = 1: out_ij = X0 t_ij Y0^T; a single non-zero in X, Y and t lands exactly where Eqs. 8-9 say."""
    o, v, nr, ns = 2, 5, 3, 4
    X, Y, t = _xy_problem(o, v, 1, nr, ns, 31)
    ref = np.einsum("rc,ijcd,sd->ijrs", X[0], t, Y[0])
    assert rel(oracle.ladder_xy(X, Y, t), ref) < 1e-15
    X = np.zeros((2, nr, v)); Y = np.zeros((2, ns, v)); t = np.zeros((o, o, v, v))
    X[1, 2, 3] = 2.0; Y[1, 0, 4] = 3.0; t[1, 0, 3, 4] = 5.0
    out = oracle.ladder_xy(X, Y, t)
    assert out[1, 0, 2, 0] == 30.0 and np.count_nonzero(out) == 1
    Y[:] = 0.0; Y[0, 0, 4] = 3.0                                     # different Cholesky vector: no contribution
    assert np.count_nonzero(oracle.ladder_xy(X, Y, t)) == 0


def test_xy_sampled_equals_full(oracle):
    X, Y, t = _xy_problem(3, 5, 4, 2, 6, 41)
    full = oracle.ladder_xy(X, Y, t)
    rs = [(0, 0), (1, 5), (0, 5), (1, 0), (1, 3)]
    ij = [(0, 0), (2, 2), (0, 2), (2, 0), (1, 2)]
    got = oracle.ladder_xy_sampled(X, Y, t, rs, ij)
    for q, (r_, s_) in enumerate(rs):
        for p_, (i, j) in enumerate(ij):
            assert got[q, p_] == full[i, j, r_, s_]


def test_xy_output_sizes_are_table1(oracle):
    """Table 1, third row: the output of "abcd,ecfd->efab" has o^3 v elements (Eq. 9's shape)."""
    X, Y, t = _xy_problem(2, 3, 2, 2, 3, 1)
    assert oracle.ladder_xy(X, Y, t).size == 2 ** 3 * 3
    for K, (o, v, x) in gen.PAPER_SHAPES.items():
        n3 = {300: 94921875, 400: 300000000, 500: 732421875}[K]
        assert o * o * o * v == n3


# ------------------------------------------------------------------------------------------ 8-fold symmetry mode
@pytest.mark.parametrize("o,v,x", [(2, 4, 3), (1, 1, 2), (3, 5, 4), (2, 6, 1)])
def test_symm_equals_full_for_symmetric_L_only(oracle, o, v, x):
    """<ab|cd> = <cd|ab> holds iff L is symmetric in its orbital indices: the triangle-used-twice evaluation
    equals Eq. 6 for symmetric L (t without any symmetry, R0 non-zero) and differs for unsymmetric L."""
    r = np.random.default_rng(70 + v)
    L = r.standard_normal((x, v, v))
    Ls = L + L.transpose(0, 2, 1)
    t = r.standard_normal((o, o, v, v))
    R0 = r.standard_normal((o, o, v, v))
    assert rel(oracle.ladder_symm(Ls, t, R0), oracle.ladder_full(Ls, t, R0)) < 1e-14
    if v > 1:
        assert rel(oracle.ladder_symm(L, t), oracle.ladder_full(L, t)) > 1e-3


def test_symm_on_unsymmetric_L_is_the_mirrored_upper_triangle(oracle):
    """What the symmetric mode computes when its precondition is violated: the ladder of V'[(ab),(cd)] = V[min(ab,cd),
    max(ab,cd)] (explicit integrals from oracle_eri, mirrored in NumPy)."""
    o, v, x = 2, 4, 3
    r = np.random.default_rng(8)
    L, t = r.standard_normal((x, v, v)), r.standard_normal((o, o, v, v))
    V = oracle.eri(L).reshape(v * v, v * v)
    Vm = np.triu(V) + np.triu(V, 1).T
    ref = (t.reshape(o * o, v * v) @ Vm.T).reshape(o, o, v, v)
    assert rel(oracle.ladder_symm(L, t), ref) < 1e-14
    assert rel(oracle.ladder_dense(Vm.reshape(v, v, v, v), t), ref) < 1e-14
