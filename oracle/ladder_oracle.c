/*
 * ladder_oracle.c -- CPU oracle for the Cholesky particle-particle ladder of spin-free CCD/CCSD.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the slow, plain, obviously-correct statement of what the hot
 * path computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may build, load or call it.  It shares no code with the CUDA library (paper_2310_04559_b200/csrc):
 * no headers, no helpers, no tables.  Parity status: PINNED (tests/test_oracle_pins.py: brute force,
 * explicit (ac|bd), nchol = 1 closed form, separable closed form, symmetry, linearity/bilinearity,
 * projections, NumPy einsum cross-check, Table 1 size arithmetic; each later entry point lists its own pins).
 *
 * What it computes (Sec. 2 Eq. 6, with the Cholesky form of Eq. 5):
 *
 *     R[i,j,a,b] += sum_{c,d} ( sum_P L[P,a,c] * L[P,b,d] ) * t[i,j,c,d]
 *
 * Layouts (row-major, 0-based, IEEE binary64): L[P][a][c] (x*v*v), t[i][j][c][d] and R[i][j][a][b]
 * (o*o*v*v).  The paper stores t_new[i,a,j,b]; the mapping t_paper[i,c,j,d] = t[i,j,c,d],
 * t_new_paper[i,a,j,b] = R[i,j,a,b] is reading 8 of DESIGN.md.  "+=" is reading 1.
 *
 * The method reaches exactly this finite sum (the kernels only re-associate it), so the oracle is the
 * definition evaluated in the paper's own for-loop order: for each a (and b) build the
 * integral slab, then contract it with t.  All sums are accumulated in `long double` (x87 80-bit on the
 * x86 hosts this runs on), rounded to double once, so the oracle is the more exact side.
 * No BLAS, no blocking, no reordering beyond that.  OpenMP only distributes independent (a,b) pairs.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (never -ffast-math).  See build() in oracle/__init__.py.
 */
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double acc_t;

#define IDX3(P, a, c, v) (((size_t)(P) * (size_t)(v) + (size_t)(a)) * (size_t)(v) + (size_t)(c))
#define IDX4(i, j, a, b, o, v) \
    ((((size_t)(i) * (size_t)(o) + (size_t)(j)) * (size_t)(v) + (size_t)(a)) * (size_t)(v) + (size_t)(b))

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* Eq. 5 for one fixed (a,b):  V[c][d] = sum_P L[P,a,c] L[P,b,d]  (the integral <ab|cd>). */
static void eri_slab(int v, int x, const double *L, int a, int b, acc_t *V)
{
    size_t vv = (size_t)v * (size_t)v;
    for (size_t k = 0; k < vv; ++k) V[k] = 0.0L;
    for (int P = 0; P < x; ++P) {
        const double *La = L + IDX3(P, a, 0, v);
        const double *Lb = L + IDX3(P, b, 0, v);
        for (int c = 0; c < v; ++c) {
            acc_t lac = (acc_t)La[c];
            acc_t *Vc = V + (size_t)c * (size_t)v;
            for (int d = 0; d < v; ++d) Vc[d] += lac * (acc_t)Lb[d];
        }
    }
}

/* Eq. 4 / Eq. 6 for one fixed (a,b) and (i,j):  sum_{cd} <ab|cd> t_ij^cd. */
static acc_t contract_slab(int v, const acc_t *V, const double *tij)
{
    acc_t s = 0.0L;
    size_t vv = (size_t)v * (size_t)v;
    for (size_t k = 0; k < vv; ++k) s += V[k] * (acc_t)tij[k];
    return s;
}

/* Full evaluation, R += ladder(L, t).  Cost 2 v^4 (x + o^2).  PAPER.md:58 (Eq. 6), order of 107-114. */
int oracle_ladder_full(int o, int v, int x, const double *L, const double *t, double *R)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !R) return -1;
    size_t vv = (size_t)v * (size_t)v;
    int fail = 0;
#pragma omp parallel
    {
        acc_t *V = (acc_t *)malloc(vv * sizeof(acc_t));
        if (!V) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (long ab = 0; ab < (long)vv; ++ab) {
                int a = (int)(ab / v), b = (int)(ab % v);
                eri_slab(v, x, L, a, b, V);
                for (int i = 0; i < o; ++i)
                    for (int j = 0; j < o; ++j) {
                        acc_t s = contract_slab(v, V, t + IDX4(i, j, 0, 0, o, v));
                        R[IDX4(i, j, a, b, o, v)] += (double)s;
                    }
            }
            free(V);
        }
    }
    return fail ? -2 : 0;
}

/*
 * Exchange variant (Sec. 6.2 Eq. 7; the paper's recipe "abcd,edfc->eafb"):
 *
 *     E[i,j,a,b] += sum_{c,d} ( sum_P L[P,a,d] * L[P,b,c] ) * t[i,j,c,d]
 *
 * "Not present when working in a spin-free representation", benchmarked by the paper for
 * completeness; SURVEY.md 8(f) NEXT-2.  Written out literally in the same for-loop order as the ladder: for each
 * (a,b) the slab W[c][d] = sum_P L[P,a,d] L[P,b,c], then the contraction with t_ij.  Parity status: PINNED
 * (tests/test_oracle_pins.py: NumPy einsum "Pad,Pbc,ijcd->ijab", E[i,j,a,b] == ladder[i,j,b,a],
 * E(L, t) == ladder(L, t with c and d swapped), separable closed form).
 */
int oracle_ladder_exchange(int o, int v, int x, const double *L, const double *t, double *R)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !R) return -1;
    size_t vv = (size_t)v * (size_t)v;
    int fail = 0;
#pragma omp parallel
    {
        acc_t *W = (acc_t *)malloc(vv * sizeof(acc_t));
        if (!W) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (long ab = 0; ab < (long)vv; ++ab) {
                int a = (int)(ab / v), b = (int)(ab % v);
                for (size_t k = 0; k < vv; ++k) W[k] = 0.0L;
                for (int P = 0; P < x; ++P) {
                    const double *La = L + IDX3(P, a, 0, v);      /* L[P,a,d], d = 0..v-1 */
                    const double *Lb = L + IDX3(P, b, 0, v);      /* L[P,b,c], c = 0..v-1 */
                    for (int c = 0; c < v; ++c) {
                        acc_t lbc = (acc_t)Lb[c];
                        acc_t *Wc = W + (size_t)c * (size_t)v;
                        for (int d = 0; d < v; ++d) Wc[d] += (acc_t)La[d] * lbc;
                    }
                }
                for (int i = 0; i < o; ++i)
                    for (int j = 0; j < o; ++j) {
                        acc_t s = contract_slab(v, W, t + IDX4(i, j, 0, 0, o, v));
                        R[IDX4(i, j, a, b, o, v)] += (double)s;
                    }
            }
            free(W);
        }
    }
    return fail ? -2 : 0;
}

/*
 * The occupied-virtual family (Sec. 6.2 Eqs. 8-9; the paper's recipe "abcd,ecfd->efab" with
 * "abcd" = "xac,xbd").  One statement covers both equations:
 *
 *     out[i,j,r,s] += sum_{c,d} ( sum_P X[P,r,c] * Y[P,s,d] ) * t[i,j,c,d]
 *
 * X[P][r][c] (x * nr * v) and Y[P][s][d] (x * ns * v) are two independent blocks of Cholesky vectors whose
 * second orbital index is virtual; out[i][j][r][s] is o*o*nr*ns (the recipe's output order "efab").
 *   Eq. 9:  t~_ijbk = sum_xcd L_bd L_kc t_ij^cd   <=>  X = L_ov[P,k,c] (nr = o), Y = L_vv[P,b,d] (ns = v), out[i,j,k,b]
 *   Eq. 8:  t~_ijkl = sum_xcd L_kc L_ld t_ij^cd   <=>  X = Y = L_ov (nr = ns = o),                       out[i,j,k,l]
 *   Eq. 6:  the ladder itself                    <=>  X = Y = L_vv (nr = ns = v).
 * ("sum_{rcd}" in Eq. 8 is read as sum_{xcd}, reading 6; the output order is DESIGN.md reading 17.)
 * Written in the same for-loop order as the ladder: for each (r,s) the slab W[c][d], then the contraction with
 * t_ij.  Parity status: PINNED (tests/test_oracle_pins.py: the paper's einsum string on explicit integrals, Eqs. 8
 * and 9 as literal einsums, reduction to oracle_ladder_full for X = Y = L, row slicing, x = 1 closed form
 * X0 t_ij Y0^T, unit placement, hand-worked golden, Table 1's o^3 v integers).
 */
static void xy_slab(int v, int x, int nr, int ns, const double *X, const double *Y, int r, int s, acc_t *W)
{
    size_t vv = (size_t)v * (size_t)v;
    for (size_t k = 0; k < vv; ++k) W[k] = 0.0L;
    for (int P = 0; P < x; ++P) {
        const double *Xr = X + ((size_t)P * (size_t)nr + (size_t)r) * (size_t)v;   /* X[P,r,c], c = 0..v-1 */
        const double *Ys = Y + ((size_t)P * (size_t)ns + (size_t)s) * (size_t)v;   /* Y[P,s,d], d = 0..v-1 */
        for (int c = 0; c < v; ++c) {
            acc_t xrc = (acc_t)Xr[c];
            acc_t *Wc = W + (size_t)c * (size_t)v;
            for (int d = 0; d < v; ++d) Wc[d] += xrc * (acc_t)Ys[d];
        }
    }
}

int oracle_ladder_xy(int o, int v, int x, int nr, int ns, const double *X, const double *Y, const double *t,
                     double *out)
{
    if (o <= 0 || v <= 0 || x <= 0 || nr <= 0 || ns <= 0 || !X || !Y || !t || !out) return -1;
    size_t vv = (size_t)v * (size_t)v;
    int fail = 0;
#pragma omp parallel
    {
        acc_t *W = (acc_t *)malloc(vv * sizeof(acc_t));
        if (!W) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (long rs = 0; rs < (long)nr * (long)ns; ++rs) {
                int r = (int)(rs / ns), s = (int)(rs % ns);
                xy_slab(v, x, nr, ns, X, Y, r, s, W);
                for (int i = 0; i < o; ++i)
                    for (int j = 0; j < o; ++j) {
                        acc_t q = contract_slab(v, W, t + IDX4(i, j, 0, 0, o, v));
                        out[(((size_t)i * (size_t)o + (size_t)j) * (size_t)nr + (size_t)r) * (size_t)ns + (size_t)s] +=
                            (double)q;
                    }
            }
            free(W);
        }
    }
    return fail ? -2 : 0;
}

/* Same arithmetic at listed (r,s) x (i,j) pairs only (no out0): res[q*n_ij + p] for rs[2q], rs[2q+1] and ij[2p], ij[2p+1]. */
int oracle_ladder_xy_sampled(int o, int v, int x, int nr, int ns, const double *X, const double *Y, const double *t,
                             int n_rs, const int *rs, int n_ij, const int *ij, double *res)
{
    if (o <= 0 || v <= 0 || x <= 0 || nr <= 0 || ns <= 0 || !X || !Y || !t || !res || n_rs < 0 || n_ij < 0) return -1;
    for (int q = 0; q < n_rs; ++q)
        if (rs[2 * q] < 0 || rs[2 * q] >= nr || rs[2 * q + 1] < 0 || rs[2 * q + 1] >= ns) return -1;
    for (int p = 0; p < n_ij; ++p)
        if (ij[2 * p] < 0 || ij[2 * p] >= o || ij[2 * p + 1] < 0 || ij[2 * p + 1] >= o) return -1;
    size_t vv = (size_t)v * (size_t)v;
    int fail = 0;
#pragma omp parallel
    {
        acc_t *W = (acc_t *)malloc(vv * sizeof(acc_t));
        if (!W) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int q = 0; q < n_rs; ++q) {
                xy_slab(v, x, nr, ns, X, Y, rs[2 * q], rs[2 * q + 1], W);
                for (int p = 0; p < n_ij; ++p)
                    res[(size_t)q * (size_t)n_ij + (size_t)p] =
                        (double)contract_slab(v, W, t + IDX4(ij[2 * p], ij[2 * p + 1], 0, 0, o, v));
            }
            free(W);
        }
    }
    return fail ? -2 : 0;
}

/*
 * The 8-fold-symmetry evaluation (Sec. 2: "both Cholesky vectors ... are identical ... 8-fold
 * permutational symmetry").  When L[P,a,c] = L[P,c,a] the integrals obey
 * <ab|cd> = <cd|ab>, i.e. the matrix V[(ab),(cd)] is symmetric, so only its upper triangle (ab) <= (cd) (pairs
 * ordered as ab = a*v + b) is built and every off-diagonal element is used twice, step by step:
 *
 *     for (a,b) <= (c,d):   V = sum_P L[P,a,c] L[P,b,d]
 *                           R[i,j,a,b] += V * t[i,j,c,d]
 *                           R[i,j,c,d] += V * t[i,j,a,b]      if (a,b) != (c,d)
 *
 * It ASSUMES the symmetry: for a symmetric L it must equal oracle_ladder_full, for an unsymmetric L it must NOT
 * (it then evaluates the ladder of the symmetrised integral matrix V'[(ab),(cd)] = V[min, max]).  Parity status:
 * PINNED (tests/test_oracle_pins.py: == full for symmetric L with unsymmetric t, != full for unsymmetric L, and for
 * unsymmetric L == the dense ladder of the explicitly mirrored upper triangle of oracle_eri).  Tiny sizes (O(v^4 (x + o^2))
 * with a serial outer loop).
 */
int oracle_ladder_symm(int o, int v, int x, const double *L, const double *t, double *R)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !R) return -1;
    size_t vv = (size_t)v * (size_t)v, oo = (size_t)o * (size_t)o;
    acc_t *acc = (acc_t *)calloc(oo * vv, sizeof(acc_t));     /* long-double image of the ladder part of R */
    if (!acc) return -2;
    for (size_t ab = 0; ab < vv; ++ab) {
        int a = (int)(ab / (size_t)v), b = (int)(ab % (size_t)v);
        for (size_t cd = ab; cd < vv; ++cd) {
            int c = (int)(cd / (size_t)v), d = (int)(cd % (size_t)v);
            acc_t V = 0.0L;
            for (int P = 0; P < x; ++P) V += (acc_t)L[IDX3(P, a, c, v)] * (acc_t)L[IDX3(P, b, d, v)];
            for (size_t ij = 0; ij < oo; ++ij) {
                acc[ij * vv + ab] += V * (acc_t)t[ij * vv + cd];
                if (cd != ab) acc[ij * vv + cd] += V * (acc_t)t[ij * vv + ab];
            }
        }
    }
    for (size_t k = 0; k < oo * vv; ++k) R[k] += (double)acc[k];
    free(acc);
    return 0;
}

/* Sampled evaluation for sizes where the full one takes days: out[s*n_ij + r] = ladder value (without
 * any R0) at (a,b) = ab[2s], ab[2s+1] and (i,j) = ij[2r], ij[2r+1].  Same arithmetic as the full one. */
int oracle_ladder_sampled(int o, int v, int x, const double *L, const double *t,
                          int n_ab, const int *ab, int n_ij, const int *ij, double *out)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !out || n_ab < 0 || n_ij < 0) return -1;
    for (int s = 0; s < n_ab; ++s)
        if (ab[2 * s] < 0 || ab[2 * s] >= v || ab[2 * s + 1] < 0 || ab[2 * s + 1] >= v) return -1;
    for (int r = 0; r < n_ij; ++r)
        if (ij[2 * r] < 0 || ij[2 * r] >= o || ij[2 * r + 1] < 0 || ij[2 * r + 1] >= o) return -1;
    size_t vv = (size_t)v * (size_t)v;
    int fail = 0;
#pragma omp parallel
    {
        acc_t *V = (acc_t *)malloc(vv * sizeof(acc_t));
        if (!V) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int s = 0; s < n_ab; ++s) {
                eri_slab(v, x, L, ab[2 * s], ab[2 * s + 1], V);
                for (int r = 0; r < n_ij; ++r) {
                    acc_t q = contract_slab(v, V, t + IDX4(ij[2 * r], ij[2 * r + 1], 0, 0, o, v));
                    out[(size_t)s * (size_t)n_ij + (size_t)r] = (double)q;
                }
            }
            free(V);
        }
    }
    return fail ? -2 : 0;
}

/* Literal seven-index sum of Eq. 6 with no intermediate at all: o^2 v^4 x multiply-adds.  Tiny sizes. */
int oracle_ladder_brute(int o, int v, int x, const double *L, const double *t, double *R)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !R) return -1;
    for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j)
            for (int a = 0; a < v; ++a)
                for (int b = 0; b < v; ++b) {
                    acc_t s = 0.0L;
                    for (int c = 0; c < v; ++c)
                        for (int d = 0; d < v; ++d) {
                            acc_t tcd = (acc_t)t[IDX4(i, j, c, d, o, v)];
                            for (int P = 0; P < x; ++P)
                                s += (acc_t)L[IDX3(P, a, c, v)] * (acc_t)L[IDX3(P, b, d, v)] * tcd;
                        }
                    R[IDX4(i, j, a, b, o, v)] += (double)s;
                }
    return 0;
}

/* Explicit integral tensor of Eq. 5:  V[a][b][c][d] = <ab|cd> = sum_P L[P,a,c] L[P,b,d].
 * v^4 doubles -- tiny sizes only (this is the array the hot path must never materialise). */
int oracle_eri(int v, int x, const double *L, double *V)
{
    if (v <= 0 || x <= 0 || !L || !V) return -1;
    size_t vv = (size_t)v * (size_t)v;
    acc_t *slab = (acc_t *)malloc(vv * sizeof(acc_t));
    if (!slab) return -2;
    for (int a = 0; a < v; ++a)
        for (int b = 0; b < v; ++b) {
            eri_slab(v, x, L, a, b, slab);
            double *dst = V + ((size_t)a * (size_t)v + (size_t)b) * vv;
            for (size_t k = 0; k < vv; ++k) dst[k] = (double)slab[k];
        }
    free(slab);
    return 0;
}

/* Dense ladder of Eq. 4:  R[i,j,a,b] += sum_cd <ab|cd> t_ij^cd with V[a][b][c][d] given. */
int oracle_ladder_dense(int o, int v, const double *V, const double *t, double *R)
{
    if (o <= 0 || v <= 0 || !V || !t || !R) return -1;
    size_t vv = (size_t)v * (size_t)v;
    for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j)
            for (int a = 0; a < v; ++a)
                for (int b = 0; b < v; ++b) {
                    const double *Vab = V + ((size_t)a * (size_t)v + (size_t)b) * vv;
                    const double *tij = t + IDX4(i, j, 0, 0, o, v);
                    acc_t s = 0.0L;
                    for (size_t k = 0; k < vv; ++k) s += (acc_t)Vab[k] * (acc_t)tij[k];
                    R[IDX4(i, j, a, b, o, v)] += (double)s;
                }
    return 0;
}

/* Step a0 of the hot path (reading 10): symmetric / antisymmetric packing of the amplitudes,
 *   tp[ij][(c<=d)] = t[ij,c,d] + t[ij,d,c] (c<d),  = t[ij,c,c] (c==d);   tm[ij][(c<d)] = t[ij,c,d] - t[ij,d,c].
 * Pair index of (c<=d): c*v - c*(c-1)/2 + (d-c); of (c<d) within tm: c*(v-1) - c*(c-1)/2 + (d-c-1). */
int oracle_pack_tpm(int o, int v, const double *t, double *tp, double *tm)
{
    if (o <= 0 || v <= 0 || !t || !tp || !tm) return -1;
    size_t np = (size_t)v * (size_t)(v + 1) / 2, nm = (size_t)v * (size_t)(v - 1) / 2;
    for (size_t ij = 0; ij < (size_t)o * (size_t)o; ++ij) {
        const double *tij = t + ij * (size_t)v * (size_t)v;
        size_t kp = 0, km = 0;
        for (int c = 0; c < v; ++c)
            for (int d = c; d < v; ++d) {
                double tcd = tij[(size_t)c * v + d], tdc = tij[(size_t)d * v + c];
                if (c == d) {
                    tp[ij * np + kp++] = tcd;
                } else {
                    tp[ij * np + kp++] = tcd + tdc;
                    tm[ij * nm + km++] = tcd - tdc;
                }
            }
    }
    return 0;
}

/* The t+/t- split evaluation, step by step as in DESIGN.md reading 10 (not in the paper; north_star):
 *   V+-[ab,cd] = 1/2 [ (ac|bd) +- (ad|bc) ],  R+_ab = sum_{c<=d} V+ t+,  R-_ab = sum_{c<d} V- t-,
 *   R_ab += R+ + R-,  R_ba += R+ - R- (a<b),  R_aa += R+.
 * Must equal oracle_ladder_full for ANY L and t (pin in tests). */
int oracle_ladder_split(int o, int v, int x, const double *L, const double *t, double *R)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !R) return -1;
    size_t vv = (size_t)v * (size_t)v;
    acc_t *Vab = (acc_t *)malloc(vv * sizeof(acc_t));
    if (!Vab) return -2;
    for (int a = 0; a < v; ++a)
        for (int b = a; b < v; ++b) {
            eri_slab(v, x, L, a, b, Vab);           /* Vab[c][d] = (ac|bd); (ad|bc) = Vab[d][c] */
            for (int i = 0; i < o; ++i)
                for (int j = 0; j < o; ++j) {
                    const double *tij = t + IDX4(i, j, 0, 0, o, v);
                    acc_t rp = 0.0L, rm = 0.0L;
                    for (int c = 0; c < v; ++c) {
                        rp += Vab[(size_t)c * v + c] * (acc_t)tij[(size_t)c * v + c];
                        for (int d = c + 1; d < v; ++d) {
                            acc_t vcd = Vab[(size_t)c * v + d], vdc = Vab[(size_t)d * v + c];
                            acc_t tcd = (acc_t)tij[(size_t)c * v + d], tdc = (acc_t)tij[(size_t)d * v + c];
                            rp += 0.5L * (vcd + vdc) * (tcd + tdc);
                            rm += 0.5L * (vcd - vdc) * (tcd - tdc);
                        }
                    }
                    if (a == b) {
                        R[IDX4(i, j, a, a, o, v)] += (double)rp;
                    } else {
                        R[IDX4(i, j, a, b, o, v)] += (double)(rp + rm);
                        R[IDX4(i, j, b, a, o, v)] += (double)(rp - rm);
                    }
                }
        }
    free(Vab);
    return 0;
}

/* Whole-tensor projection over the occupied pair (pin P7a):
 *   out[a][b] = sum_ij u_i w_j ladder(L,t)[i,j,a,b] = sum_P ( L_P  Tt  L_P^T )[a][b],  Tt = sum_ij u_i w_j t_ij.
 * Cost O(o^2 v^2 + x v^3): evaluated through the right-hand side. */
int oracle_project_occ(int o, int v, int x, const double *L, const double *t,
                       const double *u, const double *w, double *out)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !u || !w || !out) return -1;
    size_t vv = (size_t)v * (size_t)v;
    acc_t *Tt = (acc_t *)calloc(vv, sizeof(acc_t));
    acc_t *acc = (acc_t *)calloc(vv, sizeof(acc_t));
    if (!Tt || !acc) { free(Tt); free(acc); return -2; }
    for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j) {
            acc_t f = (acc_t)u[i] * (acc_t)w[j];
            const double *tij = t + IDX4(i, j, 0, 0, o, v);
            for (size_t k = 0; k < vv; ++k) Tt[k] += f * (acc_t)tij[k];
        }
#pragma omp parallel
    {
        acc_t *W = (acc_t *)malloc(vv * sizeof(acc_t));
        acc_t *mine = (acc_t *)calloc(vv, sizeof(acc_t));
#pragma omp for schedule(dynamic, 1)
        for (int P = 0; P < x; ++P) {
            const double *LP = L + IDX3(P, 0, 0, v);
            /* W[a][d] = sum_c L_P[a][c] Tt[c][d] */
            for (size_t k = 0; k < vv; ++k) W[k] = 0.0L;
            for (int a = 0; a < v; ++a)
                for (int c = 0; c < v; ++c) {
                    acc_t l = (acc_t)LP[(size_t)a * v + c];
                    for (int d = 0; d < v; ++d) W[(size_t)a * v + d] += l * Tt[(size_t)c * v + d];
                }
            /* mine[a][b] += sum_d W[a][d] L_P[b][d] */
            for (int a = 0; a < v; ++a)
                for (int b = 0; b < v; ++b) {
                    acc_t s = 0.0L;
                    for (int d = 0; d < v; ++d) s += W[(size_t)a * v + d] * (acc_t)LP[(size_t)b * v + d];
                    mine[(size_t)a * v + b] += s;
                }
        }
#pragma omp critical
        for (size_t k = 0; k < vv; ++k) acc[k] += mine[k];
        free(W);
        free(mine);
    }
    for (size_t k = 0; k < vv; ++k) out[k] = (double)acc[k];
    free(Tt);
    free(acc);
    return 0;
}

/* Whole-tensor projection over the virtual pair (pin P7b):
 *   out[i][j] = sum_ab p_a q_b ladder(L,t)[i,j,a,b] = sum_cd t_ij^cd Wh[c][d],
 *   Wh[c][d] = sum_P (p^T L_P)[c] (q^T L_P)[d].   Cost O(x v^2 + o^2 v^2). */
int oracle_project_virt(int o, int v, int x, const double *L, const double *t,
                        const double *p, const double *q, double *out)
{
    if (o <= 0 || v <= 0 || x <= 0 || !L || !t || !p || !q || !out) return -1;
    size_t vv = (size_t)v * (size_t)v;
    acc_t *Wh = (acc_t *)calloc(vv, sizeof(acc_t));
    acc_t *pl = (acc_t *)malloc((size_t)v * sizeof(acc_t));
    acc_t *ql = (acc_t *)malloc((size_t)v * sizeof(acc_t));
    if (!Wh || !pl || !ql) { free(Wh); free(pl); free(ql); return -2; }
    for (int P = 0; P < x; ++P) {
        const double *LP = L + IDX3(P, 0, 0, v);
        for (int c = 0; c < v; ++c) { pl[c] = 0.0L; ql[c] = 0.0L; }
        for (int a = 0; a < v; ++a)
            for (int c = 0; c < v; ++c) {
                pl[c] += (acc_t)p[a] * (acc_t)LP[(size_t)a * v + c];
                ql[c] += (acc_t)q[a] * (acc_t)LP[(size_t)a * v + c];
            }
        for (int c = 0; c < v; ++c)
            for (int d = 0; d < v; ++d) Wh[(size_t)c * v + d] += pl[c] * ql[d];
    }
    for (int i = 0; i < o; ++i)
        for (int j = 0; j < o; ++j)
            out[(size_t)i * o + j] = (double)contract_slab(v, Wh, t + IDX4(i, j, 0, 0, o, v));
    free(Wh);
    free(pl);
    free(ql);
    return 0;
}
