"""Seeded synthetic inputs for the Cholesky vvvv ladder (shared by the oracle side and the CUDA side).

This module holds *none* of the ladder's arithmetic (Eq. 6): it only manufactures the
operands L, t and an optional non-zero R0, bit-identically for whoever asks, from a counter-based
generator defined here.  Both the CPU oracle (tests) and the CUDA library (tests, bench.py) are fed the
very same host arrays; nothing here imports `oracle/` or the CUDA package.

Recipe (BASELINE.json configs[0], readings 11-13 and 16 of DESIGN.md):

* ``L[P,a,c] = L[P,c,a] = g * exp(-3 P / nchol)`` with one draw ``g ~ N(0,1)`` per ``(P, a<=c)``;
* ``M[Q,i,a] ~ N(0, sigma=0.1)``, ``nQ = 60``; ``e_occ ~ U[-2,-0.5]``; ``e_virt ~ U[0.2,3]``;
* ``t[i,j,a,b] = (sum_Q M[Q,i,a] M[Q,j,b]) / (e_i + e_j - e_a - e_b)``, so ``t[i,j,a,b] == t[j,i,b,a]``
  holds *bitwise* (the numerator is explicitly symmetrised, the denominator is evaluated as
  ``(e_i+e_j)-(e_a+e_b)``).

The paper's own timing workloads are iid random arrays with ``nchol = 5K``; `paper_shaped`
gives those shapes with iid N(0,1) entries (no symmetry at all), which is also what the parity tests use to
make sure the library assumes neither symmetry.

Counter-based generator: ``bits(seed, stream, n) = mix64(key(seed, stream) + n * GOLDEN)`` with the
splitmix64 finaliser; uniforms take the top 53 bits; normals are Box-Muller on counters ``2n, 2n+1``.
Everything is evaluated on the host with NumPy (libm of the host only).
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "CONFIGS", "PAPER_SHAPES", "config_sizes", "ladder_flops", "uniform01", "normal01",
    "cholesky_vectors", "cholesky_block", "amplitudes", "noise", "make_inputs", "paper_shaped",
]

# BASELINE.json configs[k] -> (nocc, nvirt, nchol); seed == k.
CONFIGS = {
    0: (5, 20, 60),
    1: (20, 120, 400),
    2: (40, 300, 1000),
    3: (50, 420, 1400),
    4: (64, 520, 1800),
}

# PAPER.md:312 / Table 1: v = int(3K/4), o = K - v, x = 5K.
PAPER_SHAPES = {300: (75, 225, 1500), 400: (100, 300, 2000), 500: (125, 375, 2500)}

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_STREAM_MUL = np.uint64(0xD1B54A32D192ED03)

STREAM_L, STREAM_M, STREAM_EOCC, STREAM_EVIRT, STREAM_R0, STREAM_T_IID, STREAM_LOV = 1, 2, 3, 4, 5, 6, 7
NQ = 60


def config_sizes(k: int):
    return CONFIGS[int(k)]


def ladder_flops(nocc: int, nvirt: int, nchol: int) -> int:
    """Algorithmic flops of one full (non-split) evaluation: 2 v^4 (x + o^2)."""
    v2 = nvirt * nvirt
    return 2 * v2 * v2 * (nchol + nocc * nocc)


def _mix64(z: np.ndarray) -> np.ndarray:
    z = z.copy()
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def _key(seed: int, stream: int) -> np.uint64:
    with np.errstate(over="ignore"):
        s = _mix64(np.array([np.uint64(seed) + _GOLDEN], dtype=np.uint64))
        s ^= np.uint64(stream) * _STREAM_MUL
        return _mix64(s)[0]


def _bits(seed: int, stream: int, counters: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        return _mix64(_key(seed, stream) + counters.astype(np.uint64) * _GOLDEN)


def uniform01(seed: int, stream: int, counters: np.ndarray) -> np.ndarray:
    """U[0,1) with 53 random bits, one value per counter."""
    return (_bits(seed, stream, counters) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(seed: int, stream: int, counters: np.ndarray) -> np.ndarray:
    """N(0,1) by Box-Muller on counters (2n, 2n+1)."""
    c = counters.astype(np.uint64)
    two = np.uint64(2)
    with np.errstate(over="ignore"):
        b1 = _bits(seed, stream, c * two)
        b2 = _bits(seed, stream, c * two + np.uint64(1))
    u1 = ((b1 >> np.uint64(11)).astype(np.float64) + 1.0) * (1.0 / 9007199254740992.0)   # (0,1]
    u2 = (b2 >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)           # [0,1)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos((2.0 * np.pi) * u2)


def cholesky_vectors(seed: int, nvirt: int, nchol: int, symmetric: bool = True) -> np.ndarray:
    """L[P,a,c], shape (nchol, nvirt, nvirt), C-contiguous float64.

    symmetric=True: one N(0,1) draw per (P, a<=c), mirrored, times exp(-3P/nchol) (BASELINE.json).
    symmetric=False: an independent draw per (P,a,c), same decay (used to prove no symmetry is assumed).
    """
    v = int(nvirt)
    L = np.empty((nchol, v, v), dtype=np.float64)
    a = np.arange(v, dtype=np.uint64)
    lo = np.minimum(a[:, None], a[None, :])
    hi = np.maximum(a[:, None], a[None, :])
    if symmetric:
        within = lo * np.uint64(v) + hi          # canonical counter of the pair (min,max)
    else:
        within = a[:, None] * np.uint64(v) + a[None, :]
    vv = np.uint64(v * v)
    for P in range(nchol):
        g = normal01(seed, STREAM_L, np.uint64(P) * vv + within)
        L[P] = g * np.exp(-3.0 * P / nchol)
    return L


def cholesky_block(seed: int, nrows: int, nvirt: int, nchol: int) -> np.ndarray:
    """A rectangular block of Cholesky vectors, e.g. the occupied-virtual block L_ov[P,k,c] of PAPER.md:288-298
    (Eqs. 8-9): shape (nchol, nrows, nvirt), iid N(0,1) entries with the same decay exp(-3P/nchol) as `cholesky_vectors`
    (an off-diagonal orbital block has no symmetry of its own)."""
    n = int(nrows) * int(nvirt)
    B = np.empty((nchol, int(nrows), int(nvirt)), dtype=np.float64)
    within = np.arange(n, dtype=np.uint64)
    for P in range(nchol):
        g = normal01(seed, STREAM_LOV, np.uint64(P) * np.uint64(n) + within)
        B[P] = (g * np.exp(-3.0 * P / nchol)).reshape(nrows, nvirt)
    return B


def amplitudes(seed: int, nocc: int, nvirt: int) -> np.ndarray:
    """t[i,j,a,b] = g_iajb / (e_i+e_j-e_a-e_b), shape (o,o,v,v); t[i,j,a,b] == t[j,i,b,a] bitwise."""
    o, v = int(nocc), int(nvirt)
    M = 0.1 * normal01(seed, STREAM_M, np.arange(NQ * o * v, dtype=np.uint64)).reshape(NQ, o * v)
    e_occ = -2.0 + 1.5 * uniform01(seed, STREAM_EOCC, np.arange(o, dtype=np.uint64))
    e_virt = 0.2 + 2.8 * uniform01(seed, STREAM_EVIRT, np.arange(v, dtype=np.uint64))
    t = np.empty((o, o, v, v), dtype=np.float64)
    Mq = M.reshape(NQ, o, v)
    eab = e_virt[:, None] + e_virt[None, :]
    Mflat = Mq.reshape(NQ, o * v)
    for i in range(o):
        # g[a,(j,b)] = sum_Q M[Q,i,a] M[Q,j,b]
        g = (Mq[:, i, :].T @ Mflat).reshape(v, o, v).transpose(1, 0, 2)          # (j,a,b)
        den = (e_occ[i] + e_occ)[:, None, None] - eab[None, :, :]                 # (e_i+e_j)-(e_a+e_b)
        t[i] = g / den
    # Make t[i,j,a,b] == t[j,i,b,a] hold bitwise whatever the BLAS blocking did: the i<j half is kept,
    # the i>j half is its mirror, the i==j blocks are symmetrised in (a,b).
    for i in range(o):
        for j in range(i):
            t[i, j] = t[j, i].T
        d = t[i, i]
        t[i, i] = 0.5 * (d + d.T)
    return t


def noise(seed: int, stream: int, shape, scale: float = 1.0) -> np.ndarray:
    """iid N(0, scale) array of the given shape (used for R0 and for the unsymmetric test operands)."""
    n = int(np.prod(shape))
    out = np.empty(n, dtype=np.float64)
    step = 1 << 22
    for s in range(0, n, step):
        e = min(n, s + step)
        out[s:e] = normal01(seed, stream, np.arange(s, e, dtype=np.uint64))
    if scale != 1.0:
        out *= scale
    return out.reshape(shape)


def make_inputs(nocc: int, nvirt: int, nchol: int, seed: int, *, symmetric: bool = True, r0: bool = False):
    """(L, t, R0) for the BASELINE.json generators.  R0 is zeros unless r0=True (then seeded noise)."""
    L = cholesky_vectors(seed, nvirt, nchol, symmetric=symmetric)
    if symmetric:
        t = amplitudes(seed, nocc, nvirt)
    else:
        t = noise(seed, STREAM_T_IID, (nocc, nocc, nvirt, nvirt), 0.05)
    if r0:
        R0 = noise(seed, STREAM_R0, (nocc, nocc, nvirt, nvirt), 1.0)
    else:
        R0 = np.zeros((nocc, nocc, nvirt, nvirt), dtype=np.float64)
    return L, t, R0


def paper_shaped(K: int, seed: int):
    """iid N(0,1) operands with the paper's benchmark shapes: no symmetry."""
    o, v, x = PAPER_SHAPES[K]
    L = noise(seed, STREAM_L, (x, v, v), 1.0)
    t = noise(seed, STREAM_T_IID, (o, o, v, v), 1.0)
    return L, t
