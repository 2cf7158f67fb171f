"""ctypes front end of the CPU oracle (oracle/ladder_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
``--impl reference`` legs.  The product package (paper_2310_04559_b200) never imports this module and this
module never imports the product package.  Argument marshalling only -- every number comes out of the C file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ladder_oracle.c")
_LIB = os.path.join(_HERE, "libladder_oracle.so")

_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp (no -ffast-math) -> oracle/libladder_oracle.so.  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        c_int = ctypes.c_int
        lib.oracle_num_threads.restype = c_int
        lib.oracle_set_num_threads.argtypes = [c_int]
        lib.oracle_set_num_threads.restype = None
        for name in ("oracle_ladder_full", "oracle_ladder_brute", "oracle_ladder_split", "oracle_ladder_exchange",
                     "oracle_ladder_symm"):
            f = getattr(lib, name)
            f.argtypes = [c_int, c_int, c_int, _dp, _dp, _dp]
            f.restype = c_int
        lib.oracle_ladder_sampled.argtypes = [c_int, c_int, c_int, _dp, _dp, c_int, _ip, c_int, _ip, _dp]
        lib.oracle_ladder_sampled.restype = c_int
        lib.oracle_ladder_xy.argtypes = [c_int, c_int, c_int, c_int, c_int, _dp, _dp, _dp, _dp]
        lib.oracle_ladder_xy.restype = c_int
        lib.oracle_ladder_xy_sampled.argtypes = [c_int, c_int, c_int, c_int, c_int, _dp, _dp, _dp, c_int, _ip, c_int,
                                                 _ip, _dp]
        lib.oracle_ladder_xy_sampled.restype = c_int
        lib.oracle_eri.argtypes = [c_int, c_int, _dp, _dp]
        lib.oracle_eri.restype = c_int
        lib.oracle_ladder_dense.argtypes = [c_int, c_int, _dp, _dp, _dp]
        lib.oracle_ladder_dense.restype = c_int
        lib.oracle_pack_tpm.argtypes = [c_int, c_int, _dp, _dp, _dp]
        lib.oracle_pack_tpm.restype = c_int
        lib.oracle_project_occ.argtypes = [c_int, c_int, c_int, _dp, _dp, _dp, _dp, _dp]
        lib.oracle_project_occ.restype = c_int
        lib.oracle_project_virt.argtypes = [c_int, c_int, c_int, _dp, _dp, _dp, _dp, _dp]
        lib.oracle_project_virt.restype = c_int
        _lib = lib
    return _lib


def _d(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _i(a: np.ndarray):
    assert a.dtype == np.int32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_ip)


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"{what} failed with status {rc}")


def _sizes(L: np.ndarray, t: np.ndarray):
    x, v, v2 = L.shape
    o, o2, v3, v4 = t.shape
    assert v == v2 == v3 == v4 and o == o2, (L.shape, t.shape)
    return o, v, x


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def ladder_full(L, t, R0=None) -> np.ndarray:
    """R0 + ladder(L, t); R0 defaults to zeros.  Returns a new array (o,o,v,v)."""
    L, t = _c(L), _c(t)
    o, v, x = _sizes(L, t)
    R = np.zeros((o, o, v, v)) if R0 is None else _c(R0).copy()
    _check(_load().oracle_ladder_full(o, v, x, _d(L), _d(t), _d(R)), "oracle_ladder_full")
    return R


def ladder_brute(L, t, R0=None) -> np.ndarray:
    L, t = _c(L), _c(t)
    o, v, x = _sizes(L, t)
    R = np.zeros((o, o, v, v)) if R0 is None else _c(R0).copy()
    _check(_load().oracle_ladder_brute(o, v, x, _d(L), _d(t), _d(R)), "oracle_ladder_brute")
    return R


def ladder_exchange(L, t, R0=None) -> np.ndarray:
    """R0 + exchange(L, t): E[i,j,a,b] = sum_cd (sum_P L[P,a,d] L[P,b,c]) t[i,j,c,d]  (Eq. 7)."""
    L, t = _c(L), _c(t)
    o, v, x = _sizes(L, t)
    R = np.zeros((o, o, v, v)) if R0 is None else _c(R0).copy()
    _check(_load().oracle_ladder_exchange(o, v, x, _d(L), _d(t), _d(R)), "oracle_ladder_exchange")
    return R


def ladder_symm(L, t, R0=None) -> np.ndarray:
    """R0 + the 8-fold-symmetry evaluation (upper triangle of V[(ab),(cd)] used twice): equals
    ladder_full only when L[P,a,c] == L[P,c,a]."""
    L, t = _c(L), _c(t)
    o, v, x = _sizes(L, t)
    R = np.zeros((o, o, v, v)) if R0 is None else _c(R0).copy()
    _check(_load().oracle_ladder_symm(o, v, x, _d(L), _d(t), _d(R)), "oracle_ladder_symm")
    return R


def _xy_sizes(X, Y, t):
    x, nr, v = X.shape
    x2, ns, v2 = Y.shape
    o, o2, v3, v4 = t.shape
    assert x == x2 and v == v2 == v3 == v4 and o == o2, (X.shape, Y.shape, t.shape)
    return o, v, x, nr, ns


def ladder_xy(X, Y, t, out0=None) -> np.ndarray:
    """out0 + sum_cd (sum_P X[P,r,c] Y[P,s,d]) t[i,j,c,d] as out[i,j,r,s]  (Eqs. 8-9: "abcd,ecfd->efab")."""
    X, Y, t = _c(X), _c(Y), _c(t)
    o, v, x, nr, ns = _xy_sizes(X, Y, t)
    out = np.zeros((o, o, nr, ns)) if out0 is None else _c(out0).copy()
    _check(_load().oracle_ladder_xy(o, v, x, nr, ns, _d(X), _d(Y), _d(t), _d(out)), "oracle_ladder_xy")
    return out


def ladder_xy_sampled(X, Y, t, rs, ij) -> np.ndarray:
    """ladder_xy(X, Y, t)[i,j,r,s] at the listed pairs: rs (n_rs,2) and ij (n_ij,2) -> (n_rs, n_ij)."""
    X, Y, t = _c(X), _c(Y), _c(t)
    o, v, x, nr, ns = _xy_sizes(X, Y, t)
    rs = np.ascontiguousarray(rs, dtype=np.int32).reshape(-1, 2)
    ij = np.ascontiguousarray(ij, dtype=np.int32).reshape(-1, 2)
    res = np.zeros((rs.shape[0], ij.shape[0]))
    _check(_load().oracle_ladder_xy_sampled(o, v, x, nr, ns, _d(X), _d(Y), _d(t), rs.shape[0], _i(rs), ij.shape[0],
                                            _i(ij), _d(res)), "oracle_ladder_xy_sampled")
    return res


def ladder_split(L, t, R0=None) -> np.ndarray:
    L, t = _c(L), _c(t)
    o, v, x = _sizes(L, t)
    R = np.zeros((o, o, v, v)) if R0 is None else _c(R0).copy()
    _check(_load().oracle_ladder_split(o, v, x, _d(L), _d(t), _d(R)), "oracle_ladder_split")
    return R


def ladder_sampled(L, t, ab, ij) -> np.ndarray:
    """ladder(L,t)[i,j,a,b] (no R0) at the listed pairs: ab (n_ab,2) and ij (n_ij,2) -> (n_ab, n_ij)."""
    L, t = _c(L), _c(t)
    o, v, x = _sizes(L, t)
    ab = np.ascontiguousarray(ab, dtype=np.int32).reshape(-1, 2)
    ij = np.ascontiguousarray(ij, dtype=np.int32).reshape(-1, 2)
    out = np.zeros((ab.shape[0], ij.shape[0]))
    _check(_load().oracle_ladder_sampled(o, v, x, _d(L), _d(t), ab.shape[0], _i(ab), ij.shape[0], _i(ij),
                                         _d(out)), "oracle_ladder_sampled")
    return out


def eri(L) -> np.ndarray:
    """Explicit <ab|cd> = sum_P L[P,a,c] L[P,b,d] as V[a,b,c,d] (tiny sizes)."""
    L = _c(L)
    x, v, _ = L.shape
    V = np.zeros((v, v, v, v))
    _check(_load().oracle_eri(v, x, _d(L), _d(V)), "oracle_eri")
    return V


def ladder_dense(V, t, R0=None) -> np.ndarray:
    V, t = _c(V), _c(t)
    o, v = t.shape[0], t.shape[2]
    R = np.zeros((o, o, v, v)) if R0 is None else _c(R0).copy()
    _check(_load().oracle_ladder_dense(o, v, _d(V), _d(t), _d(R)), "oracle_ladder_dense")
    return R


def pack_tpm(t):
    t = _c(t)
    o, v = t.shape[0], t.shape[2]
    tp = np.zeros((o * o, v * (v + 1) // 2))
    tm = np.zeros((o * o, max(1, v * (v - 1) // 2)))
    _check(_load().oracle_pack_tpm(o, v, _d(t), _d(tp), _d(tm)), "oracle_pack_tpm")
    return tp, tm[:, : v * (v - 1) // 2]


def project_occ(L, t, u, w) -> np.ndarray:
    L, t, u, w = _c(L), _c(t), _c(u), _c(w)
    o, v, x = _sizes(L, t)
    out = np.zeros((v, v))
    _check(_load().oracle_project_occ(o, v, x, _d(L), _d(t), _d(u), _d(w), _d(out)), "oracle_project_occ")
    return out


def project_virt(L, t, p, q) -> np.ndarray:
    L, t, p, q = _c(L), _c(t), _c(p), _c(q)
    o, v, x = _sizes(L, t)
    out = np.zeros((o, o))
    _check(_load().oracle_project_virt(o, v, x, _d(L), _d(t), _d(p), _d(q), _d(out)), "oracle_project_virt")
    return out
