"""Thin ctypes binding of include/cc_ladder.h -- same names, argument marshalling only.

Every step of the hot path runs inside libcc_ladder.so (hand-written sm_100a kernels).  PyTorch appears only
as the owner of device memory and streams.  There is no CPU fallback: if the shared library is missing the
import fails, and without a B200 `cc_ladder_plan` raises.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcc_ladder.so")

# status codes / option keys (mirrors of include/cc_ladder.h)
CC_LADDER_OK = 0
CC_LADDER_EINVAL = -1
CC_LADDER_EARCH = -2
CC_LADDER_EWORKSPACE = -3
CC_LADDER_ECUDA = -4
CC_LADDER_ENOMEM = -5
CC_LADDER_ESCRATCH = -6
CC_LADDER_STATIC_SCRATCH_BYTES = 33554432

CC_LADDER_OPT_SPLIT = 1
CC_LADDER_OPT_ALGO = 2
CC_LADDER_OPT_NUM_CTAS = 3
CC_LADDER_OPT_SUPERTILE = 4
CC_LADDER_OPT_TILE = 5
CC_LADDER_OPT_EXCHANGE = 6
CC_LADDER_OPT_LAYOUT = 7
CC_LADDER_OPT_XY_ROWS_X = 8
CC_LADDER_OPT_XY_ROWS_Y = 9
CC_LADDER_OPT_HOST_BUDGET = 10
CC_LADDER_OPT_INDEX_BITS = 11
CC_LADDER_OPT_SYMM_L = 12
CC_LADDER_OPT_SCHEDULE = 13
CC_LADDER_OPT_HOST_BLOCK_ROWS = 14
CC_LADDER_SCHEDULE_DYNAMIC = 0
CC_LADDER_SCHEDULE_STATIC = 1
CC_LADDER_LAYOUT_IJAB = 0
CC_LADDER_LAYOUT_IAJB = 1

CC_LADDER_ALGO_FUSED = 0
CC_LADDER_ALGO_SIMPLE = 1

CC_LADDER_INFO_NUM_TILES = 1
CC_LADDER_INFO_KERNEL_LAUNCHES = 2
CC_LADDER_INFO_FLOPS_EXECUTED = 3
CC_LADDER_INFO_FLOPS_FULL = 4
CC_LADDER_INFO_NUM_SMS = 5
CC_LADDER_INFO_SMEM_BYTES = 6
CC_LADDER_INFO_TILE_SHAPE = 7
CC_LADDER_INFO_SUPERTILE_SHAPE = 8
CC_LADDER_INFO_INDEX_BITS = 9
CC_LADDER_INFO_HOST_CHUNKS = 10

EXPORTS = (
    "cc_ladder_plan", "cc_ladder_set_option", "cc_ladder_get_option", "cc_ladder_get_info",
    "cc_ladder_workspace_bytes", "cc_ladder_set_workspace", "cc_ladder", "cc_ladder_xy", "cc_ladder_host",
    "cc_ladder_fp64_peak", "cc_ladder_check_symmetric",
    "cc_ladder_split_static", "cc_ladder_split_static_bytes", "cc_ladder_static_scratch_bytes",
    "cc_ladder_split_static_error",
    "cc_ladder_destroy", "cc_ladder_status_string", "cc_ladder_last_cuda_error", "cc_ladder_version",
)


class CCLadderError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str = ""):
        self.status = status
        msg = f"{what}: status {status} ({status_string(status)})"
        if detail:
            msg += f" [{detail}]"
        super().__init__(msg)


def _load() -> ctypes.CDLL:
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2310_04559_b200.build` "
            "(nvcc, sm_100a).  There is no fallback path.")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i, ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong
    lib.cc_ladder_plan.argtypes = [ctypes.POINTER(vp), i, i, i]
    lib.cc_ladder_plan.restype = i
    lib.cc_ladder_set_option.argtypes = [vp, i, ll]
    lib.cc_ladder_set_option.restype = i
    lib.cc_ladder_get_option.argtypes = [vp, i, ctypes.POINTER(ll)]
    lib.cc_ladder_get_option.restype = i
    lib.cc_ladder_get_info.argtypes = [vp, i, ctypes.POINTER(ll)]
    lib.cc_ladder_get_info.restype = i
    lib.cc_ladder_workspace_bytes.argtypes = [vp]
    lib.cc_ladder_workspace_bytes.restype = ctypes.c_size_t
    lib.cc_ladder_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
    lib.cc_ladder_set_workspace.restype = i
    lib.cc_ladder.argtypes = [vp, vp, vp, vp, vp]
    lib.cc_ladder.restype = i
    lib.cc_ladder_xy.argtypes = [vp, vp, ll, ll, i, vp, ll, ll, i, vp, vp, vp]
    lib.cc_ladder_xy.restype = i
    lib.cc_ladder_fp64_peak.argtypes = [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), vp]
    lib.cc_ladder_fp64_peak.restype = i
    lib.cc_ladder_check_symmetric.argtypes = [vp, vp, ctypes.POINTER(ll), vp]
    lib.cc_ladder_check_symmetric.restype = i
    lib.cc_ladder_host.argtypes = [vp, vp, vp, vp]
    lib.cc_ladder_host.restype = i
    lib.cc_ladder_split_static.argtypes = [i, i, i, vp, vp, vp, vp]
    lib.cc_ladder_split_static.restype = i
    lib.cc_ladder_split_static_bytes.argtypes = [i, i]
    lib.cc_ladder_split_static_bytes.restype = ctypes.c_size_t
    lib.cc_ladder_static_scratch_bytes.argtypes = []
    lib.cc_ladder_static_scratch_bytes.restype = ctypes.c_size_t
    lib.cc_ladder_split_static_error.argtypes = []
    lib.cc_ladder_split_static_error.restype = ctypes.c_char_p
    lib.cc_ladder_destroy.argtypes = [vp]
    lib.cc_ladder_destroy.restype = i
    lib.cc_ladder_status_string.argtypes = [i]
    lib.cc_ladder_status_string.restype = ctypes.c_char_p
    lib.cc_ladder_last_cuda_error.argtypes = [vp]
    lib.cc_ladder_last_cuda_error.restype = ctypes.c_char_p
    lib.cc_ladder_version.argtypes = []
    lib.cc_ladder_version.restype = i
    return lib


_lib = _load()


def library_path() -> str:
    return _LIB_PATH


def status_string(status: int) -> str:
    return _lib.cc_ladder_status_string(int(status)).decode()


def cc_ladder_version() -> int:
    return int(_lib.cc_ladder_version())


def _check(rc: int, what: str, plan=None):
    if rc != CC_LADDER_OK:
        detail = _lib.cc_ladder_last_cuda_error(plan).decode() if plan else ""
        raise CCLadderError(rc, what, detail)


def _ptr(x) -> int:
    """Address of a torch tensor / numpy array / raw int, without looking at its contents."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if hasattr(x, "ctypes"):
        return int(x.ctypes.data)
    raise TypeError(f"cannot take the address of {type(x)!r}")


def cc_ladder_plan(nocc: int, nvirt: int, nchol: int) -> int:
    """-> opaque plan handle (int).  Raises CCLadderError (no device / not sm_100 / bad sizes)."""
    h = ctypes.c_void_p()
    _check(_lib.cc_ladder_plan(ctypes.byref(h), int(nocc), int(nvirt), int(nchol)), "cc_ladder_plan")
    return h.value


def cc_ladder_set_option(plan: int, key: int, value: int) -> None:
    _check(_lib.cc_ladder_set_option(plan, int(key), int(value)), "cc_ladder_set_option", plan)


def cc_ladder_get_option(plan: int, key: int) -> int:
    v = ctypes.c_longlong()
    _check(_lib.cc_ladder_get_option(plan, int(key), ctypes.byref(v)), "cc_ladder_get_option", plan)
    return int(v.value)


def cc_ladder_get_info(plan: int, key: int) -> int:
    v = ctypes.c_longlong()
    _check(_lib.cc_ladder_get_info(plan, int(key), ctypes.byref(v)), "cc_ladder_get_info", plan)
    return int(v.value)


def cc_ladder_workspace_bytes(plan: int) -> int:
    return int(_lib.cc_ladder_workspace_bytes(plan))


def cc_ladder_set_workspace(plan: int, dev_ptr, nbytes: int) -> None:
    _check(_lib.cc_ladder_set_workspace(plan, _ptr(dev_ptr), int(nbytes)), "cc_ladder_set_workspace", plan)


def cc_ladder(plan: int, L, t, R, stream=0) -> None:
    """R += ladder(L, t) on device buffers (torch CUDA tensors or raw device addresses); enqueues on `stream`."""
    if hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    _check(_lib.cc_ladder(plan, _ptr(L), _ptr(t), _ptr(R), int(stream)), "cc_ladder", plan)


def cc_ladder_xy(plan: int, X, x_pstride: int, x_rstride: int, nr: int, Y, y_pstride: int, y_rstride: int, ns: int,
                 t, out, stream=0) -> None:
    """out[i,j,r,s] += sum_cd (sum_P X[P,r,c] Y[P,s,d]) t[i,j,c,d] on device buffers (Eqs. 8-9)."""
    if hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    _check(_lib.cc_ladder_xy(plan, _ptr(X), int(x_pstride), int(x_rstride), int(nr), _ptr(Y), int(y_pstride),
                             int(y_rstride), int(ns), _ptr(t), _ptr(out), int(stream)), "cc_ladder_xy", plan)


def cc_ladder_check_symmetric(plan: int, L, stream=0) -> int:
    """-> number of (P, a < c) with L[P,a,c] != L[P,c,a] on the device array L (0: CC_LADDER_OPT_SYMM_L may be used)."""
    if hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    n = ctypes.c_longlong()
    _check(_lib.cc_ladder_check_symmetric(plan, _ptr(L), ctypes.byref(n), int(stream)), "cc_ladder_check_symmetric", plan)
    return int(n.value)


def cc_ladder_fp64_peak(stream=0):
    """-> (TFLOP/s, flop/clk/SM) of a register-only DMMA loop on the current device (the roofline denominator)."""
    if hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    a, b = ctypes.c_double(), ctypes.c_double()
    _check(_lib.cc_ladder_fp64_peak(ctypes.byref(a), ctypes.byref(b), int(stream)), "cc_ladder_fp64_peak")
    return float(a.value), float(b.value)


def cc_ladder_host(plan: int, L, t, R) -> None:
    """R += ladder(L, t) on HOST buffers (numpy arrays / pinned torch CPU tensors); blocking."""
    _check(_lib.cc_ladder_host(plan, _ptr(L), _ptr(t), _ptr(R)), "cc_ladder_host", plan)


def cc_ladder_split_static(nocc: int, nvirt: int, nchol: int, L, t, R, stream=0) -> None:
    """R += ladder(L, t) in split mode on device buffers, scratch in the library's static device array: no plan, no
    workspace, no allocation.  Raises CCLadderError(CC_LADDER_ESCRATCH) beyond cc_ladder_static_scratch_bytes()."""
    if hasattr(stream, "cuda_stream"):
        stream = stream.cuda_stream
    rc = _lib.cc_ladder_split_static(int(nocc), int(nvirt), int(nchol), _ptr(L), _ptr(t), _ptr(R), int(stream))
    if rc != CC_LADDER_OK:
        raise CCLadderError(rc, "cc_ladder_split_static", _lib.cc_ladder_split_static_error().decode())


def cc_ladder_split_static_bytes(nocc: int, nvirt: int) -> int:
    return int(_lib.cc_ladder_split_static_bytes(int(nocc), int(nvirt)))


def cc_ladder_static_scratch_bytes() -> int:
    return int(_lib.cc_ladder_static_scratch_bytes())


def cc_ladder_split_static_error() -> str:
    return _lib.cc_ladder_split_static_error().decode()


def cc_ladder_destroy(plan: int) -> None:
    _check(_lib.cc_ladder_destroy(plan), "cc_ladder_destroy")
