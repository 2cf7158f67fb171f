"""B200-native Cholesky vvvv ladder: R[i,j,a,b] += sum_cd (sum_P L[P,a,c] L[P,b,d]) t[i,j,c,d].

(arXiv:2310.04559, Eq. 6.)  The product is the C-ABI shared library `libcc_ladder.so` (include/cc_ladder.h,
csrc/*.cu, hand-written sm_100a kernels); this package is its ctypes binding plus the in-tree build step.

The binding is loaded on first use so that `paper_2310_04559_b200.build` can be imported (and run) in a clean
tree; any use of the API without the built library raises ImportError -- there is no fallback path.
"""
import importlib as _importlib


def __getattr__(name):
    if name.startswith("__"):
        raise AttributeError(name)
    if name == "build":
        return _importlib.import_module(".build", __name__)
    binding = _importlib.import_module(".binding", __name__)
    if name == "binding":
        return binding
    try:
        return getattr(binding, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None
