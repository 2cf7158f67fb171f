"""B200-native Cholesky vvvv ladder: R[i,j,a,b] += sum_cd (sum_P L[P,a,c] L[P,b,d]) t[i,j,c,d].

(arXiv:2310.04559, Eq. 6.)  The product is the C-ABI shared library `libcc_ladder.so` (include/cc_ladder.h,
csrc/*.cu, hand-written sm_100a kernels); this package is its ctypes binding plus the in-tree build step.
"""
from .binding import *  # noqa: F401,F403
from .binding import (CCLadderError, cc_ladder, cc_ladder_destroy, cc_ladder_get_info,  # noqa: F401
                      cc_ladder_get_option, cc_ladder_host, cc_ladder_plan, cc_ladder_set_option,
                      cc_ladder_set_workspace, cc_ladder_version, cc_ladder_workspace_bytes, library_path,
                      status_string)
