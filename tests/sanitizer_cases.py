"""Small ladders through the C ABI for `compute-sanitizer` (memcheck / racecheck / synccheck), SURVEY.md section 4 (T4).

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Every tile shape, odd nvirt (8-byte copies), ragged tiles in all four dimensions, a ragged last row chunk, several
tiles per CTA (ring phases wrap, the stage ring / Vs hand-over is exercised) and the split mode's CTA pairs.
Each case is also checked against the oracle, so a run under the sanitizer is a parity run too.
"""
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import ladder_inputs as gen   # noqa: E402
import oracle                 # noqa: E402
import paper_2310_04559_b200 as cl   # noqa: E402

# (nocc, nvirt, nchol, tile, split, exchange, layout)
CASES = [(3, 20, 21, 1, 0, 0, 0), (2, 33, 18, 1, 0, 0, 0), (3, 24, 40, 2, 0, 0, 0), (2, 40, 9, 3, 0, 0, 0),
         (9, 26, 70, 3, 0, 0, 0), (12, 18, 20, 1, 0, 0, 0), (3, 34, 20, 0, 1, 0, 0), (2, 17, 5, 0, 1, 0, 0),
         (3, 22, 19, 0, 0, 1, 0), (10, 21, 17, 3, 0, 0, 1), (3, 18, 20, 0, 0, 1, 1)]


def main():
    for (o, v, x, tile, split, exchange, layout) in CASES:
        L, t, R0 = gen.make_inputs(o, v, x, seed=1, symmetric=False, r0=True)
        ref = oracle.ladder_exchange(L, t, R0) if exchange else oracle.ladder_full(L, t, R0)
        if layout:      # the paper's [i,a,j,b] storage
            t, R0, ref = (np.ascontiguousarray(a.transpose(0, 2, 1, 3)) for a in (t, R0, ref))
        dL, dt, dR = (torch.from_numpy(a).cuda() for a in (L, t, R0))
        plan = cl.cc_ladder_plan(o, v, x)
        try:
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_TILE, tile)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_SPLIT, split)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_EXCHANGE, exchange)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_LAYOUT, layout)
            cl.cc_ladder_set_option(plan, cl.CC_LADDER_OPT_NUM_CTAS, 6)
            nb = cl.cc_ladder_workspace_bytes(plan)
            if nb:
                ws = torch.empty(nb, dtype=torch.uint8, device="cuda")
                cl.cc_ladder_set_workspace(plan, ws, nb)
            cl.cc_ladder(plan, dL, dt, dR, torch.cuda.current_stream())
            torch.cuda.synchronize()
        finally:
            cl.cc_ladder_destroy(plan)
        err = float(np.max(np.abs(dR.cpu().numpy() - ref)) / np.max(np.abs(ref)))
        print((o, v, x, tile, split, exchange, layout), "max rel err", err, flush=True)
        assert err <= 1e-11
    print("sanitizer cases ok")


if __name__ == "__main__":
    main()
