"""One pass of every mode of the hot path on the two smallest BASELINE.json configs (tiny, small) plus two odd
shapes, each checked against the oracle -- the program `compute-sanitizer` is pointed at:

    compute-sanitizer --tool racecheck python tests/sanitizer_case.py     (one tool per gpurun call)
    compute-sanitizer --tool memcheck  python tests/sanitizer_case.py

Not collected by pytest (no test_ prefix); results are recorded in profiles/README.md.
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import paper_2603_20912_b200 as P  # noqa: E402
import ppl_inputs as I  # noqa: E402

SHAPES = [(5, 20, 60), (5, 53, 232), (4, 37, 19), (6, 64, 48)]


def main():
    n = 0
    for (o, v, x) in SHAPES:
        L = I.make_L(v, x, 1, symmetric=True)
        t2 = I.make_t2(o, v, 1, symmetric=True)
        want = oracle.full(L, t2, np.zeros((o, o, v, v)))
        Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
        for sym in (P.PPL_SYM_FULL, P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR, P.PPL_SYM_NONE):
            with P.Plan(o, v, x, 0) as plan:
                if sym == P.PPL_SYM_FULL and not plan.info()["full_available"]:
                    continue
                plan.set_symmetry(sym)
                plan.set_graph(0)
                Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
                plan.apply(Ld, td, Rd)
                torch.cuda.synchronize()
                err = float(np.abs(Rd.cpu().numpy() - want).max() / np.abs(want).max())
                print(f"({o},{v},{x}) sym {sym}: tiles {plan.info()['n_tiles']} err {err:.1e}")
                assert err <= 1e-11, err
                n += 1
    print(f"SANITIZER CASE OK ({n} applies)")


if __name__ == "__main__":
    main()
