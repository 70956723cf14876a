"""-m gpu: seeded random sweep over shapes x symmetry mode x layouts x alpha/beta x workspace cap x graph mode,
each case against the oracle (1e-11 relative; exact-integer inputs bit for bit).  Shapes are drawn without knowledge
of the planner's tile grid: odd and even nvirt, nocc and nchol from 1 up, caps that force several tiles."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _case(seed):
    rng = np.random.default_rng(seed)
    while True:
        o, v, x = int(rng.integers(1, 22)), int(rng.integers(1, 120)), int(rng.integers(1, 60))
        if o * o * v ** 4 <= 3e9:
            break
    sym = int(rng.integers(0, 4))
    graph = int(rng.integers(0, 2))
    lay_t, lay_r = str(rng.choice(["ijab", "iajb"])), str(rng.choice(["ijab", "iajb"]))
    integer = bool(rng.random() < 0.3)
    alpha, beta = (1.0, 1.0) if rng.random() < 0.4 else (float(rng.normal()), float(rng.choice([0.0, 1.0, -0.5])))
    if integer:
        alpha, beta = float(round(alpha)), float(round(beta))
    cap = 0
    if rng.random() < 0.5:
        cols = int(rng.integers(5, 80))
        cap = (3 * cols + 2 * o * o) * (v * v + 64) * 8 + 64 * o * o * cols * 8 + 8192
    seeds = [int(s) for s in rng.integers(1 << 30, size=3)]
    l_sym = bool(sym == P.PPL_SYM_FULL or rng.random() < 0.5)
    return o, v, x, sym, graph, lay_t, lay_r, integer, alpha, beta, cap, seeds, l_sym


@pytest.mark.parametrize("seed", range(48))
def test_random_case_against_oracle(seed):
    import torch

    o, v, x, sym, graph, lay_t, lay_r, integer, alpha, beta, cap, seeds, l_sym = _case(seed)
    L = I.make_L(v, x, seeds[0], symmetric=l_sym, integer=integer)
    t2 = I.make_t2(o, v, seeds[1], symmetric=(sym != P.PPL_SYM_NONE), integer=integer)
    R0 = I.make_t2(o, v, seeds[2], symmetric=False, integer=integer)
    tl = np.ascontiguousarray(t2 if lay_t == "ijab" else t2.transpose(0, 2, 1, 3))
    Rl = np.ascontiguousarray(R0 if lay_r == "ijab" else R0.transpose(0, 2, 1, 3))
    want = oracle.full_ex(L, tl, Rl.copy(), lay_t, lay_r, alpha, beta)
    try:
        plan = P.Plan(o, v, x, cap)
    except P.PplError:
        pytest.skip("workspace cap too small for this shape")
    with plan:
        info = plan.info()
        if sym == P.PPL_SYM_FULL and not info["full_available"]:
            pytest.skip("no PPL_SYM_FULL buffers under this cap")
        try:
            plan.set_symmetry(sym)
        except P.PplError:
            pytest.skip("mode not available under this cap")
        plan.set_graph(graph)
        Ld, td, Rd = (torch.from_numpy(a).cuda() for a in (L, tl, Rl))
        plan.apply_ex(Ld, td, Rd, t2_layout=lay_t, r_layout=lay_r, alpha=alpha, beta=beta)
        torch.cuda.synchronize()
        got = Rd.cpu().numpy()
    what = dict(o=o, v=v, x=x, sym=sym, graph=graph, t2=lay_t, r=lay_r, integer=integer, alpha=alpha, beta=beta, cap=cap, info=info)
    if integer:
        assert np.array_equal(got, want), what
    else:
        assert relerr(got, want) <= TOL, what
