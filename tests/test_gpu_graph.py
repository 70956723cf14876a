"""-m gpu: the CUDA-graph replay of one apply (ppl_plan_set_graph, include/ppl.h) against plain launches and the oracle.

The graph holds the same kernels with the same arguments in the same order, so the result must be bit-identical
to the plain-launch path; replays on an unchanged key, re-captures on a changed key (pointers, options, symmetry
mode), launches into a non-default stream and a caller who captures the apply into a graph of their own are covered.
"""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11
SHAPES = [(5, 20, 60), (4, 37, 19), (5, 53, 232), (6, 64, 48)]
SYMS = [P.PPL_SYM_FULL, P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR, P.PPL_SYM_NONE]


def _inputs(o, v, x, seed=3):
    return I.make_L(v, x, seed, symmetric=True), I.make_t2(o, v, seed, symmetric=True), I.make_t2(o, v, seed + 1, symmetric=False)


def _apply(plan, L, t2, R0, n=1, stream=None, **ex):
    import torch

    Ld, td, Rd = (torch.from_numpy(a).cuda() for a in (L, t2, R0))
    for _ in range(n):
        if ex:
            plan.apply_ex(Ld, td, Rd, stream=stream, **ex)
        else:
            plan.apply(Ld, td, Rd, stream)
    torch.cuda.synchronize()
    return Rd.cpu().numpy()


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("sym", SYMS)
def test_graph_equals_plain_launches_bit_for_bit(shape, sym):
    o, v, x = shape
    L, t2, R0 = _inputs(o, v, x)
    want = oracle.full(L, t2, R0.copy())
    got = {}
    for mode in (0, 1):
        with P.Plan(o, v, x, 0) as plan:
            if sym == P.PPL_SYM_FULL and not plan.info()["full_available"]:
                pytest.skip("no PPL_SYM_FULL buffers for this shape")
            plan.set_symmetry(sym)
            plan.set_graph(mode)
            got[mode] = _apply(plan, L, t2, R0)
    assert relerr(got[1], want) <= TOL
    assert np.array_equal(got[0], got[1])


@pytest.mark.parametrize("sym", [P.PPL_SYM_FULL, P.PPL_SYM_PAIR_SA])
def test_graph_replays_accumulate(sym):
    """Three applies on the same buffers: one capture, two replays; R = R0 + 3 term."""
    o, v, x = 5, 53, 40
    L, t2, R0 = _inputs(o, v, x, seed=5)
    term = oracle.full(L, t2, np.zeros_like(R0))
    with P.Plan(o, v, x, 0) as plan:
        plan.set_symmetry(sym)
        plan.set_graph(1)
        got = _apply(plan, L, t2, R0, n=3)
    assert relerr(got, R0 + 3.0 * term) <= TOL


def test_graph_recaptures_on_new_key():
    """New R, new t2, new options and a new symmetry mode each invalidate the stored graph."""
    import torch

    o, v, x = 5, 20, 60
    L, t2a, R0 = _inputs(o, v, x, seed=7)
    t2b = I.make_t2(o, v, 8, symmetric=True)
    ta, tb = oracle.full(L, t2a, np.zeros_like(R0)), oracle.full(L, t2b, np.zeros_like(R0))
    Ld, tda, tdb = (torch.from_numpy(a).cuda() for a in (L, t2a, t2b))
    R1, R2 = torch.from_numpy(R0).cuda(), torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    with P.Plan(o, v, x, 0) as plan:
        plan.set_graph(1)
        plan.apply(Ld, tda, R1)                            # capture
        plan.apply(Ld, tda, R2)                            # new R
        plan.apply(Ld, tdb, R2)                            # new t2
        plan.apply_ex(Ld, tda, R2, alpha=2.0, beta=-1.0)   # new options: R2 = -(ta + tb) + 2 ta
        plan.apply_ex(Ld, tda, R2, alpha=2.0, beta=-1.0)   # replay:      R2 = -(ta - tb) + 2 ta
        plan.set_symmetry(P.PPL_SYM_PAIR)
        plan.apply(Ld, tdb, R1)                            # new mode, old pointers
        plan.set_graph(0)
        plan.apply(Ld, tdb, R1)                            # plain launches behind graph launches on the same stream
        torch.cuda.synchronize()
    assert relerr(R1.cpu().numpy(), R0 + ta + 2.0 * tb) <= TOL
    assert relerr(R2.cpu().numpy(), ta + tb) <= TOL


def test_graph_on_side_stream_and_auto_mode():
    import torch

    o, v, x = 5, 53, 232  # config 'small': below the auto threshold
    L, t2, R0 = _inputs(o, v, x, seed=9)
    want = oracle.full(L, t2, R0.copy())
    s = torch.cuda.Stream()
    with P.Plan(o, v, x, 0) as plan:  # default mode -1
        with torch.cuda.stream(s):
            got = _apply(plan, L, t2, R0, stream=s)
    assert relerr(got, want) <= TOL


@pytest.mark.parametrize("sym", [P.PPL_SYM_FULL, P.PPL_SYM_PAIR_SA])
def test_caller_captures_the_apply(sym):
    """A caller capturing `stream` gets the plain launches (side-stream forks and joins included) in their own graph."""
    import torch

    o, v, x = 5, 53, 40
    L, t2, R0 = _inputs(o, v, x, seed=11)
    term = oracle.full(L, t2, np.zeros_like(R0))
    Ld, td, Rd = (torch.from_numpy(a).cuda() for a in (L, t2, R0))
    with P.Plan(o, v, x, 0) as plan:
        plan.set_symmetry(sym)
        plan.apply(Ld, td, Rd)  # warm: lazy allocations happen outside the capture
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            plan.apply(Ld, td, Rd, torch.cuda.current_stream())
        g.replay()
        g.replay()
        torch.cuda.synchronize()
    assert relerr(Rd.cpu().numpy(), R0 + 3.0 * term) <= TOL


@pytest.mark.parametrize("sym", SYMS)
def test_graph_paper_layouts_alpha_beta(sym):
    """'icjd' -> 'iajb' with alpha / beta under the graph: the un-packed modes allocate their permuted t2 lazily,
    inside the (relaxed-mode) capture."""
    o, v, x = 4, 38, 19
    L, t2, R0 = _inputs(o, v, x, seed=13)
    tl = np.ascontiguousarray(t2.transpose(0, 2, 1, 3))
    Rl = np.ascontiguousarray(R0.transpose(0, 2, 1, 3))
    want = oracle.full_ex(L, tl, Rl.copy(), "iajb", "iajb", -0.75, 0.5)
    got = {}
    for mode in (0, 1):
        with P.Plan(o, v, x, 0) as plan:
            if sym == P.PPL_SYM_FULL and not plan.info()["full_available"]:
                pytest.skip("no PPL_SYM_FULL buffers for this shape")
            plan.set_symmetry(sym)
            plan.set_graph(mode)
            got[mode] = _apply(plan, L, tl, Rl, t2_layout="iajb", r_layout="iajb", alpha=-0.75, beta=0.5)
    assert relerr(got[1], want) <= TOL
    assert np.array_equal(got[0], got[1])
