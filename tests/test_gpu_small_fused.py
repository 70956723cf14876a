"""-m gpu: the one-kernel path of launch-bound shapes (csrc/ppl_kernels_small.cuh; nvirt <= 56, nocc <= 8: BASELINE.json's tiny
and small configs), as the product runs it, against the CPU oracle -- 1e-11 relative, exact integers bit for bit and
therefore bit-identical to the tiled path on such inputs."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import gpu_ladder, relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11
FUSED = {"no_small_fused": 0}
# every accumulator-block count NB = ceil(nvirt / 8) = 1..7, nvirt at / next to the block edges, odd and even, one-element
# cases, nchol below / at / above the 16-wide k tile and the 3-stage ring, nocc 1..8
SHAPES = [(1, 1, 1), (2, 1, 3), (1, 5, 1), (3, 7, 5), (2, 8, 16), (5, 9, 17), (4, 16, 33), (5, 20, 60), (3, 23, 48), (8, 24, 50),
          (6, 25, 7), (2, 32, 64), (7, 33, 20), (5, 40, 100), (3, 41, 31), (4, 48, 16), (5, 53, 232), (8, 55, 40), (2, 56, 90)]


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("sym", [None, P.PPL_SYM_NONE, P.PPL_SYM_PAIR])
def test_fused_path_parity(shape, sym):
    o, v, x = shape
    symmetric = sym != P.PPL_SYM_NONE
    L = I.make_L(v, x, 13, symmetric=False)          # the fused path never uses L's symmetry, in any mode
    t2 = I.make_t2(o, v, 13, symmetric=symmetric)
    R0 = I.make_t2(o, v, 14, symmetric=False)
    want = oracle.full(L, t2, R0.copy())
    got, info = gpu_ladder(L, t2, R0=R0.copy(), sym=sym, return_info=True, debug=FUSED)
    assert info["small_fused"] == 1 and info["launches_per_apply"] == 1 + (v & 1), info  # + the padded copy for odd nvirt
    assert relerr(got, want) <= TOL, info


@pytest.mark.parametrize("shape", [(5, 20, 60), (5, 53, 232), (3, 41, 31), (8, 24, 50), (2, 56, 90)])
def test_fused_path_exact_integers_equal_the_tiled_path_bit_for_bit(shape):
    o, v, x = shape
    L = I.make_L(v, x, 15, symmetric=True, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 15, symmetric=True, integer=True)
    want = oracle.full(L, t2)
    fused, info = gpu_ladder(L, t2, return_info=True, debug=FUSED)
    assert info["small_fused"] == 1
    assert np.array_equal(fused, want)
    for sym in (P.PPL_SYM_PAIR_SA, P.PPL_SYM_FULL, P.PPL_SYM_PAIR):
        tiled, info_t = gpu_ladder(L, t2, sym=sym, return_info=True, debug={"no_small_fused": 1})
        assert info_t["small_fused"] == 0 and info_t["launches_per_apply"] > 1
        assert np.array_equal(tiled, fused), sym


@pytest.mark.parametrize("t2_layout,r_layout", [("iajb", "iajb"), ("ijab", "iajb"), ("iajb", "ijab")])
def test_fused_path_layouts_alpha_beta_overwrite(t2_layout, r_layout):
    import torch

    o, v, x = 4, 37, 19
    L = I.make_L(v, x, 17, symmetric=False)
    t2 = I.make_t2(o, v, 17, symmetric=True)
    R0 = I.make_t2(o, v, 18, symmetric=False)
    to = lambda a, lay: np.ascontiguousarray(a if lay == "ijab" else a.transpose(0, 2, 1, 3))
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(to(t2, t2_layout)).cuda()
    with P.Plan(o, v, x, debug=FUSED) as plan:
        assert plan.info()["small_fused"] == 1
        for alpha, beta, start in ((-0.75, 0.5, R0), (2.0, 0.0, np.full_like(R0, np.nan))):
            want = oracle.full_ex(L, to(t2, t2_layout), to(np.nan_to_num(start), r_layout).copy(), t2_layout, r_layout, alpha, beta)
            Rd = torch.from_numpy(to(start, r_layout)).cuda()
            plan.apply_ex(Ld, td, Rd, t2_layout=t2_layout, r_layout=r_layout, alpha=alpha, beta=beta)
            torch.cuda.synchronize()
            assert relerr(Rd.cpu().numpy(), want) <= TOL, (alpha, beta)


def test_fused_path_zero_t2_repeat_and_which_shapes_take_it():
    import torch

    o, v, x = 5, 20, 60
    L, t2 = I.make_config("tiny", seed=0)
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    R0 = I.make_t2(o, v, 19, symmetric=False)
    with P.Plan(o, v, x, debug=FUSED) as plan:
        Rd = torch.from_numpy(R0.copy()).cuda()
        plan.apply(Ld, torch.zeros_like(td), Rd)     # t2 == 0: R bitwise unchanged (A15)
        torch.cuda.synchronize()
        assert np.array_equal(Rd.cpu().numpy(), R0)
        Rd.zero_()
        for _ in range(3):
            plan.apply(Ld, td, Rd)
        prof = plan.apply_profiled(Ld, td, Rd)
        torch.cuda.synchronize()
        assert relerr(Rd.cpu().numpy(), 4.0 * oracle.full(L, t2)) <= TOL
        assert prof["n_step0"] in (1, 2) and prof["n_step1"] == 0 and prof["total_ms"] > 0
    # the path is for launch-bound shapes only
    assert P.ppl_plan_dry(5, 53, 232, debug=FUSED)["small_fused"] == 1
    assert P.ppl_plan_dry(5, 57, 232, debug=FUSED)["small_fused"] == 0      # nvirt > 56: W_ab no longer fits the accumulators
    assert P.ppl_plan_dry(9, 40, 100, debug=FUSED)["small_fused"] == 0      # nocc > 8
    assert P.ppl_plan_dry(5, 53, 4000, debug=FUSED)["small_fused"] == 0     # not launch-bound any more
    assert P.ppl_plan_dry(5, 53, 232, debug={"no_small_fused": 1})["small_fused"] == 0


@pytest.mark.parametrize("shape", [(5, 20, 60), (5, 53, 232), (3, 41, 31), (1, 5, 1)])
def test_fused_path_checks_its_inputs_inside_the_same_launch(shape):
    """PPL_OPT_VERIFY_INPUTS = 1 on the one-kernel path: the first CTAs of the launch scan the inputs; a violation is reported
    by the next call on the plan, a clean apply by none -- over many back-to-back applies (the sequence word), and again
    after the mode no longer relies on the violated symmetry."""
    import torch

    o, v, x = shape
    L = I.make_L(v, x, 23, symmetric=True)
    t2 = I.make_t2(o, v, 23, symmetric=True)
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    bad_t = torch.from_numpy(I.make_t2(o, v, 24, symmetric=False)).cuda()
    bad_L = torch.from_numpy(I.make_L(v, x, 24, symmetric=False)).cuda()
    with P.Plan(o, v, x, debug=FUSED) as plan:
        info = plan.info()
        assert info["small_fused"] == 1
        Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
        for _ in range(20):
            plan.apply(Ld, td, Rd)
        assert plan.verify_status() == 0
        torch.cuda.synchronize()
        assert relerr(Rd.cpu().numpy(), 20.0 * oracle.full(L, t2)) <= TOL
        if o > 1 or v > 1:  # (a 1 x 1 x 1 x 1 t2 is pair-symmetric whatever it holds)
            plan.apply(Ld, bad_t, Rd)
            with pytest.raises(P.PplError) as e:  # the next call reports it if the check has finished by then, else the one
                plan.apply(Ld, td, Rd)            # after: a call never waits for the check of the apply just before it
                plan.apply(Ld, td, Rd)
            assert e.value.code == P.PPL_ERR_PRECONDITION
            plan.verify_status()                 # (drains a clean check the first of the two calls may have queued)
            plan.apply(Ld, td, Rd)               # cleared: a clean apply goes through again
            assert plan.verify_status() == 0
            plan.apply(Ld, bad_t, Rd)            # and a device that has finished reports at the very next call
            torch.cuda.synchronize()
            with pytest.raises(P.PplError) as e:
                plan.apply(Ld, td, Rd)
            assert e.value.code == P.PPL_ERR_PRECONDITION
        # L is not verified on this path (it does not use L[P,a,c] = L[P,c,a]: the result is right for any L) ...
        Rd.zero_()
        plan.apply(bad_L, td, Rd)
        assert plan.verify_status() == 0
        torch.cuda.synchronize()
        assert relerr(Rd.cpu().numpy(), oracle.full(bad_L.cpu().numpy(), t2)) <= TOL
        if info["symmetry"] == P.PPL_SYM_FULL and v > 1:  # ... except by the synchronous mode, which checks what the mode names
            plan.set_verify(2)
            with pytest.raises(P.PplError) as e:
                plan.apply(bad_L, td, Rd)
            assert e.value.code == P.PPL_ERR_PRECONDITION
            plan.set_verify(1)
        plan.set_symmetry(P.PPL_SYM_NONE)        # nothing assumed: nothing checked, nothing reported
        plan.apply(bad_L, bad_t, Rd)
        assert plan.verify_status() == 0
        torch.cuda.synchronize()
