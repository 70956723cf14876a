"""-m gpu: PPL_OPT_VERIFY_INPUTS -- the default plan relies on L[P,a,c] == L[P,c,a] and on pair-symmetric
t2; an apply on inputs that violate a precondition of the plan's mode must not pass silently (VERDICT r01 / ADVICE r01)."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import relerr

pytestmark = pytest.mark.gpu


def _dev(*arrays):
    import torch

    return [torch.from_numpy(a).cuda() for a in arrays]


@pytest.mark.parametrize("shape", [(3, 96, 8), (4, 53, 12), (3, 130, 5)])
def test_default_plan_reports_a_non_symmetric_L_from_the_next_call(shape):
    import torch

    o, v, x = shape
    Ls, Ln = I.make_L(v, x, 3, symmetric=True), I.make_L(v, x, 3, symmetric=False)
    t2 = I.make_t2(o, v, 3, symmetric=True)
    Lsd, Lnd, td = _dev(Ls, Ln, t2)
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    plan = P.Plan(o, v, x)
    assert plan.info()["symmetry"] == P.PPL_SYM_FULL
    plan.apply(Lsd, td, Rd)           # fine
    plan.apply(Lnd, td, Rd)           # queued; the violation is found by the check at its head
    with pytest.raises(P.PplError) as e:
        plan.apply(Lsd, td, Rd)       # ... and reported by the next call
    assert e.value.code == P.PPL_ERR_PRECONDITION
    # the error state is cleared by the report: the plan keeps working
    Rd.zero_()
    plan.apply(Lsd, td, Rd)
    assert plan.verify_status() == 0
    torch.cuda.synchronize()
    assert relerr(Rd.cpu().numpy(), oracle.full(Ls, t2)) <= 1e-11
    # ppl_plan_verify_status and ppl_destroy report it too
    plan.apply(Lnd, td, Rd)
    with pytest.raises(P.PplError) as e:
        plan.verify_status()
    assert e.value.code == P.PPL_ERR_PRECONDITION
    plan.apply(Lnd, td, Rd)
    with pytest.raises(P.PplError) as e:
        plan.destroy()
    assert e.value.code == P.PPL_ERR_PRECONDITION


def test_synchronous_mode_leaves_R_untouched_and_t2_is_checked_in_every_symmetric_mode():
    import torch

    o, v, x = 4, 64, 10
    Ls = I.make_L(v, x, 5, symmetric=True)
    ts, tn = I.make_t2(o, v, 5, symmetric=True), I.make_t2(o, v, 5, symmetric=False)
    Lsd, tsd, tnd = _dev(Ls, ts, tn)
    R0 = I.make_t2(o, v, 6, symmetric=False)
    for sym in (P.PPL_SYM_FULL, P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR):
        with P.Plan(o, v, x) as plan:
            plan.set_symmetry(sym)
            plan.set_verify(2)
            Rd = torch.from_numpy(R0.copy()).cuda()
            with pytest.raises(P.PplError) as e:
                plan.apply(Lsd, tnd, Rd)
            assert e.value.code == P.PPL_ERR_PRECONDITION
            torch.cuda.synchronize()
            assert np.array_equal(Rd.cpu().numpy(), R0)  # nothing was queued
            plan.apply(Lsd, tsd, Rd)
            torch.cuda.synchronize()
            assert relerr(Rd.cpu().numpy(), oracle.full(Ls, ts, R0.copy())) <= 1e-11
    # both storage orders of t2 are checked in place
    with P.Plan(o, v, x) as plan:
        plan.set_verify(2)
        for arr, ok in ((ts, True), (tn, False)):
            td = torch.from_numpy(np.ascontiguousarray(arr.transpose(0, 2, 1, 3))).cuda()
            Rd = torch.zeros((o, v, o, v), dtype=torch.float64, device="cuda")
            if ok:
                plan.apply_ex(Lsd, td, Rd, t2_layout="iajb", r_layout="iajb")
            else:
                with pytest.raises(P.PplError):
                    plan.apply_ex(Lsd, td, Rd, t2_layout="iajb", r_layout="iajb")
    # PPL_SYM_NONE has no precondition; verify = 0 switches the check off
    with P.Plan(o, v, x) as plan:
        plan.set_symmetry(P.PPL_SYM_NONE)
        Ln = torch.from_numpy(I.make_L(v, x, 5, symmetric=False)).cuda()
        Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
        plan.apply(Ln, tnd, Rd)
        plan.apply(Ln, tnd, Rd)
        assert plan.verify_status() == 0
    with P.Plan(o, v, x) as plan:
        plan.set_verify(0)
        Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
        plan.apply(Lsd, tnd, Rd)
        plan.apply(Lsd, tnd, Rd)
        assert plan.verify_status() == 0


def test_a_single_wrong_element_is_found_anywhere():
    """One element of L (resp. t2) off by one ulp, at block corners and in the ragged edge of the 32 x 32 check tiles."""
    import torch

    o, v, x = 3, 70, 4
    Ls, ts = I.make_L(v, x, 7, symmetric=True), I.make_t2(o, v, 7, symmetric=True)
    with P.Plan(o, v, x) as plan:
        plan.set_verify(2)
        Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
        for (P_, a, c) in ((0, 0, 1), (3, 69, 0), (1, 31, 32), (2, 64, 69), (3, 33, 5)):
            L = Ls.copy()
            L[P_, a, c] = np.nextafter(L[P_, a, c], np.inf)
            with pytest.raises(P.PplError):
                plan.apply(torch.from_numpy(L).cuda(), torch.from_numpy(ts).cuda(), Rd)
        for (i, j, c, d) in ((0, 0, 0, 1), (0, 2, 69, 69), (2, 1, 32, 31), (1, 1, 64, 3)):
            t = ts.copy()
            t[i, j, c, d] = np.nextafter(t[i, j, c, d], np.inf)
            with pytest.raises(P.PplError):
                plan.apply(torch.from_numpy(Ls).cuda(), torch.from_numpy(t).cuda(), Rd)
        plan.apply(torch.from_numpy(Ls).cuda(), torch.from_numpy(ts).cuda(), Rd)  # and the clean inputs pass


def test_host_entry_point_reports_at_once():
    o, v, x = 3, 96, 6
    Ln = I.make_L(v, x, 9, symmetric=False)
    t2 = I.make_t2(o, v, 9, symmetric=True)
    R = np.zeros((o, o, v, v))
    with P.Plan(o, v, x) as plan:
        with pytest.raises(P.PplError) as e:
            plan.apply_host(Ln, t2, R)
        assert e.value.code == P.PPL_ERR_PRECONDITION
