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


@pytest.mark.parametrize("shape,chunk_mb", [((6, 96, 6), 1), ((6, 96, 6), 0), ((5, 53, 7), 1), ((4, 130, 5), 1)])
def test_host_entry_point_checks_t2_chunk_by_chunk_in_the_default_mode(shape, chunk_mb):
    """ppl_apply_host in PPL_SYM_FULL streams t2 through staging buffers and packs only its rows i <= j, so a
    t2 that is not pair-symmetric used to give a wrong R with PPL_OK.  Now the rows i >= j of every chunk are compared with
    what their mirror images packed (k_check_t2_rows); 1 MiB staging buffers put a row and its image into different chunks
    on different streams."""
    o, v, x = shape
    L = I.make_L(v, x, 21, symmetric=True)
    ts = I.make_t2(o, v, 21, symmetric=True)
    dbg = {"host_chunk_mb": chunk_mb} if chunk_mb else None
    with P.Plan(o, v, x, debug=dbg) as plan:
        assert plan.info()["symmetry"] == P.PPL_SYM_FULL
        R = np.zeros((o, o, v, v))
        plan.apply_host(L, ts, R)  # clean inputs pass, and the result is the oracle's
        assert relerr(R, oracle.full(L, ts)) <= 1e-11
        # one wrong element: in a row i > j (never read by the packing), in a row i < j, in the antisymmetric part of a
        # diagonal row, in the last row, on the diagonal c == d of a row i > j
        for (i, j, c, d) in [(o - 1, 0, 3, v - 2), (0, o - 1, v - 1, 0), (2, 2, 1, v - 1), (o - 1, o - 2, 0, 1), (3, 1, 7, 7)]:
            t = ts.copy()
            t[i, j, c, d] += 1e-9
            with pytest.raises(P.PplError) as e:
                plan.apply_host(L, t, np.zeros((o, o, v, v)))
            assert e.value.code == P.PPL_ERR_PRECONDITION, (i, j, c, d)
        # a fully unstructured t2, in the synchronous mode as well
        tn = I.make_t2(o, v, 22, symmetric=False)
        for mode in (1, 2):
            plan.set_verify(mode)
            with pytest.raises(P.PplError) as e:
                plan.apply_host(L, tn, np.zeros((o, o, v, v)))
            assert e.value.code == P.PPL_ERR_PRECONDITION
        # the report clears the state; the caller may vouch for its inputs instead
        plan.set_verify(0)
        plan.apply_host(L, tn, np.zeros((o, o, v, v)))
        plan.set_verify(1)
        R = np.zeros((o, o, v, v))
        plan.apply_host(L, ts, R)
        assert relerr(R, oracle.full(L, ts)) <= 1e-11


def test_with_block_does_not_mask_the_callers_exception_and_checks_survive_their_stream():
    """(1) Plan.__exit__ used to raise PPL_ERR_PRECONDITION from destroy() over an exception already leaving the
    with-block; (2) on the one-kernel path the outstanding checks are now followed by events of their own, so a caller may
    issue applies on different streams and destroy a stream while a check is still outstanding."""
    import torch

    o, v, x = 5, 20, 60
    L = I.make_L(v, x, 1, symmetric=True)
    ts, tn = I.make_t2(o, v, 1, symmetric=True), I.make_t2(o, v, 1, symmetric=False)
    Ld, tsd, tnd = _dev(L, ts, tn)
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    with pytest.raises(KeyError):
        with P.Plan(o, v, x, debug={"no_small_fused": 0}) as plan:
            assert plan.info()["small_fused"] == 1
            plan.apply(Ld, tnd, Rd)  # violation, still unreported when the block is left ...
            raise KeyError("the caller's own error")  # ... by this exception, which must come out
    with P.Plan(o, v, x, debug={"no_small_fused": 0}) as plan:
        s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
        torch.cuda.synchronize()
        plan.apply(Ld, tsd, Rd, s1)
        s2.wait_stream(s1)           # one apply of a plan in flight at a time (include/ppl.h, Threading)
        plan.apply(Ld, tnd, Rd, s2)  # two checks outstanding, on two streams
        del s1, s2                   # (torch returns them to its pool; an event would survive a destroyed stream as well)
        with pytest.raises(P.PplError) as e:
            plan.verify_status()
        assert e.value.code == P.PPL_ERR_PRECONDITION
        torch.cuda.synchronize()
        Rd.zero_()
        plan.apply(Ld, tsd, Rd)
        assert plan.verify_status() == 0
        torch.cuda.synchronize()
        assert relerr(Rd.cpu().numpy(), oracle.full(L, ts)) <= 1e-11
