"""-m gpu: the widened entry points against the CPU oracle.

  NEXT-1  ppl_apply_ex: t2 / R in the paper's storage orders ('icjd' -> 'iajb') and in
          BASELINE.json's ('ijab'), R = beta*R + alpha*term, beta == 0 overwrites without reading R;
  NEXT-3  ppl_apply_dense: step 1 alone on caller-supplied dense integrals ('abcd,ecfd->efab');
  NEXT-4  PPL_SYM_PAIR_SA (symmetric / antisymmetric packed step 1) is covered by the parametrised
          parity tests in test_gpu_parity.py / test_gpu_fullsize.py; here: its flop accounting.
Same tolerance as everywhere: max|diff| <= 1e-11 * max|want|; exact-integer inputs bit for bit.
"""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11
SYMS = [P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR, P.PPL_SYM_NONE]


def _to_layout(a, layout):
    """[i,j,p,q] -> the requested storage order (a copy, C-contiguous)."""
    return np.ascontiguousarray(a if layout == "ijab" else a.transpose(0, 2, 1, 3))


def _run_ex(L, t2, R0, sym, t2_layout, r_layout, alpha, beta, cap=0):
    import torch

    x, v, _ = L.shape
    o = t2.shape[0]
    Ld = torch.from_numpy(L).cuda()
    td = torch.from_numpy(_to_layout(t2, t2_layout)).cuda()
    Rd = torch.from_numpy(_to_layout(R0, r_layout)).cuda()
    with P.Plan(o, v, x, cap) as plan:
        plan.set_symmetry(sym)
        plan.apply_ex(Ld, td, Rd, t2_layout=t2_layout, r_layout=r_layout, alpha=alpha, beta=beta)
        torch.cuda.synchronize()
        info = plan.info()
    return Rd.cpu().numpy(), info


@pytest.mark.parametrize("shape,cap_cols", [((5, 20, 60), 0), ((4, 37, 19), 60), ((7, 26, 30), 90), ((5, 53, 40), 0)])
@pytest.mark.parametrize("sym", SYMS)
@pytest.mark.parametrize("t2_layout,r_layout", [("iajb", "iajb"), ("ijab", "iajb"), ("iajb", "ijab")])
def test_apply_ex_layouts_alpha_beta(shape, cap_cols, sym, t2_layout, r_layout):
    o, v, x = shape
    symmetric = sym != P.PPL_SYM_NONE
    L = I.make_L(v, x, 11, symmetric=False)
    t2 = I.make_t2(o, v, 11, symmetric=symmetric)
    R0 = I.make_t2(o, v, 12, symmetric=False)
    alpha, beta = -0.75, 0.5
    want = oracle.full_ex(L, _to_layout(t2, t2_layout), _to_layout(R0, r_layout).copy(), t2_layout, r_layout, alpha, beta)
    cap = 0 if cap_cols == 0 else (3 * cap_cols + 2 * o * o) * (v * v + 64) * 8 + 64 * o * o * cap_cols * 8 + 8192
    got, info = _run_ex(L, t2, R0, sym, t2_layout, r_layout, alpha, beta, cap)
    assert got.shape == want.shape
    assert relerr(got, want) <= TOL, info
    if cap_cols:
        assert info["n_tiles"] > 1, info


@pytest.mark.parametrize("sym", SYMS)
@pytest.mark.parametrize("r_layout", ["ijab", "iajb"])
def test_apply_ex_beta_zero_overwrites_without_reading_R(sym, r_layout):
    o, v, x = 4, 30, 12
    L = I.make_L(v, x, 21, symmetric=False)
    t2 = I.make_t2(o, v, 21, symmetric=sym != P.PPL_SYM_NONE)
    R0 = np.full((o, o, v, v), np.nan)
    want = oracle.full_ex(L, t2, np.zeros_like(_to_layout(R0, r_layout)), "ijab", r_layout, 2.0, 0.0)
    got, info = _run_ex(L, t2, R0, sym, "ijab", r_layout, 2.0, 0.0, cap=(200 + 2 * o * o) * (v * v + 64) * 8 + (1 << 20))
    assert np.isfinite(got).all(), "beta == 0 must not read R (NaN on entry)"
    assert relerr(got, want) <= TOL, info


@pytest.mark.parametrize("sym", SYMS)
def test_apply_ex_exact_integers_paper_layouts(sym):
    o, v, x = 6, 34, 21
    L = I.make_L(v, x, 31, symmetric=sym != P.PPL_SYM_NONE, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 31, symmetric=sym != P.PPL_SYM_NONE, integer=True)
    R0 = I.make_t2(o, v, 32, symmetric=False, integer=True)
    want = oracle.full_ex(L, _to_layout(t2, "iajb"), _to_layout(R0, "iajb").copy(), "iajb", "iajb", 3.0, -2.0)
    got, _ = _run_ex(L, t2, R0, sym, "iajb", "iajb", 3.0, -2.0, cap=(150 + 2 * o * o) * (v * v + 64) * 8 + (1 << 20))
    assert np.array_equal(got, want)


def test_apply_ex_null_opts_equals_apply_and_bad_layout_is_rejected():
    import ctypes

    import torch

    L, t2 = I.make_config("tiny", seed=0)
    o, v, x = I.CONFIGS["tiny"]
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    R1 = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    R2 = torch.zeros_like(R1)
    with P.Plan(o, v, x) as plan:
        plan.apply(Ld, td, R1)
        rc = P.lib().ppl_apply_ex(plan._h, Ld.data_ptr(), td.data_ptr(), R2.data_ptr(), None, None)
        assert rc == P.PPL_OK
        torch.cuda.synchronize()
        assert torch.equal(R1, R2)
        bad = P.binding.ppl_opts_t(7, 0, 1.0, 1.0)
        assert P.lib().ppl_apply_ex(plan._h, Ld.data_ptr(), td.data_ptr(), R2.data_ptr(), ctypes.byref(bad), None) == P.PPL_ERR_INVALID_ARG


# ---------------------------------------------------------------------------------------------------
# NEXT-3: dense integrals, step 1 alone
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape", [(5, 20, 3), (3, 23, 2), (9, 30, 4)])
@pytest.mark.parametrize("layouts", [("ijab", "ijab"), ("iajb", "iajb")])
def test_apply_dense_slabs_match_the_definition(shape, layouts):
    """eri[a,b,c,d] random (no symmetry at all): R[i,j,a,b] = beta R + alpha sum_cd eri[a,b,c,d] t2[i,j,c,d],
    fed slab by slab; the expected value is the definition as a matrix product in numpy (fp64)."""
    import torch

    o, v, x = shape
    t2_layout, r_layout = layouts
    eri = I.make_vec(v**4, 5, 300).reshape(v, v, v, v)
    t2 = I.make_t2(o, v, 51, symmetric=False)
    R0 = I.make_t2(o, v, 52, symmetric=False)
    alpha, beta = 1.25, -1.0
    want = beta * R0 + alpha * (t2.reshape(o * o, v * v) @ eri.reshape(v * v, v * v).T).reshape(o, o, v, v)
    td = torch.from_numpy(_to_layout(t2, t2_layout)).cuda()
    Rd = torch.from_numpy(_to_layout(R0, r_layout)).cuda()
    with P.Plan(o, v, x) as plan:
        a0 = 0
        for na in (1, 7, v):  # ragged slabs
            na = min(na, v - a0)
            if na <= 0:
                break
            slab = torch.from_numpy(np.ascontiguousarray(eri[a0:a0 + na])).cuda()
            plan.apply_dense(slab, a0, td, Rd, t2_layout=t2_layout, r_layout=r_layout, alpha=alpha, beta=beta)
            a0 += na
        torch.cuda.synchronize()
        assert a0 == v
    got = Rd.cpu().numpy()
    assert relerr(got, _to_layout(want, r_layout)) <= TOL


def test_apply_dense_on_cholesky_integrals_equals_oracle():
    """With eri = (ac|bd) built on the host from L, the dense route must reproduce the ladder oracle."""
    import torch

    o, v, x = 5, 20, 60
    L, t2 = I.make_config("tiny", seed=0)
    eri = np.ascontiguousarray(np.einsum("Pac,Pbd->abcd", L, L))
    want = oracle.full(L, t2)
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    with P.Plan(o, v, x) as plan:
        plan.apply_dense(torch.from_numpy(eri).cuda(), 0, torch.from_numpy(t2).cuda(), Rd)
        torch.cuda.synchronize()
    assert relerr(Rd.cpu().numpy(), want) <= TOL


# ---------------------------------------------------------------------------------------------------
# NEXT-4: flop accounting of the packed mode
# ---------------------------------------------------------------------------------------------------
def test_sa_mode_is_default_and_halves_step1_flops():
    o, v, x = 12, 40, 64
    with P.Plan(o, v, x) as plan:
        sa = plan.info()
        assert sa["symmetry"] == P.PPL_SYM_PAIR_SA
        plan.set_symmetry(P.PPL_SYM_PAIR)
        pair = plan.info()
        plan.set_symmetry(P.PPL_SYM_NONE)
        none = plan.info()
    assert sa["flops_step0"] == pair["flops_step0"]
    mp, mm, kp, km = o * (o + 1) // 2, o * (o - 1) // 2, v * (v + 1) // 2, v * (v - 1) // 2
    assert (sa["sa_rows_plus"], sa["sa_rows_minus"], sa["sa_k_plus"], sa["sa_k_minus"]) == (mp, mm, kp, km)
    ratio = sa["flops_step1"] / pair["flops_step1"]
    assert abs(ratio - (mp * kp + mm * km) / (o * o * v * v)) < 1e-12 and 0.5 <= ratio < 0.52
    assert none["flops_executed"] == none["flops_nominal"]
