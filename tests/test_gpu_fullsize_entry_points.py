"""-m gpu: the widened entry points at the `large` shape of BASELINE.json (nocc 40, nvirt 400, nchol 1600), against the
oracle on sampled columns (VERDICT r02 "weak" 1: until round 3 they had met the oracle only at nvirt <= 130).

  ppl_apply_ex        the paper's storage orders 'icjd' -> 'iajb', alpha != 1, beta = 0 over a
                      NaN-filled R, in the default mode -- the strided addressing of the pack / unpack kernels at 2 GB arrays
  ppl_generate_eri -> ppl_apply_dense on two slabs of 16 a's (8.2 GB of <ab|cd> each)
  ppl_contract_pair   on the ladder's two strings: 'xac,xbd->acbd' with a 2 GB output, and 'abcd,ecfd->efab' with t2 stored
                      'ecfd' (the generic gather route, K = 160 000, split-K partials)
The full oracle is unaffordable here (164 TFLOP); oracle.columns / oracle.contract_pair on sampled (a,b) are exact
per-column definitions.  Tolerance: 1e-11 max|.| as everywhere.
"""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I

pytestmark = pytest.mark.gpu
TOL = 1e-11
O, V, X = I.CONFIGS["large"]


@pytest.fixture(scope="module")
def large_inputs():
    return I.make_L(V, X, 0), I.make_t2(O, V, 0)


def _relerr(got, want):
    return float(np.abs(got - want).max() / np.abs(want).max())


def test_apply_ex_paper_layouts_alpha_beta0_at_large(large_inputs):
    import torch

    L, t2 = large_inputs
    Ld = torch.from_numpy(L).cuda()
    t_icjd = torch.from_numpy(t2).cuda().permute(0, 2, 1, 3).contiguous()  # t2[i,j,c,d] stored [i][c][j][d]
    R_iajb = torch.full((O, V, O, V), float("nan"), dtype=torch.float64, device="cuda")  # beta = 0 must not read it
    alpha = -0.625
    with P.Plan(O, V, X) as plan:
        assert plan.info()["symmetry"] == P.PPL_SYM_FULL
        plan.apply_ex(Ld, t_icjd, R_iajb, "iajb", "iajb", alpha=alpha, beta=0.0)
        torch.cuda.synchronize()
    assert bool(torch.isfinite(R_iajb).all())
    pairs = I.sample_pairs(V, 160, seed=3)
    want = alpha * oracle.columns(L, t2, pairs)  # [n, o, o]
    a = torch.from_numpy(pairs[:, 0].astype(np.int64)).cuda()
    b = torch.from_numpy(pairs[:, 1].astype(np.int64)).cuda()
    got = R_iajb[:, a, :, b]  # advanced indices separated by a slice: result [n, o(i), o(j)]
    assert _relerr(got.cpu().numpy(), want) <= TOL
    # the pair symmetry of the result holds in this storage order too: R[i,a,j,b] == R[j,b,i,a], every entry
    assert torch.equal(R_iajb, R_iajb.permute(2, 3, 0, 1))


def test_generate_eri_then_apply_dense_on_two_slabs_at_large(large_inputs):
    import torch

    L, t2 = large_inputs
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    Rd = torch.zeros((O, O, V, V), dtype=torch.float64, device="cuda")
    na = 16
    eri = torch.empty((na, V, V, V), dtype=torch.float64, device="cuda")  # 8.2 GB
    rng = np.random.default_rng(5)
    with P.Plan(O, V, X) as plan:
        for a0 in (0, V - na):
            plan.generate_eri(Ld, a0, na, eri)
            plan.apply_dense(eri, a0, td, Rd)  # R[:, :, a0:a0+na, :] += the slab's share of the ladder
            torch.cuda.synchronize()
            # a few integrals of the slab against eq. 5 directly: <ab|cd> = sum_P L[P,a,c] L[P,b,d]
            for _ in range(6):
                al, b, c, d = (int(rng.integers(na)), *(int(t) for t in rng.integers(V, size=3)))
                want = float(np.dot(L[:, a0 + al, c], L[:, b, d]))
                assert abs(float(eri[al, b, c, d]) - want) <= 1e-12 * max(1.0, abs(want))
    pairs = np.array([(a, int(b)) for a0 in (0, V - na) for a in (a0, a0 + 7, a0 + na - 1) for b in rng.integers(V, size=8)])
    want = oracle.columns(L, t2, pairs)
    a = torch.from_numpy(pairs[:, 0].astype(np.int64)).cuda()
    b = torch.from_numpy(pairs[:, 1].astype(np.int64)).cuda()
    got = Rd[:, :, a, b].permute(2, 0, 1).contiguous().cpu().numpy()
    assert _relerr(got, want) <= TOL
    assert float(Rd[:, :, na : V - na, :].abs().max()) == 0.0  # a's outside the two slabs were not touched


def test_contract_pair_on_the_ladder_strings_at_large_sizes(large_inputs):
    import torch

    L, t2 = large_inputs
    Ld = torch.from_numpy(L).cuda()
    # step 0, 4 a's: output [4][400][400][400] = 2.05 GB ('acbd' order); operands are slices of L
    a0, na = 200, 4
    A = Ld[:, a0 : a0 + na, :].contiguous()
    W = P.ppl_contract_pair("xac,xbd->acbd", A, Ld)
    torch.cuda.synchronize()
    assert W.numel() * 8 > 2 * 10**9
    rng = np.random.default_rng(7)
    for _ in range(4):
        al, b = int(rng.integers(na)), int(rng.integers(V))
        want = oracle.contract_pair("xac,xbd->acbd", np.ascontiguousarray(L[:, a0 + al : a0 + al + 1, :]), np.ascontiguousarray(L[:, b : b + 1, :]))
        got = W[al, :, b, :].cpu().numpy()  # [c][d]
        assert _relerr(got, want[0, :, 0, :]) <= TOL
    # step 1 with t2 stored 'ecfd' (the paper's own order): generic gather route, K = nvirt^2 = 160 000
    eri = torch.from_numpy(I.make_vec(na * V * V * V, 11, 60).reshape(na, V, V, V)).cuda()
    t_ecfd = torch.from_numpy(t2).cuda().permute(0, 2, 1, 3).contiguous()
    C = P.ppl_contract_pair("abcd,ecfd->efab", eri, t_ecfd)
    torch.cuda.synchronize()
    t_host = np.ascontiguousarray(t2.transpose(0, 2, 1, 3))
    for _ in range(4):
        al, b = int(rng.integers(na)), int(rng.integers(V))
        sub = np.ascontiguousarray(eri[al : al + 1, b : b + 1].cpu().numpy())
        want = oracle.contract_pair("abcd,ecfd->efab", sub, t_host)  # [e][f][1][1]
        assert _relerr(C[:, :, al, b].cpu().numpy(), want[:, :, 0, 0]) <= TOL
    # and the no-allocation entry point on the same request (tables 16 (M + N + K) = 2.6 MB of its 32 MiB)
    C2 = torch.full_like(C, float("nan"))
    P.ppl_contract_pair_noalloc("abcd,ecfd->efab", eri, t_ecfd, C2)
    torch.cuda.synchronize()
    assert _relerr(C2.cpu().numpy(), C.cpu().numpy()) <= TOL
