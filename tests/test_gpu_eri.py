"""-m gpu: ppl_generate_eri -- step 0 alone ('xac,xbd->acbd'; eq. 5) -- against
oracle.eri_slab, element by element (1e-11 relative; exact-integer inputs bit for bit), and its duality with
ppl_apply_dense: generate a slab, contract it, compare with the ladder oracle."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11


def _generate(o, v, x, L, a0, na, poison=True):
    import torch

    Ld = torch.from_numpy(L).cuda()
    eri = torch.full((na, v, v, v), float("nan") if poison else 0.0, dtype=torch.float64, device="cuda")
    with P.Plan(o, v, x, 0) as plan:
        plan.generate_eri(Ld, a0, na, eri)
        torch.cuda.synchronize()
    return eri.cpu().numpy()


@pytest.mark.parametrize("shape", [(1, 1, 1), (2, 5, 1), (3, 7, 5), (2, 16, 4), (4, 37, 19), (3, 40, 33), (5, 53, 40), (2, 66, 70)])
@pytest.mark.parametrize("symmetric", [False, True])
def test_generate_eri_parity(shape, symmetric):
    o, v, x = shape
    L = I.make_L(v, x, 21, symmetric=symmetric)
    for a0, na in sorted({(0, v), (v // 3, v - v // 3), (v - 1, 1)}):
        got = _generate(o, v, x, L, a0, na)  # NaN-filled on entry: every element must be written
        want = oracle.eri_slab(L, a0, na)
        assert got.shape == want.shape
        assert relerr(got, want) <= TOL, (a0, na)


@pytest.mark.parametrize("shape", [(2, 20, 9), (3, 37, 12), (2, 72, 30)])
def test_generate_eri_exact_integers_bit_for_bit(shape):
    o, v, x = shape
    L = I.make_L(v, x, 22, symmetric=False, integer=True)
    assert np.array_equal(_generate(o, v, x, L, 0, v), oracle.eri_slab(L, 0, v))


def test_generate_eri_slab_of_more_than_64_and_bad_arguments():
    import torch

    o, v, x = 2, 70, 8  # the slab is cut into pieces of 64 a's
    L = I.make_L(v, x, 23, symmetric=False)
    assert relerr(_generate(o, v, x, L, 0, v), oracle.eri_slab(L, 0, v)) <= TOL
    Ld = torch.from_numpy(L).cuda()
    eri = torch.zeros((2, v, v, v), dtype=torch.float64, device="cuda")
    with P.Plan(o, v, x, 0) as plan:
        for a0, na in ((-1, 2), (v - 1, 2), (0, 0)):
            with pytest.raises(P.PplError):
                lib_rc = P.binding.lib().ppl_generate_eri(plan._h, Ld.data_ptr(), a0, na, eri.data_ptr(), None)
                P.binding._check(lib_rc, "ppl_generate_eri")


@pytest.mark.parametrize("shape", [(4, 24, 17), (5, 53, 40)])
def test_generate_then_apply_dense_equals_the_ladder(shape):
    """The dense / Cholesky duality: 'xac,xbd->acbd' then 'abcd,ecfd->efab' slab by slab is the pp-ladder."""
    import torch

    o, v, x = shape
    L = I.make_L(v, x, 24, symmetric=False)
    t2 = I.make_t2(o, v, 24, symmetric=False)
    R0 = I.make_t2(o, v, 25, symmetric=False)
    want = oracle.full(L, t2, R0.copy())
    Ld, td, Rd = (torch.from_numpy(a).cuda() for a in (L, t2, R0))
    na = 7
    with P.Plan(o, v, x, 0) as plan:
        for a0 in range(0, v, na):
            n = min(na, v - a0)
            eri = torch.empty((n, v, v, v), dtype=torch.float64, device="cuda")
            plan.generate_eri(Ld, a0, n, eri)
            plan.apply_dense(eri, a0, td, Rd)
        torch.cuda.synchronize()
    assert relerr(Rd.cpu().numpy(), want) <= TOL
