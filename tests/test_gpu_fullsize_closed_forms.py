"""-m gpu: EVERY entry of R at BASELINE.json's full sizes, in the launch configuration bench.py times, against closed
forms of eq. 6 that need no oracle run ("any size incl. XL"):

  P3  identity L:  L[P] = s_P * 1  =>  (ac|bd) = (sum_P s_P^2) delta_ac delta_bd  =>  R = (sum_P s_P^2) * t2.
      With dyadic s_P and even-integer t2 every product and partial sum is exactly representable: bit for bit.
  P4  rank-1 L:    L[P,a,c] = alpha_P u_a u_c  =>  R[i,j,a,b] = |alpha|^2 u_a u_b (u^T T_ij u); 1e-11 * max|R|.
  tagged L == 1:   (ac|bd) = nchol  =>  R[i,j,a,b] = nchol * sum_cd t2[i,j,c,d] for every (a,b); t2 tags every
      (row, 16-wide k-tile) pair, so a fragment read from a stale pipeline slot or a neighbouring row changes the integer
      result (the pattern that exposed the ring-slot race of round 1) -- here in the symmetric modes too.
The right-hand sides are evaluated on the device with plain torch FP64 ops of the test (never by the library).
Inputs are seeded and generated on the device (pair-symmetric by construction: T + T^T over (i,j),(c,d))."""
import pytest

import paper_2603_20912_b200 as P
import ppl_inputs as I

pytestmark = pytest.mark.gpu
TOL = 1e-11
SYMS = {"default": None, "pair_sa": P.PPL_SYM_PAIR_SA, "pair": P.PPL_SYM_PAIR}


def _fits(name):
    import torch

    o, v, x = I.CONFIGS[name]
    need = (x * v * v + 3 * o * o * v * v) * 8 + (70e9 if name == "xl" else 25e9 if name == "large" else 6e9)
    return torch.cuda.mem_get_info()[0] > need


def _pair_symmetric(o, v, seed, integer):
    import torch

    g = torch.Generator(device="cuda").manual_seed(seed)
    if integer:
        T = torch.randint(-2, 3, (o, o, v, v), device="cuda", generator=g).to(torch.float64)
        return (2.0 * (T + T.permute(1, 0, 3, 2))).contiguous()  # even integers: (t2[cd] +- t2[dc]) / 2 stays exact
    T = 0.1 * torch.randn((o, o, v, v), dtype=torch.float64, device="cuda", generator=g)
    return (T + T.permute(1, 0, 3, 2)).contiguous()


def _apply(name, sym, L, t2):
    import torch

    o, v, x = I.CONFIGS[name]
    R = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    with P.Plan(o, v, x) as plan:
        if sym is not None:
            plan.set_symmetry(sym)
        assert plan.info()["symmetry"] == (P.PPL_SYM_FULL if sym is None else sym)
        plan.apply(L, t2, R)
        assert plan.verify_status() == 0  # the library's own input check agrees that the inputs are symmetric
        torch.cuda.synchronize()
    return R


@pytest.mark.parametrize("name,mode", [("medium", "default"), ("medium", "pair_sa"), ("medium", "pair"), ("large", "default"),
                                       ("large", "pair_sa"), ("xl", "default")])
def test_P3_identity_L_every_entry_bit_for_bit(name, mode):
    import torch

    if not _fits(name):
        pytest.skip("not enough device memory")
    o, v, x = I.CONFIGS[name]
    s = torch.tensor([1.0, 0.5, -2.0, 0.25, -1.0, 4.0, -0.5], dtype=torch.float64, device="cuda")[torch.arange(x, device="cuda") % 7]
    L = torch.zeros((x, v, v), dtype=torch.float64, device="cuda")
    idx = torch.arange(v, device="cuda")
    L[:, idx, idx] = s[:, None]
    t2 = _pair_symmetric(o, v, 31, integer=True)
    R = _apply(name, SYMS[mode], L, t2)
    want = float((s * s).sum().item()) * t2  # sum of dyadic squares: exact
    assert int((R != want).sum().item()) == 0


@pytest.mark.parametrize("name,mode", [("medium", "default"), ("medium", "pair_sa"), ("large", "default"), ("large", "pair"),
                                       ("xl", "default")])
def test_P4_rank1_L_every_entry(name, mode):
    import torch

    if not _fits(name):
        pytest.skip("not enough device memory")
    o, v, x = I.CONFIGS[name]
    g = torch.Generator(device="cuda").manual_seed(32)
    alpha = torch.randn(x, dtype=torch.float64, device="cuda", generator=g) * torch.exp(-3.0 * torch.arange(x, device="cuda") / x)
    u = torch.randn(v, dtype=torch.float64, device="cuda", generator=g)
    L = (alpha[:, None, None] * (u[:, None] * u[None, :])[None]).contiguous()  # symmetric in (a, c)
    t2 = _pair_symmetric(o, v, 33, integer=False)
    R = _apply(name, SYMS[mode], L, t2)
    q = torch.einsum("ijcd,d->ijc", t2, u)
    q = torch.einsum("ijc,c->ij", q, u)                      # u^T T_ij u
    want = float((alpha * alpha).sum().item()) * q[:, :, None, None] * (u[:, None] * u[None, :])[None, None]
    err = float((R - want).abs().max().item()) / float(want.abs().max().item())
    assert err <= TOL, err


@pytest.mark.parametrize("name,mode", [("medium", "default"), ("medium", "pair_sa"), ("medium", "pair"), ("large", "default")])
def test_tagged_constant_L_every_entry_bit_for_bit(name, mode):
    import torch

    if not _fits(name):
        pytest.skip("not enough device memory")
    o, v, x = I.CONFIGS[name]
    vv = v * v
    L = torch.ones((x, v, v), dtype=torch.float64, device="cuda")
    m_idx = torch.arange(o * o, device="cuda", dtype=torch.float64).reshape(o * o, 1)
    ktag = (torch.arange(vv, device="cuda") // 16).to(torch.float64)
    T = (ktag.reshape(1, vv) + 1000.0 * m_idx).reshape(o, o, v, v)
    t2 = (2.0 * (T + T.permute(1, 0, 3, 2))).contiguous()    # pair-symmetric, even integers
    want = (x * t2.sum(dim=(2, 3))).reshape(o, o, 1, 1)       # exact integers < 2^53
    for rep in range(2):
        R = _apply(name, SYMS[mode], L, t2)
        assert int((R != want).sum().item()) == 0, rep
