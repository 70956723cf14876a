"""-m gpu: the CUDA path (C ABI -> sm_100a kernels) against the CPU oracle, element by element on
the same seeded inputs.  Tolerance (north_star, reading A14): max|R_gpu - R_oracle| <= 1e-11 *
max|R_oracle| over the compared entries, R zero on entry; exact-integer inputs must match bit for
bit.  Full element-wise parity on configs 0-2 shapes that the oracle finishes in seconds; sampled
columns + full-coverage projections at the large sizes (tests/test_gpu_fullsize.py)."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import gpu_ladder, relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11


def test_native_library_is_loaded_and_device_is_b200():
    import torch

    assert torch.cuda.is_available()
    assert torch.cuda.get_device_capability(0)[0] == 10
    P.lib()
    maps = open("/proc/self/maps").read()
    assert "libppl.so" in maps, "native CUDA library not loaded"


def test_dmma_fragment_layout():
    """One mma.sync.m8n8k4.f64 with the fragment layout the kernels assume equals A @ B exactly."""
    import torch

    A = np.arange(1, 33, dtype=np.float64).reshape(8, 4)
    B = ((np.arange(32) * 7) % 11 - 3).astype(np.float64).reshape(4, 8)
    C = torch.zeros((8, 8), dtype=torch.float64, device="cuda")
    P.ppl_debug_dmma_layout(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C)
    assert np.array_equal(C.cpu().numpy(), A @ B)


@pytest.mark.parametrize("name", ["tiny", "small"])
@pytest.mark.parametrize("sym", [P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR, P.PPL_SYM_NONE])
def test_configs_0_1_full_parity(name, sym):
    L, t2 = I.make_config(name, seed=0)
    want = oracle.full(L, t2)
    got, info = gpu_ladder(L, t2, sym=sym, return_info=True)
    assert relerr(got, want) <= TOL, info


# shapes chosen to span several CTA tiles (128x128x16), ragged m/n/k tails, odd nvirt (8-byte copy
# path), nocc^2 > 128, and -- through the workspace cap -- several (a,b) tiles with a ragged edge
SHAPES = [
    (1, 1, 1), (2, 1, 3), (1, 5, 1), (3, 7, 5), (2, 16, 4), (3, 24, 17), (12, 18, 9),
    (4, 37, 19), (3, 40, 33), (13, 22, 40), (6, 50, 70),
]


def _cap(o, v, cap_cols, sym):
    """workspace cap in units of W columns (v*v*8 bytes each) + room for partials (+ the packed
    amplitudes and the un-folded step-0 tile in PPL_SYM_PAIR_SA): forces small tiles"""
    if cap_cols == 0:
        return 0
    cap = cap_cols * v * v * 8 + 64 * o * o * cap_cols * 8 + 4096
    if sym == P.PPL_SYM_PAIR_SA:
        cap += (o * o + cap_cols) * (v * v + 64) * 8 + 4096
    return cap


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("sym", [P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR, P.PPL_SYM_NONE])
@pytest.mark.parametrize("cap_cols", [0, 40, 7])
def test_shapes_full_parity(shape, sym, cap_cols):
    o, v, x = shape
    symmetric = sym != P.PPL_SYM_NONE
    L = I.make_L(v, x, seed=5, symmetric=symmetric)  # non-symmetric L in general mode
    t2 = I.make_t2(o, v, seed=5, symmetric=symmetric)
    if sym != P.PPL_SYM_NONE:  # the pair modes need pair-symmetric t2 only: L stays non-symmetric
        L = I.make_L(v, x, seed=5, symmetric=False)
    want = oracle.full(L, t2)
    cap = _cap(o, v, cap_cols, sym)
    try:
        got, info = gpu_ladder(L, t2, sym=sym, workspace_bytes=cap, return_info=True)
    except P.PplError as e:
        assert e.code == P.PPL_ERR_WORKSPACE_TOO_SMALL and cap_cols == 7
        pytest.skip("cap below the minimum plan for this shape")
    assert info["symmetry"] == sym
    assert relerr(got, want) <= TOL, info
    if cap_cols and cap < v**4 * 8:  # the cap cannot hold the whole W: the plan must have tiled it
        assert info["n_tiles"] > 1 and info["workspace_bytes"] <= cap, info


def test_pair_mode_is_symmetric_and_general_mode_detects_asymmetry():
    o, v, x = 4, 30, 12
    L = I.make_L(v, x, 9, symmetric=False)
    tn = I.make_t2(o, v, 9, symmetric=False)
    Rn = gpu_ladder(L, tn, sym=P.PPL_SYM_NONE, workspace_bytes=60 * v * v * 8 + (1 << 20))
    assert relerr(Rn, oracle.full(L, tn)) <= TOL
    assert relerr(Rn, Rn.transpose(1, 0, 3, 2)) > 1e-3  # negative control: asymmetric t2 -> asymmetric R


def test_accumulate_semantics_and_zero_t2():
    o, v, x = 5, 20, 60
    L, t2 = I.make_config("tiny", seed=0)
    R0 = I.make_t2(o, v, 77, symmetric=False)
    got = gpu_ladder(L, t2, R0=R0.copy())
    want = oracle.full(L, t2, R0.copy())
    assert relerr(got, want) <= TOL
    # t2 == 0 leaves R bitwise unchanged
    got0 = gpu_ladder(L, np.zeros_like(t2), R0=R0.copy())
    assert np.array_equal(got0, R0)


@pytest.mark.parametrize("shape,cap_cols", [((5, 20, 60), 0), ((5, 53, 40), 0), ((4, 37, 19), 40), ((12, 18, 9), 7)])
@pytest.mark.parametrize("sym", [P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR, P.PPL_SYM_NONE])
def test_exact_integers_bit_for_bit(shape, cap_cols, sym):
    """Small-integer inputs: every product and partial sum is exact in binary64, so any summation
    order gives the same bits -> separates logic bugs (tile edges, mirror, split-K) from rounding."""
    o, v, x = shape
    symmetric = sym != P.PPL_SYM_NONE
    L = I.make_L(v, x, 41, symmetric=symmetric, integer=True)
    t2 = I.make_t2(o, v, 41, symmetric=symmetric, integer=True)
    if sym == P.PPL_SYM_PAIR_SA:
        t2 *= 2.0  # tau+- = (t2[cd] +- t2[dc]) / 2 stays an exact integer
    got = gpu_ladder(L, t2, sym=sym, workspace_bytes=_cap(o, v, cap_cols, sym))
    assert np.array_equal(got, oracle.full(L, t2))


@pytest.mark.parametrize("shape", [(24, 64, 128), (16, 72, 200), (30, 48, 260)])
@pytest.mark.parametrize("sym", [P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR])
def test_persistent_ring_many_items_per_cta(shape, sym):
    """Regression for a shared-memory WAR race in the persistent TMA kernels: every CTA runs several
    work items back to back and every item has more k-tiles than the ring has stages, so slots are
    refilled across item boundaries while other warps are in their epilogue.  Exact-integer inputs:
    any stale or early fragment changes the bits.  Repeated, because the race was timing dependent."""
    o, v, x = shape
    L = I.make_L(v, x, 43, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 43, integer=True)
    want = oracle.full(L, t2)
    for rep in range(6):
        got, info = gpu_ladder(L, t2, sym=sym, return_info=True)
        assert np.array_equal(got, want), (rep, info)


def test_check_inputs_flags():
    import torch

    o, v, x = 3, 12, 5
    Ls, ts = I.make_L(v, x, 3), I.make_t2(o, v, 3)
    Ln, tn = I.make_L(v, x, 3, symmetric=False), I.make_t2(o, v, 3, symmetric=False)
    with P.Plan(o, v, x) as plan:
        assert plan.check_inputs(torch.from_numpy(Ls).cuda(), torch.from_numpy(ts).cuda()) == 0
        assert plan.check_inputs(torch.from_numpy(Ln).cuda(), torch.from_numpy(ts).cuda()) == 1
        with pytest.raises(P.PplError) as ei:
            plan.check_inputs(torch.from_numpy(Ls).cuda(), torch.from_numpy(tn).cuda())
        assert ei.value.code == P.PPL_ERR_PRECONDITION
        plan.set_symmetry(P.PPL_SYM_NONE)
        assert plan.check_inputs(torch.from_numpy(Ls).cuda(), torch.from_numpy(tn).cuda()) == 2


def test_stream_ordering_and_repeated_apply():
    """apply is asynchronous and ordered on the caller's stream; two applies add the term twice."""
    import torch

    L, t2 = I.make_config("tiny", seed=0)
    o, v, x = 5, 20, 60
    want = oracle.full(L, t2)
    s = torch.cuda.Stream()
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    torch.cuda.synchronize()
    with P.Plan(o, v, x) as plan, torch.cuda.stream(s):
        Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
        plan.apply(Ld, td, Rd)        # uses torch's current stream = s
        Rd.mul_(0.5)                  # ordered after the apply on s
        plan.apply(Ld, td, Rd)
        s.synchronize()
    assert relerr(Rd.cpu().numpy(), 1.5 * want) <= TOL


def test_host_entry_point():
    L, t2 = I.make_config("tiny", seed=0)
    R = np.zeros((5, 5, 20, 20))
    with P.Plan(5, 20, 60) as plan:
        h2d, d2h = plan.apply_host(L, t2, R)
    assert h2d == L.nbytes + t2.nbytes + R.nbytes and d2h == R.nbytes
    assert relerr(R, oracle.full(L, t2)) <= TOL


def test_workspace_too_small_and_bad_pointers():
    with pytest.raises(P.PplError) as ei:
        P.ppl_plan(5, 20, 60, workspace_bytes=1000)
    assert ei.value.code == P.PPL_ERR_WORKSPACE_TOO_SMALL
    with P.Plan(5, 20, 60) as plan:
        assert P.lib().ppl_apply(plan._h, None, None, None, None) == P.PPL_ERR_INVALID_ARG


@pytest.mark.parametrize("shape", [(5, 20, 60), (5, 53, 232), (7, 81, 300), (20, 200, 800), (12, 18, 9)])
def test_dry_planner_equals_the_device_plan(shape):
    """ppl_plan_dry (the planner alone, tests/test_planner_cpu.py) and ppl_plan on the device agree field by field."""
    import torch

    with P.Plan(*shape) as plan:
        dev = plan.info()
    dry = P.ppl_plan_dry(*shape, device_free_bytes=torch.cuda.mem_get_info()[0], num_sms=torch.cuda.get_device_properties(0).multi_processor_count)
    assert dry == dev
