"""ppl_apply_host in the un-packed modes (the paper's own setting, on the
unstructured arrays of its benchmark): t2 resident, L whole or streamed as row panels, R streamed as slabs
(PPL_SYM_NONE) or resident (PPL_SYM_PAIR).  Every case against the CPU oracle at the north_star tolerance; exact-integer
inputs bit for bit.  Nothing here is symmetric unless the mode needs it."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11

# (shape, tile edge): several rows of tiles, a ragged last block, rings that wrap (tiles > ring), one-tile plans
CASES = [((6, 96, 40), 16), ((4, 70, 33), 16), ((5, 58, 24), 20), ((3, 64, 17), 64), ((7, 34, 50), 5), ((2, 130, 12), 48)]


@pytest.mark.parametrize("panels", [1, 2])
@pytest.mark.parametrize("shape,T", CASES)
def test_none_mode_streams_L_panels_and_R_slabs(shape, T, panels):
    """PPL_SYM_NONE, non-symmetric L and t2, R non-zero on entry; two calls through the same buffers (+= twice)."""
    o, v, x = shape
    L = I.make_L(v, x, seed=11, symmetric=False)
    t2 = I.make_t2(o, v, seed=11, symmetric=False)
    R0 = I.make_vec(o * o * v * v, 11, 40).reshape(o, o, v, v)
    want = oracle.full(L, t2)
    R = R0.copy()
    with P.Plan(o, v, x, debug=dict(tile_edge=T, host_panels=panels, no_small_fused=1)) as plan:
        plan.set_symmetry(P.PPL_SYM_NONE)
        info = plan.info()
        nblk = info["n_ablocks"]
        assert info["n_tiles"] == nblk * nblk
        for rep in range(2):
            h2d, d2h = plan.apply_host(L, t2, R)
            assert d2h == R.nbytes  # every slab travels out once
            if panels == 1:  # row panel per row of tiles + a column panel per off-diagonal tile; t2 and the R slabs once
                assert h2d == t2.nbytes + R.nbytes + L.nbytes * nblk
            else:
                assert h2d == t2.nbytes + R.nbytes + L.nbytes
            assert relerr(R - R0, (rep + 1) * want) <= TOL, rep


@pytest.mark.parametrize("panels", [1, 2])
@pytest.mark.parametrize("shape,T", CASES[:4])
def test_pair_mode_streams_L_panels_R_resident(shape, T, panels):
    """PPL_SYM_PAIR: pair-symmetric t2, ANY L (non-symmetric here); the mirror writes reach every slab, R stays resident."""
    o, v, x = shape
    L = I.make_L(v, x, seed=12, symmetric=False)
    t2 = I.make_t2(o, v, seed=12, symmetric=True)
    want = oracle.full(L, t2)
    R = np.zeros((o, o, v, v))
    with P.Plan(o, v, x, debug=dict(tile_edge=T, host_panels=panels, no_small_fused=1)) as plan:
        plan.set_symmetry(P.PPL_SYM_PAIR)
        nblk = plan.info()["n_ablocks"]
        h2d, d2h = plan.apply_host(L, t2, R)
        assert d2h == R.nbytes
        if panels == 1:  # tiles a-block <= b-block: a row panel per row, a column panel per off-diagonal tile
            per_block = x * v * 8 * min(T, v)
            assert h2d <= t2.nbytes + R.nbytes + per_block * (nblk + nblk * (nblk - 1) // 2)
        assert relerr(R, want) <= TOL


def test_pair_mode_reports_a_violated_precondition():
    o, v, x = 4, 64, 20
    L = I.make_L(v, x, seed=13, symmetric=False)
    t2 = I.make_t2(o, v, seed=13, symmetric=False)
    R = np.zeros((o, o, v, v))
    with P.Plan(o, v, x, debug=dict(tile_edge=16, host_panels=1, no_small_fused=1)) as plan:
        plan.set_symmetry(P.PPL_SYM_PAIR)
        with pytest.raises(P.PplError) as e:
            plan.apply_host(L, t2, R)
        assert e.value.code == P.PPL_ERR_PRECONDITION
        plan.set_symmetry(P.PPL_SYM_NONE)  # the same arrays are fine where nothing is assumed
        R[:] = 0
        plan.apply_host(L, t2, R)
    assert relerr(R, oracle.full(L, t2)) <= TOL


@pytest.mark.parametrize("mode", ["none", "pair"])
def test_exact_integers_bit_for_bit(mode):
    o, v, x = 5, 72, 14
    L = I.make_L(v, x, 21, symmetric=False, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 21, symmetric=(mode == "pair"), integer=True)
    R = np.zeros((o, o, v, v))
    with P.Plan(o, v, x, debug=dict(tile_edge=16, host_panels=1, no_small_fused=1)) as plan:
        plan.set_symmetry(P.PPL_SYM_NONE if mode == "none" else P.PPL_SYM_PAIR)
        plan.apply_host(L, t2, R)
    assert np.array_equal(R, oracle.full(L, t2))


def test_panels_and_whole_L_agree_bit_for_bit():
    """The same kernels on the same numbers in the same order: where L sits changes nothing."""
    o, v, x = 5, 80, 37
    L = I.make_L(v, x, seed=31, symmetric=False)
    t2 = I.make_t2(o, v, seed=31, symmetric=False)
    got = []
    for panels in (1, 2):
        R = np.zeros((o, o, v, v))
        with P.Plan(o, v, x, debug=dict(tile_edge=16, host_panels=panels, no_small_fused=1)) as plan:
            plan.set_symmetry(P.PPL_SYM_NONE)
            plan.apply_host(L, t2, R)
        got.append(R)
    assert np.array_equal(got[0], got[1])
    Rd = np.zeros((o, o, v, v))
    import torch

    with P.Plan(o, v, x, debug=dict(tile_edge=16, no_small_fused=1)) as plan:  # and the device-resident apply
        plan.set_symmetry(P.PPL_SYM_NONE)
        plan.set_graph(0)
        Rt = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
        plan.apply(torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda(), Rt)
        torch.cuda.synchronize()
        Rd = Rt.cpu().numpy()
    assert np.array_equal(got[0], Rd)


def test_odd_nvirt_takes_the_whole_copy_route():
    o, v, x = 4, 53, 30
    L = I.make_L(v, x, seed=41, symmetric=False)
    t2 = I.make_t2(o, v, seed=41, symmetric=False)
    R = np.zeros((o, o, v, v))
    with P.Plan(o, v, x, debug=dict(no_small_fused=1)) as plan:
        plan.set_symmetry(P.PPL_SYM_NONE)
        h2d, d2h = plan.apply_host(L, t2, R)
    assert h2d == L.nbytes + 2 * R.nbytes and d2h == R.nbytes
    assert relerr(R, oracle.full(L, t2)) <= TOL
