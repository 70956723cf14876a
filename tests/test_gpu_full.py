"""-m gpu: PPL_SYM_FULL (full 8-fold ERI symmetry: slabs of 16 a's, symmetric S+- used twice, step 0
restricted to d-block >= b-block; include/ppl.h) against the CPU oracle.  The mode needs symmetric L and
pair-symmetric t2; odd nvirt runs in the geometry of nvirt + 1 with a zero pad index (L copied into 16-byte aligned
rows for TMA).  Same tolerance as everywhere (1e-11 relative, exact integers bit
for bit).  The identity behind it is pinned on the CPU (test_oracle_pins.py::test_full_symmetry_hook_identity)."""
import numpy as np
import pytest

import oracle
import paper_2603_20912_b200 as P
import ppl_inputs as I
from gpu_util import gpu_ladder, relerr

pytestmark = pytest.mark.gpu
TOL = 1e-11

# even nvirt; one slab (v <= 16), several slabs, ragged last slab (v % 16 != 0), nocc^2 > 128, one/two-element edges;
# odd nvirt (padded to nvirt + 1): below / at / above a 16-block edge, the small config's 53, one-element edges
SHAPES = [(1, 2, 1), (2, 16, 4), (12, 18, 9), (3, 24, 17), (5, 20, 60), (3, 40, 33), (13, 22, 40), (6, 50, 70),
          (4, 66, 30), (9, 100, 24), (24, 64, 128), (2, 130, 20),
          (2, 3, 2), (3, 15, 7), (4, 17, 9), (5, 31, 12), (3, 33, 20), (5, 53, 232), (7, 97, 30), (2, 129, 16), (1, 5, 1)]


# the two forms of the W+- tiles and of the diagonal d-blocks of step 0 (include/ppl.h, ppl_debug_opts_t): the product's
# (runs of the packed pair index; 9 packed chunks per diagonal block) and the round-1 form (rectangular tiles with zero
# rows; 16 plain chunks), which the memory-tight form still uses
FORMS = {"range+packed": {}, "rect+plain": {"full_rect_tiles": 1, "full_no_diag_pack": 1},
         "range+plain": {"full_no_diag_pack": 1}, "rect+packed": {"full_rect_tiles": 1}}


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("tbg", [128, 32, 16])
@pytest.mark.parametrize("form", ["range+packed", "rect+plain"])
def test_full_mode_parity(shape, tbg, form):
    o, v, x = shape
    L = I.make_L(v, x, seed=21, symmetric=True)
    t2 = I.make_t2(o, v, seed=21, symmetric=True)
    want = oracle.full(L, t2)
    got, info = gpu_ladder(L, t2, sym=P.PPL_SYM_FULL, return_info=True, debug=dict(FORMS[form], full_tbg=tbg))
    assert info["symmetry"] == P.PPL_SYM_FULL and info["full_available"] == 1
    assert info["full_tbg"] == min(tbg, (v + 15) // 16 * 16)
    assert relerr(got, want) <= TOL, info


@pytest.mark.parametrize("shape", [(5, 20, 60), (4, 38, 19), (12, 18, 9), (24, 64, 128), (7, 82, 33), (3, 130, 12), (9, 100, 24),
                                   (4, 37, 19), (6, 81, 33), (3, 113, 12), (5, 53, 40)])
@pytest.mark.parametrize("tbg", [128, 16])
@pytest.mark.parametrize("form", sorted(FORMS))
def test_full_mode_exact_integers_bit_for_bit(shape, tbg, form):
    o, v, x = shape
    L = I.make_L(v, x, 41, symmetric=True, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 41, symmetric=True, integer=True)  # tau+- (and t2[cc]/2) stay exact integers
    want = oracle.full(L, t2)
    for rep in range(2):
        got = gpu_ladder(L, t2, sym=P.PPL_SYM_FULL, debug=dict(FORMS[form], full_tbg=tbg))
        assert np.array_equal(got, want), rep


@pytest.mark.parametrize("nvirt", [36, 35])
def test_full_mode_accumulates_and_handles_layouts_alpha_beta(nvirt):
    import torch

    o, v, x = 4, nvirt, 19
    L = I.make_L(v, x, 11, symmetric=True)
    t2 = I.make_t2(o, v, 11, symmetric=True)
    R0 = I.make_t2(o, v, 12, symmetric=False)
    got = gpu_ladder(L, t2, R0=R0.copy(), sym=P.PPL_SYM_FULL)
    assert relerr(got, oracle.full(L, t2, R0.copy())) <= TOL
    for t2_layout, r_layout in (("iajb", "iajb"), ("ijab", "iajb"), ("iajb", "ijab")):
        to = lambda a, lay: np.ascontiguousarray(a if lay == "ijab" else a.transpose(0, 2, 1, 3))
        alpha, beta = -0.75, 0.5
        want = oracle.full_ex(L, to(t2, t2_layout), to(R0, r_layout).copy(), t2_layout, r_layout, alpha, beta)
        Ld, td, Rd = torch.from_numpy(L).cuda(), torch.from_numpy(to(t2, t2_layout)).cuda(), torch.from_numpy(to(R0, r_layout)).cuda()
        with P.Plan(o, v, x) as plan:
            plan.set_symmetry(P.PPL_SYM_FULL)
            plan.apply_ex(Ld, td, Rd, t2_layout=t2_layout, r_layout=r_layout, alpha=alpha, beta=beta)
            torch.cuda.synchronize()
        assert relerr(Rd.cpu().numpy(), want) <= TOL, (t2_layout, r_layout)
    # beta == 0 overwrites without reading R (NaN on entry must not leak)
    Rn = torch.full((o, o, v, v), float("nan"), dtype=torch.float64, device="cuda")
    with P.Plan(o, v, x) as plan:
        plan.set_symmetry(P.PPL_SYM_FULL)
        plan.apply_ex(torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda(), Rn, alpha=1.0, beta=0.0)
        torch.cuda.synchronize()
    assert relerr(Rn.cpu().numpy(), oracle.full(L, t2)) <= TOL


def test_full_mode_preconditions_default_and_availability():
    import torch

    # default: PPL_SYM_FULL from nvirt = 52 up (odd nvirt included: padded geometry), PPL_SYM_PAIR_SA below
    with P.Plan(3, 96, 8) as plan:
        assert plan.info()["symmetry"] == P.PPL_SYM_FULL
    with P.Plan(3, 40, 8) as plan:
        info = plan.info()
        assert info["symmetry"] == P.PPL_SYM_PAIR_SA and info["full_available"] == 1
    with P.Plan(3, 97, 8) as plan:
        info = plan.info()
        assert info["symmetry"] == P.PPL_SYM_FULL and info["full_available"] == 1 and info["nvirt"] == 97
    with P.Plan(3, 53, 8) as plan:
        info = plan.info()
        assert info["symmetry"] == P.PPL_SYM_FULL and info["full_available"] == 1
    with P.Plan(3, 51, 8) as plan:
        info = plan.info()
        assert info["symmetry"] == P.PPL_SYM_PAIR_SA and info["full_available"] == 1
    # a cap that holds the PPL_SYM_PAIR_SA plan but not the 16 x nvirt^3 strip: the plan falls back
    o, v, x = 3, 96, 8
    with P.Plan(o, v, x, 40 << 20) as plan:
        info = plan.info()
        assert info["full_available"] == 0 and info["symmetry"] == P.PPL_SYM_PAIR_SA and info["workspace_bytes"] <= 40 << 20
    # ppl_check_inputs: a non-symmetric L violates the precondition of PPL_SYM_FULL only
    Ln = torch.from_numpy(I.make_L(v, x, 3, symmetric=False)).cuda()
    Ls = torch.from_numpy(I.make_L(v, x, 3, symmetric=True)).cuda()
    t2 = torch.from_numpy(I.make_t2(o, v, 3, symmetric=True)).cuda()
    with P.Plan(o, v, x) as plan:
        assert plan.check_inputs(Ls, t2) == 0
        with pytest.raises(P.PplError) as e:
            plan.check_inputs(Ln, t2)
        assert e.value.code == P.PPL_ERR_PRECONDITION
        plan.set_symmetry(P.PPL_SYM_PAIR_SA)
        assert plan.check_inputs(Ln, t2) == 1  # reported, not required


def test_full_mode_flop_accounting():
    """Executed flops: step 0 about 1/8 and step 1 about 1/4 of nominal (plus block-edge overheads)."""
    o, v, x = 20, 200, 800
    with P.Plan(o, v, x) as plan:
        info = plan.info()
    assert info["symmetry"] == P.PPL_SYM_FULL
    nom0, nom1 = 2.0 * x * v**4, 2.0 * o * o * v**4
    # the 16-blocks on the diagonals (d-block == b-block, c-block == a-block) are computed whole: + O(16/nvirt)
    assert 0.125 <= info["flops_step0"] / nom0 <= 0.19, info
    assert 0.25 <= info["flops_step1"] / nom1 <= 0.32, info


def test_full_mode_repeated_apply_and_stream_ordering():
    import torch

    o, v, x = 6, 48, 20
    L = I.make_L(v, x, 5, symmetric=True, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 5, symmetric=True, integer=True)
    want = oracle.full(L, t2)
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    with P.Plan(o, v, x) as plan:
        plan.set_symmetry(P.PPL_SYM_FULL)
        with torch.cuda.stream(s):
            for _ in range(3):
                plan.apply(Ld, td, Rd, s)
            Rd.mul_(0.5)  # ordered after the applies on the same stream
        s.synchronize()
    assert np.array_equal(Rd.cpu().numpy(), 1.5 * want)


@pytest.mark.parametrize("shape,chunk_mb", [((6, 96, 40), 1), ((9, 100, 24), 1), ((5, 130, 20), 1), ((4, 98, 30), 1024),
                                            ((6, 97, 40), 1), ((5, 131, 20), 1)])
def test_host_entry_point_streams_t2_and_R_in_chunks(shape, chunk_mb):
    """ppl_apply_host in PPL_SYM_FULL: t2 and R never sit on the device whole; they pass through
    two staging buffers of `chunk_mb` (several chunks, ragged last one, odd chunk counts) and R accumulates (+=)."""
    o, v, x = shape
    L = I.make_L(v, x, seed=61, symmetric=True)
    t2 = I.make_t2(o, v, seed=61, symmetric=True)
    R0 = I.make_vec(o * o * v * v, 61, 40).reshape(o, o, v, v)
    want = oracle.full(L, t2)
    R = R0.copy()
    with P.Plan(o, v, x, debug=dict(host_chunk_mb=chunk_mb)) as plan:
        assert plan.info()["symmetry"] == P.PPL_SYM_FULL
        for rep in range(2):  # the staging buffers are reused; the second call adds the term again
            h2d, d2h = plan.apply_host(L, t2, R)
            assert h2d == L.nbytes + t2.nbytes + R.nbytes and d2h == R.nbytes
            assert relerr(R - R0, (rep + 1) * want) <= TOL, rep


def test_host_entry_point_exact_integers_chunked():
    o, v, x = 7, 98, 12
    L = I.make_L(v, x, 43, symmetric=True, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 43, symmetric=True, integer=True)
    R = np.zeros((o, o, v, v))
    with P.Plan(o, v, x, debug=dict(host_chunk_mb=1)) as plan:
        plan.apply_host(L, t2, R)
    assert np.array_equal(R, oracle.full(L, t2))


@pytest.mark.parametrize("shape", [(6, 96, 40), (4, 130, 12), (5, 53, 40)])
def test_one_and_two_strips_agree_bit_for_bit(shape):
    """Two strips (step 0 of slab k+1 on its own stream while slab k is folded; the default while a strip is <= 2 GiB)
    and one strip (large, XL) run the same kernels on the same arguments in the same per-buffer order."""
    import torch

    o, v, x = shape
    L = I.make_L(v, x, 71, symmetric=True)
    t2 = I.make_t2(o, v, 71, symmetric=True)
    want = oracle.full(L, t2)
    Ld, td = torch.from_numpy(L).cuda(), torch.from_numpy(t2).cuda()
    got = {}
    for strips in ("1", "2"):
        with P.Plan(o, v, x, 0, debug=dict(full_strips=int(strips))) as plan:
            plan.set_symmetry(P.PPL_SYM_FULL)
            plan.set_graph(0)
            Rd = torch.zeros((o, o, v, v), dtype=torch.float64, device="cuda")
            for _ in range(2):  # twice: events and strips are reused across applies
                plan.apply(Ld, td, Rd)
            torch.cuda.synchronize()
            got[strips] = (Rd.cpu().numpy(), plan.info()["workspace_bytes"])
    assert got["2"][1] > got["1"][1]  # the second strip was really allocated
    assert np.abs(got["2"][0] - 2.0 * want).max() <= 1e-11 * np.abs(2.0 * want).max()
    assert np.array_equal(got["1"][0], got["2"][0])


@pytest.mark.parametrize("shape", [(1, 2, 1), (2, 16, 4), (12, 18, 9), (5, 20, 60), (3, 40, 33), (6, 50, 70), (5, 53, 40), (4, 98, 30), (7, 130, 20)])
@pytest.mark.parametrize("tbg,strips", [(16, 2), (32, 1), (256, 2)])
def test_memory_tight_mode_parity(shape, tbg, strips):
    """PPL_SYM_FULL with a strip of one (slab; b-group) tile: step 0 per tile on the full (b, d) rectangle (no image),
    the fold and the GEMMs unchanged.  Forced here (debug option full_tight); taken by the planner when 16 v^3 does not fit."""
    o, v, x = shape
    L = I.make_L(v, x, 81, symmetric=True)
    t2 = I.make_t2(o, v, 81, symmetric=True)
    R0 = I.make_vec(o * o * v * v, 82, 40).reshape(o, o, v, v)
    want = oracle.full(L, t2, R0.copy())
    got, info = gpu_ladder(L, t2, R0=R0.copy(), sym=P.PPL_SYM_FULL, return_info=True,
                           debug=dict(full_tight=1, full_tbg=tbg, full_strips=strips))
    assert info["full_tight"] == 1 and info["symmetry"] == P.PPL_SYM_FULL, info
    assert relerr(got, want) <= 1e-11, info


@pytest.mark.parametrize("shape", [(5, 20, 60), (4, 38, 19), (24, 64, 128), (7, 82, 33), (3, 130, 12), (5, 53, 40)])
def test_memory_tight_mode_exact_integers_and_flops(shape):
    o, v, x = shape
    L = I.make_L(v, x, 83, symmetric=True, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 83, symmetric=True, integer=True)
    want = oracle.full(L, t2)
    # the reference in the round-1 form (rectangular tiles, plain diagonal chunks): the tight form shares its step 1
    ref, info_ref = gpu_ladder(L, t2, sym=P.PPL_SYM_FULL, return_info=True,
                               debug=dict(full_tbg=32, full_rect_tiles=1, full_no_diag_pack=1))
    got, info = gpu_ladder(L, t2, sym=P.PPL_SYM_FULL, return_info=True, debug=dict(full_tight=1, full_tbg=32))
    assert info["full_tight"] == 1 and info_ref["full_tight"] == 0
    assert np.array_equal(got, want) and np.array_equal(ref, want)
    # same step 1; step 0 on the full rectangle: more than the image mode, at most about twice it
    assert info["flops_step1"] == info_ref["flops_step1"]
    assert info_ref["flops_step0"] <= info["flops_step0"] <= 2.0 * info_ref["flops_step0"]  # equal when one CTA tile covers either
    if v >= 64:
        assert info["flops_step0"] > 1.2 * info_ref["flops_step0"]
    assert info["full_workspace_bytes"] < info_ref["full_workspace_bytes"] or v <= 32


def test_memory_tight_mode_is_what_a_small_cap_gets():
    """Under a cap that has no room for the 16 v^3 strip the planner keeps the 8-fold path in its memory-tight form."""
    import torch

    o, v, x = 6, 128, 40
    L = I.make_L(v, x, 85, symmetric=True)
    t2 = I.make_t2(o, v, 85, symmetric=True)
    want = oracle.full(L, t2)
    with P.Plan(o, v, x, 0) as plan:
        roomy = plan.info()
    assert roomy["full_available"] == 1 and roomy["full_tight"] == 0
    free = torch.cuda.mem_get_info()[0]
    cap = roomy["workspace_bytes"]
    while True:  # shrink the cap until the planner (asked without the device) gives up the 16 v^3 strip (268 MB here)
        cap -= 32 << 20
        dry = P.ppl_plan_dry(o, v, x, workspace_bytes=cap, device_free_bytes=free)
        assert dry["full_available"] == 1, "the tight mode should come before PPL_SYM_FULL is lost"
        if dry["full_tight"]:
            break
    got, info = gpu_ladder(L, t2, sym=P.PPL_SYM_FULL, workspace_bytes=cap, return_info=True)
    assert info["full_tight"] == 1 and info["workspace_bytes"] <= cap, info
    assert relerr(got, want) <= 1e-11
    assert dry["full_tbg"] == info["full_tbg"] and dry["n_tiles"] == info["n_tiles"]


@pytest.mark.parametrize("shape", [(6, 96, 40), (5, 131, 20), (7, 98, 12)])
def test_host_entry_point_in_the_memory_tight_form(shape):
    """ppl_apply_host (t2 and R streamed in chunks) on a plan whose PPL_SYM_FULL buffers are the one-tile-strip kind."""
    o, v, x = shape
    L = I.make_L(v, x, 91, symmetric=True, integer=True)
    t2 = 2.0 * I.make_t2(o, v, 91, symmetric=True, integer=True)
    R0 = I.make_vec(o * o * v * v, 92, 40, integer=True).reshape(o, o, v, v)
    want = oracle.full(L, t2, R0.copy())
    R = R0.copy()
    with P.Plan(o, v, x, debug=dict(host_chunk_mb=1, full_tight=1, full_tbg=32)) as plan:
        info = plan.info()
        assert info["symmetry"] == P.PPL_SYM_FULL and info["full_tight"] == 1
        plan.apply_host(L, t2, R)
    assert np.array_equal(R, want)
