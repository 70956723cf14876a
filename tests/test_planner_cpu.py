"""-m "not gpu": the planner (the analogue of the paper's memory functions, Table 1 / Fig. 3,
PAPER.md:99-116, 134) through ppl_plan_dry -- the host half of ppl_plan for a stated device, no CUDA call.

Checked here, without a GPU: the flop accounting bench.py's `value` and `roofline` rest on (F_nom = 2 x v^4 + 2 o^2 v^4;
F_exec per symmetry mode, recomputed from the tile grid), tile counts, the packed geometry, workspace caps and the
fallbacks under them, and that the plans recorded from the B200 runs (profiles/r01_large_full.md) are reproduced.
"""
import pytest

import paper_2603_20912_b200 as P

CONFIGS = {"tiny": (5, 20, 60), "small": (5, 53, 232), "medium": (20, 200, 800), "large": (40, 400, 1600), "xl": (60, 600, 2400)}
SHAPES = list(CONFIGS.values()) + [(1, 1, 1), (2, 1, 3), (1, 5, 1), (3, 7, 5), (7, 81, 300), (10, 100, 400), (12, 18, 9), (100, 700, 4000)]


def f_nom(o, v, x):
    return 2.0 * x * v ** 4 + 2.0 * o * o * v ** 4


def tile_edges(v, T):
    return [min(T, v - a0) for a0 in range(0, v, T)]


@pytest.mark.parametrize("shape", SHAPES)
def test_nominal_flops_and_unpacked_modes(shape):
    o, v, x = shape
    none = P.ppl_plan_dry(o, v, x, mode=P.PPL_SYM_NONE)
    pair = P.ppl_plan_dry(o, v, x, mode=P.PPL_SYM_PAIR)
    for d in (none, pair):
        assert (d["nocc"], d["nvirt"], d["nchol"]) == shape
        assert d["flops_nominal"] == f_nom(o, v, x)
        assert d["flops_executed"] == d["flops_step0"] + d["flops_step1"]
        assert d["ta"] == d["tb"] and 1 <= d["ta"] <= v and 1 <= d["ring"] <= 3 and d["splitk"] >= 1
    # no symmetry: every (A, B) tile runs, executed == nominal
    e = tile_edges(v, none["ta"])
    assert none["n_tiles"] == len(e) ** 2
    assert none["flops_executed"] == pytest.approx(f_nom(o, v, x), rel=1e-12)
    # pair symmetry: tiles A <= B only (F_exec = F_nom (nb+1)/(2 nb) when T divides v)
    e = tile_edges(v, pair["ta"])
    nb = len(e)
    assert pair["n_tiles"] == nb * (nb + 1) // 2
    cols = sum(e[i] * e[j] for i in range(nb) for j in range(i, nb))
    assert pair["flops_step0"] == pytest.approx(2.0 * x * cols * v * v, rel=1e-12)
    assert pair["flops_step1"] == pytest.approx(2.0 * o * o * cols * v * v, rel=1e-12)
    if v % pair["ta"] == 0:
        assert pair["flops_executed"] == pytest.approx(f_nom(o, v, x) * (nb + 1) / (2 * nb), rel=1e-12)


@pytest.mark.parametrize("shape", SHAPES)
def test_packed_geometry_and_pair_sa_accounting(shape):
    o, v, x = shape
    d = P.ppl_plan_dry(o, v, x, mode=P.PPL_SYM_PAIR_SA)
    vp = v + (v & 1)  # packed operands live in the geometry of nvirt rounded up to even (DESIGN 6.1)
    assert d["vec16"] == (1 if v % 2 == 0 else 0)
    assert (d["sa_rows_plus"], d["sa_rows_minus"]) == (o * (o + 1) // 2, o * (o - 1) // 2)
    assert (d["sa_k_plus"], d["sa_k_minus"]) == (vp * (vp + 1) // 2, vp * (vp - 1) // 2)
    e = tile_edges(v, d["ta"])
    cols = sum(e[i] * e[j] for i in range(len(e)) for j in range(i, len(e)))
    assert d["flops_step0"] == pytest.approx(2.0 * x * cols * v * v, rel=1e-12)  # step 0 as in PPL_SYM_PAIR
    want1 = 2.0 * cols * (d["sa_rows_plus"] * d["sa_k_plus"] + d["sa_rows_minus"] * d["sa_k_minus"])
    assert d["flops_step1"] == pytest.approx(want1, rel=1e-12)                    # a quarter of nominal, asymptotically
    for key in ("sa_tile_m_plus", "sa_tile_m_minus", "step1_tile_m"):
        assert d[key] % 16 == 0 and 16 <= d[key] <= 160  # CTA tile rows 16*NI, NI = 1..10


@pytest.mark.parametrize("name", ["small", "medium", "large", "xl"])
def test_full_mode_accounting(name):
    o, v, x = CONFIGS[name]
    d = P.ppl_plan_dry(o, v, x)
    assert d["symmetry"] == P.PPL_SYM_FULL and d["full_available"] == 1  # the default from nvirt = 52
    vp = v + (v & 1)
    assert d["full_slabs"] == (vp + 15) // 16 and d["ta"] == 16
    assert d["full_tbg"] % 16 == 0 and d["n_tiles"] >= d["full_slabs"]
    n0, n1 = 2.0 * x * v ** 4, 2.0 * o * o * v ** 4
    # the 8-fold symmetry bounds the saving: never below 1/8 (step 0) and 1/4 (step 1) of nominal; the excess is the
    # block granularity (16-wide slabs, 128-wide CTA tiles, zero rows of diagonal blocks) and shrinks with nvirt
    hi0, hi1 = {"small": (3.5, 1.7), "medium": (1.45, 1.12), "large": (1.15, 1.04), "xl": (1.14, 1.04)}[name]
    assert 1.0 <= d["flops_step0"] / (n0 / 8) <= hi0
    assert 1.0 <= d["flops_step1"] / (n1 / 4) <= hi1
    # per apply: pack [+ pad of L for odd nvirt] + one step 0 per slab + per tile (fold, 2-4 GEMMs, 2 reductions) + unpack
    lo = 2 + d["full_slabs"] + 4 * d["n_tiles"]
    assert lo <= d["launches_per_apply"] <= 3 + d["full_slabs"] + 7 * d["n_tiles"]
    assert d["full_workspace_bytes"] <= d["workspace_bytes"]


def test_plans_recorded_on_the_b200_are_reproduced():
    """profiles/r01_large_full.md / bench lines of round 1 (B200, 148 SMs): the same plan comes out without the device."""
    large = P.ppl_plan_dry(40, 400, 1600)
    assert (large["ta"], large["full_tbg"], large["n_tiles"], large["full_slabs"], large["splitk"]) == (16, 256, 34, 25, 15)
    assert large["launches_per_apply"] == 263 and large["workspace_bytes"] == 22777048064
    assert large["flops_executed"] == 32683249664000.0 and large["flops_nominal"] == 163840000000000.0
    xl = P.ppl_plan_dry(60, 600, 2400)
    assert (xl["n_tiles"], xl["full_slabs"], xl["splitk"], xl["workspace_bytes"]) == (66, 38, 9, 66028931072)
    assert xl["flops_executed"] == 329273179299840.0
    medium = P.ppl_plan_dry(20, 200, 800)
    assert (medium["full_tbg"], medium["n_tiles"], medium["splitk"]) == (208, 13, 11) and medium["flops_executed"] == 803177799680.0
    tiny = P.ppl_plan_dry(5, 20, 60)  # below nvirt = 52: PPL_SYM_PAIR_SA, one tile
    assert (tiny["symmetry"], tiny["n_tiles"], tiny["ta"], tiny["launches_per_apply"]) == (P.PPL_SYM_PAIR_SA, 1, 20, 6)


def test_workspace_caps_and_fallbacks():
    o, v, x = CONFIGS["large"]
    auto = P.ppl_plan_dry(o, v, x)
    prev = auto["workspace_bytes"]
    for gb in (64, 24, 12, 6, 3, 1):
        cap = gb << 30
        d = P.ppl_plan_dry(o, v, x, workspace_bytes=cap)
        assert d["workspace_bytes"] <= cap
        assert d["workspace_bytes"] <= prev  # a smaller cap never plans a larger workspace
        prev = d["workspace_bytes"]
        if not d["full_available"]:
            assert d["symmetry"] in (P.PPL_SYM_PAIR_SA, P.PPL_SYM_PAIR)
            with pytest.raises(P.PplError):
                P.ppl_plan_dry(o, v, x, workspace_bytes=cap, mode=P.PPL_SYM_FULL)
    assert P.ppl_plan_dry(o, v, x, workspace_bytes=3 << 30)["full_available"] == 0   # the 8.2 GB strip does not fit
    with pytest.raises(P.PplError):
        P.ppl_plan_dry(o, v, x, workspace_bytes=1 << 20)                              # not even one tile
    # a device with little free memory behaves like a cap
    small_dev = P.ppl_plan_dry(o, v, x, device_free_bytes=4 << 30)
    assert small_dev["workspace_bytes"] <= 0.9 * (4 << 30) and small_dev["full_available"] == 0
    # near the HBM limit (DESIGN 6.2): (80, 800, 3200) with 82 GB of inputs resident leaves no room for the 65.5 GB strip
    # of PPL_SYM_FULL: the plan keeps the 8-fold path in its memory-tight form (a strip of one (slab; b-group) tile)
    big = P.ppl_plan_dry(80, 800, 3200, device_free_bytes=(178 - 82) << 30)
    assert big["full_available"] == 1 and big["full_tight"] == 1 and big["symmetry"] == P.PPL_SYM_FULL
    assert big["workspace_bytes"] <= 0.9 * ((178 - 82) << 30)
    n0, n1 = 2.0 * 3200 * 800 ** 4, 2.0 * 6400 * 800 ** 4
    assert 2.0 <= big["flops_step0"] / (n0 / 8) <= 2.3    # the full (b, d) rectangle: a quarter of nominal, not an eighth
    assert 1.0 <= big["flops_step1"] / (n1 / 4) <= 1.04   # step 1 as in the roomy plan
    # between "fits" and "PPL_SYM_FULL lost" there is always the tight form
    seen_tight = False
    for mb in range(22000, 2000, -500):
        d = P.ppl_plan_dry(o, v, x, workspace_bytes=mb << 20)
        seen_tight = seen_tight or d["full_tight"] == 1
        if not d["full_available"]:
            break
        assert d["full_tight"] in (0, 1) and d["symmetry"] == P.PPL_SYM_FULL
    assert seen_tight


@pytest.mark.parametrize("sms", [1, 8, 132, 148, 160])
def test_other_sm_counts_and_bad_arguments(sms):
    d = P.ppl_plan_dry(20, 200, 800, num_sms=sms)
    assert d["flops_nominal"] == f_nom(20, 200, 800) and d["splitk"] >= 1 and d["n_tiles"] >= 1
    for bad in ((0, 10, 10), (10, 0, 10), (10, 10, 0), (5, 40000, 5), (40000, 5, 5)):
        with pytest.raises(P.PplError):
            P.ppl_plan_dry(*bad, num_sms=sms)
    with pytest.raises(P.PplError):
        P.ppl_plan_dry(5, 20, 60, num_sms=0)
    with pytest.raises(P.PplError):
        P.ppl_plan_dry(5, 20, 60, mode=7)
