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


def kplus(c, d, v):
    """Packed index of the pair (c <= d): restated from DESIGN.md 6.1 (row c starts so that the index has the parity of d)."""
    return c * v - c * (c + 1) // 2 + (c + 1) // 2 + d


def kminus(c, d, v):
    return c * (2 * v - c - 1) // 2 - c + c // 2 + d


def full_mode_flops_from_the_grid(o, v, x, tbg=256, rect=False, plain_diag=False):
    """PPL_SYM_FULL's executed flops recomputed from the tile grid as DESIGN.md 6.2 describes it (even nvirt):
    step 0: per slab of 16 a's a GEMM of (8 c x 16 a_l = 128)-row tiles x (8 chunks of 16 d = 128)-column tiles over nchol;
    step 1: per W+- tile use 1 (rows of tau x tile rows x packed columns J >= (A0, A0)) and use 2 (rows of tau x packed
    columns J >= (A0 + 16, A0 + 16) x tile rows), counted as the CTA tiles run them (rows in 8s, columns in 128s, k in 16s)."""
    Mp, Mm = o * (o + 1) // 2, o * (o - 1) // 2
    Kp, Km = kplus(v - 1, v - 1, v) + 1, (kminus(v - 2, v - 1, v) + 1 if v >= 2 else 0)
    up = lambda a, b: (a + b - 1) // b * b
    gemm = lambda M, ncols, kr: 0 if min(M, ncols, kr) <= 0 else 2.0 * up(M, 8) * up(ncols, 128) * up(kr, 16)
    f0 = f1 = 0.0
    for A0 in range(0, v, 16):
        r, ta = v - A0, min(16, v - A0)
        dL = A0 + (v - 1 - A0) // 16 * 16
        w = v - dL
        reverse = w < 16 and w * ((r + 15) // 16) < r
        chunks = 0
        for d0 in range(A0, v, 16):
            if reverse and d0 == dL:
                break
            packed = (not plain_diag) and v >= 16 and d0 + 16 <= v
            chunks += (d0 if packed else min(d0 + 16, v)) - A0
        if reverse:
            chunks += w * ((dL - A0) // 16 + 1)
        if not plain_diag and v >= 16:
            chunks += 9 * len([d0 for d0 in range(A0, v, 16) if d0 + 16 <= v])
        f0 += 2.0 * x * (128 * ((r + 7) // 8)) * (128 * ((chunks + 7) // 8))
        c1 = min(A0 + 16, v)
        k0p, k0m = kplus(A0, A0, v), (kminus(A0, A0 + 1, v) - 1 if A0 + 1 < v else Km)
        k1p, k1m = (kplus(c1, c1, v) if c1 < v else Kp), (kminus(c1, c1 + 1, v) - 1 if c1 + 1 < v else Km)
        tiles = []  # (use-1 rows +, -, use-2 rows +, -)
        if rect:
            nblk, per = (r + 15) // 16, tbg // 16
            ng = (nblk + per - 1) // per
            for gi in range(ng):
                N = 16 * 16 * (nblk // ng + (1 if gi < nblk % ng else 0))
                tiles.append((N, N, N, N))
        else:
            lo, hi = k0p, kplus(A0 + ta - 1, v - 1, v) + 1
            NT = 16 * tbg
            ng = (hi - lo + NT - 1) // NT
            chunk = min(NT, up((hi - lo + ng - 1) // ng, 128))
            for kp0 in range(lo, hi, chunk):
                np_ = min(kp0 + chunk, hi) - kp0
                ms = [kminus(a, b, v) for a in range(A0, A0 + ta) for b in range(a + 1, v) if kp0 <= kplus(a, b, v) < kp0 + np_]
                nm = (max(ms) + 1 - (min(ms) & ~1)) if ms else 0
                tiles.append((np_, nm, up(np_, 16), up(nm, 16)))
        for (n1p, n1m, n2p, n2m) in tiles:
            f1 += gemm(Mp, n1p, Kp - k0p) + gemm(Mm, n1m, Km - k0m)
            f1 += gemm(Mp, Kp - (k1p & ~15), n2p) + gemm(Mm, Km - (k1m & ~15), n2m)
    return f0, f1


@pytest.mark.parametrize("name", ["medium", "large", "xl"])
@pytest.mark.parametrize("form", [{}, {"full_rect_tiles": 1, "full_no_diag_pack": 1}, {"full_no_diag_pack": 1}, {"full_rect_tiles": 1}])
def test_full_mode_executed_and_useful_flops_recomputed_from_the_tile_grid(name, form):
    o, v, x = CONFIGS[name]
    d = P.ppl_plan_dry(o, v, x, debug=form)
    f0, f1 = full_mode_flops_from_the_grid(o, v, x, tbg=d["full_tbg"], rect=bool(form.get("full_rect_tiles")),
                                           plain_diag=bool(form.get("full_no_diag_pack")))
    assert d["flops_step0"] == pytest.approx(f0, rel=1e-12)
    assert d["flops_step1"] == pytest.approx(f1, rel=1e-12)
    # useful: the unique (ac|bd) of the 8-fold symmetry, and the whole symmetric S+- applied once (include/ppl.h)
    P2, Q2, Mp, Mm = v * (v + 1) // 2, v * (v - 1) // 2, o * (o + 1) // 2, o * (o - 1) // 2
    assert d["flops_useful_step0"] == pytest.approx(2.0 * x * P2 * (P2 + 1) / 2, rel=1e-12)
    assert d["flops_useful_step1"] == pytest.approx(2.0 * (Mp * P2 * P2 + Mm * Q2 * Q2), rel=1e-12)
    assert d["flops_useful"] == d["flops_useful_step0"] + d["flops_useful_step1"] <= d["flops_executed"]


def test_executed_over_useful_targets():
    """launched / useful flops of the default mode.  Round 1: 1.064 / 1.059 / 1.255."""
    ratio = {}
    for name in ("large", "xl", "medium"):
        d = P.ppl_plan_dry(*CONFIGS[name])
        ratio[name] = d["flops_executed"] / d["flops_useful"]
    assert ratio["xl"] <= 1.03 and ratio["large"] <= 1.045 and ratio["medium"] <= 1.12, ratio
    old = P.ppl_plan_dry(*CONFIGS["medium"], debug={"full_rect_tiles": 1, "full_no_diag_pack": 1})
    assert old["flops_executed"] / old["flops_useful"] > ratio["medium"] + 0.08


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
    # block granularity (16-wide slabs, 128-wide CTA tiles) and shrinks with nvirt
    hi0, hi1 = {"small": (3.0, 1.7), "medium": (1.25, 1.08), "large": (1.10, 1.04), "xl": (1.07, 1.03)}[name]
    assert 1.0 <= d["flops_step0"] / (n0 / 8) <= hi0
    assert 1.0 <= d["flops_step1"] / (n1 / 4) <= hi1
    # per apply: pack, diagonal-block pack [+ pad of L for odd nvirt] + one step 0 per slab + per tile (fold, 2-4 GEMMs, 2 reductions) + unpack
    lo = 3 + d["full_slabs"] + 4 * d["n_tiles"]
    assert lo <= d["launches_per_apply"] <= 4 + d["full_slabs"] + 7 * d["n_tiles"]
    assert d["full_workspace_bytes"] <= d["workspace_bytes"]


def test_plans_recorded_on_the_b200_are_reproduced():
    """Bench lines of round 2 (B200, 148 SMs; gpurun_out/c2_bench_*.json): the same plan comes out without the device."""
    large = P.ppl_plan_dry(40, 400, 1600)
    assert (large["ta"], large["full_tbg"], large["n_tiles"], large["full_slabs"], large["splitk"]) == (16, 256, 34, 25, 15)
    assert large["launches_per_apply"] == 264 and large["workspace_bytes"] == 22866753536
    assert large["flops_executed"] == 32103848542208.0 and large["flops_nominal"] == 163840000000000.0
    xl = P.ppl_plan_dry(60, 600, 2400)
    assert (xl["n_tiles"], xl["full_slabs"], xl["splitk"], xl["workspace_bytes"]) == (66, 38, 15, 66550880768)
    assert xl["flops_executed"] == 319215647883264.0
    medium = P.ppl_plan_dry(20, 200, 800)
    assert (medium["full_tbg"], medium["n_tiles"], medium["splitk"]) == (208, 13, 11) and medium["flops_executed"] == 719121612800.0
    # the round-1 form of the tiles (debug options) still plans what round 1 recorded (profiles/r01_large_full.md)
    r1 = P.ppl_plan_dry(40, 400, 1600, debug={"full_rect_tiles": 1, "full_no_diag_pack": 1})
    assert (r1["n_tiles"], r1["launches_per_apply"]) == (34, 263)
    tiny = P.ppl_plan_dry(5, 20, 60, debug={"no_small_fused": 1})  # the tiled plan below nvirt = 52: PPL_SYM_PAIR_SA, one tile
    assert (tiny["symmetry"], tiny["n_tiles"], tiny["ta"], tiny["launches_per_apply"]) == (P.PPL_SYM_PAIR_SA, 1, 20, 6)
    # what the product runs at tiny and small: one fused launch over (a; 4 b's) work items, pair symmetry
    for shape, items in (((5, 20, 60), sum((20 - a + 3) // 4 for a in range(20))), ((5, 53, 232), sum((53 - a + 3) // 4 for a in range(53)))):
        d = P.ppl_plan_dry(*shape, debug={"no_small_fused": 0})
        assert (d["small_fused"], d["launches_per_apply"], d["n_tiles"]) == (1, 1 + (shape[1] & 1), items)
        o, v, x = shape
        w8, pairs, k16 = (v + 7) // 8 * 8, v * (v + 1) // 2, (x + 15) // 16 * 16
        assert d["flops_step0"] == 2.0 * k16 * w8 * w8 * pairs and d["flops_step1"] == 2.0 * o * o * w8 * w8 * pairs


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


def test_planner_builds_with_gpp_alone_and_agrees_with_the_library(tmp_path):
    """csrc/ppl_plan.cpp is plain C++: no nvcc, no CUDA call, no link dependency (CUDA headers serve as type definitions
    only).  Built here with g++ into a library of its own, ppl_plan_dry gives the same answers as the one inside libppl.so."""
    import ctypes
    import os
    import shutil
    import subprocess

    from paper_2603_20912_b200 import _build
    from paper_2603_20912_b200.binding import ppl_info_t

    gpp = shutil.which("g++")
    inc = os.path.join(os.path.dirname(_build.nvcc()), "..", "include")
    so = str(tmp_path / "libppl_plan_only.so")
    subprocess.check_call([gpp, "-std=c++17", "-O2", "-shared", "-fPIC", "-I", inc, "-o", so, "ppl_plan.cpp"], cwd=_build.CSRC)
    assert "libcudart" not in subprocess.check_output(["ldd", so], text=True)
    lib = ctypes.CDLL(so)
    lib.ppl_plan_dry.restype = ctypes.c_int
    lib.ppl_plan_dry.argtypes = [ctypes.c_int] * 3 + [ctypes.c_size_t] * 2 + [ctypes.c_int] * 2 + [ctypes.POINTER(ppl_info_t)]
    for shape in ((5, 20, 60), (5, 53, 232), (20, 200, 800), (60, 600, 2400)):
        for cap in (0, 6 << 30):
            out = ppl_info_t()
            rc = lib.ppl_plan_dry(*shape, cap, 170 << 30, 148, -1, ctypes.byref(out))
            assert rc == P.PPL_OK
            assert out.asdict() == P.ppl_plan_dry(*shape, workspace_bytes=cap, debug={"no_small_fused": 0})


def test_ragged_tile_edges_down_to_a_quarter_are_candidates():
    """Un-packed modes: an edge whose last block is ragged down to T/4 competes (the cost model counts its tiles); the round-1
    rule (T/2) kept T = 16 out at nvirt = 900 and cost 4 % on the paper's Table 3 row N = 1000 (measured: 571 -> 549 s)."""
    d = P.ppl_plan_dry(100, 900, 5000, workspace_bytes=8 << 30, mode=P.PPL_SYM_NONE)
    assert (d["ta"], d["n_ablocks"], d["n_tiles"]) == (16, 57, 57 * 57)
    d = P.ppl_plan_dry(20, 200, 800, mode=P.PPL_SYM_PAIR)
    assert d["ta"] == 32 and d["n_ablocks"] == 7  # ragged last block of 8 = T/4
    for v in (97, 130, 171, 200, 333):  # and never a last block below T/4
        d = P.ppl_plan_dry(6, v, 64, mode=P.PPL_SYM_NONE, debug={"no_small_fused": 1})
        T = d["ta"]
        nblk = (v + T - 1) // T
        assert nblk == 1 or 4 * (v - (nblk - 1) * T) >= T, (v, T)
