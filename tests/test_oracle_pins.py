"""Pins for the CPU oracle (oracle/ppl_oracle.c) -- CPU only, no GPU, no CUDA path.

The paper prints no worked numerical example of the ladder term, so the oracle is pinned to what
the paper's equations and the mathematics fix:

  hand-worked 2x2 example of eq. (6)                    tests/golden/hand_2x2.txt
  brute force, two ways (explicit W; 7-index long double)   P1   (north_star i)
  nchol = 1  ->  R_ij = L0 T_ij L0^T (library matmul)        P2   (north_star v)
  identity L ->  R = (sum s_P^2) t2                          P3
  rank-1 L   ->  closed form                                 P4
  unit impulse -> R[i0,j0,a,b] = sum_P L[P,a,c0] L[P,b,d0]   P5   (pairing a-c, b-d: reading A2)
  linearity, zero, accumulate semantics                      P6   (north_star ii, iii)
  output pair symmetry + negative control                    P7   (north_star iv)
  projection identity (oracle.project vs oracle.full)        P8
  exact integers vs int64 arithmetic, bit for bit            P9
  numpy einsum 'Pac,Pbd,ijcd->ijab' and the paper's two-step tensordot  P10

Each pin is chosen so that a plausible mistake (dropped term, wrong sign or index, transposed
operand, wrong pairing, overwrite instead of accumulate) fails at least one of them.
"""
import os

import numpy as np
import pytest

import oracle
import ppl_inputs as I

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
RTOL = 1e-13  # oracle vs another FP64 evaluation order: ~1e-15 expected, 1e-13 asserted

ODD_SHAPES = [(1, 1, 1), (2, 1, 3), (1, 5, 1), (3, 7, 5), (2, 9, 4), (3, 6, 7)]


def rel(a, b):
    m = np.abs(b).max()
    return np.abs(a - b).max() / (m if m > 0 else 1.0)


def rand_inputs(o, v, x, seed=1, symmetric=False, integer=False):
    return I.make_L(v, x, seed, symmetric, integer), I.make_t2(o, v, seed, symmetric, integer)


# ----------------------------------------------------------------------------- golden fixtures
def _read_hand():
    d = {}
    for line in open(os.path.join(GOLD, "hand_2x2.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *vals = line.split()
        d[k] = np.array([float(s) for s in vals])
    return d


@pytest.mark.parametrize("fn", ["full", "bruteforce_w", "bruteforce_direct", "columns", "project"])
def test_hand_worked_2x2(fn):
    """eq. (6), by hand; non-symmetric L and t so the pairing and operand order matter."""
    d = _read_hand()
    L = d["L"].reshape(1, 2, 2).copy()
    t2 = d["t2"].reshape(1, 1, 2, 2).copy()
    want, bad = d["R"].reshape(2, 2), d["Rbad"].reshape(2, 2)
    if fn == "columns":
        pairs = [(0, 0), (0, 1), (1, 0), (1, 1)]
        got = oracle.columns(L, t2, pairs).reshape(2, 2)
    elif fn == "project":
        got = np.empty((2, 2))
        for a in range(2):
            for b in range(2):
                got[a, b] = oracle.project(L, t2, np.eye(2)[a], np.eye(2)[b])[0][0, 0]
    else:
        got = getattr(oracle, fn)(L, t2)[0, 0]
    assert np.array_equal(got, want)  # small integers: exact
    assert not np.array_equal(got, bad)


def test_golden_tiny_samples():
    """Regression anchor: entries of config 0 written by tests/golden/make_golden.py (oracle only)."""
    L, t2 = I.make_config("tiny", seed=0)
    R = oracle.full(L, t2)
    n = 0
    for line in open(os.path.join(GOLD, "oracle_tiny_samples.txt")):
        if line.startswith("#"):
            continue
        i, j, a, b, hx, _ = line.split()
        want = float.fromhex(hx)
        assert abs(R[int(i), int(j), int(a), int(b)] - want) <= 1e-12 * 21.65
        n += 1
    assert n == 7


# ----------------------------------------------------------------------------- P1 brute force
@pytest.mark.parametrize("shape", [(5, 20, 60)] + ODD_SHAPES)
@pytest.mark.parametrize("symmetric", [True, False])
def test_P1_bruteforce(shape, symmetric):
    o, v, x = shape
    L, t2 = rand_inputs(o, v, x, seed=3, symmetric=symmetric)
    R = oracle.full(L, t2)
    assert rel(R, oracle.bruteforce_w(L, t2)) <= RTOL
    assert rel(R, oracle.bruteforce_direct(L, t2)) <= RTOL


def test_P1_columns_equal_full():
    L, t2 = rand_inputs(3, 11, 9, seed=5)
    R = oracle.full(L, t2)
    pairs = [(a, b) for a in range(11) for b in range(11)]
    C = oracle.columns(L, t2, pairs)  # [121, 3, 3]
    assert np.array_equal(C.reshape(11, 11, 3, 3).transpose(2, 3, 0, 1), R)  # same code path, same order


# ----------------------------------------------------------------------------- P2 nchol = 1
@pytest.mark.parametrize("shape", [(5, 20, 1), (5, 53, 1), (2, 7, 1)])
def test_P2_nchol1_triple_product(shape):
    o, v, _ = shape
    L, t2 = rand_inputs(o, v, 1, seed=7, symmetric=False)
    R = oracle.full(L, t2)
    want = np.matmul(np.matmul(L[0], t2), L[0].T)  # R_ij = L0 T_ij L0^T  (textbook triple product)
    assert rel(R, want) <= RTOL
    # transposed operand must fail (the test has power)
    assert rel(R, np.matmul(np.matmul(L[0].T, t2), L[0])) > 1e-3


# ----------------------------------------------------------------------------- P3 identity L
def test_P3_identity_L():
    o, v, x = 4, 13, 6
    s = np.arange(1, x + 1, dtype=np.float64) * 0.5
    L = np.ascontiguousarray(s[:, None, None] * np.eye(v)[None])
    t2 = I.make_t2(o, v, 11, symmetric=False)
    R = oracle.full(L, t2)
    assert rel(R, (s**2).sum() * t2) <= RTOL


# ----------------------------------------------------------------------------- P4 rank-1 L
def test_P4_rank1_L():
    o, v, x = 3, 17, 5
    al = I.make_vec(x, 1, 20)
    u = I.make_vec(v, 1, 21)
    L = np.ascontiguousarray(al[:, None, None] * u[None, :, None] * u[None, None, :])
    t2 = I.make_t2(o, v, 13, symmetric=False)
    R = oracle.full(L, t2)
    utu = np.einsum("c,ijcd,d->ij", u, t2, u)
    want = (al**2).sum() * utu[:, :, None, None] * u[None, None, :, None] * u[None, None, None, :]
    assert rel(R, want) <= RTOL


# ----------------------------------------------------------------------------- P5 unit impulse
def test_P5_impulse_pins_index_pairing():
    o, v, x = 3, 8, 6
    L = I.make_L(v, x, 17, symmetric=False)
    i0, j0, c0, d0 = 1, 2, 3, 5
    t2 = np.zeros((o, o, v, v))
    t2[i0, j0, c0, d0] = 1.0
    R = oracle.full(L, t2)
    want = np.einsum("Pa,Pb->ab", L[:, :, c0], L[:, :, d0])  # sum_P L[P,a,c0] L[P,b,d0]
    assert rel(R[i0, j0], want) <= RTOL
    wrong = np.einsum("Pa,Pb->ab", L[:, :, d0], L[:, :, c0])  # (ad|bc) pairing
    assert rel(R[i0, j0], wrong) > 1e-3
    mask = np.ones((o, o), bool)
    mask[i0, j0] = False
    assert np.all(R[mask] == 0.0)  # no cross-talk between (i,j) blocks


# ----------------------------------------------------------------------------- P6 linearity / zero / accumulate
def test_P6_linearity_zero_accumulate():
    o, v, x = 3, 9, 7
    L = I.make_L(v, x, 19, symmetric=False)
    t = I.make_t2(o, v, 19, symmetric=False)
    tp = I.make_t2(o, v, 23, symmetric=False)
    al, be = 0.75, -1.5
    lhs = oracle.full(L, al * t + be * tp)
    rhs = al * oracle.full(L, t) + be * oracle.full(L, tp)
    assert rel(lhs, rhs) <= RTOL
    # zero t2 leaves R bitwise unchanged
    R0 = I.make_t2(o, v, 29, symmetric=False)
    R = R0.copy()
    oracle.full(L, np.zeros_like(t), R)
    assert np.array_equal(R, R0)
    # accumulate (+=, coefficient 1): R_in + term, and calling twice adds twice
    R = R0.copy()
    oracle.full(L, t, R)
    term = oracle.full(L, t)
    assert rel(R - R0, term) <= 1e-12
    oracle.full(L, t, R)
    assert rel(R - R0, 2 * term) <= 1e-12


# ----------------------------------------------------------------------------- P7 output symmetry
def test_P7_pair_symmetry_and_negative_control():
    o, v, x = 4, 10, 8
    L = I.make_L(v, x, 31, symmetric=False)  # holds for ANY L
    ts = I.make_t2(o, v, 31, symmetric=True)
    assert np.array_equal(ts, ts.transpose(1, 0, 3, 2))
    R = oracle.full(L, ts)
    assert rel(R, R.transpose(1, 0, 3, 2)) <= RTOL
    tn = I.make_t2(o, v, 31, symmetric=False)
    Rn = oracle.full(L, tn)
    assert rel(Rn, Rn.transpose(1, 0, 3, 2)) > 1e-3  # non-symmetric t2 breaks it


# ----------------------------------------------------------------------------- P8 projection
@pytest.mark.parametrize("shape", [(5, 20, 60), (3, 7, 5)])
def test_P8_projection_matches_full(shape):
    o, v, x = shape
    L, t2 = rand_inputs(o, v, x, seed=37, symmetric=False)
    R = oracle.full(L, t2)
    for k in range(4):
        u, w = I.make_vec(v, 37, 40 + 2 * k), I.make_vec(v, 37, 41 + 2 * k)
        got, scale = oracle.project(L, t2, u, w)
        want = np.einsum("a,ijab,b->ij", u, R, w)
        assert np.abs(got - want).max() <= 1e-13 * scale.max()
    # and against an independent numpy evaluation of the identity's right-hand side
    u, w = I.make_vec(v, 37, 50), I.make_vec(v, 37, 51)
    M = np.einsum("Pc,Pd->cd", np.einsum("a,Pac->Pc", u, L), np.einsum("b,Pbd->Pd", w, L))
    got, _ = oracle.project(L, t2, u, w)
    assert rel(got, np.einsum("cd,ijcd->ij", M, t2)) <= RTOL


# ----------------------------------------------------------------------------- P9 exact integers
@pytest.mark.parametrize("shape", [(5, 20, 60), (3, 7, 5), (5, 53, 16)])
def test_P9_exact_integers(shape):
    o, v, x = shape
    L, t2 = rand_inputs(o, v, x, seed=41, symmetric=True, integer=True)
    Li, ti = L.astype(np.int64), t2.astype(np.int64)
    W = np.einsum("Pac,Pbd->abcd", Li, Li)
    want = np.einsum("abcd,ijcd->ijab", W, ti)  # int64: exact
    for fn in (oracle.full, oracle.bruteforce_direct):
        if fn is oracle.bruteforce_direct and v > 20:
            continue
        got = fn(L, t2)
        assert np.array_equal(got, want.astype(np.float64))  # bit for bit, any summation order


# ----------------------------------------------------------------------------- P10 other opinions
@pytest.mark.parametrize("name", ["tiny", "small"])
def test_P10_numpy_einsum_and_paper_tensordot(name):
    L, t2 = I.make_config(name, seed=0)
    R = oracle.full(L, t2)
    if name == "tiny":  # numpy's einsum path is slow (no BLAS) beyond tiny sizes
        assert rel(R, np.einsum("Pac,Pbd,ijcd->ijab", L, L, t2, optimize=True)) <= RTOL
    # the paper's two steps with its axes: tensordot over x, then over (c,d)
    W = np.tensordot(L, L, axes=(0, 0))  # [a,c,b,d]
    out = np.tensordot(W, t2, axes=([1, 3], [2, 3]))  # [a,b,i,j]
    assert rel(R, out.transpose(2, 3, 0, 1)) <= RTOL


def test_oracle_self_error_bound():
    """The FP64 oracle vs the long-double 7-index sum on config 0: its own rounding error, which
    the 1e-11 GPU tolerance must dominate by orders of magnitude (reading A13)."""
    L, t2 = I.make_config("tiny", seed=0)
    assert rel(oracle.full(L, t2), oracle.bruteforce_direct(L, t2)) <= 1e-14


# ----------------------------------------------------------------------------- input recipe
def test_input_recipe():
    """BASELINE.json configs: symmetric L with exp(-3P/nchol) decay, t2 ~ N(0,1e-2) pair-symmetric."""
    o, v, x = 5, 53, 232
    L, t2 = I.make_config("small", seed=0)
    assert L.shape == (x, v, v) and t2.shape == (o, o, v, v)
    assert np.array_equal(L, L.transpose(0, 2, 1))
    assert np.array_equal(t2, t2.transpose(1, 0, 3, 2))
    assert abs(t2.std() - 0.1) < 0.003 and abs(t2.mean()) < 0.003
    sd = L.reshape(x, -1).std(axis=1)
    want = np.exp(-3.0 * np.arange(x) / x)
    assert np.all(np.abs(sd / want - 1.0) < 0.08)
    # seeded and reproducible; different seeds differ
    assert np.array_equal(L, I.make_L(v, x, 0))
    assert not np.array_equal(L, I.make_L(v, x, 1))
    p = I.sample_pairs(400, 64, seed=0)
    assert p.min() >= 0 and p.max() < 400 and len({tuple(r) for r in p}) == len(p)


# ------------------------------------------------------------------ NEXT-1: paper layouts, alpha/beta
@pytest.mark.parametrize("shape", [(3, 4, 5), (2, 7, 3), (1, 1, 1), (4, 3, 2)])
def test_full_ex_is_the_papers_einsum_string(shape):
    """PAPER.md:75 prints the contraction as 'xac,xbd,icjd->iajb': evaluate exactly that string with
    numpy on arrays stored the paper's way and compare with oracle.full_ex in every layout combination."""
    o, v, x = shape
    L = I.make_L(v, x, 3, symmetric=False)
    t_ijcd = I.make_t2(o, v, 3, symmetric=False)
    t_icjd = np.ascontiguousarray(t_ijcd.transpose(0, 2, 1, 3))
    want_iajb = np.einsum("xac,xbd,icjd->iajb", L, L, t_icjd)
    want_ijab = np.ascontiguousarray(want_iajb.transpose(0, 2, 1, 3))
    for tl, t in (("ijab", t_ijcd), ("iajb", t_icjd)):
        for rl, want in (("ijab", want_ijab), ("iajb", want_iajb)):
            assert rel(oracle.full_ex(L, t, None, tl, rl), want) <= RTOL
    # the 'ijab'/'ijab' case is oracle.full itself
    assert rel(oracle.full_ex(L, t_ijcd), oracle.full(L, t_ijcd)) <= RTOL


def test_full_ex_alpha_beta_and_overwrite():
    o, v, x = 3, 5, 4
    L, t = rand_inputs(o, v, x, seed=5)
    term = oracle.full(L, t)
    R0 = I.make_vec(o * o * v * v, 5, 40).reshape(o, o, v, v)
    got = oracle.full_ex(L, t, R0.copy(), alpha=-0.5, beta=2.0)
    assert rel(got, 2.0 * R0 - 0.5 * term) <= RTOL
    # beta = 0 overwrites and never reads R (NaN on entry must not propagate)
    got = oracle.full_ex(L, t, np.full((o, o, v, v), np.nan), alpha=3.0, beta=0.0)
    assert np.isfinite(got).all() and rel(got, 3.0 * term) <= RTOL
    # wrong-layout negative control: reading 'icjd' storage as 'ijcd' gives a different answer
    o, v, x = 3, 3, 2  # o == v so the shapes coincide and only the index meaning differs
    L, t = rand_inputs(o, v, x, seed=6)
    a = oracle.full_ex(L, t, None, "ijab", "ijab")
    b = oracle.full_ex(L, t.reshape(o, v, o, v), None, "iajb", "ijab")
    assert rel(a, b) > 1e-3


# ------------------------------------------------ NEXT-4: symmetric / antisymmetric repacking identity
@pytest.mark.parametrize("shape", [(3, 5, 4), (4, 6, 3), (1, 4, 2), (2, 1, 3)])
def test_symmetric_antisymmetric_packing_identity(shape):
    """For pair-symmetric t2 (t[i,j,c,d] = t[j,i,d,c]) and ANY L the term splits as
         R[i,j,a,b] = R+ + R-,  R[j,i,a,b] = R+ - R-   (i <= j),
         R+-[ij,ab] = sum_{c<=d} W+-[ab,cd] tau+-[ij,cd],
         W+-[ab,cd] = (ac|bd) +- (ad|bc)  (c<d; W+[ab,cc] = (ac|bc)),
         tau+-[ij,cd] = (t[ij,cd] +- t[ij,dc]) / 2  (c<d; tau+[ij,cc] = t[ij,cc])
    -- the packing the CUDA path's PPL_SYM_PAIR_SA mode uses.  Built here with numpy from
    the definitions and checked against the oracle, so the identity itself is pinned on the CPU."""
    o, v, x = shape
    L = I.make_L(v, x, 9, symmetric=False)
    t = I.make_t2(o, v, 9, symmetric=True)
    want = oracle.full(L, t)
    X = np.einsum("Pac,Pbd->abcd", L, L)
    cu, du = np.triu_indices(v)
    cs, ds = np.triu_indices(v, 1)
    off = (cu != du).astype(np.float64)
    Wp = X[:, :, cu, du] + off * X[:, :, du, cu]
    Wm = X[:, :, cs, ds] - X[:, :, ds, cs]
    tp = np.where(cu == du, 1.0, 0.5) * (t[:, :, cu, du] + off * t[:, :, du, cu])
    tm = 0.5 * (t[:, :, cs, ds] - t[:, :, ds, cs])
    Rp = np.einsum("abk,ijk->ijab", Wp, tp)
    Rm = np.einsum("abk,ijk->ijab", Wm, tm)
    got = np.zeros_like(want)
    for i in range(o):
        for j in range(i, o):
            got[i, j] = Rp[i, j] + Rm[i, j]
            if i != j:
                got[j, i] = Rp[i, j] - Rm[i, j]
    assert rel(got, want) <= RTOL
    # negative control: without pair symmetry the reconstruction from i <= j fails
    if o > 1 and v > 1:
        tn = I.make_t2(o, v, 9, symmetric=False)
        wantn = oracle.full(L, tn)
        tpn = np.where(cu == du, 1.0, 0.5) * (tn[:, :, cu, du] + off * tn[:, :, du, cu])
        tmn = 0.5 * (tn[:, :, cs, ds] - tn[:, :, ds, cs])
        Rpn = np.einsum("abk,ijk->ijab", Wp, tpn)
        Rmn = np.einsum("abk,ijk->ijab", Wm, tmn)
        gotn = np.zeros_like(wantn)
        for i in range(o):
            for j in range(i, o):
                gotn[i, j] = Rpn[i, j] + Rmn[i, j]
                if i != j:
                    gotn[j, i] = Rpn[i, j] - Rmn[i, j]
        assert rel(gotn, wantn) > 1e-3


# ------------------------------------------------ full 8-fold symmetry: the "hook" decomposition of PPL_SYM_FULL
def _kp(c, d, v):
    return c * v - c * (c - 1) // 2 + (d - c)


def _km(c, d, v):
    return c * (2 * v - c - 1) // 2 + (d - c - 1)


def _full_symmetry_emulation(L, t2, T):
    """The data flow of the CUDA path's PPL_SYM_FULL mode (include/ppl.h), step by step in numpy:
    a-blocks of T; for slab A only integrals with all four indices >= A0 are formed; the packed
    S+-[(a<=b)][(c<=d)] = (ac|bd) +- (ad|bc) rows of the slab are used once as rows (contraction over
    (c,d) with c >= A0) and once as columns (outputs (c,d) with c >= A0+T)."""
    x, v, _ = L.shape
    o = t2.shape[0]
    Kp, Km, Mp, Mm = v * (v + 1) // 2, v * (v - 1) // 2, o * (o + 1) // 2, o * (o - 1) // 2
    taup, taum = np.zeros((Mp, Kp)), np.zeros((max(Mm, 1), max(Km, 1)))
    for i in range(o):
        for j in range(i, o):
            for c in range(v):
                taup[_kp(i, j, o), _kp(c, c, v)] = 0.5 * t2[i, j, c, c]
                for d in range(c + 1, v):
                    taup[_kp(i, j, o), _kp(c, d, v)] = 0.5 * (t2[i, j, c, d] + t2[i, j, d, c])
                    if i < j:
                        taum[_km(i, j, o), _km(c, d, v)] = 0.5 * (t2[i, j, c, d] - t2[i, j, d, c])
    Rp, Rm = np.zeros((Mp, Kp)), np.zeros((max(Mm, 1), max(Km, 1)))
    for A0 in range(0, v, T):
        ta = min(T, v - A0)
        c1 = A0 + ta
        X = np.einsum("Pac,Pbd->abcd", L[:, A0:c1, A0:], L[:, A0:, A0:])  # (ac|bd), b, c, d >= A0 only
        k0p, k1p = _kp(A0, A0, v), _kp(c1, c1, v)
        k0m, k1m = A0 * (2 * v - A0 - 1) // 2, c1 * (2 * v - c1 - 1) // 2
        for al in range(ta):
            a = A0 + al
            for b in range(a, v):
                Xab = X[al, b - A0]
                wp, wm = np.zeros(Kp), np.zeros(max(Km, 1))
                for c in range(A0, v):
                    for d in range(c, v):
                        wp[_kp(c, d, v)] = Xab[c - A0, d - A0] + Xab[d - A0, c - A0]
                        if c < d:
                            wm[_km(c, d, v)] = Xab[c - A0, d - A0] - Xab[d - A0, c - A0]
                Rp[:, _kp(a, b, v)] += taup[:, k0p:] @ wp[k0p:]             # use 1
                Rp[:, k1p:] += np.outer(taup[:, _kp(a, b, v)], wp[k1p:])    # use 2
                if a < b and Mm > 0:
                    Rm[:, _km(a, b, v)] += taum[:, k0m:Km] @ wm[k0m:Km]
                    Rm[:, k1m:Km] += np.outer(taum[:, _km(a, b, v)], wm[k1m:Km])
    R = np.zeros_like(t2)
    for i in range(o):
        for j in range(i, o):
            for a in range(v):
                for b in range(a, v):
                    rp = Rp[_kp(i, j, o), _kp(a, b, v)]
                    rm = Rm[_km(i, j, o), _km(a, b, v)] if (i < j and a < b) else 0.0
                    R[i, j, a, b] = R[j, i, b, a] = rp + rm
                    R[j, i, a, b] = R[i, j, b, a] = rp - rm
    return R


@pytest.mark.parametrize("shape,T", [((3, 7, 5), 3), ((2, 5, 4), 2), ((4, 9, 6), 4), ((1, 4, 3), 2), ((3, 6, 2), 6), ((2, 1, 3), 1)])
def test_full_symmetry_hook_identity(shape, T):
    """With L[P,a,c] = L[P,c,a] AND pair-symmetric t2 the whole term follows from the integrals
    (ac|bd) with a in block A and b, c, d >= A0 alone (1/8 of the v^4 tensor), because
    S+-[(ab)][(cd)] = (ac|bd) +- (ad|bc) is symmetric in its two pair indices.  Pinned against the oracle;
    negative controls: a non-symmetric L, or a non-pair-symmetric t2, breaks it."""
    o, v, x = shape
    L = I.make_L(v, x, 13, symmetric=True)
    t = I.make_t2(o, v, 13, symmetric=True)
    assert rel(_full_symmetry_emulation(L, t, T), oracle.full(L, t)) <= RTOL
    if v > 2 and T < v:
        Ln = I.make_L(v, x, 13, symmetric=False)
        assert rel(_full_symmetry_emulation(Ln, t, T), oracle.full(Ln, t)) > 1e-3
    if o > 1 and v > 1:
        tn = I.make_t2(o, v, 13, symmetric=False)
        assert rel(_full_symmetry_emulation(L, tn, T), oracle.full(L, tn)) > 1e-3


# ----------------------------------------------------------------------------- step 0 alone: oracle.eri_slab
def test_eri_slab_hand_worked_2x2():
    """eq. (5), by hand with the L of tests/golden/hand_2x2.txt (nchol = 1): <ab|cd> = L[a,c] L[b,d].
    L is not symmetric, so the other pairing L[a,d] L[b,c] gives a different tensor (negative control)."""
    L = _read_hand()["L"].reshape(1, 2, 2).copy()
    eri = oracle.eri_slab(L, 0, 2)
    # a b c d -> L[a,c] L[b,d]; L = [[1,2],[3,4]]
    want = np.array([[[[1, 2], [2, 4]], [[3, 4], [6, 8]]], [[[3, 6], [4, 8]], [[9, 12], [12, 16]]]], dtype=float)
    assert np.array_equal(eri, want)
    bad = np.einsum("ad,bc->abcd", L[0], L[0])
    assert not np.array_equal(eri, bad)


@pytest.mark.parametrize("shape", [(1, 1), (5, 1), (7, 5), (9, 4), (20, 60), (53, 17)])
def test_eri_slab_against_einsum_and_outer_product(shape):
    v, x = shape
    L = I.make_L(v, x, 3, symmetric=False)
    for a0, na in {(0, v), (v // 2, v - v // 2), (v - 1, 1), (0, 1)}:
        eri = oracle.eri_slab(L, a0, na)
        want = np.einsum("Pac,Pbd->abcd", L[:, a0:a0 + na, :], L, optimize=True)  # library contraction, own summation order
        assert rel(eri, want) <= RTOL
    # nchol = 1: a single product per entry, so the outer product is reproduced bit for bit
    e1 = oracle.eri_slab(L[:1].copy(), 0, v)
    assert np.array_equal(e1, np.einsum("ac,bd->abcd", L[0], L[0]))


def test_eri_slab_contracted_with_t2_reproduces_the_ladder():
    """'abcd,ijcd->ijab' on the slab is the ladder term (eq. 4): ties eri_slab to the pinned oracle.full."""
    o, v, x = 3, 11, 6
    L, t2 = rand_inputs(o, v, x, seed=4)
    R = oracle.full(L, t2)
    for a0, na in ((0, 4), (4, 7)):
        eri = oracle.eri_slab(L, a0, na)
        got = np.tensordot(t2, eri, axes=([2, 3], [2, 3]))  # [i,j,al,b]
        assert rel(got, R[:, :, a0:a0 + na, :]) <= RTOL


def test_eri_slab_symmetries_and_exact_integers():
    v, x = 10, 7
    Ls = I.make_L(v, x, 5, symmetric=True, integer=True)
    e = oracle.eri_slab(Ls, 0, v)
    want = np.einsum("Pac,Pbd->abcd", Ls.astype(np.int64), Ls.astype(np.int64))
    assert np.array_equal(e, want.astype(float))  # exact integers: any summation order gives the same bits
    # real orbitals: the 8-fold symmetry of (ac|bd) in the <ab|cd> order
    assert np.array_equal(e, e.transpose(2, 1, 0, 3))  # a <-> c
    assert np.array_equal(e, e.transpose(0, 3, 2, 1))  # b <-> d
    assert np.array_equal(e, e.transpose(1, 0, 3, 2))  # (ac) <-> (bd)
    Ln = I.make_L(v, x, 5, symmetric=False, integer=True)
    en = oracle.eri_slab(Ln, 0, v)
    assert np.array_equal(en, en.transpose(1, 0, 3, 2))       # holds for any L
    assert not np.array_equal(en, en.transpose(2, 1, 0, 3))   # needs L[P,a,c] = L[P,c,a]: negative control
