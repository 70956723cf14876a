"""-m "not gpu": pins of oracle.contract_pair -- the generic two-operand contraction 'op0,op1->out' the paper builds its
generic batching recipe on (the ladder's own steps are the strings of PAPER.md:118-120).  The oracle is
the einsum definition written out as one loop nest; it is pinned here by what does not depend on it: a hand-worked
example (tests/golden/contract_pair_hand.txt), numpy's einsum / tensordot / matmul, closed-form special cases, exact
integer arithmetic, and the ladder oracle itself (two pair contractions in the paper's order reproduce oracle.full)."""
import os

import numpy as np
import pytest

import oracle
import ppl_inputs as I

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "contract_pair_hand.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, *vals = line.split()
        out[name] = np.array([float(t) for t in vals])
    return out


def _rand(shape, seed):
    return I.make_vec(int(np.prod(shape)), seed, 50).reshape(shape)


def test_hand_worked_examples_of_the_papers_two_steps():
    g = _golden()
    A, B = g["A"].reshape(2, 2, 2), g["B"].reshape(2, 2, 2)
    C = oracle.contract_pair("xac,xbd->acbd", A, B)
    for name in ("C0000", "C0110", "C1001", "C1111", "C0100"):
        idx = tuple(int(ch) for ch in name[1:])
        assert C[idx] == g[name][0], name
    # negative control: the same products filed in 'abcd' order land elsewhere
    Cbad = oracle.contract_pair("xac,xbd->abcd", A, B)
    assert Cbad[0, 1, 0, 0] == g["C0100bad"][0] and Cbad[0, 1, 0, 0] != C[0, 1, 0, 0]
    a, b, c, d = np.meshgrid(*[np.arange(2)] * 4, indexing="ij")
    X = (1 + a + 2 * b + 4 * c + 8 * d).astype(np.float64)  # X[a][b][c][d]
    e, c2, f, d2 = np.meshgrid(*[np.arange(2)] * 4, indexing="ij")
    T = ((e + 1) * (f + 2) - c2 * d2).astype(np.float64)    # T[e][c][f][d]
    R = oracle.contract_pair("abcd,ecfd->efab", np.ascontiguousarray(X), np.ascontiguousarray(T))
    assert R[0, 0, 0, 0] == g["R0000"][0] and R[1, 0, 0, 1] == g["R1001"][0]


STRINGS = [
    ("xac,xbd->acbd", (5, 3, 4), (5, 2, 6)),          # the paper's step 0
    ("abcd,ecfd->efab", (3, 2, 4, 5), (2, 4, 3, 5)),  # the paper's step 1
    ("abcd,efcd->efab", (3, 2, 4, 5), (2, 3, 4, 5)),  # step 1 with t2 stored [i,j,c,d] (BASELINE.json's layout)
    ("xac,icjd->xajd", (4, 3, 5), (2, 5, 3, 6)),      # a Cholesky factor against an amplitude: one summed index in the middle
    ("ik,kj->ij", (7, 5), (5, 6)),                    # matmul
    ("ki,kj->ij", (5, 7), (5, 6)),
    ("ik,jk->ij", (7, 5), (6, 5)),
    ("i,j->ji", (4,), (3,)),                          # outer product, transposed output
    ("abc,abc->", (3, 4, 2), (3, 4, 2)),              # full inner product
    ("abc,dcb->ad", (3, 4, 2), (5, 2, 4)),            # summed indices in different orders in the two operands
    ("xab,xcd->dbca", (3, 2, 4), (3, 5, 2)),          # permuted output
    ("abcd,cd->ab", (2, 3, 4, 5), (4, 5)),
]


@pytest.mark.parametrize("subs,sa,sb", STRINGS)
def test_against_numpy_einsum(subs, sa, sb):
    A, B = _rand(sa, 1), _rand(sb, 2)
    want = np.einsum(subs, A, B)
    got = oracle.contract_pair(subs, A, B)
    assert got.shape == want.shape
    assert np.abs(got - want).max() <= 1e-13 * max(1.0, np.abs(want).max())


def test_special_cases_that_reduce_to_library_routines():
    A, B = _rand((6, 9), 3), _rand((9, 4), 4)
    assert np.allclose(oracle.contract_pair("ik,kj->ij", A, B), A @ B, rtol=0, atol=1e-13)
    u, w = _rand((5,), 5), _rand((7,), 6)
    assert np.array_equal(oracle.contract_pair("i,j->ij", u, w), np.outer(u, w))  # one product per entry: bit for bit
    # nchol = 1: step 0 is an outer product of the two matrices, bit for bit
    La, Lb = _rand((1, 3, 4), 7), _rand((1, 2, 5), 8)
    want = La[0][:, :, None, None] * Lb[0][None, None, :, :]
    assert np.array_equal(oracle.contract_pair("xac,xbd->acbd", La, Lb), want)
    # tensordot with the paper's axes: tensordot(chol_1, chol_2, axes=(0, 0)) is 'xac,xbd->acbd'
    A3, B3 = _rand((4, 3, 5), 9), _rand((4, 2, 6), 10)
    assert np.allclose(oracle.contract_pair("xac,xbd->acbd", A3, B3), np.tensordot(A3, B3, axes=(0, 0)), rtol=0, atol=1e-13)


def test_exact_integers_bit_for_bit():
    A = I.make_vec(4 * 3 * 5, 11, 51, integer=True).reshape(4, 3, 5)
    B = I.make_vec(2 * 5 * 3 * 6, 12, 52, integer=True).reshape(2, 5, 3, 6)
    want = np.einsum("xac,icjd->xajd", A.astype(np.int64), B.astype(np.int64)).astype(np.float64)
    assert np.array_equal(oracle.contract_pair("xac,icjd->xajd", A, B), want)


def test_alpha_beta_and_overwrite():
    A, B = _rand((3, 4, 5), 13), _rand((3, 2, 6), 14)
    C0 = _rand((4, 5, 2, 6), 15)
    term = np.einsum("xac,xbd->acbd", A, B)
    got = oracle.contract_pair("xac,xbd->acbd", A, B, C0.copy(), alpha=-0.5, beta=2.0)
    assert np.abs(got - (2.0 * C0 - 0.5 * term)).max() <= 1e-13
    nan = np.full((4, 5, 2, 6), np.nan)
    got = oracle.contract_pair("xac,xbd->acbd", A, B, nan, alpha=1.0, beta=0.0)  # beta == 0: C is not read
    assert np.abs(got - term).max() <= 1e-13


def test_two_pair_contractions_in_the_papers_order_are_the_ladder():
    """step 0 'xac,xbd->acbd', step 1 'acbd,ecfd->efab' (t2 stored [e,f,c,d] here)."""
    o, v, x = 3, 6, 7
    L = I.make_L(v, x, 5, symmetric=False)
    t2 = I.make_t2(o, v, 5, symmetric=False)
    W = oracle.contract_pair("xac,xbd->acbd", L, L)
    R = oracle.contract_pair("acbd,efcd->efab", W, t2)
    want = oracle.full(L, t2)
    assert np.abs(R - want).max() <= 1e-13 * np.abs(want).max()


@pytest.mark.parametrize("bad", ["ab,bc", "ab,bc->ad", "aa,ab->b", "ab->ab", "ab,bc,cd->ad", "a1,b->ab"])
def test_malformed_requests_are_refused(bad):
    with pytest.raises((RuntimeError, ValueError, AssertionError, KeyError)):
        oracle.contract_pair(bad, np.zeros((2, 2)), np.zeros((2, 2)))
