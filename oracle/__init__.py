"""ctypes loader for the CPU oracle (oracle/ppl_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s
cpu_baseline / ``--impl reference`` legs.  Never imported by ``paper_2603_20912_b200`` (the CUDA
path), and imports nothing from it.  Arrays are numpy float64, C-contiguous, host memory.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libppl_oracle.so")
_SRC = os.path.join(_HERE, "ppl_oracle.c")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O3, host ISA, OpenMP).  Building it is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O3", "-march=native", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"],
            cwd=_HERE,
        )
    return _SO


_lib = None
_dp = ctypes.POINTER(ctypes.c_double)


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i, i64 = ctypes.c_int, ctypes.c_int64
        lib.ppl_oracle_num_threads.restype = i
        for name in ("ppl_oracle_full", "ppl_oracle_bruteforce_w", "ppl_oracle_bruteforce_direct"):
            f = getattr(lib, name)
            f.argtypes = [i, i, i, _dp, _dp, _dp]
            f.restype = i
        lib.ppl_oracle_columns.argtypes = [i, i, i, _dp, _dp, i64, ctypes.POINTER(ctypes.c_int32), _dp]
        lib.ppl_oracle_columns.restype = i
        lib.ppl_oracle_project.argtypes = [i, i, i, _dp, _dp, _dp, _dp, _dp, _dp]
        lib.ppl_oracle_project.restype = i
        lib.ppl_oracle_full_ex.argtypes = [i, i, i, _dp, _dp, _dp, i, i, ctypes.c_double, ctypes.c_double]
        lib.ppl_oracle_full_ex.restype = i
        lib.ppl_oracle_eri_slab.argtypes = [i, i, _dp, i, i, _dp]
        lib.ppl_oracle_eri_slab.restype = i
        lib.ppl_oracle_contract_pair.argtypes = [ctypes.c_char_p, ctypes.POINTER(i64), ctypes.POINTER(i64), _dp, _dp, _dp,
                                                 ctypes.c_double, ctypes.c_double]
        lib.ppl_oracle_contract_pair.restype = i
        _lib = lib
    return _lib


def _chk(a: np.ndarray, shape) -> np.ndarray:
    assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous, "need C-contiguous float64"
    assert tuple(a.shape) == tuple(shape), f"shape {a.shape} != {shape}"
    return a


def _p(a: np.ndarray):
    return a.ctypes.data_as(_dp)


def _dims(L: np.ndarray, t2: np.ndarray):
    x, v, v2 = L.shape
    o = t2.shape[0]
    _chk(L, (x, v, v))
    _chk(t2, (o, o, v, v))
    return o, v, x


def num_threads() -> int:
    return int(_load().ppl_oracle_num_threads())


def _run3(fn, L, t2, R):
    o, v, x = _dims(L, t2)
    R = np.zeros((o, o, v, v)) if R is None else _chk(R, (o, o, v, v))
    rc = fn(o, v, x, _p(L), _p(t2), _p(R))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return R


def full(L, t2, R=None):
    """R[i,j,a,b] += sum_cd sum_P L[P,a,c] L[P,b,d] t2[i,j,c,d]; R=None starts from zeros."""
    return _run3(_load().ppl_oracle_full, L, t2, R)


def bruteforce_w(L, t2, R=None):
    return _run3(_load().ppl_oracle_bruteforce_w, L, t2, R)


def bruteforce_direct(L, t2, R=None):
    return _run3(_load().ppl_oracle_bruteforce_direct, L, t2, R)


def columns(L, t2, pairs) -> np.ndarray:
    """Bare ladder term at the (a,b) pairs: returns [npairs, nocc, nocc]."""
    o, v, x = _dims(L, t2)
    pairs = np.ascontiguousarray(pairs, dtype=np.int32).reshape(-1, 2)
    out = np.empty((pairs.shape[0], o, o), dtype=np.float64)
    rc = _load().ppl_oracle_columns(o, v, x, _p(L), _p(t2), pairs.shape[0],
                                    pairs.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _p(out))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return out


def project(L, t2, u, w):
    """(sum_ab u_a w_b R[i,j,a,b], sum_cd |M_cd||t2_ijcd|) from the definition, long double."""
    o, v, x = _dims(L, t2)
    u = _chk(np.ascontiguousarray(u, dtype=np.float64), (v,))
    w = _chk(np.ascontiguousarray(w, dtype=np.float64), (v,))
    out = np.empty((o, o), dtype=np.float64)
    absout = np.empty((o, o), dtype=np.float64)
    rc = _load().ppl_oracle_project(o, v, x, _p(L), _p(t2), _p(u), _p(w), _p(out), _p(absout))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return out, absout


LAYOUTS = {"ijab": 0, "iajb": 1}


def full_ex(L, t2, R=None, t2_layout="ijab", r_layout="ijab", alpha=1.0, beta=1.0):
    """R = beta*R + alpha*term with t2 / R stored 'ijab' ([i,j,c,d]) or 'iajb' ([i,c,j,d], the paper's
    'icjd' -> 'iajb').  Shapes follow the layouts; R=None starts from zeros."""
    x, v, _ = L.shape
    o = t2.shape[0]
    shp = {"ijab": (o, o, v, v), "iajb": (o, v, o, v)}
    _chk(L, (x, v, v))
    _chk(t2, shp[t2_layout])
    R = np.zeros(shp[r_layout]) if R is None else _chk(R, shp[r_layout])
    rc = _load().ppl_oracle_full_ex(o, v, x, _p(L), _p(t2), _p(R), LAYOUTS[t2_layout], LAYOUTS[r_layout],
                                    float(alpha), float(beta))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return R


def eri_slab(L, a0: int, na: int) -> np.ndarray:
    """eri[al,b,c,d] = <ab|cd> = sum_P L[P,a0+al,c] L[P,b,d]: step 0 alone ('xac,xbd->acbd'),
    stored in the order of the paper's dense variant 'abcd'."""
    x, v, _ = L.shape
    _chk(L, (x, v, v))
    out = np.empty((na, v, v, v))
    rc = _load().ppl_oracle_eri_slab(v, x, _p(L), int(a0), int(na), _p(out))
    if rc:
        raise RuntimeError(f"oracle error {rc}")
    return out


def contract_pair(subscripts: str, A: np.ndarray, B: np.ndarray, C: np.ndarray | None = None, alpha=1.0, beta=0.0) -> np.ndarray:
    """C = beta*C + alpha * einsum(subscripts, A, B) from the definition ('op0,op1->out'); one loop
    nest over every index letter, plain double accumulation.  C=None: a fresh output (beta is then 0)."""
    ins, out = subscripts.replace(" ", "").split("->")
    s0, s1 = ins.split(",")
    assert A.dtype == np.float64 and B.dtype == np.float64 and A.flags.c_contiguous and B.flags.c_contiguous
    assert A.ndim == len(s0) and B.ndim == len(s1)
    ext = dict(zip(s0, A.shape))
    ext.update(zip(s1, B.shape))
    shape = tuple(ext[c] for c in out)
    if C is None:
        C, beta = np.zeros(shape), 0.0
    _chk(C, shape)
    d0 = (ctypes.c_int64 * max(A.ndim, 1))(*A.shape)
    d1 = (ctypes.c_int64 * max(B.ndim, 1))(*B.shape)
    rc = _load().ppl_oracle_contract_pair(subscripts.encode(), d0, d1, _p(A), _p(B), _p(C), float(alpha), float(beta))
    if rc:
        raise RuntimeError(f"oracle error {rc}: malformed contraction {subscripts!r}")
    return C
