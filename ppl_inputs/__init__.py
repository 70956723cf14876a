"""Seeded synthetic inputs for the pp-ladder path (host buffers, numpy float64).

A module of its own: it contains none of the method's arithmetic and is the only code shared by
the CPU oracle's tests and the CUDA path's tests/bench (both read the same host buffers).
Recipe and readings: see ``ppl_inputs.c`` and DESIGN.md ("Input recipe").
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libppl_inputs.so")
_SRC = os.path.join(_HERE, "ppl_inputs.c")

# BASELINE.json "configs": (nocc, nvirt, nchol)
CONFIGS = {
    "tiny": (5, 20, 60),
    "small": (5, 53, 232),
    "medium": (20, 200, 800),
    "large": (40, 400, 1600),
    "xl": (60, 600, 2400),
}
CONFIG_ORDER = ["tiny", "small", "medium", "large", "xl"]
# Shapes of the paper's own synthetic ladder benchmark (Table 3; N = nocc + nvirt basis functions,
# nchol = 5N): host-resident operands, a second workload.  Not BASELINE.json configs.
TABLE3_SHAPES = {
    "table3_n800_o100": (100, 700, 4000),
    "table3_n900_o100": (100, 800, 4500),
    "table3_n800_o150": (150, 650, 4000),  # PAPER.md:440-441 (nvec = 5 N = 4000; 166 GB of host operands)
    "table3_n1000_o100": (100, 900, 5000),  # PAPER.md:432-433 (162 GB of host operands)
    "table3_n1000_o50": (50, 950, 10000),   # PAPER.md:448-449 (nvec = 10 N: the row with the paper's best derived rate)
}


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _SO, _SRC, "-lm"], cwd=_HERE
        )
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.ppl_inputs_fill_L.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_uint64, ctypes.c_int, ctypes.c_int]
        lib.ppl_inputs_fill_L.restype = None
        lib.ppl_inputs_fill_t2.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_uint64, ctypes.c_int, ctypes.c_int]
        lib.ppl_inputs_fill_t2.restype = None
        lib.ppl_inputs_fill_vec.argtypes = [dp, ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int]
        lib.ppl_inputs_fill_vec.restype = None
        _lib = lib
    return _lib


def _ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def make_L(nvirt: int, nchol: int, seed: int = 0, symmetric: bool = True, integer: bool = False,
           out: np.ndarray | None = None) -> np.ndarray:
    """L[nchol, nvirt, nvirt] (row-major float64). ``out`` lets the caller supply (pinned) memory."""
    L = np.empty((nchol, nvirt, nvirt), dtype=np.float64) if out is None else out
    assert L.dtype == np.float64 and L.flags.c_contiguous and L.shape == (nchol, nvirt, nvirt)
    _load().ppl_inputs_fill_L(_ptr(L), nvirt, nchol, seed, int(symmetric), int(integer))
    return L


def make_t2(nocc: int, nvirt: int, seed: int = 0, symmetric: bool = True, integer: bool = False,
            out: np.ndarray | None = None) -> np.ndarray:
    """t2[nocc, nocc, nvirt, nvirt] (row-major float64)."""
    t2 = np.empty((nocc, nocc, nvirt, nvirt), dtype=np.float64) if out is None else out
    assert t2.dtype == np.float64 and t2.flags.c_contiguous and t2.shape == (nocc, nocc, nvirt, nvirt)
    _load().ppl_inputs_fill_t2(_ptr(t2), nocc, nvirt, seed, int(symmetric), int(integer))
    return t2


def make_vec(n: int, seed: int, tag: int, integer: bool = False, uniform: bool = False) -> np.ndarray:
    """Test vector of n draws from stream ``tag`` (>= 16): N(0,1), small integers, or U(0,1)."""
    x = np.empty(n, dtype=np.float64)
    _load().ppl_inputs_fill_vec(_ptr(x), n, seed, tag, 2 if uniform else int(integer))
    return x


def make_config(name: str, seed: int = 0, symmetric: bool = True, integer: bool = False):
    o, v, x = CONFIGS[name]
    return make_L(v, x, seed, symmetric, integer), make_t2(o, v, seed, symmetric, integer)


def sample_pairs(nvirt: int, k: int, seed: int = 0) -> np.ndarray:
    """(a,b) columns for sampled parity: a deterministic edge/diagonal set plus k seeded-random
    pairs and their transposes; chosen without any knowledge of the planner's tile grid
    (SURVEY.md 8(c) P11).  Returns int32 [n,2], unique rows."""
    v = nvirt
    det = [(0, 0), (0, v - 1), (v - 1, 0), (v - 1, v - 1)]
    for a in sorted({v // 7, v // 3, v // 2, (2 * v) // 3, v - 2} & set(range(v))):
        for b in (a - 1, a, a + 1):
            if 0 <= b < v:
                det.append((a, b))
    u = make_vec(2 * k, seed, 77, uniform=True)
    idx = np.minimum((u * v).astype(np.int64), v - 1).reshape(k, 2) if k else np.zeros((0, 2), np.int64)
    pairs = det + [(int(a), int(b)) for a, b in idx] + [(int(b), int(a)) for a, b in idx[: k // 4]]
    seen, uniq = set(), []
    for p in pairs:
        if p not in seen:
            seen.add(p)
            uniq.append(p)
    return np.asarray(uniq, dtype=np.int32).reshape(-1, 2)
