"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU,
exports every symbol include/ppl.h declares, and FAILS LOUDLY (no fallback) when no B200 is there."""
import ctypes
import os
import re

import pytest

import paper_2603_20912_b200 as P

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "ppl.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ppl_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    so = P.build()
    assert os.path.exists(so)
    lib = ctypes.CDLL(so)
    declared = _declared_symbols()
    assert {"ppl_plan", "ppl_apply", "ppl_destroy"} <= set(declared)
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in ppl.h but not exported"
    assert sorted(P.SYMBOLS) == declared  # the binding mirrors the header one to one


def test_error_strings_and_null_destroy():
    lib = P.lib()
    for code in range(0, 8):
        assert lib.ppl_error_string(code)
    assert lib.ppl_destroy(None) == P.PPL_OK


def test_no_fallback_without_gpu():
    import torch

    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the no-GPU refusal is checked on the CPU box")
    with pytest.raises(P.PplError) as ei:
        P.ppl_plan(5, 20, 60)
    assert ei.value.code == P.PPL_ERR_UNSUPPORTED_DEVICE
    with pytest.raises(P.PplError):
        P.ppl_probe_fp64_peak()


def test_invalid_dims_rejected():
    for dims in [(0, 5, 5), (5, 0, 5), (5, 5, 0), (-1, 2, 2), (5, 50000, 5)]:
        with pytest.raises(P.PplError) as ei:
            P.ppl_plan(*dims)
        assert ei.value.code in (P.PPL_ERR_INVALID_ARG, P.PPL_ERR_UNSUPPORTED_DEVICE)
    assert P.lib().ppl_apply(None, None, None, None, None) == P.PPL_ERR_INVALID_ARG


def test_product_does_not_import_oracle():
    """The CUDA path and the oracle share no code and do not import each other."""
    pkg = os.path.join(ROOT, "paper_2603_20912_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "ppl_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2603_20912_b200" not in txt and "ppl_kernels" not in txt and "ppl.h" not in txt, f
