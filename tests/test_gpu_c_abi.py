"""-m gpu: the C ABI from a caller that is not Python.  tests/c_abi_example.cu (CUDA runtime + include/ppl.h, no
torch) is compiled with nvcc, linked against the in-tree libppl.so and run: ppl_plan / ppl_plan_set_symmetry /
ppl_apply in all four modes and ppl_generate_eri against closed forms that are exact in FP64 (identity-like L:
R = R0 + (sum_P s_P^2) t2; SURVEY 8(c) pin P3), with caller-owned cudaMalloc buffers and a caller-created stream."""
import os
import subprocess
import sys

import pytest

import paper_2603_20912_b200 as P

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


@pytest.mark.parametrize("shape", [(6, 64, 24), (3, 53, 10), (5, 20, 60)])
def test_c_caller(shape, tmp_path):
    so = P.build()
    exe = str(tmp_path / "c_abi_example")
    libdir = os.path.dirname(so)
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O2", "-std=c++17", "-I", os.path.join(ROOT, "include"), os.path.join(HERE, "c_abi_example.cu"), "-o", exe,
           "-L", libdir, "-l:" + os.path.basename(so), "-Xlinker", "-rpath=" + libdir]
    subprocess.check_call(cmd)
    out = subprocess.run([exe] + [str(n) for n in shape], capture_output=True, text=True, timeout=300)
    sys.stdout.write(out.stdout)
    sys.stderr.write(out.stderr)
    assert out.returncode == 0, out.stdout + out.stderr
    assert "C ABI EXAMPLE OK" in out.stdout
