"""The host planner (csrc/ppl_plan.cpp, plain C++) under AddressSanitizer + UndefinedBehaviorSanitizer (
VERDICT r02 "missing" 4).  compute-sanitizer is closed on this GPU pool, but the planner needs no GPU: it is compiled here with
g++ -fsanitize=address,undefined together with tests/planner_sanitizer_driver.cpp, which walks ppl_plan_dry_ex over shapes x
modes x caps x debug knobs.  The command is the one in CMD below; a sanitizer report aborts the driver."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CSRC = os.path.join(ROOT, "paper_2603_20912_b200", "csrc")


def test_planner_is_clean_under_asan_and_ubsan(tmp_path):
    gxx = shutil.which("g++")
    if not gxx:
        pytest.skip("no g++")
    exe = str(tmp_path / "planner_sanitizer_driver")
    CMD = [gxx, "-std=c++17", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer",
           "-I/usr/local/cuda/include", os.path.join(ROOT, "tests", "planner_sanitizer_driver.cpp"), os.path.join(CSRC, "ppl_plan.cpp"),
           "-o", exe]
    subprocess.check_call(CMD)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "no report" in r.stdout
