"""ASan + UBSan over the host-side native code (CPU only): the oracle (oracle/rt_oracle.cpp) and the
library's host logic (csrc/spline_fit.cpp + the constant folding of csrc/rt_params.h through tests/host_shim.cpp) are
compiled with ``-fsanitize=address,undefined -fno-sanitize-recover=all`` and driven by tests/sanitize_run.py in a
subprocess with the sanitizer runtime preloaded; any report fails the test.  (``compute-sanitizer`` over the kernels is
closed on the GPU pool: DESIGN.md section 7.)"""
import os
import subprocess
import sys
from pathlib import Path

import pytest

HERE = Path(__file__).resolve().parent
ROOT = HERE.parent
SAN = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]


def _gcc_file(name: str) -> str:
    return subprocess.run(["gcc", f"-print-file-name={name}"], capture_output=True, text=True, check=True).stdout.strip()


def test_oracle_and_host_logic_run_clean_under_asan_and_ubsan(tmp_path):
    asan, ubsan = _gcc_file("libasan.so"), _gcc_file("libubsan.so")
    if not (os.path.isabs(asan) and os.path.exists(asan)):
        pytest.skip("libasan is not installed")
    oracle_so, shim_so = tmp_path / "librt_oracle_san.so", tmp_path / "libspline_shim_san.so"
    base = ["g++", "-std=c++17", "-ffp-contract=off", "-fPIC", "-shared", *SAN]
    subprocess.run([*base, "-fopenmp", "-Wno-misleading-indentation", str(ROOT / "oracle" / "rt_oracle.cpp"), "-o",
                    str(oracle_so)], check=True)
    subprocess.run([*base, str(HERE / "host_shim.cpp"), str(ROOT / "paper_2508_15967_b200" / "csrc" / "spline_fit.cpp"),
                    "-o", str(shim_so)], check=True)
    env = dict(os.environ, RT_ORACLE_LIB=str(oracle_so),
               LD_PRELOAD=" ".join(p for p in (asan, ubsan) if os.path.isabs(p) and os.path.exists(p)),
               ASAN_OPTIONS="detect_leaks=0:halt_on_error=1:abort_on_error=0", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, str(HERE / "sanitize_run.py"), str(shim_so)], env=env, capture_output=True, text=True,
                       timeout=600)
    report = r.stdout + r.stderr
    assert r.returncode == 0, report[-4000:]
    assert "sanitize_run ok" in r.stdout
    assert "AddressSanitizer" not in report and "runtime error:" not in report, report[-4000:]
