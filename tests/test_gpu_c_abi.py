"""-m gpu: a plain C99 client (tests/c_abi/trk_c_smoke.c) built with gcc against include/trk.h and libtrk.so -- the boundary
is a C ABI, not a Python extension: no torch, no CUDA headers, host buffers only."""
import os
import subprocess

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_client_runs_the_served_request(tmp_path):
    from paper_2501_05520_b200 import LIB_PATH, lib
    lib()                                                            # fails loudly if libtrk.so is not built
    pkg = os.path.dirname(LIB_PATH)
    exe = str(tmp_path / "trk_c_smoke")
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
           os.path.join(ROOT, "tests", "c_abi", "trk_c_smoke.c"), "-o", exe, "-L", pkg, "-ltrk", "-lm", f"-Wl,-rpath,{pkg}"]
    b = subprocess.run(cmd, capture_output=True, text=True)
    assert b.returncode == 0, b.stderr
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.startswith("OK ")
    print(r.stdout.strip())
