"""The C ABI used as shipped, by a C program that moves data (tests/c/abi_gpu.c): pools created, filled, migrated in two
stages, fused through a pinned host buffer, scattered, read back — and compared, inside the C program, with files
written by tests/golden/make_abi_gpu_case.py, which calls only `synth` and `oracle`.  No Python in the data path."""
import os
import shutil
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_client_migrates_packs_and_unpacks_bit_exactly(tmp_path):
    gcc = shutil.which("gcc")
    if not gcc:
        pytest.skip("gcc unavailable")
    from paper_2406_03243_b200 import build
    build.build()
    case = str(tmp_path / "case")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "golden", "make_abi_gpu_case.py"), case],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    libdir = os.path.join(ROOT, "paper_2406_03243_b200")
    exe = str(tmp_path / "abi_gpu")
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Wextra", "-Werror", "-pedantic", "-D_POSIX_C_SOURCE=200112L",
                        "-I", os.path.join(ROOT, "include"), os.path.join(ROOT, "tests", "c", "abi_gpu.c"), "-o", exe,
                        "-L", libdir, "-lllx", "-Wl,-rpath," + libdir], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    r = subprocess.run([exe, case], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "abi_gpu ok" in r.stdout, r.stdout + r.stderr
