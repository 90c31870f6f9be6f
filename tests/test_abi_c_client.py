"""include/sift.h used from plain C (gcc, no Python types anywhere near the calls): tests/abi_c/abi_smoke.c."""
import os
import subprocess

import pytest

from paper_2606_09441_b200 import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "tests", "abi_c", "abi_smoke.c")


def _compile(tmp_path):
    lib = build.build_library()
    exe = os.path.join(str(tmp_path), "abi_smoke")
    cuda_lib = "/usr/local/cuda/lib64"
    cmd = ["gcc", "-std=c99", "-O1", "-Wall", "-I", os.path.join(ROOT, "include"), SRC, "-o", exe, lib,
           "-L", cuda_lib, "-lcudart", "-lm", f"-Wl,-rpath,{os.path.dirname(lib)}", f"-Wl,-rpath,{cuda_lib}"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    return exe


def test_c_client_host_calls(tmp_path):
    r = subprocess.run([_compile(tmp_path), "host"], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and "abi_smoke host ok" in r.stdout, r.stdout + r.stderr


@pytest.mark.gpu
def test_c_client_decode_and_attention(tmp_path):
    r = subprocess.run([_compile(tmp_path), "gpu"], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0 and "abi_smoke gpu ok" in r.stdout, r.stdout + r.stderr
