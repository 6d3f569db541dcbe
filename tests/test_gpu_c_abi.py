"""The C ABI end to end from plain C on the GPU: tests/c/abi_gpu.c (C99, only include/lumen_kv.h
and the CUDA runtime's C API) packs to HBM, to pinned host memory zero-copy and staged, restores
under fresh page tables, and checks every word against an address-coded fill -- no Python, no
torch and no oracle in the loop."""
import os
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
pytestmark = pytest.mark.gpu


def test_pack_and_restore_from_plain_c(tmp_path):
    from paper_2606_17787_b200 import build
    so = build.build()
    cuda = Path(os.environ.get("CUDA_HOME", "/usr/local/cuda"))
    exe = tmp_path / "abi_gpu"
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror", "-Wno-attributes",
                           "-O1", "-I", str(ROOT / "include"), "-isystem", str(cuda / "include"),
                           str(ROOT / "tests" / "c" / "abi_gpu.c"), "-o", str(exe),
                           "-L", str(so.parent), "-l:liblumen_kv.so", f"-Wl,-rpath,{so.parent}",
                           "-L", str(cuda / "lib64"), "-lcudart", f"-Wl,-rpath,{cuda / 'lib64'}"])
    out = subprocess.run([str(exe)], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stdout + out.stderr
    assert out.stdout.strip() == "c abi gpu ok"
