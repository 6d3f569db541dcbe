"""include/lumen_kv.h is a C header: compile tests/c/abi_smoke.c as strict C99 against it, link
the in-tree liblumen_kv.so and run the host-side entry points from plain C (no GPU needed)."""
import subprocess
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent


def test_header_compiles_as_c99_and_links(tmp_path):
    from paper_2606_17787_b200 import build
    so = build.build()
    exe = tmp_path / "abi_smoke"
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Wextra", "-Werror",
                           "-Wno-attributes", "-I", str(ROOT / "include"),
                           str(ROOT / "tests" / "c" / "abi_smoke.c"), "-o", str(exe),
                           "-L", str(so.parent), "-l:liblumen_kv.so", f"-Wl,-rpath,{so.parent}"])
    out = subprocess.run([str(exe)], capture_output=True, text=True, timeout=60)
    assert out.returncode == 0, out.stderr
    assert out.stdout.strip() == "c abi ok"
