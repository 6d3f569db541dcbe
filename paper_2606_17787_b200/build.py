"""Build liblumen_kv.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2606_17787_b200.build [--force]

The library has no torch or Python dependency: plain C ABI (include/lumen_kv.h),
static cudart.  The .so is git-ignored but travels to the GPU box with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
SO = PKG / "liblumen_kv.so"
SOURCES = [CSRC / "lib.cu", CSRC / "stager.cu", CSRC / "ckpt.cu", CSRC / "recover.cu", CSRC / "kernels.cu", CSRC / "tags.cu", CSRC / "noalloc.cu", CSRC / "plan.cpp", CSRC / "store.cpp", CSRC / "placement.cpp"]
HEADERS = [CSRC / "plan.hpp", CSRC / "kernels.hpp", CSRC / "internal.hpp", ROOT / "include" / "lumen_kv.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-Wall,-Wextra,-fvisibility=hidden",
    "-Xptxas", "-v",
    "-shared", "-cudart", "static",
]


def nvcc() -> str:
    cand = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return cand if Path(cand).exists() else "nvcc"


def stale() -> bool:
    if not SO.exists():
        return True
    t = SO.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES + HEADERS + [Path(__file__)])


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not stale():
        return SO
    tmp = SO.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc(), *NVCC_FLAGS, "-I", str(ROOT / "include"), "-I", str(CSRC),
           "-o", str(tmp), *map(str, SOURCES)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building liblumen_kv.so")
    log = (" ".join(cmd) + "\n" + res.stdout + res.stderr).replace(str(tmp), str(SO))
    log = "\n".join(l for l in log.split("\n") if "Compile time" not in l)   # keep the log deterministic
    (PKG / "build_ptxas.log").write_text(log.replace(str(ROOT) + "/", ""))
    if verbose:
        print(res.stdout + res.stderr)
    os.replace(tmp, SO)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
