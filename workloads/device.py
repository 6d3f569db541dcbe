"""Device-side helpers for tests and bench: build/load workloads/libkvfill.so and fill
torch CUDA tensors with the pattern g of workloads/content.py.  Test tooling only."""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "csrc" / "kvfill.cu"
_SO = _HERE / "libkvfill.so"
_lib = None


_PROBE_SRC = _HERE / "csrc" / "dramprobe.cu"
_PROBE_SO = _HERE / "libdramprobe.so"
_probe = None


def _nvcc_shared(src: Path, so: Path, force: bool) -> None:
    if force or not so.exists() or so.stat().st_mtime < src.stat().st_mtime:
        nvcc = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
        tmp = so.with_suffix(f".so.tmp{os.getpid()}")
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
                               "-Xcompiler", "-fPIC,-fvisibility=hidden", "-shared", "-cudart", "static",
                               "-o", str(tmp), str(src)])
        os.replace(tmp, so)


def build(force: bool = False) -> Path:
    _nvcc_shared(_SRC, _SO, force)
    _nvcc_shared(_PROBE_SRC, _PROBE_SO, force)
    return _SO


def dram_probe(mode: str, src, dst, nbytes: int, stream: int = 0) -> None:
    """Plain streaming read / write / copy over contiguous device buffers (csrc/dramprobe.cu)."""
    global _probe
    if _probe is None:
        _probe = ctypes.CDLL(str(_PROBE_SO))
        _probe.dramprobe_run.restype = ctypes.c_int
        _probe.dramprobe_run.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                                         ctypes.c_void_p, ctypes.c_void_p]
    if isinstance(mode, int):
        rc = _probe.dramprobe_run(mode, src.data_ptr(), dst.data_ptr(), int(nbytes), None, stream)
        if rc:
            raise RuntimeError(f"dramprobe_run({mode}) failed ({rc})")
        return
    rc = _probe.dramprobe_run({"read": 0, "write": 1, "copy": 2, "copy_pf4k": 3, "copy_pf32k": 4, "copy_5cta": 5, "copy_4cta": 6, "copy_persistent": 7, "copy_persistent_pf": 8}[mode], src.data_ptr(), dst.data_ptr(),
                              int(nbytes), None, stream)
    if rc:
        raise RuntimeError(f"dramprobe_run({mode}) failed ({rc})")


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        if not _SO.exists():
            raise ImportError(f"{_SO} missing: run workloads.device.build()")
        _lib = ctypes.CDLL(str(_SO))
        vp, i64, u64 = ctypes.c_void_p, ctypes.c_int64, ctypes.c_uint64
        _lib.kvfill_fill.restype = ctypes.c_int
        _lib.kvfill_fill.argtypes = [vp, i64, i64, u64, u64, vp]
        _lib.kvfill_page_checksums.restype = ctypes.c_int
        _lib.kvfill_page_checksums.argtypes = [vp, i64, i64, vp, vp]
    return _lib


def fill_plane(t, seed: int, plane: int, stream: int = 0) -> None:
    """t: contiguous torch CUDA tensor viewed as 16-bit words; fills words [0, numel)."""
    n_words = t.numel() * t.element_size() // 2
    rc = lib().kvfill_fill(t.data_ptr(), 0, n_words, seed & 0xFFFFFFFFFFFFFFFF, plane, stream)
    if rc:
        raise RuntimeError(f"kvfill_fill failed ({rc})")


def fill_words(t, first_word: int, seed: int, plane: int, stream: int = 0) -> None:
    """Fills t (a chunk of a larger logical array) with words [first_word, first_word + n) of
    g(seed, plane, .): lets a host-resident checkpoint be generated chunk by chunk on the device."""
    n_words = t.numel() * t.element_size() // 2
    if first_word % 4:
        raise ValueError("first_word must be a multiple of 4 (one 64-bit hash = 4 words)")
    rc = lib().kvfill_fill(t.data_ptr(), int(first_word), n_words, seed & 0xFFFFFFFFFFFFFFFF, plane,
                           stream)
    if rc:
        raise RuntimeError(f"kvfill_fill failed ({rc})")


def fill_host_checkpoint(host_buf, nbytes: int, seed: int, plane: int, chunk_bytes: int = 1 << 30):
    """host_buf[:nbytes] (pinned uint8 tensor) <- g(seed, plane, word index), generated on the
    device in chunks and copied down (a 72 GiB checkpoint would take minutes with numpy)."""
    import torch
    scratch = torch.empty(min(chunk_bytes, max(nbytes, 8)), dtype=torch.uint8, device="cuda")
    at = 0
    while at < nbytes:
        n = min(scratch.numel(), nbytes - at)
        fill_words(scratch[:n], at // 2, seed, plane)
        host_buf[at: at + n].copy_(scratch[:n], non_blocking=True)
        torch.cuda.synchronize()
        at += n
    del scratch


def page_checksums(t, n_pages: int, page_bytes: int, stream: int = 0):
    import torch
    out = torch.empty(n_pages, dtype=torch.int64, device=t.device)
    rc = lib().kvfill_page_checksums(t.data_ptr(), n_pages, page_bytes, out.data_ptr(), stream)
    if rc:
        raise RuntimeError(f"kvfill_page_checksums failed ({rc})")
    return out


_registered = {}


def host_mem_available():
    """MemAvailable of /proc/meminfo in bytes (None if unreadable)."""
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable:"):
                return int(line.split()[1]) * 1024
    except OSError:
        pass
    return None


def pinned_exact(nbytes: int):
    """Page-locked host tensor of exactly nbytes (torch's pinned allocator rounds sizes up
    to a power of two, which doubles a 32 GiB + guard-band buffer).  Registers a pageable
    tensor with cudaHostRegister; call unpin(t) when done."""
    import torch
    avail = host_mem_available()
    if avail is not None and int(nbytes) > avail - (4 << 30):
        # page-locking more than the box has would get the process (or the box) killed
        raise RuntimeError(f"pinned_exact({nbytes}): only {avail} bytes of host memory available")
    t = torch.empty(int(nbytes), dtype=torch.uint8)
    rc = torch.cuda.cudart().cudaHostRegister(t.data_ptr(), t.numel(), 0)
    if int(rc) != 0:
        raise RuntimeError(f"cudaHostRegister({nbytes}) failed: {rc}")
    _registered[t.data_ptr()] = t
    return t


def unpin(t) -> None:
    import torch
    if _registered.pop(t.data_ptr(), None) is not None:
        torch.cuda.cudart().cudaHostUnregister(t.data_ptr())
