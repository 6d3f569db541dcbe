"""workloads -- seeded synthetic inputs shared by the oracle tests and the CUDA path.

This package holds NO pack/unpack arithmetic: only (a) the *structure* of the
synthetic KV workloads (request lengths, page tables, delta ranges, free
lists) drawn from numpy PCG64 streams, and (b) the pool *content* generator
g(seed, plane, word index) -> uint16, a counter-based SplitMix64 finaliser
implemented twice (numpy here, CUDA in csrc/kvfill.cu) and cross-checked in
tests/test_gpu_fill.py before any parity test relies on it.

The inputs stand in for the KV state the paper's ShareGPT / Splitwise-Conv
runs would produce: only lengths and page scatter matter to the
path, and the recipe for each BASELINE.json config is in DESIGN.md section 4.
"""
from .gen import (MASTER_SEED, Workload, substream, cfg0_tiny, cfg1_qwen14b,
                  cfg2_qwen32b, cfg3_burst, cfg4_longctx, random_mid, random_tiny)
from .content import g_words, fill_plane_np

__all__ = ["MASTER_SEED", "Workload", "substream", "cfg0_tiny", "cfg1_qwen14b",
           "cfg2_qwen32b", "cfg3_burst", "cfg4_longctx", "random_mid", "random_tiny",
           "g_words", "fill_plane_np"]
