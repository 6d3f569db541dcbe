"""Differential fuzz of the CUDA path against the oracle: random geometries (workloads.random_mid /
random_tiny) x kernels x descriptor paths x buffer kinds (HBM, mapped host, staged ring) x
MERGE_ADJACENT x L2-prefetch distances x parameter size classes, every case compared word for word
(whole destination pools included).  Runs for LUMEN_FUZZ_SECONDS (default 25 s, about 250 cases); a
500 s run of the same loop (4,947 cases) is what round 2 was checked with."""
import os
import time

import pytest

from workloads import random_mid, random_tiny, substream

pytestmark = pytest.mark.gpu


def test_random_cases_against_the_oracle():
    from tests import gpu_util as G
    from tests.test_gpu_parity import run_case, run_staged_case
    G.build_all()
    lk = G.lk
    budget = float(os.environ.get("LUMEN_FUZZ_SECONDS", "25"))
    seed = int(os.environ.get("LUMEN_FUZZ_SEED", "1"))
    rng = substream(seed, "fuzz")
    t0, n = time.time(), 0
    try:
        while time.time() - t0 < budget:
            w = random_mid(rng) if rng.random() < 0.7 else random_tiny(rng)
            L, H, D, S, N = w.geom
            row = H * D * 2
            if row % 16:
                continue
            kernel = str(rng.choice(["warp", "warp_upload", "bulk", "auto"]))
            where = str(rng.choice(["device", "host"]))
            merge = bool(rng.integers(0, 2))
            pf = int(rng.choice([-1, 0, 1, 16, 100]))
            lk.lumen_kv_set_option("prefetch", pf)
            lk.lumen_kv_set_option("inline_max_runs", int(rng.choice([0, 256, 1024])))
            what = (n, w.geom, len(w.reqs), kernel, where, merge, pf)
            try:
                if rng.random() < 0.25 and w.tokens > 0:
                    # a run (tokens inside one page, cut at 32 KiB) always fits a slot
                    slot = max(row, min(S * row, 32768)) * int(rng.integers(1, 5))
                    run_staged_case(G, w, slot, int(rng.integers(2, 5)), seed=n,
                                    kernel=kernel if kernel != "warp" else "auto")
                else:
                    run_case(G, w, kernel, where, merge=merge, seed=n)
            except Exception as e:                                   # name the case before failing
                raise AssertionError(f"fuzz case {what}: {e!r}") from e
            n += 1
    finally:
        lk.lumen_kv_set_option("prefetch", 16)
        lk.lumen_kv_set_option("inline_max_runs", 1024)
    assert n > 20, n
