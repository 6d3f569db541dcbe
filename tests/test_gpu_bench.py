"""bench.py's headline at the driver's step count: the timed region must be bound by the two
kernels, not by the host (NVML polls between the event records made the
driver-run step 4x slower than the kernels at --steps 20)."""
import gc
import json
import subprocess
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent
pytestmark = pytest.mark.gpu


def test_headline_step_is_kernel_bound_at_20_steps():
    import torch
    gc.collect()
    torch.cuda.empty_cache()                       # the bench process needs the 146.5 GiB pool
    free_b, _ = torch.cuda.mem_get_info()
    if free_b < (100 << 30):
        pytest.skip("GPU memory is held by another test process")
    res = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--steps", "20", "--warmup", "5", "--no-e2e",
                          "--no-cpu-baseline", "--no-large"], capture_output=True, text=True, cwd=ROOT,
                         timeout=600)
    assert res.returncode == 0, res.stderr[-2000:]
    line = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    r = line["roofline"]
    kernels = r["pack_ms"] + r["unpack_ms"]
    assert line["steps"] == 20 and line["gpu_launches"] == 40
    assert not line["host_bound"]
    assert line["host_enqueue_ms_per_step"] < kernels
    assert line["ms_per_step"] <= 1.15 * kernels, (line["ms_per_step"], kernels)
    assert line["clocks"]["samples"] >= 1
    assert line["aligned_delta_variant"]["runs_per_plan"] == 64
    assert r["traffic_source"] is None or "profiles/" in r["traffic_source"]
