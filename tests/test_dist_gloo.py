"""N > 1 path on CPU (world_size 2, gloo): the path shards with no exchange step
(SURVEY.md section 8(e)), so what is covered here is the host logic of
`bench.py --gpus N`: per-rank seeds give independent replicas, the job time is the max
over ranks, `value` aggregates all ranks, and the reference arm runs on rank 0 only."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, str(ROOT))
    import bench
    from workloads import MASTER_SEED, cfg1_qwen14b

    assert bench.rank_env() == (rank, world, rank)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seed = bench.replica_seed(MASTER_SEED, rank)
    w = cfg1_qwen14b(seed, L=2, N=4000, n_reqs=8, grow_iters=4)
    # each rank's "device time": rank r took 10 + 5 r ms
    ms_local = 10.0 + 5.0 * rank
    ms = bench.max_over_ranks(ms_local, dist, "cpu")
    value = bench.job_payload_gbps(world, 3, w.payload_bytes, ms)
    # gather the structure of every replica to compare on rank 0
    pts = [None] * world
    dist.all_gather_object(pts, [pt.tolist() for pt, _, _ in w.reqs])
    lens = [None] * world
    dist.all_gather_object(lens, w.meta["lens"])
    dist.barrier()
    if rank == 0:
        Path(out_dir, "r0.json").write_text(json.dumps(
            {"ms": ms, "value": value, "P": w.payload_bytes, "pts": pts, "lens": lens}))
    dist.destroy_process_group()


def test_replicas_world2_gloo(tmp_path):
    world, port = 2, _free_port()
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    r = json.loads((tmp_path / "r0.json").read_text())
    assert r["ms"] == 15.0                               # max over ranks, not rank 0's 10 ms
    # 8 requests x 16 tokens x 2 L x 2 KiB rows, packed + restored, 3 steps, 2 ranks
    P = 8 * 16 * 2 * 2 * 2048
    assert r["P"] == P
    assert r["value"] == 2 * 3 * 2 * P / 15e-3 / 1e9
    # independent replicas: different lengths and different page tables per rank
    assert r["lens"][0] != r["lens"][1]
    assert r["pts"][0] != r["pts"][1]
    # a replica's page tables never reuse a page (rank-local pools are disjoint by construction)
    for rank_pts in r["pts"]:
        flat = np.concatenate([np.asarray(p) for p in rank_pts])
        assert np.unique(flat).size == flat.size


def test_single_process_defaults(monkeypatch):
    sys.path.insert(0, str(ROOT))
    import bench
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert bench.rank_env() == (0, 1, 0)
    assert bench.max_over_ranks(7.5, None, "cpu") == 7.5
    assert bench.job_payload_gbps(1, 10, 10**9, 1000.0) == 20.0


def test_reference_arm_runs_on_rank0_only():
    """Under torchrun the other ranks exit 0 without work or output."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    p = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "1", "--warmup", "1"], env=env, capture_output=True, text=True,
                       timeout=120)
    assert p.returncode == 0 and p.stdout.strip() == ""


def test_cuda_arm_fails_loudly_without_gpu():
    if torch.cuda.is_available():
        return
    p = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--steps", "1"],
                       capture_output=True, text=True, timeout=300)
    assert p.returncode != 0
    assert "no CPU path" in p.stderr
