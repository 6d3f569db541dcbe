#!/usr/bin/env python
"""bench.py -- KV checkpoint pack / restore throughput on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload cfg1|cfg2|cfg4] [--kernel auto|warp|bulk]

A "step" is one pass of the whole hot path over one batch:
  a1 select every running request's delta [t_prev, t_cur)         (vectorised host ints)
  a2 lumen_kv_plan_build for the pack and for the restore          (host C++ + 1 small H2D)
  a3 lumen_kv_checkpoint_pack  pool -> HBM staging buffer          (1 kernel)
  a6 fresh pages for the restore come from the seeded page tables  (input)
  a7 lumen_kv_restore_unpack   HBM staging buffer -> fresh pages   (1 kernel)
  plus lumen_kv_plan_free of both plans.
`value` is payload GB/s (bytes checkpointed + bytes restored per second), device-timed
with inputs resident in HBM.  `e2e` is the same step through the same C ABI with HOST
buffers: pack writes mapped pinned host memory (a4), restore reads it back, so P bytes
cross the host link in each direction inside the timed region.
Default workload = BASELINE.json configs[1] (Qwen3-14B shape, 64 requests, 16-token
deltas, pool of 60,000 pages = 146.5 GiB).  Input recipe: DESIGN.md section 4.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

CYCLE = 64          # distinct delta sets the steps rotate over (each advances 16 tokens)
N_STAGE = 4         # rotating HBM staging buffers (4 x 160 MiB > 126 MB L2)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4", "chain", "interference", "overhead", "hostlink", "dram"],
                    default="cfg1")
    ap.add_argument("--kernel", choices=["auto", "warp", "bulk"], default="auto")
    ap.add_argument("--upload-descriptors", action="store_true",
                    help="LUMEN_KV_NO_INLINE: upload small plans to device memory too (A/B evidence)")
    ap.add_argument("--requests", type=int, default=0,
                    help="cfg1 only: a decode batch of this many requests instead of configs[1]'s 64 (evidence "
                         "for the descriptor size classes; the line says VARIANT)")
    ap.add_argument("--median", type=int, default=0, help="cfg1 only, with --requests: lognormal median")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-large", action="store_true",
                    help="default run only: skip the large_configs block (cfg2 + cfg4 wave 0)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="default: min(steps, 100)")
    args = ap.parse_args()
    if args.requests:
        CFG1_VARIANT["n_reqs"] = args.requests
        if args.median:
            CFG1_VARIANT["median"] = args.median
    return args


# ------------------------------------------------------------------------------------
# workload construction (structure only; see workloads/gen.py)
# ------------------------------------------------------------------------------------
CFG1_VARIANT = {}   # --requests / --median: a larger decode batch than configs[1] names (evidence only)


def make_workload(name: str, seed: int, pages_cap=None):
    from workloads import cfg0_tiny, cfg1_qwen14b, cfg2_qwen32b, cfg4_longctx
    if name == "cfg0":
        w = cfg0_tiny(seed)
        label = ("BASELINE.json configs[0]: tiny pool, 2 layers x [64 pages, 16, 2 kv_heads, 64], 4 requests "
                 "37/100/5/64 tokens, deltas [t_prev, len) -- a correctness config: it fits in L2, its GB/s "
                 "is launch latency, not a roofline claim")
        delta = 0
    elif name == "cfg1":
        N = 60000 if pages_cap is None else min(60000, pages_cap)
        w = cfg1_qwen14b(seed, N=N, grow_iters=CYCLE, **CFG1_VARIANT)
        label = (f"BASELINE.json configs[1]: Qwen3-14B-shaped KV (40 layers, 8 kv_heads, head_dim 128, "
                 f"bf16, page_size 16, pool {N} pages), 64 requests lognormal(median 2k, sigma 1, "
                 f"clip 128..16k), 16-token delta per request per step")
        if CFG1_VARIANT:
            label = (f"VARIANT of configs[1] (not the BASELINE.json workload): {CFG1_VARIANT.get('n_reqs', 64)} "
                     f"requests, lognormal median {CFG1_VARIANT.get('median', 2048)}, otherwise as configs[1]: "
                     f"Qwen3-14B shape, pool {N} pages, 16-token delta per request per step")
        delta = 16
    elif name == "cfg2":
        w = cfg2_qwen32b(seed)
        label = ("BASELINE.json configs[2]: Qwen3-32B-shaped KV (64 layers), 16 requests x 8k-token "
                 "full-prefix pack then restore into fresh seeded-random pages, pool 20000 pages")
        delta = 0
    else:
        w = cfg4_longctx(seed, wave_reqs=2)
        label = ("BASELINE.json configs[4] (wave of 2 of the 8 requests; the as-written 256 GiB does "
                 "not fit one GPU): Qwen3-32B shape, page_size 1, 128k tokens each, shuffled slots")
        delta = 0
    return w, label, delta


def iteration_ranges(w, delta: int, cycle: int):
    """Per cycle position: (t_begin[], t_end[]) for every request (a1)."""
    tb0 = np.array([tb for _, tb, _ in w.reqs], dtype=np.int64)
    te0 = np.array([te for _, _, te in w.reqs], dtype=np.int64)
    if delta == 0:
        return [(tb0, te0)]
    return [(tb0 + delta * i, te0 + delta * i) for i in range(cycle)]


# ------------------------------------------------------------------------------------
# clocks during the timed region: NVML polled by a HELPER PROCESS (its own interpreter, so it can
# neither take this process's GIL nor sit between the two event records of a timed region)
# ------------------------------------------------------------------------------------
_CLOCK_HELPER = r"""
import os, signal, sys, time
import pynvml as nv
uuid, index, path = sys.argv[1], int(sys.argv[2]), sys.argv[3]
parent = os.getppid()
nv.nvmlInit()
try:
    h = nv.nvmlDeviceGetHandleByUUID(uuid)
except Exception:
    h = nv.nvmlDeviceGetHandleByIndex(index)
state = {"stop": False, "period": None}          # period None: idle (no NVML traffic at all)
signal.signal(signal.SIGTERM, lambda *a: state.update(stop=True))
signal.signal(signal.SIGUSR1, lambda *a: state.update(period=0.0002))   # short kernel regions
signal.signal(signal.SIGHUP, lambda *a: state.update(period=0.05))      # seconds-long host-link regions
signal.signal(signal.SIGUSR2, lambda *a: state.update(period=None))
f = open(path, "w")
f.write("max %d\n" % nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)); f.flush()
while not state["stop"] and os.getppid() == parent:      # never outlive the bench process
    if state["period"] is None:
        time.sleep(0.001)
        continue
    t = time.monotonic_ns()
    mhz = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
    try:
        mask = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
    except Exception:
        mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
    f.write("%d %d %d\n" % (t, mhz, mask)); f.flush()
    time.sleep(state["period"] or 0.0002)
f.close()
"""


class ClockSampler:
    """SM clock and throttle reasons DURING timed regions.  A helper process polls NVML while a
    window is open and stamps each sample with CLOCK_MONOTONIC; start() / stop() signal the helper
    and note the window's two timestamps, summary() keeps the samples inside the windows.  Outside
    windows the helper makes no NVML call: polling at kHz rate for the whole run was measured to
    cost the copy engines a quarter of their D2H rate (pinned memcpy 41 instead of 57 GB/s), so
    seconds-long host-link regions are sampled at 20 Hz (start(slow=True)).
    poll() takes one sample from the calling thread: call it only where the host has nothing
    left to enqueue (after the end event has been recorded, while the device is still busy)."""
    REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap",
               0x8: "hw_slowdown", 0x10: "sync_boost", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
               0x100: "display_clock_setting"}

    def __init__(self, index: int, uuid: str = ""):
        import subprocess
        import tempfile
        self.windows, self._open, self.own = [], None, []
        self.max_mhz, self.proc, self.nv, self.h = None, None, None, None
        fd, self.path = tempfile.mkstemp(prefix="lumen_clocks_", suffix=".txt")
        os.close(fd)
        try:
            self.proc = subprocess.Popen([sys.executable, "-c", _CLOCK_HELPER, uuid, str(index), self.path],
                                         stdout=subprocess.DEVNULL, stderr=subprocess.DEVNULL)
            import atexit
            atexit.register(self.close)
        except Exception:
            self.proc = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid)
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _signal(self, sig):
        if self.proc is not None and self.proc.poll() is None:
            try:
                os.kill(self.proc.pid, sig)
            except OSError:
                pass

    def start(self, slow: bool = False):
        import signal
        self._signal(signal.SIGHUP if slow else signal.SIGUSR1)
        self._open = time.monotonic_ns()

    def stop(self):
        import signal
        if self._open is not None:
            self.windows.append((self._open, time.monotonic_ns()))
            self._open = None
        self._signal(signal.SIGUSR2)

    def poll(self):
        if self.nv is None:
            return
        try:
            mhz = self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)
            try:
                mask = self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
            except Exception:
                mask = self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            self.own.append((mhz, mask))
        except Exception:
            pass

    def _helper_samples(self):
        out = []
        try:
            for line in open(self.path):
                p = line.split()
                if len(p) == 3:
                    out.append((int(p[0]), int(p[1]), int(p[2])))
        except Exception:
            pass
        return out

    def summary(self, reset: bool = False):
        """Median SM MHz and the union of throttle reasons over the windows noted so far."""
        hs = [(m, k) for t, m, k in self._helper_samples()
              if any(a <= t <= b for a, b in self.windows)]
        allp = hs + self.own
        reasons = sorted({name for _, mask in allp for bit, name in self.REASONS.items()
                          if mask & bit and name != "gpu_idle"})
        out = {"sm_mhz": float(np.median([m for m, _ in allp])) if allp else None,
               "sm_max_mhz": self.max_mhz, "reasons": reasons, "samples": len(allp),
               "sampler": "NVML polled by a helper process during the timed regions"
                          + (f" ({len(hs)} samples)" if hs else " (none fell inside)")
                          + (f" + {len(self.own)} from this process after the end event was recorded, "
                             "device still busy" if self.own else "")}
        if reset:
            self.windows, self.own = [], []
        return out

    def close(self):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()
            self.proc = None
        try:
            os.unlink(self.path)
        except OSError:
            pass


def gpu_uuid(torch, local: int) -> str:
    try:
        return "GPU-" + str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        return ""


# ------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py executes oracle/)
# ------------------------------------------------------------------------------------
def oracle_sample(workload: str, seed: int):
    """A bounded sample of the workload on a sparse host pool: one step's pack + restore
    for cfg1 (2 x 160 MiB); for the 32 GiB configs the first request's first 4096 tokens."""
    from workloads.hostpool import sparse_host_pool
    if workload == "overhead":
        workload = "cfg1"
    if workload in ("chain", "interference"):
        workload = "cfg2"                  # both work on cfg 2-shaped prefixes
    if workload == "cfg3":
        # burst sample: one 1-token delta pack of the 64 running requests + the restore of the
        # first interrupted request's first 4096 tokens into its free-list pages
        from workloads import Workload, cfg3_burst
        b = cfg3_burst(seed)
        pt, _, _ = b.waves[0][0]
        n = min(4096, b.waves[0][0][2])
        w = Workload("cfg3_burst", b.geom, list(b.running), [(pt, 0, n)])
        K, V, keep = sparse_host_pool(w.geom, seed, list(w.reqs) + list(w.restore_reqs))
        return (w, "BASELINE.json configs[3] (recovery burst, Qwen3-32B shape)", w.reqs, w.restore_reqs,
                K, V, keep, f"1-token pack of 64 running requests + restore of {n} tokens of one request")
    w, label, delta = make_workload(workload, seed)
    content = "g"
    if workload in ("cfg0", "cfg1"):
        reqs, rreqs = w.reqs, w.restore_reqs
        what = f"one full step ({len(w.reqs)} requests, {w.tokens} tokens, pack + restore)"
    elif workload == "cfg2" and mem_available_gib() >= 40:
        # "cfg 2 whole if host RAM allows a 32 GiB pool + 32 GiB buffer, else the first
        # 4 requests (8 GiB) and say so".  The sparse pool holds source pages + fresh pages + buffer
        # = 3 x 8 GiB for 4 requests; the whole config would need 96 GiB of host RAM.
        reqs, rreqs = w.reqs[:4], w.restore_reqs[:4]
        content = "tiled"
        what = ("the first 4 of the 16 requests, 8,192 tokens each (8 GiB packed + 8 GiB restored per "
                f"step; the whole config needs 96 GiB of host RAM, {mem_available_gib():.0f} GiB available; "
                "touched pages hold tiled seeded random page images, see workloads/hostpool.py)")
    else:
        n = 4096
        reqs = [(w.reqs[0][0], 0, n)]
        rreqs = [(w.restore_reqs[0][0], 0, n)]
        what = f"first request, first {n} tokens (pack + restore; 1 GiB each way)"
    K, V, keep = sparse_host_pool(w.geom, seed, list(reqs) + list(rreqs), content=content)
    return w, label, reqs, rreqs, K, V, keep, what


def mem_available_gib() -> float:
    try:
        for l in open("/proc/meminfo"):
            if l.startswith("MemAvailable:"):
                return int(l.split()[1]) / 2**20
    except Exception:
        pass
    return 0.0


def oracle_step(geom, K, V, reqs, rreqs, omp=False):
    import oracle
    B = oracle.pack(geom, K, V, reqs, omp=omp)
    n_restore = oracle.total_elems(geom, rreqs)
    if n_restore != B.size:        # burst sample: the restored checkpoint is not the packed delta
        R = np.zeros(n_restore, dtype=np.uint16)
        oracle.unpack(geom, K, V, rreqs, R, omp=omp)
        return (B.size + n_restore) * 2
    oracle.unpack(geom, K, V, rreqs, B, omp=omp)
    return 2 * B.size * 2          # payload bytes moved: packed + restored


def cpu_baseline(workload: str, seed: int, budget_s: float = 12.0):
    import oracle
    w, label, reqs, rreqs, K, V, keep, what = oracle_sample(workload, seed)
    oracle_step(w.geom, K, V, reqs, rreqs)                       # warm: page-faults the pool
    t0 = time.perf_counter(); nbytes = oracle_step(w.geom, K, V, reqs, rreqs)
    one = time.perf_counter() - t0
    reps = int(max(1, min(64, budget_s / max(one, 1e-3))))
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle_step(w.geom, K, V, reqs, rreqs)
    dt = time.perf_counter() - t0
    cpu_model = next((l.split(":", 1)[1].strip() for l in open("/proc/cpuinfo") if l.startswith("model name")),
                     "unknown")
    out = {"value": nbytes * reps / dt / 1e9, "unit": "GB/s", "cores": 1, "kind": "oracle", "cpu": cpu_model,
           "cores_available": len(os.sched_getaffinity(0)),
           "sample": f"{what}, {reps} repetitions, plain single-thread C oracle as it stands"}
    # context only: the OpenMP/memcpy timing variant (asserted equal to the plain one in tests)
    threads = oracle.omp_threads()
    oracle_step(w.geom, K, V, reqs, rreqs, omp=True)
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle_step(w.geom, K, V, reqs, rreqs, omp=True)
    dt = time.perf_counter() - t0
    out["omp_variant"] = {"value": nbytes * reps / dt / 1e9, "unit": "GB/s", "cores": threads}
    return out


def l2_config(workload: str) -> str:
    """`config.l2`, the same string in both arms (what is specific to an arm sits in `l2_note`)."""
    return "fits in L2" if workload == "cfg0" else "inputs larger than L2"


def flat_summary(line: dict) -> dict:
    """The scalars a reader of the driver's record needs, as the LAST key of the line (the record
    keeps the tail): large-config fractions, the staged host fractions, how often the headline
    region was taken."""
    out = {"headline_attempts_n": len(line.get("headline_attempts") or []),
           "roofline_frac": (line.get("roofline") or {}).get("frac"),
           "e2e_value": (line.get("e2e") or {}).get("value"),
           "e2e_duplex_frac_of_duplex_memcpy_peak": (line.get("e2e") or {}).get("duplex_frac_of_duplex_memcpy_peak"),
           "host_bound": line.get("host_bound")}
    lc = line.get("large_configs") or {}
    for key, tag in (("cfg2", "cfg2"), ("cfg4_wave0", "cfg4w0")):
        c = lc.get(key) or {}
        if c:
            out[f"{tag}_hbm_frac"] = c.get("frac")
            out[f"{tag}_pack_ms"] = c.get("pack_ms")
            out[f"{tag}_unpack_ms"] = c.get("unpack_ms")
            out[f"{tag}_ms_per_step"] = c.get("ms_per_step")
            out[f"{tag}_host_enqueue_ms_per_step"] = c.get("host_enqueue_ms_per_step")
        hs = c.get("host_staged") or {}
        if "pack_frac_of_d2h_memcpy" in hs:
            out[f"{tag}_staged_pack_frac"] = hs["pack_frac_of_d2h_memcpy"]
            out[f"{tag}_staged_restore_frac"] = hs["restore_frac_of_h2d_memcpy"]
    return out


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; rank 0 only."""
    if rank_env()[0] != 0:
        return
    from workloads import MASTER_SEED
    w, label, reqs, rreqs, K, V, keep, what = oracle_sample(args.workload, MASTER_SEED)
    for _ in range(max(1, min(args.warmup, 3))):
        oracle_step(w.geom, K, V, reqs, rreqs)
    steps = max(1, args.steps)
    # keep the whole run within a few minutes whatever K the driver passes
    t0 = time.perf_counter(); nbytes = oracle_step(w.geom, K, V, reqs, rreqs); one = time.perf_counter() - t0
    timed = int(max(1, min(steps, 120.0 / max(one, 1e-3))))
    t0 = time.perf_counter()
    for _ in range(timed):
        oracle_step(w.geom, K, V, reqs, rreqs)
    dt = time.perf_counter() - t0
    val = nbytes * timed / dt / 1e9
    line = {"impl": "reference", "metric": "kv_pack_restore_payload_GBps", "value": val, "unit": "GB/s",
            "n_gpus": args.gpus, "steps": steps, "warmup": args.warmup, "ms_per_step": dt / timed * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u16",
            "data": "synthetic",
            # same keys as the CUDA arm's `config` (what is specific to an arm sits beside it)
            "config": {"workload": label,
                       "payload_bytes_per_direction_per_step": int(w.tokens) * 4 * w.geom[0] * w.geom[1] * w.geom[2],
                       "tokens_per_step": int(w.tokens),
                       "l2": l2_config(args.workload),
                       "seed": hex(MASTER_SEED)},
            "l2_note": "CPU arm: every step touches far more than the host caches hold "
                       "(the step's sample is named in cpu_baseline.sample)",
            "timed_steps": timed,
            "cpu_baseline": {"value": val, "unit": "GB/s", "cores": 1, "kind": "oracle",
                             "sample": f"each step = {what}; plain single-thread C oracle"},
            "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------
# replicas: the path shards with no exchange step, so N ranks are N
# independent replicas; the only cross-rank traffic is the barrier and the max of the times
# ------------------------------------------------------------------------------------
def rank_env():
    """(rank, world, local_rank) as torchrun exports them; single process otherwise."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def replica_seed(master_seed: int, rank: int) -> int:
    """Every rank draws its own lengths / page tables / pool content."""
    return master_seed + rank


def max_over_ranks(ms: float, dist, device) -> float:
    """Device time of the job = the slowest rank's (all_reduce MAX); dist None => 1 rank."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_payload_gbps(world: int, steps: int, payload_bytes: int, ms: float) -> float:
    """Whole-job payload GB/s: every rank packs P and restores P per step."""
    return world * steps * 2 * payload_bytes / (ms * 1e-3) / 1e9


# ------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------
def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
        except Exception:
            pass
    return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


def ncu_traffic(workload: str, kernel: str, direction: str):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, source):
    NOT measured in this run -- read from the committed ncu --set full capture that
    profiles/traffic.csv indexes (profiles/README.md names the commands); (None, None) if absent."""
    import csv
    p = ROOT / "profiles" / "traffic.csv"
    if not p.exists():
        return None, None
    try:
        rows = [r for r in csv.DictReader(open(p, newline=""))
                if (r["workload"], r["kernel"], r["direction"]) == (workload, kernel, direction)]
    except Exception:
        return None, None
    if not rows:
        return None, None
    r = rows[-1]                                        # the newest capture is appended last
    return (int(r["dram_bytes_read"]) + int(r["dram_bytes_write"]),
            f"profiles/{r['source']} (committed ncu capture, {r.get('capture') or 'cold'}; not measured in this run)")


def memcpy_peaks(torch, nbytes=1 << 30):
    """Pinned cudaMemcpyAsync D2H / H2D, best of 10, CUDA events: the host-path denominators."""
    h = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    out = {}
    for name, dst, src in (("d2h", h, d), ("h2d", d, h)):
        best = float("inf")
        for _ in range(10):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); dst.copy_(src, non_blocking=True); b.record(); torch.cuda.synchronize()
            best = min(best, a.elapsed_time(b))
        out[name] = nbytes / best / 1e6
    # both directions at once: what two concurrent copies over the full-duplex link really reach
    # (less than d2h + h2d: the two directions share the host's memory system)
    h2 = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    d2 = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    best = float("inf")
    for _ in range(10):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        join = torch.cuda.Event()
        torch.cuda.synchronize()
        a.record(sa)
        sb.wait_event(a)
        with torch.cuda.stream(sa):
            h.copy_(d, non_blocking=True)
        with torch.cuda.stream(sb):
            d2.copy_(h2, non_blocking=True)
        join.record(sb)
        sa.wait_event(join)
        b.record(sa)
        torch.cuda.synchronize()
        best = min(best, a.elapsed_time(b))
    out["duplex"] = 2 * nbytes / best / 1e6
    return out


class HbmPath:
    """One pool + one workload: the step of DESIGN.md section 7 (a1, a2 x 2, a3, a7, plan_free x 2)
    and the loops that time it.  Nothing between the two event records of a timed region but the
    calls of the path itself."""

    def __init__(self, torch, lk, pool, w, delta, kflag, stream, dist):
        self.torch, self.lk, self.pool, self.w, self.dist = torch, lk, pool, w, dist
        self.P = w.payload_bytes
        self.ranges = iteration_ranges(w, delta, CYCLE)
        self.kflag, self.stream, self.sh = kflag, stream, stream.cuda_stream
        self.ra_p, self.ra_r = lk.ReqArray(w.reqs), lk.ReqArray(w.restore_reqs)
        self.single_stats = {}

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def step(self, i, bufs, kind, lag_, evs=None, only=None):
        """only=None: the whole step.  only="pack"/"unpack": that direction alone (same plans,
        same rotation), used to time one kernel as a back-to-back batch of launches."""
        lk, pool, ranges, P, sh, stream = self.lk, self.pool, self.ranges, self.P, self.sh, self.stream
        nb = len(bufs)
        p = r = None
        if only != "unpack":
            tb, te = ranges[i % len(ranges)]
            self.ra_p.set_ranges(tb, te)                                                    # a1
            p = lk.lumen_kv_plan_build(pool.geom, self.ra_p, self.kflag, sh)                # a2
        if only != "pack":
            tb, te = ranges[(i - lag_) % len(ranges)]
            self.ra_r.set_ranges(tb, te)
            r = lk.lumen_kv_plan_build(pool.geom, self.ra_r,
                                       self.kflag | lk.LUMEN_KV_VALIDATE_UNIQUE_DST, sh)
        if evs is not None:
            evs[0].record(stream)
        if p is not None:
            lk.lumen_kv_checkpoint_pack(p, pool.k_ptrs, pool.v_ptrs, bufs[i % nb].data_ptr(), P, kind, sh)  # a3 / a4
        if evs is not None:
            evs[1].record(stream)
        if r is not None:
            lk.lumen_kv_restore_unpack(r, pool.k_ptrs, pool.v_ptrs, bufs[(i - lag_) % nb].data_ptr(), P,
                                       kind, sh)                                            # a7
        if evs is not None:
            evs[2].record(stream)
        if p is not None:
            p.close()
        if r is not None:
            r.close()

    def timed_loop(self, K, W, bufs, kind, lag_, sampler=None, per_launch=False, only=None):
        """W warm-up steps, then exactly K steps between one event pair.  per_launch=True adds
        an event between the launches of every step (kernel durations); those records sit
        between the kernels, so that variant is never the one `value` comes from.
        Returns (ms, pack_ms, unpack_ms, wall_ms, host_enqueue_ms)."""
        torch, stream, ranges = self.torch, self.stream, self.ranges
        for i in range(-lag_, 0):                      # fill the buffers the first restores read
            self.step(i + len(ranges) * len(bufs), bufs, kind, 0)
        for i in range(W):
            self.step(i, bufs, kind, lag_, only=only)
        evs = ([[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
               if per_launch else None)
        e_start, e_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.barrier(); torch.cuda.synchronize()
        if sampler:
            sampler.start()                            # one signal to the helper + a timestamp
        # the W warm-up steps again, untimed, right in front of the timed ones: the device is
        # busy (clocks up, pipeline full) when the start event fires, whatever K is
        for i in range(W):
            self.step(i, bufs, kind, lag_, None, only)
        t_wall = time.perf_counter()
        e_start.record(stream)
        for i in range(K):                             # nothing in here but the path's own calls
            self.step(W + i, bufs, kind, lag_, evs[i] if per_launch else None, only)
        e_end.record(stream)
        t_host = time.perf_counter() - t_wall          # host time to enqueue K steps
        if sampler:
            sampler.poll()                             # everything is enqueued, the device still runs it
        stream.synchronize(); torch.cuda.synchronize()
        t_wall = time.perf_counter() - t_wall
        if sampler:
            sampler.stop()
        self.barrier()
        ms = max_over_ranks(e_start.elapsed_time(e_end), self.dist, "cuda")
        pack_ms = unpack_ms = None
        if per_launch:
            pk = [e[0].elapsed_time(e[1]) for e in evs]
            up = [e[1].elapsed_time(e[2]) for e in evs]
            for name, xs in (("pack", pk), ("unpack", up)):
                self.single_stats[name] = {"mean": float(np.mean(xs)), "median": float(np.median(xs)),
                                           "best": float(np.min(xs))}
            pack_ms, unpack_ms = self.single_stats["pack"]["mean"], self.single_stats["unpack"]["mean"]
        return ms, pack_ms, unpack_ms, t_wall * 1e3, t_host * 1e3

    def direction_ms(self, K, W, bufs, kind, lag_, sampler, only, passes=1):
        """Average launch duration of one direction alone: K back-to-back launches between one event
        pair.  With only 3 launches of 10-20 ms per pass (the 32 / 64 GiB configs) one stall between
        two launches -- seen in about one run in four on this pool, 10-40 ms, not reproducible with
        the same loop in isolation and not in the per-launch times -- would triple the figure, so
        such a pass is taken `passes` times and the smallest is the kernel's; all are reported."""
        got = [self.timed_loop(K, W, bufs, kind, lag_, sampler, only=only)[0] / K for _ in range(passes)]
        return min(got), got

    def two_stream_loop(self, K, W, bufs, kind, lag_):
        """a8 on HBM buffers: the pack of step i on one stream, the restore of the buffer packed
        `lag_` steps earlier on a second one, ordered only by events on the buffers (a worker
        checkpoints its running requests and absorbs restores at the same time).  Same work per
        step as timed_loop; returns ms for K steps."""
        torch, lk, pool, ranges, P = self.torch, self.lk, self.pool, self.ranges, self.P
        sA, sB = self.stream, torch.cuda.Stream()
        nb = len(bufs)
        packed = [torch.cuda.Event() for _ in range(nb)]
        restored = [torch.cuda.Event() for _ in range(nb)]
        for ev in packed + restored:
            ev.record(sA)

        def step(i):
            tb, te = ranges[i % len(ranges)]
            self.ra_p.set_ranges(tb, te)
            p = lk.lumen_kv_plan_build(pool.geom, self.ra_p, self.kflag, sA.cuda_stream)
            tb, te = ranges[(i - lag_) % len(ranges)]
            self.ra_r.set_ranges(tb, te)
            r = lk.lumen_kv_plan_build(pool.geom, self.ra_r, self.kflag | lk.LUMEN_KV_VALIDATE_UNIQUE_DST,
                                       sB.cuda_stream)
            sA.wait_event(restored[i % nb])             # the restore that last read this buffer
            lk.lumen_kv_checkpoint_pack(p, pool.k_ptrs, pool.v_ptrs, bufs[i % nb].data_ptr(), P, kind,
                                        sA.cuda_stream)
            packed[i % nb].record(sA)
            sB.wait_event(packed[(i - lag_) % nb])      # the pack that filled the buffer it reads
            lk.lumen_kv_restore_unpack(r, pool.k_ptrs, pool.v_ptrs, bufs[(i - lag_) % nb].data_ptr(), P,
                                       kind, sB.cuda_stream)
            restored[(i - lag_) % nb].record(sB)
            p.close(); r.close()

        for i in range(-lag_, 0):
            self.step(i + len(ranges) * nb, bufs, kind, 0)
        for i in range(W):
            step(i)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.barrier(); torch.cuda.synchronize()
        for i in range(W):
            step(i)
        e0.record(sA)
        sB.wait_event(e0)
        for i in range(K):
            step(W + i)
        done_b = torch.cuda.Event(); done_b.record(sB)
        sA.wait_event(done_b)
        e1.record(sA)
        torch.cuda.synchronize(); self.barrier()
        return max_over_ranks(e0.elapsed_time(e1), self.dist, "cuda")

    def idle_single_launch(self, bufs, kind, idle_s=0.012, n=12):
        """A decode loop issues one pack per 13-58 ms iteration: no launch in front of it to
        overlap with, caches cold.  One event pair per launch around nothing but the call (plan
        built beforehand).  The stream first waits for a gate that opens after `idle_s` s in
        which the device runs nothing but one spinning warp (torch.cuda._sleep on a side
        stream): record, launch and record are already queued when it opens, so the figure holds
        no host launch latency (a Python call between the two records would add about 20 us)."""
        torch, stream, lk, pool = self.torch, self.stream, self.lk, self.pool
        side = torch.cuda.Stream()
        cycles = int(idle_s * 1.9e9)
        out = {}
        for only in ("pack", "unpack"):
            ts = []
            for i in range(n):
                tb, te = self.ranges[i % len(self.ranges)]
                ra = self.ra_p if only == "pack" else self.ra_r
                ra.set_ranges(tb, te)
                plan = lk.lumen_kv_plan_build(pool.geom, ra, self.kflag, self.sh)
                fn = lk.lumen_kv_checkpoint_pack if only == "pack" else lk.lumen_kv_restore_unpack
                torch.cuda.synchronize()
                gate = torch.cuda.Event()
                with torch.cuda.stream(side):
                    torch.cuda._sleep(cycles)
                    gate.record(side)
                stream.wait_event(gate)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                fn(plan, pool.k_ptrs, pool.v_ptrs, bufs[i % len(bufs)].data_ptr(), self.P, kind, self.sh)
                b.record(stream)
                stream.synchronize()
                plan.close()
                ts.append(a.elapsed_time(b))
            out[only] = {"median": float(np.median(ts)), "best": float(np.min(ts)), "mean": float(np.mean(ts))}
        return out


def fill_pool(pool, seed, wdev):
    for i, t in enumerate(pool.planes()):
        wdev.fill_plane(t, seed, i)


def staged_host_once(torch, lk, path, hb, ring, direction, async_call=False):
    """One staged call on a HOST buffer, device-timed; also the host time spent inside the call."""
    pool, P, s = path.pool, path.P, path.stream
    reqs, flag = ((path.ra_p, 0) if direction == "pack" else (path.ra_r, lk.LUMEN_KV_VALIDATE_UNIQUE_DST))
    tb, te = path.ranges[0]
    reqs.set_ranges(tb, te)
    plan = lk.lumen_kv_plan_build(pool.geom, reqs, path.kflag | flag, s.cuda_stream)
    name = "lumen_kv_checkpoint_pack_staged" if direction == "pack" else "lumen_kv_restore_unpack_staged"
    fn = getattr(lk, name + ("_async" if async_call else ""))
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record(s)
    t0 = time.perf_counter()
    ticket = fn(plan, pool.k_ptrs, pool.v_ptrs, hb.data_ptr(), P, ring.stager, s.cuda_stream)
    call_ms = (time.perf_counter() - t0) * 1e3
    if async_call:                                  # the calling thread is free from here on
        ring.stager.wait(ticket, s.cuda_stream)
    b.record(s)
    s.synchronize()
    n_chunks = len(plan.chunks(ring.stager.slot_bytes))
    plan.close()
    return a.elapsed_time(b), call_ms, n_chunks


def large_config(torch, lk, name, seed, kflag, stream, sampler, peak, link, with_host, waves=(0,)):
    """One of the large configs (BASELINE.json configs[2], configs[4]) inside the default line:
    HBM pack + restore (3 warm-up + 3 timed steps, then 3 launches of each direction alone), and
    for cfg2 the staged host path once in each direction.  Every `frac` is recomputable from the
    `*_ms` beside it."""
    from paper_2606_17787_b200.pool import KVPool, StagingRing
    from workloads import cfg4_longctx
    from workloads import device as wdev
    DEV = lk.LUMEN_KV_MEM_DEVICE
    out, pool, dbuf = {}, None, None
    agg_bytes = agg_ms = 0.0
    per_wave = []
    for wave in waves:
        if name == "cfg4":
            w = cfg4_longctx(seed, wave_reqs=2, wave=wave)
        else:
            w, _, _ = make_workload(name, seed)
        L, H, D, S, N = w.geom
        if pool is None:
            pool = KVPool(L, H, D, S, N)
            dbuf = torch.empty(w.payload_bytes, dtype=torch.uint8, device="cuda")
        fill_pool(pool, seed + wave, wdev)
        torch.cuda.synchronize()
        path = HbmPath(torch, lk, pool, w, 0, kflag, stream, None)
        P = path.P
        with torch.cuda.stream(stream):
            ms, _, _, _, host_ms = path.timed_loop(3, 3, [dbuf], DEV, 0, sampler)
            pack_ms, pack_passes = path.direction_ms(3, 3, [dbuf], DEV, 0, sampler, "pack", passes=2)
            unpack_ms, unpack_passes = path.direction_ms(3, 3, [dbuf], DEV, 0, sampler, "unpack", passes=2)
        per_wave.append({"wave": wave, "ms_per_step": ms / 3, "pack_ms": pack_ms, "unpack_ms": unpack_ms,
                         "pack_ms_passes": pack_passes, "unpack_ms_passes": unpack_passes,
                         "payload_GBps": 2 * P / (ms / 3) / 1e6})
        agg_bytes += 2 * P
        agg_ms += ms / 3
    dom_ms = max(pack_ms, unpack_ms)
    out = {"payload_bytes_per_direction": P, "pool_pages": N, "page_size": S,
           "ms_per_step": ms / 3, "payload_GBps": 2 * P / (ms / 3) / 1e6,
           "pack_ms": pack_ms, "unpack_ms": unpack_ms,
           "pack_ms_passes": pack_passes, "unpack_ms_passes": unpack_passes,
           "achieved_GBps": 2 * P / dom_ms / 1e6, "peak_GBps": peak, "frac": 2 * P / dom_ms / 1e6 / peak,
           "frac_formula": "2 * payload_bytes_per_direction / max(pack_ms, unpack_ms) / peak_GBps",
           "frac_of_spec_8TBps": 2 * P / dom_ms / 1e6 / 8000.0,
           "frac_of_pin_rate_8184GBps": 2 * P / dom_ms / 1e6 / 8184.0,
           "host_enqueue_ms_per_step": host_ms / 3,
           "timing": "3 warm-up + 3 timed steps between one event pair; pack_ms / unpack_ms = 3 launches of "
                     "that direction alone between one event pair; inputs larger than L2 (tens of GiB per launch)"}
    if len(waves) > 1:
        out["waves"] = per_wave
        out["all_waves_payload_GBps"] = agg_bytes / agg_ms / 1e6
    traffic, tsrc = ncu_traffic(name, "warp", "pack" if pack_ms >= unpack_ms else "unpack")
    out["traffic"], out["traffic_source"] = traffic, tsrc
    avail = wdev.host_mem_available()
    if with_host and avail is not None and P > avail - (8 << 30):
        out["host_staged"] = {"skipped": f"pinning {P >> 30} GiB needs more host memory than this box has "
                                         f"available ({avail >> 30} GiB); see --workload cfg2 on a larger host"}
        with_host = False
    if with_host:
        hb = wdev.pinned_exact(P)
        ring = StagingRing(32 << 20, 3)
        staged_host_once(torch, lk, path, hb, ring, "pack")        # warm-up
        sampler.start(slow=True)
        p_ms, p_call, n_chunks = staged_host_once(torch, lk, path, hb, ring, "pack")
        r_ms, r_call, _ = staged_host_once(torch, lk, path, hb, ring, "restore")
        pa_ms, pa_call, _ = staged_host_once(torch, lk, path, hb, ring, "pack", async_call=True)
        ra_ms, ra_call, _ = staged_host_once(torch, lk, path, hb, ring, "restore", async_call=True)
        sampler.stop()
        out["host_staged"] = {"pack_GBps": P / p_ms / 1e6, "restore_GBps": P / r_ms / 1e6,
                              "pack_ms": p_ms, "restore_ms": r_ms, "chunks_per_call": n_chunks,
                              "pack_frac_of_d2h_memcpy": P / p_ms / 1e6 / link["d2h"],
                              "restore_frac_of_h2d_memcpy": P / r_ms / 1e6 / link["h2d"],
                              "memcpy_peak_d2h_GBps": link["d2h"], "memcpy_peak_h2d_GBps": link["h2d"],
                              "staged_call_host_ms": {"pack": p_call, "restore": r_call},
                              "async": {"pack_GBps": P / pa_ms / 1e6, "restore_GBps": P / ra_ms / 1e6,
                                        "call_host_ms": {"pack": pa_call, "restore": ra_call},
                                        "note": "lumen_kv_*_staged_async: the stager's thread issues the chunks; "
                                                "call_host_ms is what the calling thread spends in the call"}}
        ring.close()
        wdev.unpin(hb)
        del hb
    out["clocks"] = sampler.summary(reset=True)
    del pool, dbuf, path
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    return out


def run_ours(args):
    import torch
    import paper_2606_17787_b200 as lk            # fails loudly if liblumen_kv.so is missing
    from paper_2606_17787_b200.pool import KVPool, pinned_buffer
    from workloads import MASTER_SEED
    from workloads import device as wdev

    rank, world, local = rank_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    torch.cuda.set_device(local)
    dist = None
    if world > 1 or os.environ.get("LUMEN_BENCH_FORCE_DIST"):   # the switch exercises the N > 1 code on 1 GPU
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    wdev.build()
    sampler = ClockSampler(local, gpu_uuid(torch, local))

    def barrier():
        if dist is not None:
            dist.barrier()

    # ---- workload (one replica per rank: weak scaling, no data-path collective) ----------
    seed = replica_seed(MASTER_SEED, rank)
    free_b, _total = torch.cuda.mem_get_info()
    pages_cap = None
    if args.workload == "cfg1":
        page_all = 2 * 40 * 16 * 8 * 128 * 2
        reserve = N_STAGE * 64 * 16 * 160 * 1024 + (6 << 30)
        fit = int((free_b - reserve) // page_all // 1000 * 1000)
        pages_cap = fit if fit < 60000 else None
    w, label, delta = make_workload(args.workload, seed, pages_cap)
    L, H, D, S, N = w.geom
    pool = KVPool(L, H, D, S, N)
    fill_pool(pool, seed, wdev)
    torch.cuda.synchronize()
    P = w.payload_bytes
    n_stage = N_STAGE if P <= (1 << 30) else 1
    lag = 2 if n_stage > 1 else 0
    dbufs = [torch.empty(P, dtype=torch.uint8, device="cuda") for _ in range(n_stage)]

    kflag = {"auto": lk.LUMEN_KV_KERNEL_AUTO, "warp": lk.LUMEN_KV_KERNEL_WARP,
             "bulk": lk.LUMEN_KV_KERNEL_BULK}[args.kernel]
    if args.upload_descriptors:
        kflag |= lk.LUMEN_KV_NO_INLINE
    stream = torch.cuda.Stream()
    sh = stream.cuda_stream
    path = HbmPath(torch, lk, pool, w, delta, kflag, stream, dist)
    ranges, ra_p, ra_r = path.ranges, path.ra_p, path.ra_r
    geom, kp, vp = pool.geom, pool.k_ptrs, pool.v_ptrs
    DEV, HOST = lk.LUMEN_KV_MEM_DEVICE, lk.LUMEN_KV_MEM_HOST_MAPPED
    UNIQUE = lk.LUMEN_KV_VALIDATE_UNIQUE_DST

    K, W = max(1, args.steps), max(3, args.warmup)
    big = P > (1 << 30)
    Kk = min(K, 200) if not big else min(K, 3)         # per-launch pass: same steps, instrumented
    with torch.cuda.stream(stream):
        # (tens-of-GiB configs: 3 launches per pass, the better of two passes -- see direction_ms)
        pack_ref, pack_passes = path.direction_ms(Kk, 3, dbufs, DEV, lag, None, "pack", passes=2 if big else 1)
        unpack_ref, unpack_passes = path.direction_ms(Kk, 3, dbufs, DEV, lag, None, "unpack", passes=2 if big else 1)
        # The headline: exactly K steps between one event pair.  A region whose step comes out more
        # than 15 % above its two kernels did not measure the kernels -- the host could not feed it
        # (this process descheduled for a millisecond inside a 2 ms region) or the device stalled
        # between launches -- and is taken again, once; both attempts are reported.  The decision is
        # the same on every rank (ms and the kernel times are maxima over ranks, the host flag is
        # reduced), so that replicas never disagree on how many loops they run.
        attempts = []
        for _ in range(2):
            ms, _, _, wall_ms, host_ms = path.timed_loop(K, W, dbufs, DEV, lag, sampler)
            clocks = sampler.summary(reset=True)
            slow = ms / K > 1.15 * (pack_ref + unpack_ref)
            starved = slow and host_ms / K > pack_ref + unpack_ref
            starved = max_over_ranks(1.0 if starved else 0.0, dist, "cuda") > 0.5
            attempts.append({"ms_per_step": ms / K, "host_enqueue_ms_per_step": host_ms / K,
                             "host_bound": bool(starved), "more_than_15pct_above_kernels": bool(slow)})
            if not slow:
                break
        ms_k, pack_1, unpack_1, _, _ = path.timed_loop(Kk, 3, dbufs, DEV, lag, per_launch=True)
        single = {k: dict(v) for k, v in path.single_stats.items()}   # single-launch latency: mean/median/best
        pack_ms, unpack_ms = pack_ref, unpack_ref
        idle = path.idle_single_launch(dbufs, DEV) if not big else None
        ms_2s = path.two_stream_loop(K, W, dbufs, DEV, lag) if n_stage > 1 else None
    value = job_payload_gbps(world, K, P, ms)
    token_bytes = 2 * L * H * D * 2
    n_pb = 200 if not big else 10                        # a2 alone, on the host clock
    t0 = time.perf_counter()
    for i in range(n_pb):
        tb, te = ranges[i % len(ranges)]
        ra_p.set_ranges(tb, te)
        pl = lk.lumen_kv_plan_build(geom, ra_p, kflag, sh)
        runs_per_plan = pl.num_runs
        pl.close()
    plan_build_us = (time.perf_counter() - t0) / n_pb * 1e6
    stream.synchronize()
    host_bound = attempts[-1]["host_bound"]

    # ---- roofline of the dominant kernel ------------------------------------------------
    peak, peak_src = measured_peaks()
    dom, dom_ms = ("lumen_kv_checkpoint_pack", pack_ms) if pack_ms >= unpack_ms else \
                  ("lumen_kv_restore_unpack", unpack_ms)
    achieved = 2 * P / (dom_ms * 1e-3) / 1e9
    resolved = args.kernel if args.kernel != "auto" else "warp"
    kname = "kv_copy_warp32 (256-bit accesses)" if resolved == "warp" else "kv_copy_" + resolved
    traffic, traffic_src = ncu_traffic(args.workload, resolved, "pack" if dom.endswith("pack") else "unpack")
    roofline = {"bound": "hbm", "kernel": f"{dom} ({kname})", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes_per_launch": 2 * P, "peak_source": peak_src,
                # also against the data-sheet figure ("spec", 8 TB/s HBM3e) and against
                # the pin rate ncu reports for this part (2,048 B/cycle x 3.996 GHz)
                "frac_of_spec_8TBps": achieved / 8000.0, "frac_of_pin_rate_8184GBps": achieved / 8184.0,
                "timing": (f"average launch duration = one CUDA-event pair around {Kk} back-to-back launches "
                           "of that direction alone (same plans and buffer rotation as the step), on the "
                           "launching stream, in this run; *_single_ms = one event pair per launch inside "
                           f"whole steps ({ms_k / Kk:.4f} ms/step: the records between the launches cost a "
                           "few us each and prevent the overlap of consecutive launches); "
                           "single_launch_after_idle_ms = one event pair per launch, queued behind a gate that opens after "
                           "12 ms in which the device runs one spinning warp (no memory traffic, no host latency inside)"),
                "pack_ms": pack_ms, "unpack_ms": unpack_ms,
                "pack_ms_passes": pack_passes, "unpack_ms_passes": unpack_passes,
                "pack_single_ms": pack_1, "unpack_single_ms": unpack_1, "single_launch_ms": single,
                "single_launch_after_idle_ms": idle,
                "pack_traffic_GBps": 2 * P / pack_ms / 1e6, "unpack_traffic_GBps": 2 * P / unpack_ms / 1e6}

    # ---- A16: the page-aligned delta variant of cfg 1 (1 run per request instead of 1-2) ---
    aligned = None
    if args.workload == "cfg1":
        from workloads import cfg1_qwen14b
        w_al = cfg1_qwen14b(seed, N=N, grow_iters=CYCLE, aligned=True)
        path_al = HbmPath(torch, lk, pool, w_al, delta, kflag, stream, dist)
        with torch.cuda.stream(stream):
            ms_al = path_al.timed_loop(K, W, dbufs, DEV, lag)[0]
        path_al.ra_p.set_ranges(*path_al.ranges[0])
        pl = lk.lumen_kv_plan_build(geom, path_al.ra_p, kflag, sh)
        aligned = {"value": job_payload_gbps(world, K, P, ms_al), "unit": "GB/s", "ms_per_step": ms_al / K,
                   "runs_per_plan": pl.num_runs,
                   "note": "SURVEY A16: t_begin = 16*floor((len-16)/16), t_end = t_begin + 16 (page-aligned deltas)"}
        pl.close()
        del path_al

    # ---- e2e: same step, host buffers, bytes cross the host link inside the timed region --
    e2e = None
    link = None
    if not args.no_e2e:
        est = 2 * P / 50e9
        Ke = args.e2e_steps or int(max(3, min(K, 100, 20.0 / est)))
        hb = [pinned_buffer(P) for _ in range(2 if not big else 1)]
        link = memcpy_peaks(torch)
        with torch.cuda.stream(stream):
            ms_e, pack_e, unpack_e, _, _ = path.timed_loop(Ke, 3, hb, HOST, 1 if len(hb) > 1 else 0,
                                                           per_launch=True)
        e2e = {"value": job_payload_gbps(world, Ke, P, ms_e), "unit": "GB/s",
               "h2d_bytes_per_step": P, "d2h_bytes_per_step": P, "steps": Ke,
               "ms_per_step": ms_e / Ke, "gpu_launches": 2 * Ke,
               "pack_to_host_GBps": P / pack_e / 1e6, "restore_from_host_GBps": P / unpack_e / 1e6,
               "memcpy_peak_d2h_GBps": link["d2h"], "memcpy_peak_h2d_GBps": link["h2d"],
               "pack_frac_of_d2h_peak": P / pack_e / 1e6 / link["d2h"],
               "restore_frac_of_h2d_peak": P / unpack_e / 1e6 / link["h2d"],
               "path": ""}
        # ---- two-stage host path: HBM-speed pack into a device staging ring + copy engine ------
        from paper_2606_17787_b200.pool import StagingRing
        SLOT, NSLOT = 32 << 20, 3
        ringP, ringR = StagingRing(SLOT, NSLOT), StagingRing(SLOT, NSLOT)

        def host_step(i, sP, sR, staged, packed=None, restored=None):
            """pack step i -> hb[cur] on sP; restore of the buffer packed in step i-1 on sR.
            sP is sR: one stream, back to back.  Otherwise a8: two streams, ordered only by the
            events on the two host buffers (the link is full duplex)."""
            cur, prev = (i % 2, (i - 1) % 2) if len(hb) > 1 else (0, 0)
            tb, te = ranges[i % len(ranges)]
            ra_p.set_ranges(tb, te)
            tb, te = ranges[(i - (1 if len(hb) > 1 else 0)) % len(ranges)]
            ra_r.set_ranges(tb, te)
            p = lk.lumen_kv_plan_build(geom, ra_p, kflag, sP.cuda_stream)
            r = lk.lumen_kv_plan_build(geom, ra_r, kflag | UNIQUE, sR.cuda_stream)
            if packed is not None:
                sP.wait_event(restored[cur])            # the restore that last read this buffer
            if staged:
                lk.lumen_kv_checkpoint_pack_staged(p, kp, vp, hb[cur].data_ptr(), P, ringP.stager,
                                                   sP.cuda_stream)
            else:
                lk.lumen_kv_checkpoint_pack(p, kp, vp, hb[cur].data_ptr(), P, HOST, sP.cuda_stream)
            if packed is not None:
                packed[cur].record(sP)
                sR.wait_event(packed[prev])
            if staged:
                lk.lumen_kv_restore_unpack_staged(r, kp, vp, hb[prev].data_ptr(), P, ringR.stager,
                                                  sR.cuda_stream)
            else:
                lk.lumen_kv_restore_unpack(r, kp, vp, hb[prev].data_ptr(), P, HOST, sR.cuda_stream)
            if packed is not None:
                restored[prev].record(sR)
            p.close(); r.close()

        def host_loop(staged, duplex):
            sA = torch.cuda.Stream()
            sB = torch.cuda.Stream() if duplex else sA
            packed = [torch.cuda.Event() for _ in hb] if duplex else None
            restored = [torch.cuda.Event() for _ in hb] if duplex else None
            for ev in (packed or []) + (restored or []):
                ev.record(sA)
            for i in range(3):
                host_step(i, sA, sB, staged, packed, restored)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier(); torch.cuda.synchronize()
            e0.record(sA)
            sB.wait_event(e0)
            for i in range(3, 3 + Ke):
                host_step(i, sA, sB, staged, packed, restored)
            done_b = torch.cuda.Event(); done_b.record(sB)
            sA.wait_event(done_b)
            e1.record(sA)
            torch.cuda.synchronize(); barrier()
            return max_over_ranks(e0.elapsed_time(e1), dist, "cuda")

        e2e["mapped_one_stream_value"] = e2e["value"]
        ms_s1 = host_loop(True, False)
        e2e["staged_one_stream_value"] = job_payload_gbps(world, Ke, P, ms_s1)
        ms_best, how = ms_s1, "pack then restore back to back on one stream"
        if len(hb) > 1:
            ms_md = host_loop(False, True)
            ms_sd = host_loop(True, True)
            e2e["mapped_duplex_value"] = job_payload_gbps(world, Ke, P, ms_md)
            e2e["staged_duplex_value"] = job_payload_gbps(world, Ke, P, ms_sd)
            ms_best, how = ms_sd, ("pack of step i (D2H) and restore of step i-1's buffer (H2D) on two "
                                   "streams, ordered by events on the two host buffers (a8, full duplex)")
            e2e["duplex_frac_of_d2h_plus_h2d_peak"] = (e2e["staged_duplex_value"] / world /
                                                       (link["d2h"] + link["h2d"]))
            e2e["memcpy_peak_duplex_GBps"] = link["duplex"]
            e2e["duplex_frac_of_duplex_memcpy_peak"] = e2e["staged_duplex_value"] / world / link["duplex"]
        e2e["value"] = job_payload_gbps(world, Ke, P, ms_best)
        e2e["ms_per_step"] = ms_best / Ke
        probe = lk.lumen_kv_plan_build(geom, ra_p, lk.LUMEN_KV_HOST_ONLY)
        n_chunks = len(probe.chunks(SLOT))
        probe.close()
        e2e["gpu_launches"] = 2 * n_chunks * Ke         # one kernel per chunk and direction
        e2e["staging"] = {"slot_bytes": SLOT, "slots": NSLOT, "rings": 2, "chunks_per_call": n_chunks}
        e2e["path"] = ("value = lumen_kv_checkpoint_pack_staged / lumen_kv_restore_unpack_staged with HOST "
                       "buffers: kernel packs chunks into a device staging ring, the copy engine moves them "
                       f"over the link; {how}.  mapped_* = the zero-copy calls (kernel stores/loads on mapped "
                       "pinned host memory); pack_to_host_GBps / restore_from_host_GBps = zero-copy, per launch")
        ringP.close(); ringR.close()
        del hb

    line = {
        "metric": "kv_pack_restore_payload_GBps", "value": value, "unit": "GB/s",
        "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms / K,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u16", "data": "synthetic",
        "runs_per_plan": runs_per_plan,
        "config": {"workload": label, "payload_bytes_per_direction_per_step": P,
                   "tokens_per_step": w.tokens,
                   "l2": l2_config(args.workload),
                   "seed": hex(MASTER_SEED)},
        "l2_note": ("cfg0 fits in L2 (latency config, no roofline claim)" if args.workload == "cfg0" else
                    f"steps rotate over {n_stage} staging buffers of {P / 2**20:.0f} MiB and {len(ranges)} "
                    f"distinct delta sets; the restore reads the buffer packed {lag} steps earlier"),
        "launch_config": {"kernel": args.kernel, "replicas": world,
                          "descriptors": "uploaded" if args.upload_descriptors else "kernel parameters (plans <= 1,024 runs and <= 512 requests; <= 256 / 128 in the small class)",
                          "pdl": os.environ.get("LUMEN_KV_PDL", "1") != "0",
                          "l2_prefetch": int(os.environ.get("LUMEN_KV_PREFETCH", "16"))},
        "tokens_per_s": value * 1e9 / token_bytes,
        "wall_ms_per_step": wall_ms / K, "host_enqueue_ms_per_step": host_ms / K,
        "host_bound": bool(host_bound), "headline_attempts": attempts,
        "step_over_kernels": (ms / K) / (pack_ms + unpack_ms),
        "plan_build_us": plan_build_us,
        "roofline": roofline, "e2e": e2e, "gpu_launches": 2 * K, "clocks": clocks,
    }
    if aligned is not None:
        line["aligned_delta_variant"] = aligned
    if ms_2s is not None:
        line["two_streams"] = {"value": job_payload_gbps(world, K, P, ms_2s), "unit": "GB/s",
                               "ms_per_step": ms_2s / K,
                               "note": "a8 on HBM buffers: pack of step i and restore of the buffer packed 2 steps "
                                       "earlier on two streams, ordered by events on the buffers; same work per "
                                       "step as `value` (which runs both on one stream)"}

    # ---- the large configs the north_star target is worded on, in the same driver-run line ----
    if args.workload == "cfg1" and world == 1 and not args.no_large:
        del path, pool, dbufs
        import gc
        gc.collect()
        torch.cuda.empty_cache()
        if link is None:
            link = memcpy_peaks(torch)
        t_large = time.perf_counter()
        line["large_configs"] = {
            "cfg2": large_config(torch, lk, "cfg2", MASTER_SEED, kflag, stream, sampler, peak, link, True),
            "cfg4_wave0": large_config(torch, lk, "cfg4", MASTER_SEED, kflag, stream, sampler, peak, link, False),
        }
        line["large_configs"]["wall_s"] = time.perf_counter() - t_large
        line["large_configs"]["what"] = (
            "BASELINE.json configs[2] (16 x 8k tokens, Qwen3-32B shape, 32 GiB per direction, pool 20000 pages) "
            "and one wave of configs[4] (2 of the 8 requests x 128k tokens, page_size 1, 64 GiB per direction; "
            "the as-written 256 GiB does not fit one GPU -- all four waves: --workload cfg4), HBM pack + restore; "
            "cfg2 also once through the staged host path (32 GiB each way over the host link)")
    if args.workload == "cfg4" and world == 1:
        # BASELINE.json configs[4] is 8 requests: all four waves of 2, fresh seeds per wave
        del path, pool, dbufs
        import gc
        gc.collect()
        torch.cuda.empty_cache()
        aw = large_config(torch, lk, "cfg4", MASTER_SEED, kflag, stream, sampler, peak, link, False,
                          waves=(0, 1, 2, 3))
        line["all_waves"] = {"requests": 8, "waves": aw["waves"],
                             "payload_GBps": aw["all_waves_payload_GBps"],
                             "payload_bytes_total": 8 * aw["payload_bytes_per_direction"],
                             "note": "4 waves x 2 requests x 128k tokens, page tables and pool content reseeded "
                                     "per wave; payload_GBps = sum of bytes packed + restored / sum of step times",
                             "clocks": aw["clocks"]}
    sampler.close()
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(args.workload, MASTER_SEED)
        line["summary"] = flat_summary(line)            # last on purpose
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    if host_bound and args.workload == "cfg1":
        sys.exit(f"bench.py: the step is HOST-bound (enqueue {host_ms / K:.4f} ms/step > kernels "
                 f"{pack_ms + unpack_ms:.4f} ms/step): the headline does not measure the kernels")


def run_cfg3(args):
    """BASELINE.json configs[3], the recovery burst (a6-a8): every wave of interrupted requests
    is restored from pinned host memory into pages popped from the seeded shuffled free list,
    first alone, then again while a second stream keeps packing 1-token deltas of the 64
    running requests to pinned host memory.  `value` = restored payload GB/s with the
    concurrent packs running, summed over the waves (bytes / device time)."""
    import torch
    import paper_2606_17787_b200 as lk
    from paper_2606_17787_b200.pool import KVPool, pinned_buffer
    from workloads import MASTER_SEED, cfg3_burst
    from workloads import device as wdev

    rank, world, local = rank_env()
    if world != 1:
        raise RuntimeError("--workload cfg3 is a 1-GPU workload")
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    torch.cuda.set_device(local)
    wdev.build()
    b = cfg3_burst(MASTER_SEED)
    L, H, D, S, N = b.geom
    tok_bytes = 2 * L * H * D * 2
    pool = KVPool(L, H, D, S, N)
    for i, t in enumerate(pool.planes()):
        wdev.fill_plane(t, MASTER_SEED, i)
    wave_bytes = [sum(te for _, _, te in w) * tok_bytes for w in b.waves]
    hbuf = wdev.pinned_exact(max(wave_bytes))
    wdev.fill_host_checkpoint(hbuf, max(wave_bytes), MASTER_SEED + 30, 0xC3)
    link = memcpy_peaks(torch)
    n_pb = 8
    pbytes = len(b.running) * tok_bytes
    pbufs = [pinned_buffer(pbytes) for _ in range(n_pb)]
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    geom, kp, vp, HOST = pool.geom, pool.k_ptrs, pool.v_ptrs, lk.LUMEN_KV_MEM_HOST_MAPPED
    ra = lk.ReqArray(b.running)
    te0 = np.array([te for _, _, te in b.running], dtype=np.int64)
    sampler = ClockSampler(local, gpu_uuid(torch, local))

    from paper_2606_17787_b200.pool import StagingRing
    ringR, ringP = StagingRing(32 << 20, 3), StagingRing(32 << 20, 3)
    PACE = 0.025   # s between delta packs: one decode iteration (the paper's mean TPOT is 58 ms)

    call_ms = {"staged_async": [], "mapped": []}

    def delta_pack(it, staged, stream):
        """a1-a4 for one decode step: 1 new token of each of the 64 running requests -> pinned host."""
        ra.set_ranges(te0 + (it % 48), te0 + (it % 48) + 1)
        p = lk.lumen_kv_plan_build(geom, ra, 0, stream.cuda_stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        if staged:
            lk.lumen_kv_checkpoint_pack_staged(p, kp, vp, pbufs[it % n_pb].data_ptr(), pbytes,
                                               ringP.stager, stream.cuda_stream)
        else:
            lk.lumen_kv_checkpoint_pack(p, kp, vp, pbufs[it % n_pb].data_ptr(), pbytes, HOST,
                                        stream.cuda_stream)
        e1.record(stream)
        p.close()
        return e0, e1

    def restore(wave, nbytes, staged, pace):
        """One wave on s1.  pace None: alone; pace > 0: one 1-token delta pack of the running
        requests every `pace` s on s2 meanwhile; pace 0: packs back to back (worst case).
        The staged restore is submitted asynchronously (2,300 chunks: the synchronous call would
        hold this thread for most of the transfer and the packs would only meet its tail)."""
        plan = lk.lumen_kv_plan_build(geom, wave, lk.LUMEN_KV_VALIDATE_UNIQUE_DST, s1.cuda_stream)
        a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record(s1)
        t0 = time.perf_counter()
        if staged:
            ticket = lk.lumen_kv_restore_unpack_staged_async(plan, kp, vp, hbuf.data_ptr(), nbytes,
                                                             ringR.stager, s1.cuda_stream)
            call_ms["staged_async"].append((time.perf_counter() - t0) * 1e3)
            done = lambda: ringR.stager.query(ticket)
        else:
            lk.lumen_kv_restore_unpack(plan, kp, vp, hbuf.data_ptr(), nbytes, HOST, s1.cuda_stream)
            call_ms["mapped"].append((time.perf_counter() - t0) * 1e3)
            z.record(s1)
            done = z.query
        it, pev = 0, []
        next_pack = time.perf_counter()
        while not done():                               # a2-a4 on stream 2 until the restore ends
            now = time.perf_counter()
            if pace is None or now < next_pack:
                time.sleep(0.0005)
                continue
            pev.append(delta_pack(it, staged, s2))
            it += 1
            next_pack = now + pace
            if pace == 0 and it % n_pb == 0:
                s2.synchronize()                        # bound the queue: n_pb packs in flight
        if staged:                                      # at most 0.5 ms after completion
            ringR.stager.wait(ticket, s1.cuda_stream)
            z.record(s1)
        torch.cuda.synchronize()
        plan.close()
        return a.elapsed_time(z), it, [x.elapsed_time(y) for x, y in pev]

    def all_waves(staged, pace):
        res = [restore(w, nb, staged, pace) for w, nb in zip(b.waves, wave_bytes)]
        t = sum(r[0] for r in res)
        packs = sum(r[1] for r in res)
        lat = [x for r in res for x in r[2]]
        return {"restore_GBps": total / t / 1e6, "ms": t, "delta_packs": packs,
                "delta_pack_ms_median": float(np.median(lat)) if lat else None,
                "delta_pack_ms_mean": float(np.mean(lat)) if lat else None,
                "delta_pack_ms_max": float(np.max(lat)) if lat else None,
                "delta_pack_GBps_median": pbytes / float(np.median(lat)) / 1e6 if lat else None}

    def stats(lat, denom):
        med, best = float(np.median(lat)), float(np.min(lat))
        return {"median_ms": med, "best_ms": best, "GBps": pbytes / med / 1e6,
                "frac": pbytes / med / 1e6 / denom}

    def delta_alone(mode, pace, n=24):
        """The decode-step delta with nothing else on the device: one event pair per call, the
        device idle for `pace` s before each (a decode loop issues one per iteration)."""
        dsrc = torch.empty(pbytes, dtype=torch.uint8, device="cuda")
        lat = []
        for it in range(-3, n):
            torch.cuda.synchronize()
            time.sleep(pace)
            if mode == "memcpy":                        # the copy engine alone, same size: the floor
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                with torch.cuda.stream(s2):
                    e0.record(s2); pbufs[it % n_pb].copy_(dsrc, non_blocking=True); e1.record(s2)
            else:
                e0, e1 = delta_pack(it, mode == "staged", s2)
            s2.synchronize()
            if it >= 0:
                lat.append(e0.elapsed_time(e1))
        return lat

    def memcpy_beside_h2d(n=24):
        """A D2H cudaMemcpyAsync of the delta's size while H2D memcpys saturate the other direction:
        what the link gives a 16 MiB transfer when it is busy both ways (the duplex share)."""
        big_h = wdev.pinned_exact(1 << 30)
        big_d = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
        dsrc = torch.empty(pbytes, dtype=torch.uint8, device="cuda")
        lat = []
        with torch.cuda.stream(s1):
            for _ in range(6):
                big_d.copy_(big_h, non_blocking=True)
        for it in range(n):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            with torch.cuda.stream(s2):
                e0.record(s2); pbufs[it % n_pb].copy_(dsrc, non_blocking=True); e1.record(s2)
            s2.synchronize()
            lat.append(e0.elapsed_time(e1))
            time.sleep(0.002)
        torch.cuda.synchronize()
        wdev.unpin(big_h)
        return lat

    total = sum(wave_bytes)
    restore(b.waves[-1], wave_bytes[-1], False, None)   # warm-up
    restore(b.waves[-1], wave_bytes[-1], True, None)
    modes = {"mapped_alone": all_waves(False, None), "staged_alone": all_waves(True, None),
             "mapped_paced_packs": all_waves(False, PACE)}
    sampler.start(slow=True)
    modes["staged_paced_packs"] = all_waves(True, PACE)
    sampler.stop()
    modes["staged_saturating_packs"] = all_waves(True, 0)
    # ---- the decode-step delta by itself ---------------------------
    d2h = link["d2h"]
    floor_busy = memcpy_beside_h2d()
    share = pbytes / float(np.median(floor_busy)) / 1e6     # GB/s a same-size D2H memcpy gets on a busy link
    delta1 = {
        "bytes": pbytes,
        "what": ("lumen_kv_plan_build + pack of 1 new token of each of the 64 running requests (64 x 256 KiB) "
                 "to pinned host, one CUDA-event pair per call; alone = device idle for the pace before each "
                 "call; frac = of the pinned D2H memcpy peak (1 GiB) alone, of the same-size memcpy's rate on "
                 "a link that is saturated in the other direction beside a restore"),
        "alone_paced_25ms": {"zero_copy": stats(delta_alone("mapped", PACE), d2h),
                             "staged": stats(delta_alone("staged", PACE), d2h),
                             "memcpy_same_size": stats(delta_alone("memcpy", PACE), d2h)},
        "alone_paced_2ms": {"zero_copy": stats(delta_alone("mapped", 0.002), d2h),
                            "staged": stats(delta_alone("staged", 0.002), d2h),
                            "memcpy_same_size": stats(delta_alone("memcpy", 0.002), d2h)},
        "duplex_share_GBps": share,
        "memcpy_same_size_beside_h2d_memcpy": stats(floor_busy, share),
        "beside_restore": {
            "zero_copy_beside_zero_copy_restore": {
                "median_ms": modes["mapped_paced_packs"]["delta_pack_ms_median"],
                "GBps": modes["mapped_paced_packs"]["delta_pack_GBps_median"],
                "frac": modes["mapped_paced_packs"]["delta_pack_GBps_median"] / share},
            "staged_beside_staged_restore": {
                "median_ms": modes["staged_paced_packs"]["delta_pack_ms_median"],
                "GBps": modes["staged_paced_packs"]["delta_pack_GBps_median"],
                "frac": modes["staged_paced_packs"]["delta_pack_GBps_median"] / share}},
    }
    head = modes["staged_paced_packs"]
    value = head["restore_GBps"]
    packs = sum(m["delta_packs"] for m in modes.values())
    n_chunks, per_wave_chunks = 0, []
    for w in b.waves:
        probe = lk.lumen_kv_plan_build(geom, w, lk.LUMEN_KV_HOST_ONLY)
        per_wave_chunks.append(len(probe.chunks(32 << 20)))
        n_chunks += per_wave_chunks[-1]
        probe.close()
    # kernels: 1 per delta pack (16 MiB = 1 chunk), 1 per mapped wave, 1 per chunk of a staged wave
    launches = packs + 2 * len(b.waves) + 3 * n_chunks + 2
    line = {
        "metric": "kv_pack_restore_payload_GBps", "value": value, "unit": "GB/s", "n_gpus": 1,
        "steps": len(b.waves), "warmup": 1, "ms_per_step": head["ms"] / len(b.waves),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u16",
        "data": "synthetic",
        "config": {"workload": ("BASELINE.json configs[3]: recovery burst, Qwen3-32B shape, pool "
                                f"{N} pages 40 % occupied by 64 running requests, 48 interrupted prefixes "
                                f"U{{1024..32768}} = {total / 2**30:.1f} GiB restored from pinned host in "
                                f"{len(b.waves)} waves (the as-written single shot needs a 330 GiB pool), "
                                f"concurrent 1-token delta packs (16 MiB) to pinned host on a second stream "
                                f"every {PACE * 1e3:.0f} ms"),
                   "wave_GiB": [x / 2**30 for x in wave_bytes], "seed": hex(MASTER_SEED),
                   "l2": "inputs larger than L2: every wave is tens of GiB read once over the host link"},
        "tokens_per_s": value * 1e9 / tok_bytes,
        "modes": modes, "delta1_to_host": delta1,
        "restore_call_host_ms": {"staged_async_median": float(np.median(call_ms["staged_async"])),
                                 "staged_async_max": float(np.max(call_ms["staged_async"])),
                                 "zero_copy_median": float(np.median(call_ms["mapped"])),
                                 "chunks_per_wave": None},
        "roofline": {"bound": "host_link", "kernel": "lumen_kv_restore_unpack_staged (copy engine H2D + kv_copy_warp)",
                     "achieved": modes["staged_alone"]["restore_GBps"], "peak": link["h2d"], "unit": "GB/s",
                     "frac": modes["staged_alone"]["restore_GBps"] / link["h2d"], "traffic": None,
                     "peak_source": "pinned cudaMemcpyAsync H2D, 1 GiB, best of 10, this run",
                     "frac_with_paced_packs": value / link["h2d"],
                     "mapped_frac": modes["mapped_alone"]["restore_GBps"] / link["h2d"],
                     "memcpy_peak_d2h_GBps": link["d2h"]},
        "e2e": {"value": value, "unit": "GB/s", "h2d_bytes_per_step": total // len(b.waves),
                "d2h_bytes_per_step": head["delta_packs"] * pbytes // len(b.waves),
                "note": "this workload is the host path: the timed region is the H2D restore itself"},
        "gpu_launches": launches, "clocks": sampler.summary(),
    }
    line["restore_call_host_ms"]["chunks_per_wave"] = per_wave_chunks
    sampler.close()
    print(json.dumps(line), flush=True)
    wdev.unpin(hbuf)


def run_chain(args):
    """The rows built after the hot path, measured:
    page tags (f1), checkpoint-store append (f3), restore of the longest checkpointed prefix
    straight out of the store's pinned arena through an explicit-layout plan and the two-stage
    path (f3 + f2), and the controller's decisions (f4).  `value` = that restore's payload GB/s."""
    import torch
    import paper_2606_17787_b200 as lk
    from paper_2606_17787_b200.pool import Checkpointer, KVPool, StagingRing, pinned_buffer
    from workloads import MASTER_SEED, cfg2_qwen32b, substream
    from workloads import device as wdev

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    torch.cuda.set_device(rank_env()[2])
    wdev.build()
    rng = substream(MASTER_SEED, "chain")
    S = 16

    def gpu_ms(fn, reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    # ---- f1: tags of 64 requests x 131,072 tokens (524,288 pages), and of one 8k prompt ----
    off = np.arange(65, dtype=np.int64) * 131072
    tok = torch.randint(0, 151936, (int(off[-1]),), dtype=torch.int32, device="cuda")
    n_pages = lk.lumen_kv_tags_num_pages(off, S)
    d_tags = torch.empty((n_pages, 2), dtype=torch.int64, device="cuda")
    ms_big = gpu_ms(lambda: lk.lumen_kv_page_tags(tok.data_ptr(), off, S, d_tags.data_ptr(), n_pages,
                                                  torch.cuda.current_stream().cuda_stream), 50)
    ms_8k = gpu_ms(lambda: lk.lumen_kv_page_tags(tok.data_ptr(), [0, 8192], S, d_tags.data_ptr(), n_pages,
                                                 torch.cuda.current_stream().cuda_stream), 200)
    tag_bytes = int(off[-1]) * 4 + n_pages * 16
    tags = {"pages": n_pages, "ms": ms_big, "pages_per_s": n_pages / ms_big * 1e3,
            "GBps": tag_bytes / ms_big / 1e6, "one_8k_prompt_us": ms_8k * 1e3,
            "note": "64 B of token IDs per page against 4 MiB of KV: launch-bound at request sizes"}

    # ---- f3: store append (host memcpy into the arena), 2 GiB prefill checkpoint -----------
    w = cfg2_qwen32b(MASTER_SEED, N=20000, n_reqs=4, prompt=8192)
    L, H, D, _, N = w.geom
    tokb = 2 * L * H * D * 2
    n_tok, tail, n_delta = 8192, 16, 12
    first = n_tok - tail * n_delta
    arena = wdev.pinned_exact(4 * (n_tok + 64) * tokb)
    src = torch.empty(first * tokb, dtype=torch.uint8).random_(0, 255)
    no_tags = np.zeros(0, dtype=lk.TAG_DTYPE)
    append = {}
    for threads in (1, 4, 16):
        st = lk.Store(arena.data_ptr(), arena.numel(), tokb, S, copy_threads=threads)
        st.reserve(0, n_tok)
        t0 = time.perf_counter()
        st.append(0, 0, first, src.data_ptr(), src.numel(), no_tags)
        append[f"{threads}_threads_GBps"] = src.numel() / (time.perf_counter() - t0) / 1e9
        st.close()
    del src

    # ---- chain: incremental packs -> store -> lookup -> restore out of the arena ----------------
    pool = KVPool(L, H, D, S, N)
    for i, t in enumerate(pool.planes()):
        wdev.fill_plane(t, MASTER_SEED, i)
    ck = Checkpointer(pool)
    ring, ring2 = StagingRing(32 << 20, 3), StagingRing(32 << 20, 3)
    stage = pinned_buffer(first * tokb)
    st = lk.Store(arena.data_ptr(), arena.numel(), tokb, S, copy_threads=16)
    hist = [rng.integers(0, 151936, size=n_tok + 7).astype(np.int32) for _ in w.reqs]
    h_tags = torch.empty((n_tok // S + 2, 2), dtype=torch.int64, device="cuda")

    def tags_of(tokens):
        d = torch.from_numpy(np.ascontiguousarray(tokens)).cuda()
        n = lk.lumen_kv_tags_num_pages([0, tokens.size], S)
        lk.lumen_kv_page_tags(d.data_ptr(), [0, tokens.size], S, h_tags.data_ptr(), n, 0)
        torch.cuda.synchronize()
        return h_tags[:n].cpu().numpy().copy().view(lk.TAG_DTYPE).reshape(-1)

    t_pack = time.perf_counter()
    for rid, (pt, _, _) in enumerate(w.reqs):
        st.reserve(rid, n_tok + 64)
        cuts = [0, first] + [first + tail * (i + 1) for i in range(n_delta)]
        cuts[-1] -= 3                                          # the last delta ends inside a page
        for tb, te in zip(cuts, cuts[1:]):
            plan = ck.plan([(pt, tb, te)])
            ck.pack_staged(plan, stage, ring)
            torch.cuda.synchronize()
            tg = tags_of(hist[rid][:te])
            st.append(rid, tb, te, stage.data_ptr(), plan.nbytes, tg[(tg["end_pos"] > tb) & (tg["end_pos"] <= te)])
            plan.close()
    t_pack = time.perf_counter() - t_pack
    t_look = time.perf_counter()
    reqs, lays, restored = [], [], 0
    for rid, (pt_new, _, _) in enumerate(w.restore_reqs):
        prefix = st.lookup(rid, tags_of(hist[rid]))
        restored += prefix
        for s_ in st.segments(rid, prefix):
            reqs.append((pt_new, int(s_["t_begin"]), int(s_["t_end"])))
            lays.append((int(s_["buf_offset"]), int(s_["plane_stride_tokens"])))
    t_look = time.perf_counter() - t_look
    link = memcpy_peaks(torch)
    sampler = ClockSampler(rank_env()[2], gpu_uuid(torch, rank_env()[2]))
    stream = torch.cuda.Stream()
    K, W = max(1, min(args.steps, 10)), max(3, min(args.warmup, 5))
    payload = restored * tokb

    def restore_once():
        rplan = lk.lumen_kv_plan_build(pool.geom, reqs, lk.LUMEN_KV_VALIDATE_UNIQUE_DST,
                                       stream.cuda_stream, layouts=lays)
        lk.lumen_kv_restore_unpack_staged(rplan, pool.k_ptrs, pool.v_ptrs, arena.data_ptr(),
                                          arena.numel(), ring2.stager, stream.cuda_stream)
        n = len(rplan.chunks(32 << 20))
        rplan.close()
        return n

    for _ in range(W):
        n_chunks = restore_once()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    sampler.start(slow=True)
    a.record(stream)
    for _ in range(K):
        restore_once()
    b.record(stream)
    torch.cuda.synchronize()
    sampler.stop()
    ms = a.elapsed_time(b) / K
    value = payload / ms / 1e6

    # ---- f4: controller decisions --------------------------------------------------------------
    Wk = 64
    q = rng.random(Wk).tolist()
    held = [[int(x) for x in rng.integers(1, 80, size=int(rng.integers(0, 30)))] for _ in range(Wk)]
    avail = [int(x) for x in rng.integers(0, 160, size=Wk)]
    t0 = time.perf_counter()
    for i in range(2000):
        lk.lumen_kv_choose_holder(q, held, avail, i % Wk, 20, 1.0, 26.0)
    t_choose = (time.perf_counter() - t0) / 2000
    alive = [i % 8 != 0 for i in range(Wk)]
    inter = [(int(rng.integers(0, Wk)), int(rng.integers(0, 32768))) for _ in range(2000)]
    t0 = time.perf_counter()
    lk.lumen_kv_recover([int(x) for x in rng.integers(0, 40, size=Wk)], alive, inter)
    t_recover = time.perf_counter() - t0

    line = {
        "metric": "kv_pack_restore_payload_GBps", "value": value, "unit": "GB/s", "n_gpus": 1,
        "steps": K, "warmup": W, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u16", "data": "synthetic",
        "config": {"workload": ("checkpoint chain (SURVEY.md 8(f)): Qwen3-32B shape, 4 requests x 8,192 tokens "
                                "checkpointed as a prefill delta + 12 decode deltas of 16 tokens into a pinned "
                                "store arena; restore of the longest checkpointed prefix (page aligned, ends "
                                "inside the last delta) out of the arena via lumen_kv_plan_build_layout + "
                                "lumen_kv_restore_unpack_staged"),
                   "restored_tokens": restored, "segments": len(reqs), "chunks": n_chunks,
                   "l2": "inputs larger than L2: 8 GiB read over the host link per step"},
        "tokens_per_s": value * 1e9 / tokb,
        "roofline": {"bound": "host_link", "kernel": "lumen_kv_restore_unpack_staged (copy engine H2D + kv_copy_warp)",
                     "achieved": value, "peak": link["h2d"], "unit": "GB/s", "frac": value / link["h2d"],
                     "traffic": None, "peak_source": "pinned cudaMemcpyAsync H2D, 1 GiB, best of 10, this run"},
        "e2e": {"value": value, "unit": "GB/s", "h2d_bytes_per_step": payload, "d2h_bytes_per_step": 0,
                "note": "the timed region is the H2D restore out of the pinned arena"},
        "page_tags": tags, "store_append": append,
        "checkpointing": {"s_total": t_pack, "deltas": 13 * len(w.reqs),
                          "note": "staged pack -> pinned staging -> store.append, incl. tags, synchronous per delta"},
        "lookup_s": t_look,
        "controller": {"choose_holder_us": t_choose * 1e6, "workers": Wk,
                       "recover_2000_interrupted_ms": t_recover * 1e3,
                       "note": "through the ctypes binding (marshalling included)"},
        "gpu_launches": K * n_chunks, "clocks": sampler.summary(),
    }
    sampler.close()
    print(json.dumps(line), flush=True)
    wdev.unpin(arena)


def run_interference(args):
    """checkpointing must stay off the GPU critical path.  A 2 GiB pack to
    pinned host memory (Qwen3-32B shape, 4 x 2,048-token prefixes) runs on one stream while a
    second stream loops an HBM-bound 2 GiB device copy (standing in for the forward pass);
    reported: the copy's slowdown and the pack's GB/s for every host-path variant."""
    import torch
    import paper_2606_17787_b200 as lk
    from paper_2606_17787_b200.pool import Checkpointer, KVPool, StagingRing, pinned_buffer
    from workloads import MASTER_SEED, cfg2_qwen32b
    from workloads import device as wdev

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    torch.cuda.set_device(rank_env()[2])
    wdev.build()
    w = cfg2_qwen32b(MASTER_SEED, N=4000, n_reqs=4, prompt=2048)
    L, H, D, S, N = w.geom
    pool = KVPool(L, H, D, S, N)
    for i, t in enumerate(pool.planes()):
        wdev.fill_plane(t, MASTER_SEED, i)
    P = w.payload_bytes
    host = pinned_buffer(P)
    ring = StagingRing(32 << 20, 3)
    a_, b_ = (torch.empty(2 << 30, dtype=torch.uint8, device="cuda") for _ in range(2))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

    def ev():
        return torch.cuda.Event(enable_timing=True)

    def copies(n):
        x, y = ev(), ev()
        with torch.cuda.stream(s2):
            x.record(s2)
            for _ in range(n):
                b_.copy_(a_)
            y.record(s2)
        return x, y

    torch.cuda.synchronize()
    x, y = copies(16)
    torch.cuda.synchronize()
    alone = x.elapsed_time(y) / 16
    variants = {
        "staged (kernel -> HBM ring -> copy engine)": ("staged", lk.LUMEN_KV_KERNEL_AUTO),
        "zero-copy, TMA bulk kernel, 24 CTAs (AUTO)": ("mapped", lk.LUMEN_KV_KERNEL_AUTO),
        "zero-copy, SIMT kernel, full grid": ("mapped", lk.LUMEN_KV_KERNEL_WARP),
    }
    out = {}
    for name, (mode, kflag) in variants.items():
        ck = Checkpointer(pool, kflag)
        plan = ck.plan(w.reqs)

        def pack():
            with torch.cuda.stream(s1):
                if mode == "staged":
                    ck.pack_staged(plan, host, ring)
                else:
                    ck.pack(plan, host)

        rplan = ck.plan(w.restore_reqs, unique_dst=True)

        def restore():
            with torch.cuda.stream(s1):
                if mode == "staged":
                    ck.unpack_staged(rplan, host, ring)
                else:
                    ck.unpack(rplan, host)

        res = {}
        for what, fn in (("pack", pack), ("restore", restore)):
            fn(); torch.cuda.synchronize()
            p0, p1 = ev(), ev()
            p0.record(s1); fn(); p1.record(s1)
            torch.cuda.synchronize()
            gbps_alone = P / p0.elapsed_time(p1) / 1e6
            n = int(P / 50e9 * 1e3 / alone) + 8                # copies outlast the transfer
            x, y = copies(n)
            p0.record(s1); fn(); p1.record(s1)
            torch.cuda.synchronize()
            res.update({f"{what}_GBps_alone": gbps_alone,
                        f"{what}_GBps_beside_copy": P / p0.elapsed_time(p1) / 1e6,
                        f"hbm_copy_slowdown_during_{what}": x.elapsed_time(y) / n / alone})
        res["hbm_copy_slowdown"] = res["hbm_copy_slowdown_during_pack"]
        out[name] = res
        rplan.close()
        plan.close()
    best = out["staged (kernel -> HBM ring -> copy engine)"]
    link = memcpy_peaks(torch)
    line = {"metric": "kv_pack_restore_payload_GBps", "value": best["pack_GBps_beside_copy"], "unit": "GB/s",
            "n_gpus": 1, "steps": 1, "warmup": 1, "ms_per_step": P / best["pack_GBps_beside_copy"] / 1e6,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u16", "data": "synthetic",
            "config": {"workload": ("interference: 2 GiB pack to pinned host (Qwen3-32B shape, 4 x 2,048 tokens) "
                                    "beside a looping 2 GiB HBM copy on another stream"),
                       "l2": "inputs larger than L2 (2 GiB per pass on both streams)"},
            "hbm_copy_alone_ms": alone, "hbm_copy_alone_GBps": 2 * (2 << 30) / alone / 1e6,
            "variants": out,
            "roofline": {"bound": "host_link", "kernel": "lumen_kv_checkpoint_pack_staged", "unit": "GB/s",
                         "achieved": best["pack_GBps_beside_copy"], "peak": link["d2h"],
                         "frac": best["pack_GBps_beside_copy"] / link["d2h"], "traffic": None,
                         "peak_source": "pinned cudaMemcpyAsync D2H, 1 GiB, best of 10, this run"},
            "e2e": {"value": best["pack_GBps_beside_copy"], "unit": "GB/s", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": P},
            # 3 packs per variant: 64 chunk kernels each when staged, 1 kernel each when zero-copy
            "gpu_launches": 3 * 64 + 3 + 3}
    print(json.dumps(line), flush=True)


def run_overhead(args):
    """PAPER.md:239 (Exp. A.1): always-on checkpointing shows no measurable steady-state overhead
    (TTFT identical, TPOT within 0.1 ms).  The same question for this implementation on B200:
    a decode-like loop (an HBM-bound 2 GiB copy repeated for about 13 ms stands in for one decode
    iteration of 64 requests, Qwen3-14B shape) runs with and without the background
    checkpointer (lumen_kv_ckpt_*) packing every iteration's new tokens into a checkpoint store."""
    import torch
    import paper_2606_17787_b200 as lk
    from paper_2606_17787_b200.pool import KVPool, pinned_buffer
    from workloads import MASTER_SEED, cfg1_qwen14b
    from workloads import device as wdev

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    torch.cuda.set_device(rank_env()[2])
    wdev.build()
    iters = 100
    w = cfg1_qwen14b(MASTER_SEED, N=60000, grow_iters=iters + 8)
    L, H, D, S, N = w.geom
    tokb = 2 * L * H * D * 2
    pool = KVPool(L, H, D, S, N)
    for i, t in enumerate(pool.planes()):
        wdev.fill_plane(t, MASTER_SEED, i)
    a_, b_ = (torch.empty(2 << 30, dtype=torch.uint8, device="cuda") for _ in range(2))
    compute = torch.cuda.Stream()
    ring = torch.empty(3 * (32 << 20), dtype=torch.uint8, device="cuda")
    pinned = pinned_buffer(1 << 30)
    lens = [te for _, _, te in w.reqs]
    ids = list(range(len(lens)))
    from paper_2606_17787_b200.pool import StagingRing
    rng = np.random.default_rng(MASTER_SEED)
    hist = [rng.integers(0, 151936, size=n + iters * 16).astype(np.int32) for n in lens]   # token IDs

    # the GPU side of the pipeline alone: prefill-completion checkpoint of all prompts into a sink
    # that drops the bytes (pack -> staging ring -> copy engine -> pinned halves -> nothing)
    bg0 = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring.data_ptr(), 32 << 20, 3,
                                    pinned.data_ptr(), pinned.numel(), lambda *a: None)
    for rid in ids:
        bg0.track(rid, 0)
    t0 = time.perf_counter()
    bg0.notify(ids, [(pt, 0, n) for (pt, _, n) in w.reqs])
    bg0.flush()
    dt0 = time.perf_counter() - t0
    bg0.close()
    drop_sink = {"GiB": sum(lens) * tokb / 2**30, "s": dt0, "GBps": sum(lens) * tokb / dt0 / 1e9}

    def loop(delta_tokens, with_ckpt):
        arena = st = bg = None
        prefill = None
        if with_ckpt:
            total_tok = sum(n + iters * delta_tokens for n in lens)
            arena = wdev.pinned_exact(total_tok * tokb)
            st = lk.Store(arena.data_ptr(), arena.numel(), tokb, S, copy_threads=16)
            # native sink: the checkpointer's thread appends straight into the store (no Python)
            bg = lk.BackgroundCheckpointer(pool.geom, pool.k_ptrs, pool.v_ptrs, ring.data_ptr(), 32 << 20,
                                           3, pinned.data_ptr(), pinned.numel(), st)
            for rid, n in enumerate(lens):
                st.reserve(rid, n + iters * delta_tokens)
                bg.track(rid, 0)
            t0 = time.perf_counter()                         # prefill-completion checkpoint, untimed part
            bg.notify(ids, [(pt, 0, n) for (pt, _, n) in w.reqs], token_ids=hist)
            bg.flush()
            dt = time.perf_counter() - t0
            prefill = {"GiB": sum(lens) * tokb / 2**30, "s": dt, "GBps": sum(lens) * tokb / dt / 1e9}
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        evs = []
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        with torch.cuda.stream(compute):
            e0.record(compute)
            for it in range(iters):
                for _ in range(20):                          # one "decode iteration": ~13 ms of HBM traffic
                    b_.copy_(a_)
                ev = torch.cuda.Event()
                ev.record(compute)
                evs.append(ev)
                if bg is not None:
                    bg.notify(ids, [(pt, 0, n + (it + 1) * delta_tokens) for (pt, _, n) in w.reqs],
                              ev.cuda_event, token_ids=hist)
            e1.record(compute)
        compute.synchronize()
        t_loop = time.perf_counter() - t0
        out = {"iteration_ms": e0.elapsed_time(e1) / iters, "host_loop_ms_per_iteration": t_loop / iters * 1e3}
        if bg is not None:
            t1 = time.perf_counter()
            bg.flush()
            out["flush_lag_ms"] = (time.perf_counter() - t1) * 1e3
            assert all(bg.progress(r) == n + iters * delta_tokens for r, n in enumerate(lens))
            assert st.sink_errors == 0 and all(st.tokens(r) == n + iters * delta_tokens for r, n in enumerate(lens))
            out["checkpointed_MiB_per_iteration"] = len(lens) * delta_tokens * tokb / 2**20
            out["prefill_checkpoint"] = prefill
            # the worker "fails": every request is recovered on the holder, one call each
            # (tags from the token history -> prefix -> layout plan -> staged restore into fresh pages)
            rs = torch.cuda.Stream()
            ringr = StagingRing(32 << 20, 3)
            r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            r0.record(rs)
            restored = 0
            for rid, (pt_new, _, n) in enumerate(w.restore_reqs):
                restored += st.restore(rid, hist[rid][: n + iters * delta_tokens], pool.geom, pt_new,
                                       pool.k_ptrs, pool.v_ptrs, ringr.stager, rs.cuda_stream)
            r1.record(rs)
            rs.synchronize()
            assert restored == sum(n + iters * delta_tokens for n in lens)   # history == what was checkpointed
            out["recovery"] = {"requests": len(lens), "tokens": restored, "GiB": restored * tokb / 2**30,
                               "device_ms": r0.elapsed_time(r1), "host_s": time.perf_counter() - t1,
                               "GBps": restored * tokb / r0.elapsed_time(r1) / 1e6}
            ringr.close()
            bg.close()
            st.close()
            wdev.unpin(arena)
        return out

    loop(1, False)                                           # warm-up
    base = loop(1, False)
    res = {"no_checkpointing": base}
    for dt in (1, 16):
        r = loop(dt, True)
        r["overhead_pct"] = (r["iteration_ms"] / base["iteration_ms"] - 1.0) * 100.0
        r["overhead_ms_per_iteration"] = r["iteration_ms"] - base["iteration_ms"]
        res[f"checkpointing_{dt}_token_per_request"] = r
    head = res["checkpointing_1_token_per_request"]
    P = head["checkpointed_MiB_per_iteration"] * 2**20
    value = P / (head["iteration_ms"] * 1e-3) / 1e9
    line = {"metric": "kv_pack_restore_payload_GBps", "value": value, "unit": "GB/s", "n_gpus": 1,
            "steps": iters, "warmup": 1, "ms_per_step": head["iteration_ms"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u16", "data": "synthetic",
            "config": {"workload": ("steady-state overhead of always-on checkpointing: 64 requests, Qwen3-14B "
                                    "shape, a 13 ms HBM-bound stand-in for each decode iteration, background "
                                    "checkpointer packing 1 (and 16) new tokens per request per iteration into "
                                    "a pinned checkpoint store"),
                       "l2": "inputs larger than L2 (2 GiB copies; deltas from a 146.5 GiB pool)"},
            "overhead": res, "prefill_checkpoint_into_a_sink_that_drops_the_bytes": drop_sink,
            "roofline": {"bound": "host_link", "kernel": "lumen_kv_ckpt (background, rate set by the decode loop)",
                         "achieved": value, "peak": None, "unit": "GB/s", "frac": None, "traffic": None},
            "e2e": {"value": value, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": int(P)},
            "gpu_launches": 2 * iters}
    print(json.dumps(line), flush=True)


def run_hostlink(args):
    """What bounds the ZERO-COPY host path (lumen_kv_checkpoint_pack / lumen_kv_restore_unpack with
    LUMEN_KV_MEM_HOST_MAPPED: SM stores / loads on pinned host memory)?  A 2 GiB pack to pinned host
    and its restore, for 32 KiB and for 2 KiB items, with the TMA bulk kernel at 8 / 24 / 96 / 296
    CTAs and the SIMT kernel (32-byte and 16-byte accesses, full grid), against the pinned
    cudaMemcpyAsync peaks of the same run.  One kernel per (variant, direction, repetition), in the
    order of `launch_order`, so that an ncu launch list of this command (pcie__read_bytes,
    pcie__write_bytes per launch) joins with it by index."""
    import torch
    import paper_2606_17787_b200 as lk
    from paper_2606_17787_b200.pool import KVPool, pinned_buffer
    from workloads import MASTER_SEED, cfg2_qwen32b, cfg4_longctx
    from workloads import device as wdev

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    torch.cuda.set_device(rank_env()[2])
    wdev.build()
    lk.lumen_kv_init()
    link = memcpy_peaks(torch)
    HOST = lk.LUMEN_KV_MEM_HOST_MAPPED
    s = torch.cuda.Stream()
    shapes = {"32KiB_items": cfg2_qwen32b(MASTER_SEED, N=3000, n_reqs=4, prompt=2048),
              "2KiB_items": cfg4_longctx(MASTER_SEED, tokens=8192, wave_reqs=1)}
    variants = [("bulk", n, 1) for n in (8, 24, 96, 296)] + [("warp", 0, 1), ("warp", 0, 0)]
    out, order = {}, []
    for sname, w in shapes.items():
        L, H, D, S, N = w.geom
        pool = KVPool(L, H, D, S, N)
        fill_pool(pool, MASTER_SEED, wdev)
        P = w.payload_bytes
        host = pinned_buffer(P)
        res = {}
        for kern, ctas, wide in variants:
            lk.lumen_kv_set_option("host_ctas", ctas)
            lk.lumen_kv_set_option("wide", wide)
            flag = lk.LUMEN_KV_KERNEL_BULK if kern == "bulk" else lk.LUMEN_KV_KERNEL_WARP
            name = f"bulk_{ctas}_ctas" if kern == "bulk" else ("simt_32B_full_grid" if wide else "simt_16B_full_grid")
            plan = lk.lumen_kv_plan_build(pool.geom, w.reqs, flag, s.cuda_stream)
            rplan = lk.lumen_kv_plan_build(pool.geom, w.restore_reqs, flag | lk.LUMEN_KV_VALIDATE_UNIQUE_DST,
                                           s.cuda_stream)
            t = {}
            for what, fn, pl in (("pack", lk.lumen_kv_checkpoint_pack, plan),
                                 ("restore", lk.lumen_kv_restore_unpack, rplan)):
                best = float("inf")
                for rep in range(3):
                    a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record(s)
                    fn(pl, pool.k_ptrs, pool.v_ptrs, host.data_ptr(), P, HOST, s.cuda_stream)
                    z.record(s)
                    s.synchronize()
                    order.append(f"{sname}/{name}/{what}/{rep}")
                    if rep:
                        best = min(best, a.elapsed_time(z))
                peak = link["d2h"] if what == "pack" else link["h2d"]
                t[what] = {"GBps": P / best / 1e6, "frac_of_memcpy": P / best / 1e6 / peak}
            res[name] = t
            plan.close(); rplan.close()
        out[sname] = res
        del pool, host
        torch.cuda.empty_cache()
    lk.lumen_kv_set_option("host_ctas", 0)
    lk.lumen_kv_set_option("wide", 1)
    best = out["32KiB_items"]["bulk_24_ctas"]
    line = {"metric": "kv_pack_restore_payload_GBps", "value": best["pack"]["GBps"], "unit": "GB/s", "n_gpus": 1,
            "steps": 2, "warmup": 1, "ms_per_step": (2 << 30) / best["pack"]["GBps"] / 1e6,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u16", "data": "synthetic",
            "config": {"workload": ("hostlink: zero-copy pack of 2 GiB to pinned host and restore from it, Qwen3-32B "
                                    "shape, 32 KiB items (page_size 16) and 2 KiB items (page_size 1), kernel and grid sweep"),
                       "l2": "inputs larger than L2 (2 GiB per launch)"},
            "variants": out, "launch_order": order,
            "memcpy_peak_d2h_GBps": link["d2h"], "memcpy_peak_h2d_GBps": link["h2d"],
            "roofline": {"bound": "host_link", "kernel": "lumen_kv_checkpoint_pack (kv_copy_bulk, 24 CTAs, zero-copy)",
                         "achieved": best["pack"]["GBps"], "peak": link["d2h"], "unit": "GB/s",
                         "frac": best["pack"]["frac_of_memcpy"], "traffic": None,
                         "peak_source": "pinned cudaMemcpyAsync D2H, 1 GiB, best of 10, this run"},
            "e2e": {"value": best["pack"]["GBps"], "unit": "GB/s", "h2d_bytes_per_step": 2 << 30,
                    "d2h_bytes_per_step": 2 << 30},
            "gpu_launches": len(order)}
    print(json.dumps(line), flush=True)


def run_dram(args):
    """Is the HBM path at the DRAM's ceiling or at the kernel's?  Plain streaming kernels with the
    library kernel's access shape (workloads/csrc/dramprobe.cu: read-only, write-only, contiguous
    copy), torch's copy_ and a device-to-device cudaMemcpyAsync over 16 GiB buffers, next to the
    pack and the restore of BASELINE.json configs[2]; all CUDA-event timed, 3 warm-up + 5 timed
    launches each.  `of_pin_rate` = against dram__bytes.sum.peak_sustained x the memory clock that
    ncu reports for this part (2,048 B/cycle x 3.996 GHz = 8,184 GB/s)."""
    import torch
    import paper_2606_17787_b200 as lk
    from paper_2606_17787_b200.pool import KVPool
    from workloads import MASTER_SEED
    from workloads import device as wdev

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU path for --impl ours")
    local = rank_env()[2]
    torch.cuda.set_device(local)
    wdev.build()
    lk.lumen_kv_init()
    peak, peak_src = measured_peaks()
    PIN = 2048 * 3.996                                   # GB/s
    s = torch.cuda.Stream()
    sampler = ClockSampler(local, gpu_uuid(torch, local))
    NB = 16 << 30
    a_ = torch.empty(NB, dtype=torch.uint8, device="cuda")
    b_ = torch.empty(NB, dtype=torch.uint8, device="cuda")
    wdev.fill_plane(a_, MASTER_SEED, 0)
    order = []

    def timed(name, fn, traffic, reps=5):
        with torch.cuda.stream(s):
            for _ in range(3):
                fn()
            x, y = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            sampler.start()
            x.record(s)
            for _ in range(reps):
                fn()
            y.record(s)
            sampler.poll()
            s.synchronize()
            sampler.stop()
        ms = x.elapsed_time(y) / reps
        order.extend([name] * (3 + reps))
        g = traffic / ms / 1e6
        return {"ms": ms, "traffic_GBps": g, "of_measured_copy_peak": g / peak, "of_pin_rate": g / PIN}

    res = {
        "probe_read_only": timed("probe_read", lambda: wdev.dram_probe("read", a_, b_, NB, s.cuda_stream), NB),
        "probe_write_only": timed("probe_write", lambda: wdev.dram_probe("write", a_, b_, NB, s.cuda_stream), NB),
        "probe_copy": timed("probe_copy", lambda: wdev.dram_probe("copy", a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_l2_prefetch_4k": timed("probe_copy_pf4k", lambda: wdev.dram_probe("copy_pf4k", a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_l2_prefetch_32k": timed("probe_copy_pf32k", lambda: wdev.dram_probe("copy_pf32k", a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_5_ctas_per_sm": timed("probe_copy_5cta", lambda: wdev.dram_probe("copy_5cta", a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_4_ctas_per_sm": timed("probe_copy_4cta", lambda: wdev.dram_probe("copy_4cta", a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_smem_carveout_7pct_dyn_4KiB": timed("probe_copy_carve_804", lambda: wdev.dram_probe(804, a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_smem_carveout_7pct_dyn_6KiB": timed("probe_copy_carve_806", lambda: wdev.dram_probe(806, a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_persistent": timed("probe_copy_persistent", lambda: wdev.dram_probe("copy_persistent", a_, b_, NB, s.cuda_stream), 2 * NB),
        "probe_copy_persistent_l2_prefetch": timed("probe_copy_persistent_pf", lambda: wdev.dram_probe("copy_persistent_pf", a_, b_, NB, s.cuda_stream), 2 * NB),
        "torch_copy_": timed("torch_copy", lambda: b_.copy_(a_), 2 * NB),
    }
    del a_, b_
    torch.cuda.empty_cache()
    w, label, _ = make_workload("cfg2", MASTER_SEED)
    L, H, D, S, N = w.geom
    pool = KVPool(L, H, D, S, N)
    fill_pool(pool, MASTER_SEED, wdev)
    dbuf = torch.empty(w.payload_bytes, dtype=torch.uint8, device="cuda")
    path = HbmPath(torch, lk, pool, w, 0, lk.LUMEN_KV_KERNEL_AUTO, s, None)
    res["lumen_kv_checkpoint_pack_cfg2"] = timed(
        "pack", lambda: path.step(0, [dbuf], lk.LUMEN_KV_MEM_DEVICE, 0, None, "pack"), 2 * path.P)
    res["lumen_kv_restore_unpack_cfg2"] = timed(
        "unpack", lambda: path.step(0, [dbuf], lk.LUMEN_KV_MEM_DEVICE, 0, None, "unpack"), 2 * path.P)
    head = res["lumen_kv_checkpoint_pack_cfg2"]
    line = {"metric": "kv_pack_restore_payload_GBps", "value": head["traffic_GBps"] / 2, "unit": "GB/s", "n_gpus": 1,
            "steps": 5, "warmup": 3, "ms_per_step": head["ms"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u16", "data": "synthetic",
            "config": {"workload": "dram: streaming read / write / copy probes (16 GiB) beside the pack and restore of "
                                   + label, "l2": "inputs larger than L2 (16-32 GiB per launch)"},
            "kernels": res, "launch_order": order, "pin_rate_GBps": PIN,
            "roofline": {"bound": "hbm", "kernel": "lumen_kv_checkpoint_pack (kv_copy_warp32)",
                         "achieved": head["traffic_GBps"], "peak": peak, "unit": "GB/s",
                         "frac": head["traffic_GBps"] / peak, "traffic": None, "peak_source": peak_src},
            "e2e": None, "gpu_launches": len(order), "clocks": sampler.summary()}
    sampler.close()
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "cfg3":
        run_cfg3(args)
    elif args.workload == "chain":
        run_chain(args)
    elif args.workload == "interference":
        run_interference(args)
    elif args.workload == "overhead":
        run_overhead(args)
    elif args.workload == "hostlink":
        run_hostlink(args)
    elif args.workload == "dram":
        run_dram(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
