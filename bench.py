#!/usr/bin/env python
"""bench.py -- SparseStack zeta=4 sketch formation on B200: GB/s of A read and fraction of the roofline.

One "step" = one complete FP16-accumulate sketch (zero-init + hash + stream A + sign/scale + RN16 +
scatter-accumulate + flush, "complete sketch") of the workload's
resident m x n FP32 matrix through the C ABI.  Default workload: BASELINE.json configs[4]'s peak
point (m = 2^25, n = 128, d = 256, zeta = 4; A = 16 GiB > L2, so no flush is needed between steps).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2|c3|c4|c5] [--variant auto|...]
    python bench.py --impl reference ...        # the CPU oracle, as it stands, on the host cores

N > 1 (torchrun): every rank sketches its own m-row shard (global row indices rank*m ...) of an
(N*m) x n matrix into a private sketch -- no data-path collective inside the scatter -- and the N
partial sketches (64 KiB each) are summed with one NCCL all-reduce.  Weak scaling.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOADS = {
    # name: (m, n, d, zeta, matrix_seed)   BASELINE.json configs[1..4]
    "c1": (4096, 16, 32, 4, 0),
    "c2": (1 << 20, 64, 128, 4, 1),
    "c3": (1 << 22, 128, 256, 4, 2),
    "c4": (1 << 23, 256, 1024, 4, 3),
    "c4-512": (1 << 23, 256, 512, 4, 3),
    "c4-2048": (1 << 23, 256, 2048, 4, 3),
    "c3-z1": (1 << 22, 128, 256, 1, 2),
    "c3-z2": (1 << 22, 128, 256, 2, 2),
    "c3-z8": (1 << 22, 128, 256, 8, 2),
    "c5": (1 << 25, 128, 256, 4, 4),
    # the paper's own headline point (Fig. 2): m = 2^21, n = 1024, d = 2n, zeta = 4, dense input;
    # BASELINE.md holds its H200 number for exactly this workload (7.11 ms complete sketch = 1208 GB/s of A)
    "e1": (1 << 21, 1024, 2048, 4, 5),
    # widths that are not 64 * 2^k (three column slices of the tensor-memory kernel)
    "w192": (1 << 22, 192, 384, 4, 6),
    "w384": (1 << 22, 384, 768, 4, 6),
    # the paper's width with sketches that still fit tensor memory (d < 2n: not a paper point)
    "n1024-d512": (1 << 21, 1024, 512, 4, 6),
    "n1024-d1024": (1 << 21, 1024, 1024, 4, 6),
    "w320": (1 << 22, 320, 640, 4, 6),
    "e1-d4096": (1 << 21, 1024, 4096, 4, 5),    # d/n = 4 of the paper's grid: 8 MiB sketch, beyond tensor memory
}
PAPER_GBPS = {"e1": (1 << 21) * 1024 * 4 / 7.11e-3 / 1e9}   # PAPER.md:322, H200 NVL (another machine: context)
L2_RED_PAYLOAD_GBPS_R01 = 6000.0   # round-1 probe (profiles/r01_red_probe.md): context only; the bench measures its own
VARIANTS = {"auto": 0, "flat_pair": 1, "flat_vec": 2, "smem": 3, "generic": 4, "tmem": 5, "small": 6}

def ncu_traffic(workload, variant):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, FROM THE COMMITTED `ncu --set full`
    CAPTURES (profiles/ncu_traffic.json: one entry per (workload, variant) with the kernel name and the profile file that
    holds the capture and its command); None where nothing was captured.  Not a measurement of this run."""
    try:
        table = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
    except (OSError, ValueError):
        return None, None
    e = table.get("%s/%s" % (workload, variant))
    return (int(e["dram_bytes_read"]) + int(e["dram_bytes_written"]), e) if e else (None, None)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM / memory clocks, board power and throttle reasons DURING the timed region (profiling recipe's clocks line), sampled
    through NVML every ~5 ms in a thread of this process (an `nvidia-smi -lms 100` child process where NVML cannot be
    loaded), so that every timed step gets the sample nearest to it and a change of regime inside a 50 ms region is visible."""

    REASONS = ((0x8, "hw_slowdown"), (0x40, "hw_thermal_slowdown"), (0x20, "sw_thermal_slowdown"), (0x4, "sw_power_cap"),
               (0x80, "hw_power_brake_slowdown"))
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,clocks.mem")

    def __init__(self, index: int, uuid: str | None = None, period_s: float = 0.005):
        self.index, self.uuid, self.period = index, uuid, period_s
        self.rows = []            # (wall time, sm MHz, mem MHz, power W, [reasons])
        self.sm_max, self.proc, self.th, self.stopflag, self.source = None, None, None, False, None

    def start(self):
        try:
            import pynvml

            pynvml.nvmlInit()
            try:
                h = pynvml.nvmlDeviceGetHandleByUUID(self.uuid if isinstance(self.uuid, bytes) else str(self.uuid).encode()) if self.uuid else None
            except Exception:
                h = None
            if h is None:
                h = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            reasons_fn = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or pynvml.nvmlDeviceGetCurrentClocksThrottleReasons

            def pump():
                while not self.stopflag:
                    try:
                        t = time.time()
                        sm = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_SM))
                        mem = float(pynvml.nvmlDeviceGetClockInfo(h, pynvml.NVML_CLOCK_MEM))
                        pw = pynvml.nvmlDeviceGetPowerUsage(h) / 1e3
                        bits = int(reasons_fn(h))
                        self.rows.append((t, sm, mem, pw, [name for bit, name in self.REASONS if bits & bit]))
                    except Exception:
                        pass
                    time.sleep(self.period)

            self.source = "nvml, %.0f ms period" % (self.period * 1e3)
            self.th = threading.Thread(target=pump, daemon=True)
            self.th.start()
            return
        except Exception:
            self.th = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi -lms 100"
            self.th = threading.Thread(target=self._pump_smi, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _pump_smi(self):
        for ln in self.proc.stdout:
            f = [x.strip() for x in ln.split(",")]
            try:
                sm, mx, pw, mem = float(f[1]), float(f[2]), float(f[3]), float(f[9])
            except (ValueError, IndexError):
                continue
            self.sm_max = mx
            names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
            self.rows.append((time.time(), sm, mem, pw, [nm for nm, val in zip(names, f[5:9]) if val.lower().startswith("active")]))

    def halt(self):
        time.sleep(0.02 if self.proc is None else 0.15)
        self.stopflag = True
        if self.proc:
            self.proc.terminate()

    def nearest(self, t: float):
        if not self.rows:
            return None
        r = min(self.rows, key=lambda row: abs(row[0] - t))
        return {"sm_mhz": r[1], "mem_mhz": r[2], "power_w": round(r[3], 1), "reasons": r[4], "dt_ms": round((r[0] - t) * 1e3, 1)}

    def summary(self, t0: float, t1: float):
        """Medians and the union of the reasons over the samples in [t0, t1] (the nearest ones when the window holds none)."""
        if self.th is None and self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no NVML and no nvidia-smi"]}
        rows = [r for r in self.rows if t0 <= r[0] <= t1]
        if not rows:
            rows = sorted(self.rows, key=lambda r: abs(r[0] - 0.5 * (t0 + t1)))[:3]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": ["no samples"], "samples": 0}

        def med(k):
            v = sorted(r[k] for r in rows)
            return v[len(v) // 2]

        return {"sm_mhz": med(1), "sm_max_mhz": self.sm_max, "reasons": sorted({x for r in rows for x in r[4]}), "samples": len(rows),
                "sm_mhz_min": min(r[1] for r in rows), "mem_mhz": med(2), "mem_mhz_min": min(r[2] for r in rows),
                "power_w": round(med(3), 1), "power_w_max": round(max(r[3] for r in rows), 1), "source": self.source}


def step_stats(ms):
    """mean / median / min / p90 of the per-step times and whether they fall into two regimes: the sorted series is cut at
    its largest relative gap; a gap above 4 % with at least two steps (and 10 % of them) on either side is flagged."""
    v = sorted(ms)
    k = len(v)
    out = {"mean": sum(v) / k, "median": v[k // 2] if k % 2 else 0.5 * (v[k // 2 - 1] + v[k // 2]), "min": v[0], "max": v[-1],
           "p90": v[min(k - 1, int(0.9 * k))], "bimodal": False}
    if k >= 4:
        gap, cut = max(((v[i + 1] / v[i] - 1.0, i + 1) for i in range(k - 1)), key=lambda g: g[0])
        need = max(2, k // 10)
        if gap > 0.04 and cut >= need and k - cut >= need:
            lo, hi = v[:cut], v[cut:]
            out.update(bimodal=True, regimes={"fast_ms": sum(lo) / len(lo), "fast_steps": len(lo), "slow_ms": sum(hi) / len(hi),
                                              "slow_steps": len(hi), "gap": gap})
    return out


def algorithmic_bytes(m, n, d, out_elem=2):
    """per input element 4 B read once; output b*d*n written once (Eq. 5's 4mn term + the sketch)."""
    return 4 * m * n + out_elem * d * n


# ------------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    """The oracle as it stands (never tuned), on the host cores, on a bounded sample of the workload."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    import numpy as np

    import oracle
    import workloads as wl

    m, n, d, zeta, mseed = WORKLOADS[args.workload]
    cores = os.cpu_count() or 1
    threads = min(cores, 64)
    sample_rows = min(m, args.ref_rows)
    A = wl.gaussian(sample_rows, n, mseed)
    seed = wl.sketch_seed(0)
    oracle.build()
    for _ in range(max(0, min(args.warmup, 1))):
        oracle.f64_sketch(seed, d, zeta, A[: sample_rows // 8], threads=threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.f64_sketch(seed, d, zeta, A, threads=threads)
    dt = (time.perf_counter() - t0) / args.steps
    gbs = sample_rows * n * 4 / dt / 1e9
    line = {
        "impl": "reference", "metric": "sketch_A_read_GBps", "value": gbs, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s (first %d of %d rows per step): SparseStack zeta=%d, m=%d, n=%d, d=%d, A FP32 N(0,1)"
                               % (args.workload, sample_rows, m, zeta, m, n, d),
                   "sample": "first %d rows per step" % sample_rows},
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": threads, "kind": "oracle",
                         "sample": "oracle FP64 mode (row-chunk-private partials, %d threads) on %d of %d rows" % (threads, sample_rows, m)},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))
    return 0


def cpu_baseline(workload, cpu_seconds=16.0):
    """The oracle as it stands on the host cores, on a bounded sample: about `cpu_seconds` of CPU work (threads x wall) in the
    all-core FP64 mode -- whole passes over the first rows of the workload, repeated -- plus ~3 s each single-threaded."""
    import numpy as np

    import oracle
    import workloads as wl

    m, n, d, zeta, mseed = WORKLOADS[workload]
    cores = os.cpu_count() or 1
    threads = min(cores, 64)
    seed = wl.sketch_seed(0)
    rows2 = int(min(m, max(1 << 12, (1 << 29) // (4 * n))))      # up to 512 MiB of A per pass
    A = wl.gaussian(rows2, n, mseed)
    oracle.f64_sketch(seed, d, zeta, A[: max(1, rows2 // 8)], threads=threads)      # page in, start the threads
    passes, t0 = 0, time.perf_counter()
    while True:
        oracle.f64_sketch(seed, d, zeta, A, threads=threads)
        passes += 1
        dt_all = time.perf_counter() - t0
        if dt_all * threads >= cpu_seconds or passes >= 4096:
            break

    def single(fn, rows, budget=3.0):
        t0 = time.perf_counter()
        fn(A[:rows])
        dt = time.perf_counter() - t0
        rows_b = int(min(rows2, max(rows, rows * budget / max(dt, 1e-4))))
        t0 = time.perf_counter()
        fn(A[:rows_b])
        return rows_b, time.perf_counter() - t0

    rows1, dt_one = single(lambda X: oracle.f64_sketch(seed, d, zeta, X, threads=1), min(rows2, 1 << 14))
    rows16, dt16 = single(lambda X: oracle.seq16_sketch(seed, d, zeta, X), min(rows2, 1 << 11))
    return {
        "value": passes * rows2 * n * 4 / dt_all / 1e9, "unit": "GB/s", "cores": threads, "kind": "oracle",
        "sample": "oracle FP64 mode, %d threads, %d passes over the first %d of %d rows (%.1f s wall = %.0f CPU-s)"
                  % (threads, passes, rows2, m, dt_all, dt_all * threads),
        "single_thread_f64_GBps": rows1 * n * 4 / dt_one / 1e9, "single_thread_f64_sample": "%d rows, %.1f s" % (rows1, dt_one),
        "single_thread_seq16_GBps": rows16 * n * 4 / dt16 / 1e9, "single_thread_seq16_sample": "%d rows, %.1f s" % (rows16, dt16),
    }


# ------------------------------------------------------------------------------------------- our arm
def run_sustained(torch, step, ms_est, seconds, sampler, a_bytes):
    """`seconds` (+15 %) of back-to-back steps with an event after every ~20 ms batch.  Returns the rate over the first half
    second, the last second and the whole run, each with the clock / power samples of that window."""
    per_batch = max(1, int(round(20.0 / max(ms_est, 1e-3))))
    batches = max(4, int(seconds * 1e3 * 1.15 / (per_batch * ms_est)) + 1)
    torch.cuda.synchronize()
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(batches + 1)]
    evs[0].record()
    for b in range(batches):
        for _ in range(per_batch):
            step()
        evs[b + 1].record()
    torch.cuda.synchronize()
    w1 = time.time()
    t = [evs[0].elapsed_time(e) * 1e-3 for e in evs]            # seconds since the first event
    total = t[-1]

    def window(lo, hi):
        idx = [i for i in range(1, len(t)) if t[i - 1] >= lo - 1e-9 and t[i] <= hi + 1e-9]
        if not idx:
            return None
        dur = t[idx[-1]] - t[idx[0] - 1]
        steps = len(idx) * per_batch
        out = {"seconds": dur, "steps": steps, "ms_per_step": dur / steps * 1e3, "GBps": steps * a_bytes / dur / 1e9}
        if sampler is not None:
            out["clocks"] = sampler.summary(w1 - (total - t[idx[0] - 1]), w1 - (total - t[idx[-1]]))
        return out

    batch_ms = [(t[i] - t[i - 1]) / per_batch * 1e3 for i in range(1, len(t))]
    return {"seconds": total, "steps": batches * per_batch, "steps_per_batch": per_batch,
            "first_half_second": window(0.0, min(0.5, total / 2)), "last_second": window(max(0.0, total - 1.0), total), "whole": window(0.0, total),
            "ms_per_step_by_batch": {"min": min(batch_ms), "median": sorted(batch_ms)[len(batch_ms) // 2], "max": max(batch_ms)},
            "batch_stats": step_stats(batch_ms),
            "note": "back-to-back complete sketches of the resident A, no L2 flush and no host work between them"}


def measure_red_payload(torch, ss, dev, d, n, replicas, variant, f32=False):
    """GB/s of RED payload the L2 atomic units take with the flat kernel's address pattern on a replicas x d x n sketch (FP16,
    or FP32 with f32=True): the widest operand the row length allows (16 / 8 / 4 bytes per lane; one column or column pair
    for flat_pair), 8 CTAs per SM, values from registers."""
    eb = 4 if f32 else 2
    if f32:
        kind, vec = (5, 4) if n % 4 == 0 else (4, 2) if n % 2 == 0 else (3, 1)
        if variant == "flat_pair":
            kind, vec = 3, 1
    else:
        if n % 2:
            return None
        kind, vec = (2, 8) if n % 8 == 0 else (1, 4) if n % 4 == 0 else (0, 2)
        if variant == "flat_pair":
            kind, vec = 0, 2
    grid = torch.cuda.get_device_properties(dev).multi_processor_count * 8
    buf = torch.zeros(replicas * d * n * eb + 16, dtype=torch.uint8, device=dev)
    ss.sketch_red_probe(buf, d, n, kind, replicas, grid, 200)
    best = 0.0
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ops = ss.sketch_red_probe(buf, d, n, kind, replicas, grid, 2000)
        e1.record()
        torch.cuda.synchronize()
        best = max(best, ops * vec * eb / (e0.elapsed_time(e1) * 1e-3) / 1e9)
    return {"payload_GBps": best, "what": "%d-byte REDs into %d partial sketches of %d x %d %s, grid %d, best of 3 x 2000 rounds"
                                          % (vec * eb, replicas, d, n, "FP32" if f32 else "FP16", grid)}


def l2_red_from_capture(entry, ms_apply):
    """L2-side reduction traffic of the dominant kernel from the committed ncu capture (profiles/ncu_traffic.json), turned
    into rates with this run's time.  None where the capture holds no RED counters."""
    if not entry or "lts_red_sectors" not in entry:
        return None
    sec = ms_apply * 1e-3
    return {"lts__t_sectors_op_red_per_s": entry["lts_red_sectors"] / sec,
            "smsp__inst_executed_op_global_red_per_s": entry.get("red_warp_inst", 0) / sec,
            "l1tex_red_payload_GBps": entry.get("red_l1tex_bytes", 0) / sec / 1e9,
            "per_launch": {k: entry[k] for k in ("lts_red_sectors", "red_warp_inst", "red_l1tex_bytes") if k in entry},
            "source": "counters per launch from the committed capture %s, divided by this run's time" % entry["profile"]}


def run_ours(args):
    import numpy as np
    import torch

    import paper_2606_20195_b200 as ss
    import workloads as wl
    from paper_2606_20195_b200.sharding import all_reduce_sketch, max_over_ranks, shard_rows

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    for _ in range(5):                 # a driver still tearing down a previous large process can fail one init
        if torch.cuda.is_available():
            break
        time.sleep(2.0)
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    dist = None
    multi = world > 1
    if "RANK" in os.environ and "WORLD_SIZE" in os.environ:
        # under torchrun the NCCL communicator is created and used even with ONE rank: the collective leg (init, FP16 / FP32
        # all-reduce of the sketch, barrier, max-over-ranks timing) then runs on whatever box this is, not only on N > 1
        import torch.distributed as dist_

        dist = dist_
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    m, n, d, zeta, mseed = WORKLOADS[args.workload]
    dev = torch.device("cuda", local)
    seed = wl.sketch_seed(0)
    sk = ss.Sketch(m * world, d, zeta, seed)   # one map over all shards; rank r owns rows [r*m, (r+1)*m)
    row_begin, shard = shard_rows(m * world, world, rank)
    assert shard == m
    A = wl.gaussian_device(m, n, mseed + 7919 * rank, dev)
    out16 = torch.empty((d, n), dtype=torch.float16, device=dev)
    out32 = torch.empty((d, n), dtype=torch.float32, device=dev)
    vid = VARIANTS[args.variant]
    plan16 = sk.plan(n, f16=True, variant=vid, rows=m, row_begin=row_begin)
    plan32 = sk.plan(n, f16=False, rows=m, row_begin=row_begin)
    small = m * n * 4 < (512 << 20)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev) if small else None

    uses_packed = plan16["hash_mode"] == 2

    def apply16():
        sk.apply_f16acc(A, out=out16, variant=vid, row_begin=row_begin, rows=m, replicas=args.replicas, hash_mode=args.hash_mode,
                        tmem_group_mode=args.tmem_group_mode)
        if dist is not None:
            all_reduce_sketch(out16, dist)   # sum of the ranks' partial sketches: one more level of the FP16 hierarchy

    def step16():
        # complete sketch ("initialization, map generation, and application"): when the scatter
        # reads precomputed hashes, the hash-pack kernel is re-run inside every timed step
        if uses_packed:
            sk.precompute_hashes()
        apply16()

    def step32():
        sk.apply_f32acc(A, out=out32, row_begin=row_begin, rows=m)
        if dist is not None:
            all_reduce_sketch(out32, dist)

    # like-for-like pairs (same privatisation on both sides): what FP16 PRECISION buys as opposed to what privatisation
    # buys (Eq. (5)): flat REDs on both sides, and tensor memory on both sides where the FP32 partial fits
    def flat16():
        sk.apply_f16acc(A, out=out16, variant=VARIANTS["flat_vec"], row_begin=row_begin, rows=m)

    def flat32():
        sk.apply_f32acc(A, out=out32, variant=VARIANTS["flat_vec"], row_begin=row_begin, rows=m)

    def tmem16():
        sk.apply_f16acc(A, out=out16, variant=VARIANTS["tmem"], row_begin=row_begin, rows=m)

    def tmem32():
        sk.apply_f32acc(A, out=out32, variant=VARIANTS["tmem"], row_begin=row_begin, rows=m)

    def can(f16, variant):
        try:
            sk.plan(n, f16=f16, variant=VARIANTS[variant], rows=m, row_begin=row_begin)
            return True
        except ss.SketchError:
            return False

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def timed(fn, steps, warmup):
        for _ in range(warmup):
            if flush is not None:
                flush.zero_()                      # warm-up steps look like timed steps (the first flush loads its own kernel)
            fn()
        barrier()
        evs = []
        l0 = ss.sketch_launch_count()
        w0 = time.time()
        for _ in range(steps):
            if flush is not None:
                flush.zero_()                      # inputs smaller than 4x L2: flush L2 between steps
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            evs.append((e0, e1))
        barrier()
        w1 = time.time()
        ms = [a.elapsed_time(b) for a, b in evs]
        # wall-clock midpoint of every step: the device ran the steps back to back up to the synchronize that returned at w1
        end = evs[0][0].elapsed_time(evs[-1][1])
        mids = [w1 - (end - 0.5 * (evs[0][0].elapsed_time(a) + evs[0][0].elapsed_time(b))) * 1e-3 for a, b in evs]
        total = max_over_ranks(sum(ms), dist, dev) if dist is not None else sum(ms)
        return total / steps, ms, ss.sketch_launch_count() - l0, (w0, w1, mids)

    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid)
    if rank == 0:
        sampler.start()
        time.sleep(0.1)
    ms16, per16, launches16, (w0, w1, mids16) = timed(step16, args.steps, args.warmup)
    clocks = sampler.summary(w1 - sum(per16) * 1e-3 - 0.005, w1 + 0.005) if rank == 0 else None
    per_step = [dict(ms=t, **(sampler.nearest(mid) or {})) for t, mid in zip(per16, mids16)] if rank == 0 else None

    # sustained operation: >= args.sustained_seconds of back-to-back complete sketches (no flush, no host work in between),
    # an event after every ~20 ms batch; the rate over the last second is what a caller streaming matrices for seconds gets
    sustained = None
    if args.sustained_seconds > 0 and not multi:
        sustained = run_sustained(torch, step16, ms16, args.sustained_seconds, sampler if rank == 0 else None, m * n * 4)
    if rank == 0:
        sampler.halt()
    ms32, _, _, _ = timed(step32, max(2, args.steps // 2), 3)
    pairs = {}
    if not args.no_pairs and not multi:
        k2 = max(2, args.steps // 2)
        if can(True, "flat_vec") and can(False, "flat_vec"):
            a16, a32 = timed(flat16, k2, 3)[0], timed(flat32, k2, 3)[0]
            pairs["flat"] = {"f16_ms": a16, "f32_ms": a32, "f16_over_f32": a32 / a16}
        if can(True, "tmem") and can(False, "tmem"):
            a16, a32 = timed(tmem16, k2, 3)[0], timed(tmem32, k2, 3)[0]
            pairs["tmem"] = {"f16_ms": a16, "f32_ms": a32, "f16_over_f32": a32 / a16}
    ms16_apply, _, _, _ = timed(apply16, max(2, args.steps // 2), 3) if uses_packed else (ms16, None, None, None)

    # second roofline term, measured in this run for the plans it bounds: result-discarding REDs with the flat kernel's
    # address pattern on this workload's own d x n and replica count, values from registers, no A loads (sketch_red_probe)
    red_probe = None
    if plan16["variant"] in ("flat_vec", "flat_pair", "generic") and not multi:
        red_probe = measure_red_payload(torch, ss, dev, d, n, max(1, int(plan16["replicas"])), plan16["variant"])

    # step a2 alone: how fast this GPU delivers A when it is only read (sketch_stream_probe; context for roofline.frac, whose
    # denominator is a COPY rate).  Plain 256-bit loads and k_tmem's TMA ring without consumers, median of 5 passes over A.
    stream_probe = {}
    if not multi and m * n * 4 >= (1 << 28):
        for key, kind in (("ld256", 0), ("tma_ring", 1)):
            ts = []
            for rep_i in range(7):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                nb = ss.sketch_stream_probe(A, kind)
                e1.record()
                torch.cuda.synchronize()
                if rep_i >= 2:
                    ts.append(e0.elapsed_time(e1))
            ts.sort()
            stream_probe[key + "_GBps"] = nb / (ts[len(ts) // 2] * 1e-3) / 1e9

    # end to end through the host-buffer entry point: pinned A on the host, H2D + kernels + D2H inside the call
    e2e = None
    if not args.no_e2e:
        try:
            Ah = torch.empty((m, n), dtype=torch.float32, pin_memory=True)
            Ah.copy_(A)
            Bh = torch.empty((d, n), dtype=torch.float16, pin_memory=True)
            torch.cuda.synchronize()

            def step_e2e():
                sk.apply_f16acc_host(Ah, out_host=Bh, variant=vid, row_begin=row_begin, rows=m)
                if dist is not None:
                    t = Bh.to(dev)
                    all_reduce_sketch(t, dist)
                    Bh.copy_(t)

            step_e2e()
            barrier()
            t0 = time.perf_counter()
            ksteps = max(1, min(args.steps, 3))
            for _ in range(ksteps):
                step_e2e()
            barrier()
            dt = (time.perf_counter() - t0) / ksteps
            if dist is not None:
                dt = max_over_ranks(dt, dist, dev)
            e2e = {"value": world * m * n * 4 / dt / 1e9, "unit": "GB/s", "h2d_bytes_per_step": m * n * 4,
                   "d2h_bytes_per_step": d * n * 2, "ms_per_step": dt * 1e3, "steps": ksteps,
                   "api": "sketch_apply_f16acc_host (pinned host A, double-buffered 256 MiB H2D chunks)"}
            # the two entry points must agree on what they computed (same variant => same partial-sum tree up to RED order)
            chk = sk.apply_f16acc(A, variant=vid, row_begin=row_begin, rows=m)
            if dist is not None:
                all_reduce_sketch(chk, dist)
            diff = (chk.float().cpu() - Bh.float()).norm() / chk.float().norm().cpu()
            e2e["rel_diff_vs_device_path"] = float(diff)
            del Ah
        except (RuntimeError, ss.SketchError) as ex:  # e.g. the box cannot pin 16 GiB
            e2e = {"value": None, "unit": "GB/s", "h2d_bytes_per_step": m * n * 4, "d2h_bytes_per_step": d * n * 2,
                   "error": str(ex)[:200]}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    peaks, peak_src = measured_peaks()
    traffic, traffic_src = ncu_traffic(args.workload, plan16["variant"])
    abytes = algorithmic_bytes(m, n, d, 2)
    gbs = world * m * n * 4 / (ms16 * 1e-3) / 1e9
    achieved = abytes / (ms16_apply * 1e-3) / 1e9    # per GPU: the event bracket holds memset + scatter (+ fold)
    hbm = float(peaks["hbm_gbs"])
    red_ops = zeta * m * n // 2
    line = {
        "metric": "sketch_A_read_GBps", "value": gbs, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms16, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (gbs / world / PAPER_GBPS[args.workload]) if args.workload in PAPER_GBPS else None,
        "dtype": "f16", "data": "synthetic",
        "config": {"workload": "%s: SparseStack zeta=%d, m=%d, n=%d, d=%d (d=2n), A FP32 row-major N(0,1) %.2f GiB per GPU, FP16-RN accumulate"
                               % (args.workload, zeta, m, n, d, m * n * 4 / 2**30),
                   "variant": plan16["variant"], "replicas": plan16["replicas"], "hash_mode": plan16["hash_mode"], "grid": plan16["grid"],
                   "l2": "input %s L2; %s" % ("<" if small else ">", "512 MiB flush write between steps" if small else "no flush needed"),
                   "sharding": ("rows; rank r hashes global rows [r*m,(r+1)*m); one NCCL all-reduce of the d x n sketch (%d rank%s)" % (world, "" if world == 1 else "s"))
                               if dist is not None else "single GPU"},
        "apply_only": {"ms_per_step": ms16_apply, "GBps": world * m * n * 4 / (ms16_apply * 1e-3) / 1e9,
                       "note": "hash-pack kernel excluded (map reused, as when A and b share one sketch, PAPER.md:356)"},
        "sketches_per_s": 1e3 / ms16,
        "contributions_per_s": zeta * m * n * world / (ms16 * 1e-3),
        "half2_updates_per_s": red_ops * world / (ms16 * 1e-3),
        "half2_updates_note": "LOGICAL count: zeta*m*n/2 two-feature FP16 adds per sketch / time.  In the tensor-memory, shared-memory and "
                              "small variants these adds happen on chip; what reaches the L2 atomic units is only the flush (l2_red below)",
        "l2_red": l2_red_from_capture(traffic_src, ms16_apply),
        "ms_per_step_stats": step_stats(per16),
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": hbm, "unit": "GB/s", "frac": achieved / hbm,
                     "traffic": traffic, "traffic_source": ("committed ncu capture %s (kernel %s)" % (traffic_src["profile"], traffic_src["kernel"])) if traffic_src else None,
                     "peak_source": peak_src,
                     "frac_of_nominal_8TBps": achieved / 8000.0,
                     "frac_of_read_only_stream": (achieved / max(stream_probe.values())) if stream_probe else None,
                     "frac_note": "`peak` is the driver's measured COPY rate (MEASURED_PEAKS.json), as the bench contract fixes; a kernel that only reads can "
                                  "exceed it, so frac may read above 1.  frac_of_read_only_stream divides by the read-only streaming rate of the same A "
                                  "measured in this run -- the actual ceiling of a complete sketch -- and stays at or below 1",
                     "frac_sustained": (sustained["last_second"]["GBps"] * abytes / (m * n * 4) / hbm) if sustained else None,
                     "read_only_stream": dict(stream_probe, note="sketch_stream_probe over the same A in this run: what a kernel that only READS can reach; "
                                                                 "`peak` is a copy rate (read + write)") if stream_probe else None,
                     "algorithmic_bytes_per_launch": abytes,
                     "note": "dominant kernel = the scatter; CUDA-event bracket on the launching stream = zero-init memset + scatter (+ replica fold), hash-pack excluded"},
        "f32acc": {"ms_per_step": ms32, "GBps": world * m * n * 4 / (ms32 * 1e-3) / 1e9, "variant": plan32["variant"],
                   "replicas": plan32["replicas"], "f16_speedup_over_f32": ms32 / ms16,
                   "like_for_like": pairs,
                   "note": "f16_speedup_over_f32 compares AUTO with AUTO; like_for_like holds both precisions on the same privatisation"},
        "e2e": e2e if e2e is not None else {"value": None, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "skipped": True},
        "gpu_launches": int(launches16),
        "clocks": clocks,
        "per_step_ms": per16,
        "per_step": per_step,
        "sustained": sustained,
        "paper_context": "H200 NVL (PAPER.md:320-322): FP16 SS zeta=4 7.11 ms for 8 GiB (1.21 TB/s), up to 1.91x its FP32 scatter",
    }
    if plan16["variant"] in ("flat_vec", "flat_pair", "generic"):
        # a flat scatter is bound by the L2 atomic units, not by HBM: 2 bytes of RED payload per contribution
        payload = 2.0 * zeta * m * n / (ms16_apply * 1e-3) / 1e9
        peak2 = red_probe["payload_GBps"] if red_probe else L2_RED_PAYLOAD_GBPS_R01
        line["roofline"]["l2_atomic"] = {"achieved": payload, "peak": peak2, "unit": "GB/s of RED payload", "frac": payload / peak2,
                                         "peak_source": ("sketch_red_probe in this run: %s" % red_probe["what"]) if red_probe
                                                        else "round-1 probe (profiles/r01_red_probe.md)",
                                         "note": "second roofline term (SURVEY 8d): the slower of HBM and L2-atomic bounds this variant"}
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(args.workload)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------- range study
def run_range_study(args):
    """BASELINE.json configs[4] (Fig. 7): A = N(0,1) * 2^k, k in {-24,-16,0,+8,+12}, RN vs SR.
    Per (k, rounding): sketch GB/s at the workload's full size, non-finite outputs, error against the FP64 oracle on
    sampled columns (entries finite in both, R18), and the oracle's per-contribution range counts on a row
    sample.  One JSON line; not the driver's bench line."""
    import numpy as np
    import torch

    import evaluation as ev
    import oracle
    import paper_2606_20195_b200 as ss
    import workloads as wl

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    m, n, d, zeta, mseed = WORKLOADS[args.workload]
    seed = wl.sketch_seed(0)
    sk = ss.Sketch(m, d, zeta, seed)
    A = wl.gaussian_device(m, n, mseed, dev)
    cols = sorted({0, 1, n // 2 - 1, n // 2, n - 2, n - 1})
    threads = min(os.cpu_count() or 1, 64)
    oracle.build()
    B0 = oracle.f64_sketch(seed, d, zeta, np.ascontiguousarray(A[:, cols].cpu().numpy()), threads=threads)  # k = 0; S(2^k A) = 2^k S A exactly
    sample = np.ascontiguousarray(A[: 1 << 16].cpu().numpy())
    out = torch.empty((d, n), dtype=torch.float16, device=dev)
    rows_out, prev = [], 0
    for k in (-24, -16, 0, 8, 12):
        A.mul_(float(2.0 ** (k - prev)))      # exact in FP32
        prev = k
        counts = oracle.range_counts(zeta, sample * np.float32(2.0 ** k))
        out_bf = torch.empty((d, n), dtype=torch.bfloat16, device=dev)
        for rname, rmode in (("RN", ss.RN), ("SR", ss.SR), ("dither", ss.DITHER), ("BF16", None)):
            if rmode is None:
                fn = lambda: sk.apply_bf16acc(A, out=out_bf)      # the BF16 control
                res, variant = out_bf, sk.plan(n, f16=2)["variant"]
            else:
                kw = dict(out=out, rounding=rmode, sr_seed=wl.sketch_seed(77))
                fn = lambda: sk.apply_f16acc(A, **kw)
                res, variant = out, sk.plan(n, rounding=rmode)["variant"]
            for _ in range(2):
                fn()
            torch.cuda.synchronize()
            reps = 5 if rname in ("RN", "BF16") else 3
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(reps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            got = res[:, cols].float().cpu().numpy().astype(np.float64)
            want = B0 * 2.0 ** k
            fin = np.isfinite(got)
            rel = ev.rel_fro(got[fin], want[fin]) if fin.any() else None
            rows_out.append({
                "k": k, "rounding": rname, "variant": variant, "ms": ms,
                "GBps": m * n * 4 / (ms * 1e-3) / 1e9,
                "nonfinite_outputs": int((~torch.isfinite(res)).sum().item()), "nan_outputs": int(torch.isnan(res).sum().item()),
                "zero_outputs": int((res == 0).sum().item()), "outputs": d * n,
                "relF_vs_f64_sampled_cols_finite": rel,
                "oracle_contribution_counts_first_65536_rows": {kk: int(v) for kk, v in counts.items()},
            })
    A.mul_(float(2.0 ** (-prev)))
    print(json.dumps({"study": "range (BASELINE.json configs[4])", "workload": "%s: m=%d n=%d d=%d zeta=%d, N(0,1) * 2^k" % (args.workload, m, n, d, zeta),
                      "sampled_columns": cols, "rows": rows_out}))
    return 0


def _time_ms(fn, reps=5, warm=2, flush=None):
    import torch

    for _ in range(warm):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        if flush is not None:
            flush.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        torch.cuda.synchronize()
        ts.append(e0.elapsed_time(e1))
    ts.sort()
    return ts[len(ts) // 2]


def run_ls_study(args):
    """SURVEY 8f NEXT-1 (Fig. 6): complete sketch-and-solve least squares on the GPU at the paper's own
    shape (m = 2^21, n = 1024, zeta = 4), both of its families, d/n in {2, 4, 8, 16, 32}: [A | b] sketched in ONE pass
    (sketch_apply_f16acc_with_rhs / _f32acc_with_rhs: A in the chosen precision, b in FP32, same map), exact widening,
    FP32 Householder QR + projection + triangular solve (cuSOLVER / cuBLAS through torch: library code, as in the paper),
    original-system residual in FP64.  Median of 5 timed solves per point.  One JSON line; not the driver's bench line."""
    import torch

    import paper_2606_20195_b200 as ss
    import workloads as wl
    from paper_2606_20195_b200 import lstsq

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    m, n, zeta = 1 << 21, 1024, 4
    fams = []
    for fam, gen in (("low_coherence", wl.ls_paper_low_coherence_device), ("coherent", wl.ls_paper_coherent_device)):
        A, b2 = gen(m, n, 6, dev)
        b = b2[:, 0].contiguous()
        bnorm = float(b.double().norm())

        def residual(x):
            acc = 0.0
            xd = x.double()
            for r0 in range(0, m, 1 << 18):
                r = A[r0:r0 + (1 << 18)].double() @ xd - b[r0:r0 + (1 << 18)].double()
                acc += float((r * r).sum())
            return acc ** 0.5 / bnorm

        rows_out = []
        for ratio in (2, 4, 8, 16, 32):
            d = ratio * n
            sk = ss.Sketch(m, d, zeta, wl.sketch_seed(0))
            W = torch.empty((d, n), dtype=torch.float32, device=dev)
            bufs = {"f16": torch.empty((d, n), dtype=torch.float16, device=dev), "f32": torch.empty((d, n), dtype=torch.float32, device=dev),
                    "bf16": torch.empty((d, n), dtype=torch.bfloat16, device=dev)}
            Sb = torch.empty((d,), dtype=torch.float32, device=dev)
            row = {"d_over_n": ratio, "d": d, "fp16_variant": sk.plan(n, f16=1)["variant"], "fp32_variant": sk.plan(n, f16=0)["variant"]}
            for prec in ("f16", "f32", "bf16"):
                solve = lambda: lstsq.sketch_and_solve(sk, A, b, prec, SA=bufs[prec], Sb=Sb, W=W)
                row["ls_ms_" + prec] = _time_ms(solve)
                row["sketch_ms_" + prec] = _time_ms(lambda: lstsq.sketch_system(sk, A, b, prec, SA=bufs[prec], Sb=Sb))
                row["residual_" + prec] = residual(solve())
            row["ls_speedup_f16_over_f32"] = row["ls_ms_f32"] / row["ls_ms_f16"]
            row["residual_increase_pct_f16"] = 100.0 * (row["residual_f16"] / row["residual_f32"] - 1.0)
            row["residual_increase_pct_bf16"] = 100.0 * (row["residual_bf16"] / row["residual_f32"] - 1.0)
            rows_out.append(row)
            del W, bufs
        fams.append({"family": fam, "rows": rows_out})
        del A, b, b2
        torch.cuda.empty_cache()
    print(json.dumps({"study": "sketch-and-solve least squares (SURVEY 8f NEXT-1)",
                      "workload": "the paper's two families (PAPER.md:362-366), m=%d n=%d zeta=%d; low-coherence: sigma linear 100->1, b = A 1 + N(0, 0.1^2); "
                                  "coherent: [I_n; 1e-3 G / sqrt(m-n)] under a row permutation, b = [x0 + N(0, 0.5^2); T x0]" % (m, n, zeta),
                      "pipeline": "one-pass [A|b] sketch -> sketch_widen -> torch.geqrf -> torch.ormqr -> solve_triangular (paper_2606_20195_b200/lstsq.py)",
                      "paper_context": "H200 NVL (PAPER.md:368-370): FP16 SS 13.921 ms at d/n=2 -> 35.016 ms at d/n=32, 1.47x / 1.44x over its FP32 pipeline, residual 0.1155 -> 0.08223, +0.34 % / +0.35 % over FP32; BF16 ~20 % above FP32 at d/n=2 (PAPER.md:396)",
                      "families": fams}))
    return 0


def run_grid_study(args):
    """the paper's complete-sketch timing grid (Fig. 2) as one command: n = 1024,
    m in {2^19, 2^20, 2^21}, d/n in {2 .. 256}, zeta in {1, 2, 4, 8}, dense (singular values linear 1000 -> 1) and coordinate
    [I_n 0]^T inputs.  Per point: complete-sketch time of the FP16 and FP32 paths (median of 5, L2 flushed when A < 512 MiB...
    never at these sizes), the variant AUTO picked, GB/s of A, fraction of the HBM peak and -- for the flat variants -- of the
    measured L2-atomic payload rate.  One JSON line; not the driver's bench line."""
    import torch

    import paper_2606_20195_b200 as ss
    import workloads as wl

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    n = 1024
    quick = args.grid == "quick"
    ms_list = (1 << 19, 1 << 21) if quick else (1 << 19, 1 << 20, 1 << 21)
    ratios = (2, 256) if quick else (2, 4, 8, 16, 32, 64, 128, 256)
    zetas = (1, 4, 8) if quick else (1, 2, 4, 8)
    peaks, peak_src = measured_peaks()
    hbm = float(peaks["hbm_gbs"])
    pts = []
    red_rates = {}
    for m in ms_list:
        for kind in ("dense", "coordinate"):
            if kind == "dense":
                A = wl.gaussian_device(m, n, 5, dev)
                A.mul_((torch.linspace(1000.0, 1.0, n, device=dev) / float(m) ** 0.5)[None, :])   # sigma linear 1000 -> 1
            else:
                A = torch.zeros((m, n), dtype=torch.float32, device=dev)
                A[:n] = torch.eye(n, device=dev)
            for ratio in ratios:
                d = ratio * n
                o16 = torch.empty((d, n), dtype=torch.float16, device=dev)
                o32 = torch.empty((d, n), dtype=torch.float32, device=dev)
                for zeta in zetas:
                    sk = ss.Sketch(m, d, zeta, wl.sketch_seed(0))
                    p16, p32 = sk.plan(n, f16=1), sk.plan(n, f16=0)
                    t16 = _time_ms(lambda: sk.apply_f16acc(A, out=o16), reps=5 if not quick else 3)
                    t32 = _time_ms(lambda: sk.apply_f32acc(A, out=o32), reps=5 if not quick else 3)
                    pt = {"m": m, "input": kind, "d_over_n": ratio, "zeta": zeta, "fp16_ms": t16, "fp32_ms": t32, "fp16_over_fp32": t32 / t16,
                          "fp16_variant": p16["variant"], "fp32_variant": p32["variant"], "fp16_GBps": m * n * 4 / t16 / 1e6,
                          "fp16_frac_hbm": (4 * m * n + 2 * d * n) / (t16 * 1e-3) / 1e9 / hbm,
                          "fp32_frac_hbm": (4 * m * n + 4 * d * n) / (t32 * 1e-3) / 1e9 / hbm}
                    for key, pl, eb, tt in (("fp16", p16, 2.0, t16), ("fp32", p32, 4.0, t32)):
                        if pl["variant"] in ("flat_vec", "flat_pair"):
                            ck = (d, pl["replicas"], pl["variant"], key)
                            if ck not in red_rates:       # the L2-atomic rate of this sketch shape, measured once per shape in this run
                                pr = measure_red_payload(torch, ss, dev, d, n, max(1, pl["replicas"]), pl["variant"], f32=key == "fp32")
                                red_rates[ck] = pr["payload_GBps"] if pr else None
                            if red_rates[ck]:
                                pt[key + "_frac_l2_atomic"] = eb * zeta * m * n / (tt * 1e-3) / 1e9 / red_rates[ck]
                                pt[key + "_l2_atomic_peak_GBps"] = red_rates[ck]
                    pts.append(pt)
                    sk.close()
                del o16, o32
            del A
            torch.cuda.empty_cache()
    print(json.dumps({"study": "paper timing grid (SURVEY 8f NEXT-2; PAPER.md:318-322)", "n": n, "hbm_peak_GBps": hbm, "peak_source": peak_src,
                      "l2_atomic_payload_GBps": "sketch_red_probe on every (d, replicas, operand) of a flat point, in this run (fp*_l2_atomic_peak_GBps)",
                      "paper_context": "H200 NVL: FP16 SS 7.11 ms at m=2^21, d=2n, zeta=4 (PAPER.md:322); FP16 up to 1.91x its FP32 scatter (PAPER.md:320)",
                      "points": pts}))
    return 0


def run_coherence_study(args):
    """The paper's geometry sweep (Sec. V-C, Fig. 5) with direct sketching of U: U(theta) =
    orth((1 - theta) Q_rand + theta [I_n 0]^T), eleven theta values, m = 2^20, n = 1024, d/n in {2, 4, 8, 16}, zeta = 4 (plus
    zeta in {1, 2, 8} at d = 2n for the rank statement of PAPER.md:352).  Per point: coherence (Eq. 2), distortion (Eq. 4) of
    the FP16 and FP32 sketches = max |sigma_i(S U) - 1| from an FP64 SVD of the returned d x n matrix, their difference, the
    smallest singular value (rank).  One JSON line; not the driver's bench line."""
    import torch

    import paper_2606_20195_b200 as ss
    import workloads as wl

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    quick = args.grid == "quick"
    m, n = (1 << 18, 256) if quick else (1 << 20, 1024)
    thetas = [0.0, 0.5, 1.0] if quick else [k / 10.0 for k in range(11)]
    cases = [(r, 4) for r in (2, 4, 8, 16)] + [(2, z) for z in (1, 2, 8)]
    sks = {(r, z): ss.Sketch(m, r * n, z, wl.sketch_seed(0)) for r, z in cases}

    def eta(SU):
        sv = torch.linalg.svdvals(SU.double())
        return float(torch.maximum((sv.max() - 1.0).abs(), (1.0 - sv.min()).abs())), float(sv.min())

    pts = []
    for theta, U, mu in wl.coherence_basis_device(m, n, thetas, 9, dev):
        for (r, z), sk in sks.items():
            e16, smin16 = eta(sk.apply_f16acc(U))
            e32, smin32 = eta(sk.apply_f32acc(U))
            pts.append({"theta": theta, "coherence": mu, "max_row_energy": mu * n / m, "d_over_n": r, "zeta": z, "eta_fp16": e16, "eta_fp32": e32,
                        "abs_diff": abs(e16 - e32), "sigma_min_fp16": smin16, "sigma_min_fp32": smin32,
                        "variant_fp16": sk.plan(n, f16=1)["variant"], "sqrt_n_over_d": (1.0 / r) ** 0.5})
        del U
    z4 = [p for p in pts if p["zeta"] == 4]
    print(json.dumps({"study": "coherence sweep with direct sketching of U (SURVEY 8f NEXT-2; PAPER.md:344-352)", "m": m, "n": n,
                      "largest_abs_diff_zeta4": max(p["abs_diff"] for p in z4),
                      "paper_context": "H200 NVL, PAPER.md:348-352: largest individual FP16-FP32 distortion difference 0.00492, largest case-median 7.80e-4; "
                                       "u sqrt(n) = 1/64 is Prop. 2's conversion-only scale; coordinate endpoint, d/n = 16: FP32 SparseStack distortion 0.364; "
                                       "at d = 2n coordinate sketches keep full rank at zeta = 4, 8 and lose it at zeta = 1 (and in the zeta = 2 runs tried)",
                      "points": pts}))
    return 0


def run_replica_study(args):
    """Conversion rule x where the partial sums live, at the workload's full size (default c5): FP16 RN / SR / dither through the
    flat REDs with P in {8, 32, 128, 256} L2-resident partial sketches and through the tensor-memory kernel -- time per complete
    sketch and relF against the FP64 oracle on sampled columns.  What AUTO's replica rule and its SR / dither rule rest on
    (DESIGN.md section 5.2).  One JSON line; not the driver's bench line."""
    import numpy as np
    import torch

    import evaluation as ev
    import oracle
    import paper_2606_20195_b200 as ss
    import workloads as wl

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    m, n, d, zeta, mseed = WORKLOADS[args.workload]
    seed = wl.sketch_seed(0)
    sk = ss.Sketch(m, d, zeta, seed)
    A = wl.gaussian_device(m, n, mseed, dev)
    cols = sorted({0, 1, n // 2 - 1, n // 2, n - 2, n - 1})
    oracle.build()
    B0 = oracle.f64_sketch(seed, d, zeta, np.ascontiguousarray(A[:, cols].cpu().numpy()), threads=min(os.cpu_count() or 1, 64))
    out = torch.empty((d, n), dtype=torch.float16, device=dev)
    rows_out = []
    for rname, rmode in (("RN", ss.RN), ("SR", ss.SR), ("dither", ss.DITHER)):
        for var, P in (("flat_vec", 8), ("flat_vec", 32), ("flat_vec", 128), ("flat_vec", 256), ("tmem", 0), ("auto", 0)):
            kw = dict(out=out, rounding=rmode, sr_seed=wl.sketch_seed(77), variant=VARIANTS[var], replicas=P)
            try:
                plan = sk.plan(n, rounding=rmode, variant=VARIANTS[var], replicas=P)
            except ss.SketchError:
                continue
            ms = _time_ms(lambda: sk.apply_f16acc(A, **kw), reps=3, warm=1)
            got = out[:, cols].float().cpu().numpy().astype(np.float64)
            rows_out.append({"rounding": rname, "requested": var, "variant": plan["variant"], "replicas": plan["replicas"], "ms": ms,
                             "GBps": m * n * 4 / ms / 1e6, "relF_vs_f64_sampled_cols": ev.rel_fro(got, B0)})
    print(json.dumps({"study": "conversion rule x partial-sum placement", "workload": "%s: m=%d n=%d d=%d zeta=%d, N(0,1)" % (args.workload, m, n, d, zeta),
                      "sampled_columns": cols, "rows": rows_out}))
    return 0


def run_graph_study(args):
    """Launch-bound config 1 (256 KiB of A): the complete FP16 and FP32 sketches captured once into a CUDA graph each (the ABI
    neither synchronises nor allocates after the first call) and replayed; per-replay time from events around 200 replays."""
    import torch

    import paper_2606_20195_b200 as ss
    import workloads as wl

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    out = []
    for name in ("c1", "c2"):
        m, n, d, zeta, mseed = WORKLOADS[name]
        A = wl.gaussian_device(m, n, mseed, dev)
        sk = ss.Sketch(m, d, zeta, wl.sketch_seed(0))
        o16 = torch.empty((d, n), dtype=torch.float16, device=dev)
        o32 = torch.empty((d, n), dtype=torch.float32, device=dev)
        row = {"workload": name, "fp16_variant": sk.plan(n, f16=1)["variant"], "fp32_variant": sk.plan(n, f16=0)["variant"]}
        st = torch.cuda.Stream()
        for key, fn in (("fp16", lambda: sk.apply_f16acc(A, out=o16, stream=st)), ("fp32", lambda: sk.apply_f32acc(A, out=o32, stream=st))):
            with torch.cuda.stream(st):
                fn()
                st.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):
                    fn()
                for _ in range(20):
                    g.replay()
                st.synchronize()
                reps = 200
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(st)
                for _ in range(reps):
                    g.replay()
                e1.record(st)
                st.synchronize()
                row[key + "_us_per_replay_warm_L2"] = e0.elapsed_time(e1) / reps * 1e3
        row["fp16_over_fp32"] = row["fp32_us_per_replay_warm_L2"] / row["fp16_us_per_replay_warm_L2"]
        out.append(row)
    print(json.dumps({"study": "CUDA-graph replay of the launch-bound configs (warm L2: back-to-back replays of a 256 KiB / 256 MiB input)", "rows": out}))
    return 0


def run_sustained_study(args):
    """Seconds-long operation (what a caller that streams one 16 GiB matrix after another sees): for c5, e1 and c2,
    --sustained-seconds (default here: 4) of back-to-back complete FP16 sketches of the resident A, rate over the first half
    second, the last second and the whole run, each with the SM / memory clocks, board power and throttle reasons NVML
    reported in that window.  One JSON line; not the driver's bench line."""
    import torch

    import paper_2606_20195_b200 as ss
    import workloads as wl

    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    peaks, peak_src = measured_peaks()
    hbm = float(peaks["hbm_gbs"])
    seconds = args.sustained_seconds if args.sustained_seconds != 2.0 else 4.0
    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(0).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(0, uuid)
    sampler.start()
    rows = []
    for w in ([args.workload] if args.workload != "c5" else ["c5", "e1", "c2"]):
        m, n, d, zeta, mseed = WORKLOADS[w]
        sk = ss.Sketch(m, d, zeta, wl.sketch_seed(0))
        A = wl.gaussian_device(m, n, mseed, dev)
        out = torch.empty((d, n), dtype=torch.float16, device=dev)
        step = lambda: sk.apply_f16acc(A, out=out)
        ms = _time_ms(step, reps=5, warm=3)
        time.sleep(1.0)                                  # start every workload from an idle board
        r = run_sustained(torch, step, ms, seconds, sampler, m * n * 4)
        scale = algorithmic_bytes(m, n, d, 2) / (m * n * 4)
        for key in ("first_half_second", "last_second", "whole"):
            if r[key]:
                r[key]["frac_of_hbm_copy_peak"] = r[key]["GBps"] * scale / hbm
        rows.append(dict(workload=w, variant=sk.plan(n)["variant"], cold_ms=ms, **r))
        sk.close()
        del A, out
        torch.cuda.empty_cache()
    sampler.halt()
    print(json.dumps({"study": "sustained operation: back-to-back complete FP16 sketches for %.1f s per workload" % seconds,
                      "hbm_peak_GBps": hbm, "peak_source": peak_src, "clock_source": sampler.source, "rows": rows}))
    return 0


def self_launch(args):
    """`python bench.py --gpus N` without a torchrun environment: re-run this very command under torch.distributed.run
    with N ranks on this node (one process per GPU, rendezvous on 127.0.0.1), so the line printed carries n_gpus = N only
    when N communicator ranks exist.  NCCL's own INFO lines stay on stderr for whoever wants to count the ranks."""
    import socket

    import torch

    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit("bench.py --gpus %d: this node has %d GPU(s)" % (args.gpus, have))
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "INFO")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus), "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd, env=env)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5", choices=sorted(WORKLOADS))
    ap.add_argument("--variant", default="auto", choices=sorted(VARIANTS))
    ap.add_argument("--replicas", type=int, default=0)
    ap.add_argument("--hash-mode", type=int, default=0)
    ap.add_argument("--tmem-group-mode", type=int, default=0, help="sketch_opts_t.tmem_group_mode (tuning: 0 = auto)")
    ap.add_argument("--study", default=None, choices=["range", "ls", "grid", "graph", "coherence", "replicas", "sustained"],
                    help="extra reports: config-5 range / rounding study; GPU sketch-and-solve least squares; the paper's timing "
                         "grid (PAPER.md:318-322); launch-bound config 1 replayed from a CUDA graph; the U(theta) coherence sweep (PAPER.md:344-352); RN / SR / dither against the number of partial sketches")
    ap.add_argument("--grid", default="full", choices=["full", "quick"], help="--study grid / coherence: every point, or the corners / a small instance")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-pairs", action="store_true", help="skip the like-for-like flat/flat and tmem/tmem FP16-vs-FP32 timings")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-rows", type=int, default=1 << 21, help="rows per step of the reference arm's bounded sample")
    ap.add_argument("--sustained-seconds", type=float, default=2.0, help="length of the back-to-back run behind `sustained` (0 = skip)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                           # timing rule: W >= 3
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.study is None:
        return self_launch(args)
    if args.study == "range":
        return run_range_study(args)
    if args.study == "ls":
        return run_ls_study(args)
    if args.study == "grid":
        return run_grid_study(args)
    if args.study == "graph":
        return run_graph_study(args)
    if args.study == "coherence":
        return run_coherence_study(args)
    if args.study == "replicas":
        return run_replica_study(args)
    if args.study == "sustained":
        return run_sustained_study(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
