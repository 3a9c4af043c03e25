#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native BCFMergesort (arXiv 1306.5076 hot path).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4a] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: bcf_sort of
BASELINE.json config 4 (2^28 uint32 keys, uniform; the configuration the metric's target is quoted
on) -- base-case ShearSort of 2^18 tiles + 18 merge rounds (partition + merge launch each).
Rank 0 prints ONE JSON line (contract in the task statement):
  value     keys/s, device-timed (CUDA events around each bcf_sort call on the launching stream; the
            input is restored from a pristine device copy before each step, outside the events),
            summed over ranks, max-over-ranks time
  e2e       same metric through bcf_sort_host with pinned HOST buffers, H2D + sort + D2H timed
  roofline  the merge kernel (18 of the 37 launches of a step): algorithmic bytes 2*4*n per launch
            over its mean launch duration (CUDA events recorded inside libbcf on the same stream)
            against the measured HBM copy bandwidth of MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle (oracle/, single thread) timed on a bounded sample of the workload
Multi-GPU: the sort does not shard without an exchange step the paper does not have; --gpus N runs N
independent replicas ("replicas only"), one process per GPU under torchrun.
`--impl reference` times the oracle alone (this tier's reference arm).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1306_5076_b200 import workloads  # noqa: E402

METRIC = "sorted keys/sec"
UNIT = "keys/s"
WORKLOADS = {
    # name: (description, log2 n default, generator)
    "cfg4a": ("BCFMergesort of 2^28 uint32 keys, uniform over [0,2^32) (BASELINE.json config 4, uniform)", 28,
              lambda n: workloads.cfg4_sort_u32("uniform", n=n)),
    "cfg4b": ("config 4, already sorted", 28, lambda n: workloads.cfg4_sort_u32("sorted", n=n)),
    "cfg4c": ("config 4, reverse sorted", 28, lambda n: workloads.cfg4_sort_u32("reverse", n=n)),
    "cfg4d": ("config 4, 256 distinct values", 28, lambda n: workloads.cfg4_sort_u32("dup256", n=n)),
    "cfg4e": ("config 4, Zipf(1.1) over [0,2^20)", 28, lambda n: workloads.cfg4_sort_u32("zipf", n=n)),
    "cfg3": ("BCFMergesort of 2^24 uint32 keys, uniform (BASELINE.json config 3)", 24,
             lambda n: workloads.cfg3_sort_u32(n=n)),
}
ORACLE_SAMPLE_LOG2 = 25   # ~15 s of single-thread CPU work


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full capture, or None."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as f:
            return json.load(f).get(kernel)
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "samples": len(sm), "reasons": sorted(reasons)}


def replica_keys(keys, rank):
    """Replicas only: rank r sorts the same recipe, rotated and re-keyed so that no two ranks share
    an input (the multiset differs, the distribution does not)."""
    if rank == 0:
        return keys
    return np.roll(keys, 7919 * rank) ^ np.uint32(rank)


def max_over_ranks(ms, world, device=None):
    """Device time of the step = the slowest rank's (contract: max over ranks)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_reference(args, rank, world):
    """This tier's reference arm: the CPU oracle as it stands, on a bounded sample per step."""
    if rank != 0:
        return
    import oracle
    desc, logn, gen = WORKLOADS[args.workload]
    n_full = 1 << (args.log2n or logn)
    n = min(n_full, 1 << ORACLE_SAMPLE_LOG2)
    keys = gen(n)   # same recipe and stream: the first n draws of the workload
    for _ in range(args.warmup and 1):
        oracle.sort_full(keys[: 1 << 16])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        out = oracle.sort_full(keys)
    dt = time.perf_counter() - t0
    assert np.all(out[:-1] <= out[1:])
    value = n * args.steps / dt
    sample = f"oracle.sort_full (ShearSort 32x32 tiles + two-finger merge rounds) on the first 2^{int(np.log2(n))} keys of the workload, per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": args.workload, "description": desc, "n": n_full, "sample_n": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4a", choices=sorted(WORKLOADS))
    ap.add_argument("--log2n", type=int, default=0, help="override the element count (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if args.steps > 3:
            args.steps = 3           # bounded: each step is ~15 s of CPU
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    import paper_1306_5076_b200 as bcf

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    args.warmup = max(args.warmup, 3)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    desc, logn, gen = WORKLOADS[args.workload]
    n = 1 << (args.log2n or logn)
    # replicas only: every rank sorts its own n keys (rank r draws from variant stream r for cfg3/4a)
    keys = replica_keys(gen(n), rank)
    src = torch.from_numpy(keys.view(np.int32)).to(dev)
    work = torch.empty_like(src)
    ws = torch.empty(bcf.workspace_bytes(bcf.binding.OP_SORT, n), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        work.copy_(src)
        bcf.sort(work, workspace=ws)
    torch.cuda.synchronize()
    out = work.cpu().numpy().view(np.uint32)
    if not np.all(out[:-1] <= out[1:]):
        raise SystemExit("bench: output not sorted")
    del out

    # ---------------- timed region: K steps, device-timed
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sampler = ClockSampler(local_rank)
    bcf.launch_counts()
    bcf.profile_enable(True)
    barrier()
    sampler.start()
    t_wall = time.perf_counter()
    for a, b in ev:
        work.copy_(src)              # restore the unsorted input (outside the events)
        a.record(stream)
        bcf.sort(work, workspace=ws)
        b.record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop()
    prof = bcf.profile_read()
    bcf.profile_enable(False)
    launches = bcf.launch_counts()
    ms = sum(a.elapsed_time(b) for a, b in ev)
    ms = max_over_ranks(ms, world, dev)
    value = world * n * args.steps / (ms * 1e-3)

    # ---------------- roofline of the dominant kernel (merge), same timed region
    peak, peak_src = measured_peak()
    m_ms, m_cnt = prof["merge"]
    rounds = m_cnt // max(args.steps, 1)
    alg_bytes = 2 * 4 * n
    achieved = alg_bytes / (m_ms / m_cnt * 1e-3) / 1e9 if m_cnt else None
    roofline = {
        "kernel": "merge_kernel<u32> (one launch = one merge round: read + write all n keys)",
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak if achieved else None, "traffic": recorded_traffic("merge"),
        "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
        "launches_timed": m_cnt, "mean_launch_ms": m_ms / m_cnt if m_cnt else None,
        "share_of_step": {k: v[0] / ms for k, v in prof.items() if v[1]},
        "whole_sort": {
            "passes": 1 + rounds,
            "frac_of_measured_peak": (1 + rounds) * alg_bytes / (ms / args.steps * 1e-3) / 1e9 / peak,
            "frac_of_nominal_8TBps": (1 + rounds) * alg_bytes / (ms / args.steps * 1e-3) / 1e9 / 8000.0,
        },
    }

    # ---------------- e2e: host buffers through bcf_sort_host, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hsrc = torch.from_numpy(keys.view(np.int32))
        hbuf = torch.empty_like(hsrc).pin_memory()
        scratch = torch.empty(bcf.workspace_bytes(bcf.binding.OP_SORT_HOST, n), dtype=torch.uint8, device=dev)
        e_steps = max(1, min(args.steps, 5))
        e_ms = 0.0
        for i in range(1 + e_steps):
            hbuf.copy_(hsrc)
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            bcf.sort_host(hbuf, scratch=scratch)
            b.record(stream)
            torch.cuda.synchronize()
            if i:
                e_ms += a.elapsed_time(b)
        e_ms = max_over_ranks(e_ms, world, dev)
        e2e = {"value": world * n * e_steps / (e_ms * 1e-3), "unit": UNIT, "steps": e_steps,
               "h2d_bytes_per_step": 4 * n, "d2h_bytes_per_step": 4 * n,
               "api": "bcf_sort_host (pinned host buffer; H2D + sort + D2H + stream sync inside the timed region)"}
        hk = hbuf.numpy().view(np.uint32)
        if not np.all(hk[:-1] <= hk[1:]):
            raise SystemExit("bench: e2e output not sorted")
        del scratch, hbuf

    # ---------------- CPU oracle beside it (rank 0, N = 1 only)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        sn = min(n, 1 << ORACLE_SAMPLE_LOG2)
        sample = keys[:sn].copy()
        t0 = time.perf_counter()
        so = oracle.sort_full(sample)
        dt = time.perf_counter() - t0
        assert np.all(so[:-1] <= so[1:])
        cpu = {"value": sn / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "host_cores_total": os.cpu_count(),
               "sample": f"oracle.sort_full on the first 2^{int(np.log2(sn))} keys of the same workload, once"}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": args.workload, "description": desc, "n": n, "bytes": 4 * n,
                       "passes": 1 + rounds, "multi_gpu": "replicas only",
                       "l2": "input (4*n bytes = 1 GiB at n = 2^28) and workspace are larger than the 126 MB L2; "
                             "the input is restored from a pristine copy before every step",
                       "timing": "CUDA events around each bcf_sort call; restore copy outside the events",
                       "wall_s_timed_region": t_wall},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(sum(launches.values())),
            "launches_by_kernel": launches, "roofline": roofline, "cpu_baseline": cpu,
        }))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
