#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native BCFMergesort (arXiv 1306.5076 hot path).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4a] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: bcf_sort of
BASELINE.json config 4 (2^28 uint32 keys, uniform; the configuration the metric's target is quoted
on) -- base case (default: long tiles of 8192 keys, one CTA of 8 warps each: tile mergesort + 3 on-chip
merge rounds; --base-case shearsort gives the paper's tile ShearSort) + the remaining merge rounds
(partition + merge launch each, one round per pass over HBM unless --rounds-per-pass 2).
Rank 0 prints ONE JSON line (contract in the task statement):
  value     keys/s, device-timed (CUDA events around each bcf_sort call on the launching stream; the
            input is restored from a pristine device copy before each step, outside the events),
            summed over ranks, max-over-ranks time
  e2e       same metric through bcf_sort_host with pinned HOST buffers, H2D + sort + D2H timed
  roofline  the merge kernel (15 of the 31 launches of a step): algorithmic bytes 2*4*n per launch
            over its mean launch duration (CUDA events recorded inside libbcf on the same stream)
            against the measured HBM copy bandwidth of MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle (oracle/, single thread) timed on a bounded sample of the workload
Multi-GPU: the sort does not shard without an exchange step the paper does not have; --gpus N runs N
independent replicas ("replicas only"), one process per GPU under torchrun.
`--impl reference` times the oracle alone (this tier's reference arm).
`other_workloads` holds short device-timed lines for the other BASELINE.json configs and for the same
configs with the other networks / pass structures (paper's ShearSort base case, tile mergesort, two merge
rounds per pass), so the headline never hides what the paper's own base case costs.
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

TILE_ALGO = "shearsort"     # --tile-algo: network bcf_sort_tiles workloads (cfg1, cfg2) run
METRIC = "sorted keys/sec"
UNIT = "keys/s"


def _keys_only(gen):
    return lambda n: (gen(n), None)


# name: (description, default log2 n, generator(n) -> (keys, vals), op, dtype)
#   op = "sort" (bcf_sort), "tiles" (bcf_sort_tiles) or ("merge", k) (bcf_merge_runs on k equal sorted runs)
WORKLOADS = {
    "cfg4a": ("BCFMergesort of 2^28 uint32 keys, uniform over [0,2^32) (BASELINE.json config 4, uniform)", 28,
              _keys_only(lambda n: workloads.cfg4_sort_u32("uniform", n=n)), "sort", "u32"),
    "cfg4b": ("config 4, already sorted", 28, _keys_only(lambda n: workloads.cfg4_sort_u32("sorted", n=n)), "sort", "u32"),
    "cfg4c": ("config 4, reverse sorted", 28, _keys_only(lambda n: workloads.cfg4_sort_u32("reverse", n=n)), "sort", "u32"),
    "cfg4d": ("config 4, 256 distinct values", 28, _keys_only(lambda n: workloads.cfg4_sort_u32("dup256", n=n)), "sort", "u32"),
    "cfg4e": ("config 4, Zipf(1.1) over [0,2^20)", 28, _keys_only(lambda n: workloads.cfg4_sort_u32("zipf", n=n)), "sort", "u32"),
    "cfg3": ("BCFMergesort of 2^24 uint32 keys, uniform (BASELINE.json config 3; fits the L2)", 24,
             _keys_only(lambda n: workloads.cfg3_sort_u32(n=n)), "sort", "u32"),
    "cfg1": ("batch tile sort, 1024 tiles of 32x32 uint32 (BASELINE.json config 1; latency-bound)", 20,
             _keys_only(lambda n: workloads.cfg1_tiles_u32(num_tiles=n // 1024)), "tiles", "u32"),
    "cfg2": ("batch tile sort, 2^16 tiles of (u32 key in [0,16), u32 value = index) (BASELINE.json config 2)", 26,
             lambda n: workloads.cfg2_tiles_u32_u32(num_tiles=n // 1024), "tiles", "u32+u32"),
    "cfg5a": ("key-value BCFMergesort of 2^26 (u64 key, u32 value) pairs (BASELINE.json config 5)", 26,
              lambda n: workloads.cfg5a_sort_u64_u32(n=n), "sort", "u64+u32"),
    "cfg5b2": ("merge-only, 2 sorted uint32 runs totalling 2^27 keys (config 5)", 27, None, ("merge", 2), "u32"),
    "cfg5b64": ("merge-only, 64 sorted uint32 runs totalling 2^27 keys (config 5)", 27, None, ("merge", 64), "u32"),
    "cfg5b1024": ("merge-only, 1024 sorted uint32 runs totalling 2^27 keys (config 5)", 27, None, ("merge", 1024), "u32"),
}
# short device-timed lines beside the headline: every other BASELINE.json config
SIDE_WORKLOADS = ("cfg4b", "cfg4c", "cfg4d", "cfg4e", "cfg5a", "cfg3", "cfg1", "cfg2", "cfg5b2", "cfg5b64", "cfg5b1024")
ORACLE_SAMPLE_LOG2 = 25   # ~6 s of single-thread CPU work


def elem_bytes(dtype):
    return {"u32": 4, "u32+u32": 8, "u64": 8, "u64+u32": 12}[dtype]


def make_input(name, n):
    """(keys, vals, run_len) host arrays of workload `name` at n elements."""
    desc, logn, gen, op, dtype = WORKLOADS[name]
    if isinstance(op, tuple):
        keys, run_len = workloads.cfg5b_merge_runs_u32(op[1], n=n)
        return keys, None, run_len
    keys, vals = gen(n)
    return keys, vals, 0


class Job:
    """One workload resident on the device: restore() the pristine input, run() one step."""

    def __init__(self, bcf, torch, dev, name, n, rank=0):
        desc, logn, gen, op, dtype = WORKLOADS[name]
        self.name, self.desc, self.op, self.dtype, self.n = name, desc, op, dtype, n
        keys, vals, self.run_len = make_input(name, n)
        if rank:
            keys = replica_keys(keys, rank, sorted_runs=self.run_len)
        self.host_keys, self.host_vals = keys, vals
        signed = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}
        self.src_k = torch.from_numpy(keys.view(signed[keys.dtype])).to(dev)
        self.src_v = None if vals is None else torch.from_numpy(vals.view(np.int32)).to(dev)
        self.k = torch.empty_like(self.src_k)
        self.v = None if vals is None else torch.empty_like(self.src_v)
        self.bcf = bcf
        kt = bcf.binding.BCF_KEY_U64 if keys.dtype == np.uint64 else bcf.binding.BCF_KEY_U32
        vt = bcf.binding.BCF_VAL_NONE if vals is None else bcf.binding.BCF_VAL_U32
        if op == "sort":
            need = bcf.workspace_bytes(bcf.binding.OP_SORT, n, kt=kt, vt=vt)
        elif op == "tiles":
            need = 0
        else:
            need = bcf.workspace_bytes(bcf.binding.OP_MERGE_RUNS, n, self.run_len, kt=kt, vt=vt)
            self.out_k = torch.empty_like(self.src_k)
        self.ws = torch.empty(max(need, 16), dtype=torch.uint8, device=dev)
        self.passes = None
        self.opts = None            # bcf_options of this job (None = library defaults)

    def restore(self):
        if self.op in ("sort", "tiles"):
            self.k.copy_(self.src_k)
            if self.v is not None:
                self.v.copy_(self.src_v)

    def run(self):
        b = self.bcf
        if self.op == "sort":
            b.sort(self.k, self.v, workspace=self.ws, opts=self.opts)
        elif self.op == "tiles":
            (b.sort_tiles_mergesort if TILE_ALGO == "mergesort" else b.sort_tiles)(self.k, self.v)
        else:
            b.merge_runs(self.src_k, self.run_len, out_keys=self.out_k, workspace=self.ws, opts=self.opts)

    def result(self):
        return self.out_k if isinstance(self.op, tuple) else self.k

    def check(self):
        """Cheap any-size property of the result (the parity tests do the real comparison)."""
        out = self.result().cpu().numpy().view(self.host_keys.dtype)
        if self.op == "tiles":
            t = out.reshape(-1, 1024)
            ok = bool(np.all(t[:, :-1] <= t[:, 1:]))
        else:
            ok = bool(np.all(out[:-1] <= out[1:]))
        if not ok:
            raise SystemExit(f"bench: output of {self.name} not sorted")
        # the same multiset as the input, by two order-independent checksums (a lost or duplicated key changes them)
        if _multiset_checksum(out) != _multiset_checksum(self.host_keys):
            raise SystemExit(f"bench: output keys of {self.name} are not a permutation of the input")
        if self.host_vals is not None and self.v is not None:
            if _multiset_checksum(self.v.cpu().numpy().view(np.uint32)) != _multiset_checksum(self.host_vals):
                raise SystemExit(f"bench: output values of {self.name} are not a permutation of the input")


def _multiset_checksum(a):
    """(sum mod 2^64, xor) of an unsigned integer array: equal for equal multisets, whatever the order."""
    a = np.ascontiguousarray(a)
    return int(a.sum(dtype=np.uint64)), int(np.bitwise_xor.reduce(a))


def _device_sorted_unsigned(torch, d):
    """d (an int32 / int64 tensor holding unsigned bit patterns) is ascending as UNSIGNED integers: flipping the
    sign bit maps unsigned order onto signed order."""
    flip = d ^ torch.iinfo(d.dtype).min
    return bool((flip[1:] >= flip[:-1]).all().item())


def _device_checksum(torch, d):
    """Order-independent checksums of a device tensor (wrapping 64-bit sums of x and of x * x)."""
    x = d.to(torch.int64)
    return int(x.sum().item()), int((x * x).sum().item())


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


def recorded_bank_conflicts():
    """Shared-memory bank-conflict counters per kernel of the committed ncu capture of THIS build
    (profiles/bank_conflicts.json, written from the ncu CSV by the command named in profiles/r3_launches.md; its `build` entry says which build):
    {kernel: {ld, st, wavefronts_ld, wavefronts_st, excess_per_instruction}}; None when no capture is committed."""
    path = os.path.join(ROOT, "profiles", "bank_conflicts.json")
    try:
        with open(path) as f:
            return json.load(f)
    except Exception:
        return None


class ClockSampler:
    """SM clock and throttle reasons sampled DURING the timed region.  The region lasts well under 100 ms, so
    the samples come from NVML in a thread of this process (a poll every ~2 ms); `nvidia-smi -lms` as a
    second process would not deliver its first line in time."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, index, torch=None):
        self.samples, self.masks, self.smax, self.err = [], [], None, None
        self.stop_flag = threading.Event()
        self.thread = None
        try:
            import pynvml
            self.nv = pynvml
            pynvml.nvmlInit()
            h = None
            try:
                uuid = str(torch.cuda.get_device_properties(index).uuid)
                h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid).encode())
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                ids = [x for x in vis.split(",") if x.strip().isdigit()]
                h = pynvml.nvmlDeviceGetHandleByIndex(int(ids[index]) if index < len(ids) else index)
            self.h = h
            self.smax = float(pynvml.nvmlDeviceGetMaxClockInfo(h, pynvml.NVML_CLOCK_SM))
            self.reasons_fn = getattr(pynvml, "nvmlDeviceGetCurrentClocksEventReasons", None) or \
                getattr(pynvml, "nvmlDeviceGetCurrentClocksThrottleReasons")
        except Exception as e:          # no NVML: the JSON line says so
            self.nv, self.err = None, "NVML unavailable: %s" % type(e).__name__

    def _poll(self):
        nv = self.nv
        while not self.stop_flag.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                self.masks.append(int(self.reasons_fn(self.h)))
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv is not None:
            self.thread = threading.Thread(target=self._poll, daemon=True)
            self.thread.start()

    def stop(self):
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": [self.err]}
        self.stop_flag.set()
        self.thread.join(timeout=2)
        mask = 0
        for m in self.masks:
            mask |= m
        reasons = sorted(name for bit, name in self.REASONS.items() if mask & bit)
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.smax,
                "samples": len(self.samples), "reasons": reasons}


def replica_keys(keys, rank, sorted_runs=0):
    """Replicas only: rank r sorts the same recipe, rotated and re-keyed so that no two ranks share
    an input (the multiset differs, the distribution does not).  Pre-sorted runs stay as they are."""
    if rank == 0 or sorted_runs:
        return keys
    return np.roll(keys, 7919 * rank) ^ keys.dtype.type(rank)


def max_over_ranks(ms, world, device=None):
    """Device time of the step = the slowest rank's (contract: max over ranks)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def oracle_run(name, keys, vals, run_len):
    """The CPU oracle on one host input of workload `name`; returns seconds."""
    import oracle
    op = WORKLOADS[name][3]
    t0 = time.perf_counter()
    if op == "sort":
        out = oracle.sort_full(keys, vals)
    elif op == "tiles":
        out = oracle.shearsort_tiles(keys, vals)
    else:
        out = oracle.merge_runs(keys, run_len)
    dt = time.perf_counter() - t0
    k = out if vals is None else out[0]
    if op != "tiles":
        assert np.all(k[:-1] <= k[1:])
    return dt


def oracle_sample(name, n_full):
    """A bounded sample of the workload for the CPU legs: the first 2^25 elements of the same recipe
    (whole tiles / whole runs), about 5-10 s of single-thread work."""
    op = WORKLOADS[name][3]
    n = min(n_full, 1 << ORACLE_SAMPLE_LOG2)
    keys, vals, run_len = make_input(name, n)
    what = {"sort": "oracle.sort_full (ShearSort 32x32 tiles + two-finger merge rounds)",
            "tiles": "oracle.shearsort_tiles"}.get(op, "oracle.merge_runs (two-finger merge rounds)")
    return keys, vals, run_len, n, f"{what} on the first 2^{int(np.log2(n))} elements of the workload recipe, 1 thread"


def run_reference(args, rank, world):
    """This tier's reference arm: the CPU oracle as it stands, on a bounded sample per step."""
    if rank != 0:
        return
    desc, logn, gen, op, dtype = WORKLOADS[args.workload]
    n_full = 1 << (args.log2n or logn)
    keys, vals, run_len, n, sample = oracle_sample(args.workload, n_full)
    if args.warmup:
        oracle_run(args.workload, keys[: 1 << 12], None if vals is None else vals[: 1 << 12], min(run_len, 1 << 11))
    dt = sum(oracle_run(args.workload, keys, vals, run_len) for _ in range(args.steps))
    value = n * args.steps / dt
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
        "config": {"workload": args.workload, "description": desc, "n": n_full, "sample_n": n},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample + ", per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def time_steps(torch, job, steps, stream, barrier):
    """Device time (ms) of `steps` steps: CUDA events around each call on the launching stream; the
    restore copy of the pristine input is outside the events."""
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    for a, b in ev:
        job.restore()
        a.record(stream)
        job.run()
        b.record(stream)
    barrier()
    return [a.elapsed_time(b) for a, b in ev]


def side_line(bcf, torch, dev, name, stream, barrier, variant=None):
    """A short device-timed measurement of another BASELINE.json config (3 warm-ups, 5 steps).
    variant: None, or a dict of per-call library options / bench settings for this line only
    ({"base_case": .., "rounds_per_pass": .., "launch_mode": .., "tile_algo": .., "label": ..})."""
    global TILE_ALGO
    saved = TILE_ALGO
    if variant:
        TILE_ALGO = variant.get("tile_algo", TILE_ALGO)
    try:
        return _side_line(bcf, torch, dev, name, stream, barrier, variant)
    finally:
        TILE_ALGO = saved


def sort_buckets_lines(bcf, torch, dev, stream):
    """BCFMergesort with the paper's bucket distribution end to end (bcf_sort_buckets, t = P = 128 = the paper's p)
    beside plain bcf_sort on the same 2^27 uint32 keys: uniform keys and keys in {0, 1} (the paper's Fig. 4a case,
    where BCFMergesortPB "has nothing more to do after rearranging the data").  3 warm-ups, 5 steps."""
    n = 1 << 27
    rng = np.random.Generator(np.random.Philox(key=workloads.seed_for(6, 1)))
    inputs = (("uniform keys", workloads.cfg4_sort_u32("uniform", n=n)),
              ("keys in {0, 1}", rng.integers(0, 2, size=n, dtype=np.uint32)))
    peak, _ = measured_peak()
    lines = []
    for dname, keys in inputs:
        src = torch.from_numpy(keys.view(np.int32)).to(dev)
        d = torch.empty_like(src)
        ws_sort = torch.empty(bcf.workspace_bytes(bcf.binding.OP_SORT, n), dtype=torch.uint8, device=dev)
        need = int(bcf.lib().bcf_sort_buckets_workspace_bytes(n, 128, 128, 1, 0))
        ws_b = torch.empty(need, dtype=torch.uint8, device=dev)
        for label, fn in (("bcf_sort (exact co-rank partitioning)", lambda: bcf.sort(d, workspace=ws_sort)),
                          ("bcf_sort_buckets, plain buckets (BCFMergesort)", lambda: bcf.sort_buckets(d, 128, workspace=ws_b)),
                          ("bcf_sort_buckets, pivot buckets (BCFMergesortPB)",
                           lambda: bcf.sort_buckets(d, 128, pivot_buckets=True, workspace=ws_b))):
            for _ in range(3):
                d.copy_(src)
                fn()
            torch.cuda.synchronize()
            # once per variant, after warm-up, for both inputs: sorted as unsigned keys, same multiset as the input
            if not _device_sorted_unsigned(torch, d):
                raise SystemExit("bench: sort_buckets output not sorted (%s, %s)" % (dname, label))
            if _device_checksum(torch, d) != _device_checksum(torch, src):
                raise SystemExit("bench: sort_buckets output is not a permutation of the input (%s, %s)" % (dname, label))
            bcf.launch_counts()
            ms = []
            for _ in range(5):
                d.copy_(src)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                fn()
                e1.record(stream)
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
            launches = bcf.launch_counts()
            t = sum(ms) / len(ms)
            lines.append({"workload": "sort_buckets", "description": "sort of 2^27 uint32 keys, " + dname, "variant": label,
                          "dtype": "u32", "n": n, "value": n / (t * 1e-3), "unit": UNIT, "ms_per_step": t, "best_ms": min(ms),
                          "gpu_launches_per_step": int(sum(launches.values())) // 5})
        del src, d, ws_sort, ws_b
        torch.cuda.empty_cache()
    return lines


def buckets_line(bcf, torch, dev, stream, pivot_buckets, zero_one=False):
    """bcf_find_buckets (Alg. 7; the paper's p = 128): 128 sorted runs totalling 2^27 uint32 keys,
    t = P = 128.  Device-timed, 3 warm-ups, 5 steps (the call allocates nothing inside the timed region
    except through torch's caching allocator, warmed up before)."""
    n, k = 1 << 27, 128
    if zero_one:
        rng = np.random.Generator(np.random.Philox(key=workloads.seed_for(6, 1)))
        keys = workloads.sorted_runs(rng.integers(0, 2, size=n, dtype=np.uint32), n // k)
        run_len = n // k
    else:
        keys, run_len = workloads.cfg5b_merge_runs_u32(k, n=n)
    d = torch.from_numpy(keys.view(np.int32)).to(dev)
    for _ in range(3):
        out = bcf.find_buckets(d, run_len, k, k, pivot_buckets=pivot_buckets)
    torch.cuda.synchronize()
    sizes = out[2].cpu().numpy().view(np.uint32)[::k].astype(np.int64)
    ms = []
    for _ in range(5):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        out = bcf.find_buckets(d, run_len, k, k, pivot_buckets=pivot_buckets)
        e1.record(stream)
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1))
    t = sum(ms) / len(ms)
    peak, _ = measured_peak()
    line = {"workload": "find_buckets", "description": "FIND-BUCKETS (Alg. 7) of 128 sorted uint32 runs totalling 2^27 keys, "
            "t = P = 128" + (", keys in {0, 1}" if zero_one else ", uniform keys"),
            "variant": "pivot buckets" if pivot_buckets else "plain", "dtype": "u32", "n": n, "value": n / (t * 1e-3),
            "unit": UNIT, "ms_per_step": t, "best_ms": min(ms), "passes": 1,
            "frac_of_measured_hbm_peak_for_pass_count": 2 * 4 * n / (t * 1e-3) / 1e9 / peak,
            "largest_bucket": int(np.diff(sizes).max()), "mean_bucket": n / (len(sizes) - 1),
            "sorted_by_distribution_alone": bool((out[0][1:] >= out[0][:-1]).all().item()) if zero_one else None}
    del d, out
    torch.cuda.empty_cache()
    return line


def colored_scan_lines(bcf, torch, dev, stream):
    """bcf_colored_prefix_sums (App. A, Figure 1): 2^28 uint32 values, colours i.i.d. uniform over d,
    for d = 1, 4, 16 and both shared-memory layouts.  Device-timed, 2 warm-ups, 5 steps each.
    Algorithmic bytes: phase 1 reads 5 n, phase 3 reads 5 n and writes 4 n = 14 n."""
    n = 1 << 28
    g = torch.Generator(device=dev)
    g.manual_seed(workloads.seed_for(7, 0))
    vals = torch.randint(-2 ** 31, 2 ** 31 - 1, (n,), dtype=torch.int32, device=dev, generator=g)
    out = torch.empty_like(vals)
    ws = torch.empty(1 << 21, dtype=torch.uint8, device=dev)
    peak, _ = measured_peak()
    lines = []
    for d in (1, 4, 16):
        cols = torch.randint(0, d, (n,), dtype=torch.uint8, device=dev, generator=g)
        for layout, lname in ((bcf.SCAN_BANK_PER_THREAD, "bank per thread (conflict-free)"),
                              (bcf.SCAN_THREAD_MAJOR, "thread-major (the layout the paper starts from)")):
            for _ in range(2):
                bcf.colored_prefix_sums(vals, cols, d, layout=layout, out=out, workspace=ws)
            ms = []
            for _ in range(5):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                bcf.colored_prefix_sums(vals, cols, d, layout=layout, out=out, workspace=ws)
                e1.record(stream)
                torch.cuda.synchronize()
                ms.append(e0.elapsed_time(e1))
            t = sum(ms) / len(ms)
            lines.append({"workload": "colored_prefix_sums", "description": "coloured prefix sums of 2^28 uint32 values, "
                          "%d colours (PAPER.md App. A)" % d, "variant": lname, "dtype": "u32", "n": n, "colors": d,
                          "value": n / (t * 1e-3), "unit": "elements/s", "ms_per_step": t, "best_ms": min(ms), "passes": 2,
                          "frac_of_measured_hbm_peak_for_pass_count": 14 * n / (t * 1e-3) / 1e9 / peak})
        del cols
    del vals, out, ws
    torch.cuda.empty_cache()
    return lines


# comparators per element of the two tile networks (include/bcf.h): ShearSort = 11 line sorts x 191 comparators per
# 32-element line; tile mergesort = 831 comparators per thread per tile of 32 x 32
TILE_COMPARATORS_PER_ELEMENT = {"shearsort": 11 * 191 / 32, "mergesort": 831 / 32}
# ALU-pipe instructions per comparator, from the SASS: u32 = VIMNMX min + max = 2; two planes = 2 subtract-with-
# borrow (IADD3 / IADD3.X into a predicate) + 3 SEL = 5 (the fourth output is formed with 2 IMADs on the FMA
# pipe, BCF_CE2_FMA_PLANES = 1); three planes = 3 + 6 SEL = 9
ALU_OPS_PER_COMPARATOR = {"u32": 2, "u32+u32": 5, "u64": 5, "u64+u32": 9}


def alu_roofline(dtype, n, tile_algo, launch_ms, sm_max_mhz=None):
    """SURVEY.md 8(d)'s second ceiling for the batch tile sorts (configs 1-2): ALU-pipe instructions the network
    issues (comparators x instructions per comparator, as built) over the launch's event time, against
    148 SMs x 64 integer lanes per clock x the SM's maximum clock."""
    sm_mhz = sm_max_mhz or 1965.0
    ops = n * TILE_COMPARATORS_PER_ELEMENT[tile_algo] * ALU_OPS_PER_COMPARATOR[dtype]
    peak_ops = 148 * 64 * sm_mhz * 1e6
    ach = ops / (launch_ms * 1e-3)
    kernel = "tile_sort_kernel (ShearSort)" if tile_algo == "shearsort" else "tile_mergesort_kernel"
    return {"kernel": kernel + ", one launch = all tiles", "bound": "alu", "achieved": ach / 1e12, "peak": peak_ops / 1e12,
            "unit": "T int-op/s", "frac": ach / peak_ops,
            "alu_ops_per_element": TILE_COMPARATORS_PER_ELEMENT[tile_algo] * ALU_OPS_PER_COMPARATOR[dtype],
            "peak_source": "148 SMs x 64 integer min/max lanes per clk x SM max clock %.0f MHz (DESIGN.md 5.1)" % sm_mhz}


def _side_line(bcf, torch, dev, name, stream, barrier, variant):
    desc, logn, gen, op, dtype = WORKLOADS[name]
    n = 1 << logn
    job = Job(bcf, torch, dev, name, n)
    if variant:
        o = {k: variant[k] for k in ("base_case", "rounds_per_pass", "launch_mode", "merge_impl") if k in variant}
        job.opts = bcf.options(**o) if o else None
    for _ in range(3):
        job.restore()
        job.run()
    torch.cuda.synchronize()
    job.check()
    bcf.launch_counts()
    ms = time_steps(torch, job, 5, stream, barrier)
    launches = bcf.launch_counts()
    t = sum(ms) / len(ms)
    rounds = (launches["merge"] + launches["merge_pagewise"]) // 5
    passes = rounds + (0 if isinstance(op, tuple) else 1)
    bytes_moved = passes * 2 * elem_bytes(dtype) * n
    peak, _ = measured_peak()
    line = {"workload": name, "description": desc, "dtype": dtype, "n": n, "value": n / (t * 1e-3), "unit": UNIT,
            "ms_per_step": t, "best_ms": min(ms), "passes": passes,
            "frac_of_measured_hbm_peak_for_pass_count": bytes_moved / (t * 1e-3) / 1e9 / peak,
            "gpu_launches_per_step": int(sum(launches.values())) // 5}
    if op == "tiles":      # one launch per step: the step's event time is the launch's
        line["alu_roofline"] = alu_roofline(dtype, n, TILE_ALGO, t)
    if variant:
        line["variant"] = variant.get("label", "")
    del job
    torch.cuda.empty_cache()
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4a", choices=sorted(WORKLOADS))
    ap.add_argument("--log2n", type=int, default=0, help="override the element count (debugging only)")
    ap.add_argument("--base-case", default="auto", choices=["auto", "shearsort", "tilemergesort", "longtiles"],
                    help="base case of bcf_sort: the paper's tile ShearSort, the tile mergesort network, long tiles "
                         "(8 tiles per CTA), or auto = the library default (long tiles for u32 keys, tile mergesort else)")
    ap.add_argument("--rounds-per-pass", type=int, default=0, choices=[0, 1, 2],
                    help="merge rounds per pass over global memory (2 = four-run kernel, 0 = the library default)")
    ap.add_argument("--launch-mode", default="auto", choices=["auto", "plain", "pdl"],
                    help="ordinary or programmatic dependent launches (auto = the library default)")
    ap.add_argument("--tile-algo", default="shearsort", choices=["shearsort", "mergesort"],
                    help="network for the batch tile sort workloads cfg1 / cfg2")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip the short lines for the other configs")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        if args.steps > 3:
            args.steps = 3           # bounded: each step is several seconds of CPU
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

    global TILE_ALGO
    TILE_ALGO = args.tile_algo
    main_opts = bcf.options(base_case={"shearsort": bcf.BASE_SHEARSORT, "tilemergesort": bcf.BASE_TILE_MERGESORT,
                                       "longtiles": bcf.BASE_LONG_TILES, "auto": bcf.BASE_AUTO}[args.base_case],
                            rounds_per_pass=args.rounds_per_pass,
                            launch_mode={"auto": bcf.LAUNCH_AUTO, "plain": bcf.LAUNCH_PLAIN, "pdl": bcf.LAUNCH_PDL}[args.launch_mode])

    desc, logn, gen, op, dtype = WORKLOADS[args.workload]
    n = 1 << (args.log2n or logn)
    eb = elem_bytes(dtype)
    # replicas only: every rank works on its own n elements of the same recipe
    job = Job(bcf, torch, dev, args.workload, n, rank)
    job.opts = main_opts
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        job.restore()
        job.run()
    torch.cuda.synchronize()
    job.check()

    # ---------------- timed region: K steps, device-timed
    sampler = ClockSampler(local_rank, torch)
    bcf.launch_counts()
    bcf.profile_enable(True)
    sampler.start()
    t_wall = time.perf_counter()
    step_ms = time_steps(torch, job, args.steps, stream, barrier)
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop()
    prof = bcf.profile_read()
    if bcf.profile_dropped():
        raise SystemExit("bench: the library's event pool overflowed (%d launches not timed): use fewer --steps"
                         % bcf.profile_dropped())
    bcf.profile_enable(False)
    launches = bcf.launch_counts()
    ms = max_over_ranks(sum(step_ms), world, dev)
    value = world * n * args.steps / (ms * 1e-3)

    # ---------------- roofline of the dominant kernel, same timed region
    peak, peak_src = measured_peak()
    dom = max((k for k in prof if prof[k][1]), key=lambda k: prof[k][0])
    d_ms, d_cnt = prof[dom]
    rounds = (prof["merge"][1] + prof["merge_pagewise"][1]) // max(args.steps, 1)
    passes = rounds + (0 if isinstance(op, tuple) else 1)
    alg_bytes = 2 * eb * n
    share = {k: v[0] / ms for k, v in prof.items() if v[1]}
    if dom == "tile_sort" and op == "tiles":
        # ALU-bound: 11 line sorts x 191 comparators x 2 min/max per 32 u32 keys,
        # integer min/max issue at 64 lanes / clk / SM.
        roofline = alu_roofline(dtype, n, TILE_ALGO, d_ms / d_cnt, clocks.get("sm_max_mhz"))
        roofline.update({"traffic": recorded_traffic("tile_sort_shearsort_cfg2") if args.workload == "cfg2" and TILE_ALGO == "shearsort" else None, "launches_timed": d_cnt, "mean_launch_ms": d_ms / d_cnt,
                         "share_of_step": share})
    else:
        m_ms, m_cnt = prof["merge"]
        achieved = alg_bytes / (m_ms / m_cnt * 1e-3) / 1e9 if m_cnt else None
        roofline = {
            "kernel": "merge kernel (one launch = one merge round: read + write all n elements)",
            "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
            "frac": achieved / peak if achieved else None, "traffic": recorded_traffic("merge"),
            "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
            "launches_timed": m_cnt, "mean_launch_ms": m_ms / m_cnt if m_cnt else None,
            "share_of_step": share,
            "whole_step": {
                "passes": passes,
                "frac_of_measured_peak": passes * alg_bytes / (ms / args.steps * 1e-3) / 1e9 / peak,
                "frac_of_nominal_8TBps": passes * alg_bytes / (ms / args.steps * 1e-3) / 1e9 / 8000.0,
            },
        }

    # ---------------- e2e: host buffers through bcf_sort_host, copies inside the timed region
    e2e = None
    if not args.no_e2e and op == "sort":
        hk_src = torch.from_numpy(job.host_keys.view(np.int64 if job.host_keys.dtype == np.uint64 else np.int32))
        hk = torch.empty_like(hk_src).pin_memory()
        hv_src = None if job.host_vals is None else torch.from_numpy(job.host_vals.view(np.int32))
        hv = None if hv_src is None else torch.empty_like(hv_src).pin_memory()
        kt = bcf.binding.BCF_KEY_U64 if job.host_keys.dtype == np.uint64 else bcf.binding.BCF_KEY_U32
        vt = bcf.binding.BCF_VAL_NONE if hv is None else bcf.binding.BCF_VAL_U32
        scratch = torch.empty(bcf.workspace_bytes(bcf.binding.OP_SORT_HOST, n, kt=kt, vt=vt), dtype=torch.uint8, device=dev)
        e_steps = max(1, min(args.steps, 5))
        e_ms = 0.0
        for i in range(1 + e_steps):
            hk.copy_(hk_src)
            if hv is not None:
                hv.copy_(hv_src)
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            bcf.sort_host(hk, hv, scratch=scratch, opts=main_opts)
            b.record(stream)
            torch.cuda.synchronize()
            if i:
                e_ms += a.elapsed_time(b)
        e_ms = max_over_ranks(e_ms, world, dev)
        e2e = {"value": world * n * e_steps / (e_ms * 1e-3), "unit": UNIT, "steps": e_steps,
               "h2d_bytes_per_step": eb * n, "d2h_bytes_per_step": eb * n,
               "api": "bcf_sort_host (pinned host buffers; H2D + sort + D2H + stream sync inside the timed region)"}
        out = hk.numpy().view(job.host_keys.dtype)
        if not np.all(out[:-1] <= out[1:]):
            raise SystemExit("bench: e2e output not sorted")
        del scratch, hk, hv

    # ---------------- CPU oracle beside it, and the other configs (rank 0, N = 1 only)
    cpu = None
    side = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        keys, vals, run_len, sn, sample = oracle_sample(args.workload, n)
        dt = oracle_run(args.workload, keys, vals, run_len)
        cpu = {"value": sn / dt, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": dt,
               "host_cores_total": os.cpu_count(), "sample": sample + ", once"}
        if op == "sort" and vals is None:
            # context only: a textbook library sort on the same sample (numpy's default sort, one thread)
            t0 = time.perf_counter()
            np.sort(keys)
            cpu["textbook_sort"] = {"what": "numpy.sort on the same sample, 1 thread", "value": sn / (time.perf_counter() - t0), "unit": UNIT}
    summary = None
    kv = None
    if rank == 0 and world == 1 and not args.no_side and args.workload == "cfg4a" and not args.log2n:
        del job
        torch.cuda.empty_cache()
        side = [side_line(bcf, torch, dev, w, stream, barrier) for w in SIDE_WORKLOADS]
        # the same configs with the other networks / pass structures the library offers
        for v in ({"base_case": bcf.BASE_SHEARSORT, "rounds_per_pass": 1, "label": "base case = the paper's tile ShearSort, one round per pass"},
                  {"base_case": bcf.BASE_TILE_MERGESORT, "rounds_per_pass": 1, "label": "base case = tile mergesort (one tile per warp), one round per pass"},
                  {"rounds_per_pass": 1, "label": "one merge round per pass (two-run kernel)"},
                  {"rounds_per_pass": 2, "label": "two merge rounds per pass (four-run kernel)"},
                  {"launch_mode": bcf.LAUNCH_PLAIN, "label": "ordinary launches"},
                  {"launch_mode": bcf.LAUNCH_PDL, "label": "programmatic dependent launches"}):
            side.append(side_line(bcf, torch, dev, "cfg4a", stream, barrier, v))
        side.append(side_line(bcf, torch, dev, "cfg1", stream, barrier, {"tile_algo": "mergesort", "label": "bcf_sort_tiles_mergesort"}))
        side.append(side_line(bcf, torch, dev, "cfg2", stream, barrier, {"tile_algo": "mergesort", "label": "bcf_sort_tiles_mergesort"}))
        side.append(buckets_line(bcf, torch, dev, stream, False))
        side.append(buckets_line(bcf, torch, dev, stream, True))
        side.append(buckets_line(bcf, torch, dev, stream, True, zero_one=True))
        side.extend(sort_buckets_lines(bcf, torch, dev, stream))
        side.extend(colored_scan_lines(bcf, torch, dev, stream))
        # every BASELINE.json config at a glance: G keys/s and fraction of the measured HBM peak for its pass count
        summary = {args.workload: [round(value / 1e9, 2), round(roofline.get("whole_step", {}).get("frac_of_measured_peak", 0.0), 3)]}
        for ln in side:
            if ln["workload"] in SIDE_WORKLOADS and "variant" not in ln:
                summary[ln["workload"]] = [round(ln["value"] / 1e9, 2), round(ln["frac_of_measured_hbm_peak_for_pass_count"], 3)]
                if "alu_roofline" in ln:    # configs 1-2: also the fraction of the ALU ceiling (third entry)
                    summary[ln["workload"]].append(round(ln["alu_roofline"]["frac"], 3))
        kv5a = next(ln for ln in side if ln["workload"] == "cfg5a" and "variant" not in ln)
        kv = {"workload": "cfg5a", "dtype": kv5a["dtype"], "n": kv5a["n"], "value": kv5a["value"], "unit": UNIT,
              "ms_per_step": kv5a["ms_per_step"], "passes": kv5a["passes"],
              "frac_of_measured_hbm_peak_for_pass_count": kv5a["frac_of_measured_hbm_peak_for_pass_count"]}

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
            "summary_gkeys_per_s_and_frac_of_hbm_peak": summary,
            "config": {"workload": args.workload, "description": desc, "n": n, "bytes": eb * n,
                       "passes": passes,
                       "base_case": None if op != "sort" else (args.base_case if args.base_case != "auto" else
                                                               "auto: " + ("longtiles" if dtype == "u32" else "tilemergesort")),
                       "tile_network": args.tile_algo if op == "tiles" else None,
                       "merge_rounds_per_pass": args.rounds_per_pass or "library default", "launch_mode": args.launch_mode,
                       "multi_gpu": "replicas only",
                       "kv": kv,
                       "l2": "input and workspace (%d MiB each) %s the 126 MB L2; the input is restored from a "
                             "pristine copy before every step" % (eb * n >> 20, "exceed" if eb * n > 126e6 else "FIT IN"),
                       "timing": "CUDA events around each library call; restore copy outside the events",
                       "best_step_ms": min(step_ms), "wall_s_timed_region": t_wall},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(sum(launches.values())),
            "launches_by_kernel": launches, "profile_launches_not_timed": bcf.profile_dropped(),
            "roofline": roofline, "bank_conflicts": recorded_bank_conflicts(), "cpu_baseline": cpu,
            "other_workloads": side,
        }))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
