#!/usr/bin/env python
"""bench.py -- PLIC solves per second on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--log2n 26]

Workload (config.workload): BASELINE.json configs[1] -- N = 2^26 cells, fp32 SoA, seed 1,
normals uniform on the unit sphere, V0 ~ U[0,1) (gen.random_sphere).  1.07 GB in + 0.27 GB
out per launch, far larger than the 126 MB L2, so consecutive steps cannot hit in cache.

A step is one plic_solve launch over the whole batch: load, mirror/sort, volume reduction,
case selection, per-case solve, sign restore, store with one
method.  All eight method variants and plic_volume (row a7) are timed the same way in the
same run (W warm-up + K timed launches each, CUDA events on the launching stream) and listed
under "methods"; the headline `value` is the fastest variant that the parity tests hold to
the 2e-5 bound -- all of them are, see tests/test_parity_gpu.py -- named in config.method.
`value` is taken in the sustained regime (300 ms of load before the first timed region; on this
pool a software power cap then holds the SM clocks at 1.5-1.85 GHz); "burst" repeats the headline
variant after 0.5 s of idle, at full clocks -- the regime MEASURED_PEAKS.json's copy bandwidth
was taken in.

Per method: `hbm_frac` against the measured copy bandwidth and `hbm_frac_nominal`
against 8 TB/s; `issue_frac` = issue slots per cell x cells/s / (SMs x 4 sub-partitions x the SM
clock sampled in that method's timed window), issue slots = warp-instructions (ncu's executed count)
+ packed fp32x2 warp-instructions (they hold the issue port for two clocks, see pipe_rates), both per
cell from the committed table profiles/instruction_counts.txt; `bound` names the larger fraction;
`issue_frac_algorithmic` is the same from SURVEY.md 8d's algorithmic operation counts (union of all case
paths) against SMs x 128 FP32 lanes x clock; `per_launch` = median and best of 20 further launches, each
between its own pair of events (2-3 % above ms_per_step: an event between two launches keeps the second
from becoming resident while the first drains).  "stream_ceiling" is the
same 4-read/1-write stream with no arithmetic (plic_solve with the blank method, d0 = V0 - 1/2);
"pipe_rates" are the instruction rates of the FMA, SFU and ALU pipes measured in this run
(plic_pipe_probe), from which the "alu" peak of the compute-bound legs is derived.

Other configs of BASELINE.json, each timed like the headline (none is part of `value`):
"divergence" = configs[2], 2^26 case-stratified cells labelled by the ORACLE (oracle.stratified:
rejection sampling on the oracle's classifier, V0 by the oracle's forward map), interleaved
(case = i mod 5: every warp holds all five cases) vs five contiguous blocks, all 8 variants;
"config4" = configs[3], 2^28 cells, half the normals snapped to an axis or face diagonal,
V0 ~ Beta(1/2,1/2) (gen.snapped_beta), all 8 variants; "curvature" = plic_curvature on configs[4]
(256^3 lattice, sphere R = 60), rotating over three copies of the lattice so that no call finds its
input in L2, with the curvature oracle beside it, and ("large") the same call on the 400 x 400 x 340
lattice of the paper's raindrop run holding a sphere of radius 120.  "paper_benchmark" is the paper's own benchmark
shape (sect. 2.6, Table 3) through plic_roundtrip_error: 2^k normals x L = 256 volumes in series per
thread, blank run (eq. 33) subtracted, ps per PLIC evaluation and E_avg (eq. 32) per method --
compute bound, for comparison with the paper's Titan Xp column (context, not the target).
"storage" lists the fp16-storage and fp64 variants of the solve.

"e2e" is the same metric through plic_solve_host with pinned HOST buffers (H2D and D2H copies
inside the timed region), next to the PCIe link's nominal and measured rates.  "cpu_baseline" /
"cpu_baseline_1core" time the fp64 oracle on all host threads / one thread.

Multi-GPU: the path has no exchange step, so rank r solves its own 2^26 cells
[r 2^26, (r+1) 2^26) of the same seeded stream, no data-path collective; `value` = all ranks'
cells / max-over-ranks time ("scaling": "weak").  Under torchrun the ranks come from the
environment; a plain `python bench.py --gpus N` (N > 1) re-launches itself under
torch.distributed.run with N ranks on 127.0.0.1.

Output: stdout carries ONE line, the compact contract line (compact_line: under 8000 bytes -- the
contract keys, `roofline`, `cpu_baseline`, `e2e`, `clocks` and a per-variant `summary`).  The full
object with every variant of every leg ("methods", "storage", "pipe_rates", "paper_benchmark",
"divergence", "config4"; 30+ KB) is written to --detail-out (default bench_detail.json, git-ignored).

--impl reference times the fp64 CPU oracle (oracle/), as it stands, on the host cores.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "plic_solves_per_second"
UNIT = "Gcells/s"
BYTES_PER_CELL = 20                      # 4 fp32 read + 1 fp32 written
WORKLOAD = "configs[1]: N=2^%d cells, fp32 SoA, seed 1, normals uniform on sphere, V0~U[0,1)"
SEED = 1
FALLBACK_HBM_GBS = 6650.0                # B200_PROFILING.md fallback


# ------------------------------------------------------------------------------------------
# distributed helpers (also exercised on CPU with gloo by tests/test_shard_gloo.py)
# ------------------------------------------------------------------------------------------
def rank_cells(per_rank: int, rank: int):
    """Weak scaling: rank r owns cells [r*per_rank, (r+1)*per_rank) of the seeded stream."""
    return rank * per_rank, (rank + 1) * per_rank


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def max_over_ranks(x: float, device="cuda") -> float:
    dist = _dist()
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device="cuda") -> float:
    dist = _dist()
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def barrier():
    dist = _dist()
    if dist is not None:
        dist.barrier()


# ------------------------------------------------------------------------------------------
# clocks: NVML sampled from a thread during the timed regions
# ------------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, torch_device_index: int, period_s: float = 0.004):
        self.samples = []          # (t, sm_mhz, reasons bitmask, power W)
        self.period = period_s
        self.ok = False
        self.sm_max = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            uuid = str(torch.cuda.get_device_properties(torch_device_index).uuid)
            if not uuid.startswith("GPU-"):
                uuid = "GPU-" + uuid
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
                idx = int(vis.split(",")[torch_device_index]) if vis and vis.split(",")[0].isdigit() \
                    else torch_device_index
                self.h = pynvml.nvmlDeviceGetHandleByIndex(idx)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:      # noqa: BLE001
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                sm = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                try:
                    pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                except Exception:
                    pw = None
                self.samples.append((time.perf_counter(), int(sm), int(rs), pw))
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.ok:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join(timeout=2.0)

    def summary(self, windows):
        """Median SM clock and the union of event reasons over samples inside `windows`
        (list of (t0, t1) perf_counter intervals = the timed regions)."""
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0,
                    "note": "NVML unavailable: %s" % getattr(self, "err", "?")}
        ins = [s for s in self.samples if any(a <= s[0] <= b for a, b in windows)]
        note = "NVML samples inside the timed regions"
        if len(ins) < 3:           # regions shorter than the sampling period: widen to the phase
            lo = min(a for a, _ in windows) - 0.05
            hi = max(b for _, b in windows) + 0.05
            ins = [s for s in self.samples if lo <= s[0] <= hi]
            note = "NVML samples over the whole timing phase (regions shorter than the sampler period)"
        if not ins:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "samples": 0, "note": note}
        clocks = sorted(s[1] for s in ins)
        mask = 0
        for s in ins:
            mask |= s[2]
        reasons = [name for bit, name in self.REASONS.items() if mask & bit]
        pw = [s[3] for s in ins if s[3] is not None]
        return {"sm_mhz": clocks[len(clocks) // 2], "sm_min_mhz": clocks[0], "sm_max_mhz": self.sm_max,
                "sm_mean_mhz": round(sum(clocks) / len(clocks), 1), "sm_top_mhz": clocks[-1],
                "reasons": reasons, "samples": len(ins), "power_w_max": max(pw) if pw else None,
                "note": note}


# ------------------------------------------------------------------------------------------
# the oracle leg (cpu_baseline and --impl reference)
# ------------------------------------------------------------------------------------------
def oracle_rate(arrays, n_cells: int, threads: int = 0):
    """Times oracle.solve on the first n_cells of the workload; returns (cells/s, seconds)."""
    import oracle
    sub = [a[:n_cells] for a in arrays]
    t0 = time.perf_counter()
    oracle.solve(*sub, threads=threads)
    dt = time.perf_counter() - t0
    return n_cells / dt, dt


def cpu_baseline(arrays, budget_s: float = 12.0, threads: int = 0):
    """The oracle as it stands on all host threads (threads=0) or on `threads` of them, for about
    budget_s seconds: a prefix of the workload sized from a calibration pass, repeated when the
    whole workload takes less."""
    import oracle
    all_threads = oracle.max_threads()       # before any call that lowers the OpenMP thread count
    N = arrays[0].shape[0]
    cal = min(N, 1 << (20 if threads == 0 else 16))
    rate, _ = oracle_rate(arrays, cal, threads)              # calibration (also warms the .so)
    n = int(min(N, max(cal, rate * budget_s)))
    passes, cells, secs = 0, 0, 0.0
    while passes == 0 or (secs < 0.8 * budget_s and passes < 64):
        _, dt = oracle_rate(arrays, n, threads)
        passes, cells, secs = passes + 1, cells + n, secs + dt
    cores = all_threads if threads == 0 else threads
    oracle.solve(arrays[0][:1], arrays[1][:1], arrays[2][:1], arrays[3][:1], threads=all_threads)   # restore
    return {"value": cells / secs / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "first %d cells of the workload x %d passes (%.1f s of fp64 bisection, %s)" % (
                n, passes, secs, "all host threads" if threads == 0 else "%d thread(s)" % threads)}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import gen
    import oracle
    N = 1 << args.log2n
    cal_n = 1 << 20
    arrays = gen.random_sphere(min(N, 1 << 24), SEED)
    rate, _ = oracle_rate(arrays, cal_n)
    # each step: a bounded sample so that (K + W) steps end within ~2 minutes
    per_step_s = max(0.25, min(4.0, 120.0 / max(1, args.steps + args.warmup)))
    n = int(min(arrays[0].shape[0], max(cal_n, rate * per_step_s)))
    for _ in range(args.warmup):
        oracle_rate(arrays, n)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_rate(arrays, n)
    dt = time.perf_counter() - t0
    value = n * args.steps / dt / 1e9
    sample = "each step = oracle.solve on the first %d cells of the workload" % n
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": WORKLOAD % args.log2n, "method": "oracle: fp64 forward map + bisection",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.max_threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------
NOMINAL_HBM_GBS = 8000.0                 # "the nominal 8 TB/s"


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs: torch copy, best of 10)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


def profile_table(name):
    """Rows of a committed profiles/*.txt table: {first column: [other columns]}; '#' lines are
    comments, a '#@ key value' line is metadata returned under '@key'."""
    rows = {}
    try:
        with open(os.path.join(ROOT, "profiles", name)) as f:
            for line in f:
                parts = line.split()
                if not parts:
                    continue
                if parts[0] == "#@" and len(parts) >= 3:
                    rows["@" + parts[1]] = parts[2:]
                elif not parts[0].startswith("#"):
                    rows[parts[0]] = parts[1:]
    except Exception:
        pass
    return rows


def csrc_digest():
    """sha1 (12 hex digits) over the kernel sources with comments and white space removed: the
    committed ncu tables carry the digest they were captured at, so a table that no longer matches
    the kernels' code is reported as stale instead of silently reused."""
    import glob
    import hashlib
    import re
    h = hashlib.sha1()
    src = os.path.join(ROOT, "paper_2006_12838_b200", "csrc")
    for f in sorted(glob.glob(os.path.join(src, "*.cu")) + glob.glob(os.path.join(src, "*.cuh"))):
        with open(f, "r", encoding="utf-8", errors="replace") as fh:
            code = re.sub(r"/\*.*?\*/", "", fh.read(), flags=re.S)
        code = re.sub(r"//[^\n]*", "", code)
        h.update(os.path.basename(f).encode() + b"\0" + re.sub(r"\s+", "", code).encode())
    return h.hexdigest()[:12]


def table_is_stale(table):
    return table.get("@csrc_sha1", ["?"])[0] != csrc_digest()


def ncu_traffic(kernel_name, cells):
    """(dram bytes per launch, provenance) of `kernel_name` from the committed ncu capture -- only
    when that capture was taken on the same number of cells, else (None, why)."""
    t = profile_table("dram_traffic.txt")
    row = t.get(kernel_name)
    cap_cells = int(t.get("@cells", ["0"])[0])
    src = "profiles/dram_traffic.txt (ncu --set full, commit %s, %d cells per launch%s)" % (
        t.get("@commit", ["?"])[0], cap_cells,
        "; STALE: the kernel sources changed since this capture" if table_is_stale(t) else "")
    if row is None:
        return None, "no ncu capture of this kernel in profiles/dram_traffic.txt"
    if cap_cells != cells:
        return None, "ncu capture is for %d cells per launch, this run uses %d" % (cap_cells, cells)
    return float(row[0]), src


def time_launches(fn, steps, warmup, stream):
    """W untimed + K timed calls of fn() on `stream`; barrier + synchronize on both sides;
    device time from CUDA events recorded on that stream.  Returns (ms total, (t0, t1) host window)."""
    import torch
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    barrier()
    torch.cuda.synchronize()
    e0 = torch.cuda.Event(enable_timing=True)
    e1 = torch.cuda.Event(enable_timing=True)
    w0 = time.perf_counter()
    e0.record(stream)
    for _ in range(steps):
        fn()
    e1.record(stream)
    torch.cuda.synchronize()
    barrier()
    torch.cuda.synchronize()
    w1 = time.perf_counter()
    return e0.elapsed_time(e1), (w0, w1)


def pcie_link(sampler):
    """Nominal PCIe rate of the GPU's link from NVML (GB/s per direction), or None."""
    try:
        nv, h = sampler.nv, sampler.h
        gen_, width = nv.nvmlDeviceGetCurrPcieLinkGeneration(h), nv.nvmlDeviceGetCurrPcieLinkWidth(h)
        per_lane = {1: 0.25, 2: 0.5, 3: 0.985, 4: 1.969, 5: 3.938, 6: 7.563}.get(int(gen_))
        return {"gen": int(gen_), "width": int(width), "nominal_gbs_per_direction": per_lane * width if per_lane else None}
    except Exception:
        return None


def per_launch_stats(fn, n, stream):
    """Median and best of n single launches, each bracketed by its own pair of CUDA events (SURVEY.md
    8d, "Timing": median and best).  Separate from the timed region of `value`: an event between two
    launches keeps the second from becoming resident while the first drains."""
    import torch
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(n + 1)]
    ev[0].record(stream)
    for i in range(n):
        fn()
        ev[i + 1].record(stream)
    torch.cuda.synchronize()
    t = sorted(ev[i].elapsed_time(ev[i + 1]) for i in range(n))
    return {"n": n, "median_ms": t[n // 2], "best_ms": t[0]}


VARIANTS = [(m, f) for f in (True, False) for m in ("analytic", "sz", "newton", "nested")]
# SURVEY.md 8d, "Algorithmic work per cell": FP32 + SFU operations of the union of all case paths
ALGORITHMIC_INST = {"analytic": 95 + 7, "sz": 95 + 7, "newton": 105 + 8, "nested": 190 + 3}


def time_variants(plic, arrays, out, steps, warmup, stream, world, sampler, sms, counts, peak, workload="configs[1]"):
    """Times the eight plic_solve variants on `arrays`; one dict per variant with both HBM fractions,
    the issue fraction at the clock sampled in its own window, and the binding roofline.  `workload`
    names the arrays (configs[k]): executed-instruction counts of the data-dependent kernels are used
    only when profiles/instruction_counts.txt was captured on that workload."""
    N = arrays[0].numel()
    res = {}
    for m, f in VARIANTS:
        name = plic.plic_method_name(plic.method_id(m, f))
        c0 = plic.plic_launch_count()
        ms, win = time_launches(lambda: plic.plic_solve(*arrays, out=out, method=m, fast=f), steps, warmup, stream)
        # kernels per timed step x steps (a call with a misaligned head or a ragged tail is two launches)
        launches = (plic.plic_launch_count() - c0) * steps // (steps + warmup)
        ms = max_over_ranks(ms) / steps
        clk = sampler.summary([win])
        gbs = BYTES_PER_CELL * N / (ms * 1e-3) / 1e9
        e = {"value": N * world / (ms * 1e-3) / 1e9, "ms_per_step": ms, "launches": launches,
             "bytes_per_cell": BYTES_PER_CELL, "hbm_gbs_per_gpu": gbs, "hbm_frac": gbs / peak,
             "hbm_frac_nominal": gbs / NOMINAL_HBM_GBS, "sm_mhz": clk.get("sm_mhz")}
        e["roofline_frac"] = e["hbm_frac"]
        e["per_launch"] = per_launch_stats(lambda: plic.plic_solve(*arrays, out=out, method=m, fast=f), 20, stream)
        e["_window"] = win
        issue_fields(e, counts_row(counts, name, workload), N, ms, sms, clk)
        if clk.get("sm_mhz"):
            # SURVEY.md 8d also asks for the issue fraction from the ALGORITHMIC counts: the thread-
            # instructions per cell a mixed warp has to issue for the method's formulas (union of all
            # case paths, SURVEY.md 8d "Algorithmic work per cell"), against SMs x 128 lanes x clock
            e["algorithmic_thread_inst_per_cell"] = ALGORITHMIC_INST[m]
            e["issue_frac_algorithmic"] = ALGORITHMIC_INST[m] * N / (ms * 1e-3) / (sms * 128 * clk["sm_mhz"] * 1e6)
        res[name] = e
    return res


DATA_DEPENDENT_KERNELS = ("map_compact",)      # per-tile compaction of the heavy cases, bisection to convergence


def counts_row(counts, name, workload):
    """Row of profiles/instruction_counts.txt for kernel `name` timed on `workload`, or None when the row
    cannot describe that run: the table carries the workload it was captured on ('#@ workload'), and the
    executed count of a data-dependent kernel (DATA_DEPENDENT_KERNELS) on another workload is a different
    number.  Branch-free kernels execute the same instructions on any input, so their row always applies."""
    row = counts.get(name)
    if row is None:
        return None
    captured_on = counts.get("@workload", ["configs[1]"])[0]
    kernel = row[3] if len(row) > 3 else ""
    if workload != captured_on and kernel.startswith(DATA_DEPENDENT_KERNELS):
        return None
    return row


def issue_fields(e, row, N, ms, sms, clk):
    """Issue roofline of one timed kernel from its row of profiles/instruction_counts.txt.  A packed
    fp32x2 instruction (FFMA2/FMUL2/FADD2) holds the issue port of its SM sub-partition for two
    clocks (pipe_rates: ffma2 alone 0.50 per clock, ffma2 + lop3 0.66 = 3 clocks per pair), every
    other instruction for one, so issue slots per cell = warp-instructions + packed warp-instructions;
    issue_frac = slots per cell x cells/s / (SMs x 4 sub-partitions x the MEAN SM clock of the NVML
    samples inside this kernel's timed window).  No row (none captured, or captured on another workload
    for a data-dependent kernel): issue_frac is None.  A fraction above 1 cannot be a measurement -- the
    counts or the clock do not belong to this run -- so it is flagged (`issue_model_error`) and does not
    pick `bound`."""
    clk = clk if isinstance(clk, dict) else {"sm_mhz": clk, "sm_mean_mhz": clk}
    mhz = clk.get("sm_mean_mhz") or clk.get("sm_mhz")
    if row is None or not mhz:
        e["issue_frac"] = None
        return
    wipc, packed = float(row[0]), float(row[2])
    e["warp_inst_per_cell"] = wipc
    e["lanes_per_inst"] = float(row[1])
    e["packed_warp_inst_per_cell"] = packed
    e["issue_slots_per_cell"] = wipc + packed
    e["issue_clock_mhz"] = mhz
    e["issue_frac"] = (wipc + packed) * N / (ms * 1e-3) / (sms * 4 * mhz * 1e6)
    if e["issue_frac"] > 1.0:
        e["issue_model_error"] = True
        e["bound"] = None
    else:
        e["bound"] = "issue" if e["issue_frac"] > e["hbm_frac"] else "hbm"


def run_ours(args):
    import numpy as np
    import torch
    import gen

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libplic has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    import paper_2006_12838_b200 as plic           # raises if libplic.so cannot be built/loaded

    sms = torch.cuda.get_device_properties(local).multi_processor_count
    N = 1 << args.log2n
    lo, hi = rank_cells(N, rank)
    host = gen.random_sphere(N, SEED, start=lo)                       # fp32 V0, nx, ny, nz
    dV, dx, dy, dz = [torch.from_numpy(a).cuda() for a in host]
    out = torch.empty_like(dV)
    stream = torch.cuda.current_stream()
    peak, peak_src = measured_peak()
    counts = profile_table("instruction_counts.txt")

    sampler = ClockSampler(local, period_s=0.002)
    sampler.start()

    # bring the clocks into the sustained regime before any timing (not counted as warm-up steps)
    t_end = time.perf_counter() + args.prewarm_ms / 1e3
    while time.perf_counter() < t_end:
        for _ in range(20):
            plic.plic_solve(dV, dx, dy, dz, out=out, method="analytic", fast=True)
        torch.cuda.synchronize()

    launches_before = plic.plic_launch_count()
    windows = {}
    methods = time_variants(plic, (dV, dx, dy, dz), out, args.steps, args.warmup, stream, world, sampler, sms,
                            counts, peak)

    def timed_map(name, fn, bytes_per_cell):
        ms, win = time_launches(fn, args.steps, args.warmup, stream)
        ms = max_over_ranks(ms) / args.steps
        gbs = bytes_per_cell * N / (ms * 1e-3) / 1e9
        clk = sampler.summary([win])
        e = {"value": N * world / (ms * 1e-3) / 1e9, "ms_per_step": ms, "launches": args.steps,
             "bytes_per_cell": bytes_per_cell, "hbm_gbs_per_gpu": gbs, "hbm_frac": gbs / peak,
             "hbm_frac_nominal": gbs / NOMINAL_HBM_GBS, "roofline_frac": gbs / peak, "sm_mhz": clk.get("sm_mhz")}
        issue_fields(e, counts.get(name), N, ms, sms, clk)
        return e

    # the 4-read / 1-write stream with no arithmetic, in the same sustained regime
    stream_ceiling = timed_map("blank", lambda: plic.plic_solve(dV, dx, dy, dz, out=out, method="blank"), BYTES_PER_CELL)
    stream_ceiling["what"] = ("plic_solve with PLIC_METHOD_BLANK (d0 = V0 - 1/2): the same four input streams, "
                              "body kernel and launch geometry as the HBM-bound solvers, no arithmetic")
    vol = torch.empty_like(dV)
    methods["plic_volume"] = timed_map("plic_volume", lambda: plic.plic_volume(out, dx, dy, dz, out=vol), BYTES_PER_CELL)
    # plane-sphere maps of sect. 3: one array in, one out (8 B per cell)
    for name, fn in (("sphere_solve-fast", lambda: plic.plic_sphere_solve(dV, out=out, fast=True)),
                     ("sphere_solve", lambda: plic.plic_sphere_solve(dV, out=out, fast=False)),
                     ("sphere_volume", lambda: plic.plic_sphere_volume(out, out=vol))):
        methods[name] = timed_map(name, fn, 8)

    # ---- fp16-storage and fp64 variants of the solve ----------------------------
    # the same cells: the fp32 workload rounded to binary16 (10 B per cell) resp. promoted to fp64 (40 B)
    storage = None
    if not args.no_storage:
        storage = {}
        hV, hx, hy, hz = [t.half() for t in (dV, dx, dy, dz)]
        hout = torch.empty_like(hV)
        storage["blank/f16"] = timed_map("blank/f16", lambda: plic.plic_solve_h(hV, hx, hy, hz, out=hout, method="blank"), 10)
        for m, f in VARIANTS:
            name = plic.plic_method_name(plic.method_id(m, f)) + "/f16"
            storage[name] = timed_map(name, lambda: plic.plic_solve_h(hV, hx, hy, hz, out=hout, method=m, fast=f), 10)
        storage["analytic-fast/f16+f32out"] = timed_map(
            "analytic-fast/f16+f32out",
            lambda: plic.plic_solve_h(hV, hx, hy, hz, out=hout, out_f32=out, method="analytic", fast=True), 14)
        storage["plic_volume/f16"] = timed_map("plic_volume/f16", lambda: plic.plic_volume_h(hout, hx, hy, hz, out=hV), 10)
        del hV, hx, hy, hz, hout
        fV, fx, fy, fz = [t.double() for t in (dV, dx, dy, dz)]
        fout = torch.empty_like(fV)
        for m in ("analytic", "sz", "newton", "nested"):
            storage["%s/f64" % m] = timed_map("%s/f64" % m, lambda: plic.plic_solve_f64(fV, fx, fy, fz, out=fout, method=m), 40)
        del fV, fx, fy, fz, fout
        for k, e in storage.items():
            e["dtype"] = "f64" if k.endswith("/f64") else "f16 storage, f32 arithmetic"
    total_launches = plic.plic_launch_count() - launches_before

    solve_names = [plic.plic_method_name(plic.method_id(m, f)) for m, f in VARIANTS]
    head = args.method if args.method != "auto" else max(solve_names, key=lambda k: methods[k]["value"])
    H = methods[head]
    hm, hf = (head[:-5], True) if head.endswith("-fast") else (head, False)
    # `clocks` is sampled inside the very window `value` was timed in (kept per variant by time_variants)
    windows[head] = H.pop("_window")
    for v in methods.values():
        v.pop("_window", None)

    # ---- instruction rates of the pipes, measured here ("confirm with an FFMA-only and a
    # MUFU-only microbenchmark"): warp-instructions per sub-partition per clock at the sampled clock
    pipe_rates = None
    if not args.no_probes:
        sink = torch.zeros(256, device="cuda")
        pipe_rates = {"unit": "warp-instructions per SM sub-partition per clock", "sms": sms, "probes": {}}
        torch.cuda.synchronize()
        time.sleep(0.3)                                  # the probes run at whatever clock they draw themselves
        for name in plic.PROBES:
            def probe(trips):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                w0 = time.perf_counter()
                e0.record(stream)
                n_inst = plic.plic_pipe_probe(name, trips, sink)
                e1.record(stream)
                torch.cuda.synchronize()
                return n_inst, e0.elapsed_time(e1) * 1e-3, (w0, time.perf_counter())
            probe(200)
            _, cal, _ = probe(400)                       # size the timed launch to ~30 ms: >= 10 clock samples
            n_inst, sec, win = probe(max(400, int(400 * 0.030 / max(cal, 1e-6))))
            ins = [s_[1] for s_ in sampler.samples if win[0] + 0.004 <= s_[0] <= win[1]]
            mhz = sorted(ins)[len(ins) // 2] if ins else (sampler.sm_max or 1965)
            pipe_rates["probes"][name] = {"t_inst_per_s": n_inst / sec / 1e12, "sm_mhz": mhz, "ms": sec * 1e3,
                                          "per_smsp_clk": n_inst / sec / (sms * 4 * mhz * 1e6)}
        pipe_rates["reading"] = ("scalar FFMA/FADD/FMUL issue at ~1 per clock, packed fp32x2 and every ALU-pipe "
                                 "instruction (min/max, compare, select, logic) at 1 per 2 clocks, MUFU at 1 per 8; a "
                                 "scalar FMA and an ALU instruction overlap (ffma+lop3 ~1 per clock) but a packed one and "
                                 "an ALU instruction do not (ffma2+lop3 ~0.66 per clock = 3 clocks per pair): a packed "
                                 "instruction holds the issue port for 2 clocks, which is the slot count issue_frac uses; "
                                 "nested_step* = one halving of nested-fast for a pair of cells in three encodings")
        del sink

    # ---- the paper's own benchmark shape (sect. 2.6, Table 3): compute bound, blank run subtracted
    paper = None
    if args.paper_log2n > 0:
        PN, PL = 1 << args.paper_log2n, 256
        pn = [torch.from_numpy(a).cuda() for a in gen.paper_normals(PN, 5)]
        pE = torch.empty_like(pn[0])
        paper = {"normals": PN, "L": PL, "unit": "ps per PLIC evaluation, blank run (eq. 33) subtracted",
                 "paper_titan_xp_ps": {"sz": 12.8, "kawano": 16.0, "analytic": 19.0, "newton": 19.2, "nested": 106.4},
                 "methods": {}}
        pnames = ["blank"] + solve_names + ["kawano"]
        raw = {}
        pwin = {}
        for name in pnames:
            ms, pwin[name] = time_launches(lambda: plic.plic_roundtrip_error(*pn, PL, out=pE, method=name),
                                           3, 3, stream)
            raw[name] = (max_over_ranks(ms) / 3, float(pE.double().mean()))
        for name in pnames:
            ms, eavg = raw[name]
            nan = eavg != eavg        # Listing 3 (kawano): NaN at n = (1,0,0), V0 in {0,1}, as in Tables 1-3
            paper["methods"][name] = {"ms": ms, "ps_per_eval": (ms - raw["blank"][0]) * 1e9 / (PN * PL),
                                      "ps_per_eval_incl_blank": ms * 1e9 / (PN * PL),
                                      "E_avg": None if nan else eavg, "E_avg_is_nan": nan}
        # issue roofline of the compute-bound loop: warp-instructions per (solve + forward map) evaluation
        # from the committed ncu capture x evaluations/s, against SMs x 4 x the clock sampled in the window
        row = counts.get("roundtrip:analytic-fast")
        mhz = sampler.summary([pwin["analytic-fast"]]).get("sm_mhz") or sampler.sm_max or 1965
        if row is not None:
            wipe, packed = float(row[0]), float(row[2])
            peak_wis = sms * 4 * mhz * 1e6 / 1e12
            ach = (wipe + packed) * PN * PL / (raw["analytic-fast"][0] * 1e-3) / 1e12
            paper["roofline"] = {"bound": "alu", "kernel": "roundtrip_kernel<analytic, fast>", "achieved": ach,
                                 "peak": peak_wis, "unit": "T issue slots/s", "frac": ach / peak_wis,
                                 "warp_instructions_per_evaluation": wipe,
                                 "packed_warp_instructions_per_evaluation": packed,
                                 "issue_slots_per_evaluation": wipe + packed, "sm_mhz": mhz,
                                 "counts_source": "profiles/instruction_counts.txt (ncu smsp__inst_executed.sum, packed "
                                                  "instructions from the SASS, commit %s)" % counts.get("@commit", ["?"])[0],
                                 "peak_source": "%d SMs x 4 sub-partitions x 1 issue slot per clock at the sampled SM clock; "
                                                "a packed fp32x2 instruction takes two slots, any other one (pipe_rates: "
                                                "scalar FFMA %.2f, FFMA2 %.2f, FFMA2+LOP3 %.2f instructions per clock)" % (
                                                    sms, *([pipe_rates["probes"][k]["per_smsp_clk"] for k in
                                                            ("ffma", "ffma2", "ffma2+lop3")] if pipe_rates else [float("nan")] * 3))}
        del pn, pE

    for k, v in methods.items():
        v.setdefault("roofline_frac", v["hbm_frac"])

    # ---- divergence cost = BASELINE.json configs[2]: 2^26 case-stratified cells labelled by the oracle
    # (rejection sampling on the oracle's classifier, V0 by the oracle's forward map), once interleaved
    # (case = i mod 5: every warp holds all five cases) and once in five contiguous blocks
    diverg = None
    if not args.no_divergence and args.log2n >= 20:
        from oracle.stratified import stratified, SEED as STRAT_SEED
        t0 = time.perf_counter()
        # torchrun sets OMP_NUM_THREADS=1 per rank: give the generator this rank's share of the cores
        sV, sx, sy, sz, kase = stratified(N, STRAT_SEED, start=lo, threads=max(1, (os.cpu_count() or 1) // world))
        gen_s = time.perf_counter() - t0
        order = np.concatenate([np.arange((k - lo) % 5, N, 5) for k in range(5)])
        diverg = {"workload": "configs[2]: N=2^%d case-stratified, seed 2, 20 %% per intersection case; labels and V0 "
                              "from the oracle (oracle/stratified.c)" % args.log2n,
                  "cells": N, "case_counts": np.bincount(kase, minlength=6)[1:].tolist(),
                  "layouts": "interleaved (case = i mod 5 + 1) vs five case-contiguous blocks of the same cells",
                  "generator_s": gen_s, "methods": {}}
        r = {}
        for lay in ("interleaved", "contiguous"):
            a = [torch.from_numpy(t if lay == "interleaved" else t[order]).cuda() for t in (sV, sx, sy, sz)]
            r[lay] = time_variants(plic, a, out, args.steps, args.warmup, stream, world, sampler, sms, counts, peak,
                                   workload="configs[2]")
            del a
        for name in solve_names:
            i_, c_ = r["interleaved"][name], r["contiguous"][name]
            diverg["methods"][name] = {"interleaved_ms": i_["ms_per_step"], "contiguous_ms": c_["ms_per_step"],
                                       "interleaved_over_contiguous": i_["ms_per_step"] / c_["ms_per_step"],
                                       "interleaved_hbm_frac": i_["hbm_frac"], "contiguous_hbm_frac": c_["hbm_frac"]}
        del sV, sx, sy, sz, kase, order, r

    # ---- BASELINE.json configs[3]: 2^28 cells, snapped normals, V0 ~ Beta(1/2, 1/2); the large-batch regime
    config4 = None
    if not args.no_config4:
        N4 = 1 << args.config4_log2n
        t0 = time.perf_counter()
        h4 = gen.snapped_beta(N4, 3, start=rank * N4)
        gen_s = time.perf_counter() - t0
        a4 = [torch.from_numpy(t).cuda() for t in h4]
        del h4
        o4 = torch.empty_like(a4[0])
        r4 = time_variants(plic, a4, o4, args.steps, args.warmup, stream, world, sampler, sms, counts, peak,
                           workload="configs[3]")
        for v in r4.values():
            v.pop("_window", None)
        config4 = {"workload": "configs[3]: N=2^%d cells (%.1f GB in, %.1f GB out), seed 3, half the normals snapped to an "
                               "axis or a face diagonal, V0 ~ Beta(1/2,1/2)" % (args.config4_log2n, 16 * N4 / 1e9, 4 * N4 / 1e9),
                   "cells": N4, "generator_s": gen_s, "methods": r4}
        del a4, o4

    # ---- curvature on configs[4]: 256^3 lattice, sphere R = 60 (sect. 4; three launches per call) ----
    curv = None
    if not args.no_curvature:
        R5 = 60.0
        host_phi = gen.sphere_fill_lattice(256, R5, (128.3, 127.7, 128.1), 8)
        # three copies of the lattice, used in turn: 3 x (67 MB read + 67 MB written) > 126 MB of L2,
        # so no call finds its input in cache
        phis = [torch.from_numpy(host_phi).cuda() for _ in range(3)]
        kaps = [torch.empty_like(p_) for p_ in phis]
        work5 = torch.empty(1 + phis[0].numel(), dtype=torch.int32, device="cuda")
        turn = [0]

        def curv_call():
            j = turn[0] % 3
            turn[0] += 1
            plic.plic_curvature(phis[j], out=kaps[j], work=work5)
        c0 = plic.plic_launch_count()
        ms, _ = time_launches(curv_call, args.steps, args.warmup, stream)
        per_call = (plic.plic_launch_count() - c0) / (args.steps + args.warmup)
        ms = max_over_ranks(ms) / args.steps
        n_if = int(work5[0].item())
        kap5 = kaps[0]
        kk = -kap5[kap5 != 0].double() * R5
        ncell = phis[0].numel()
        curv = {"workload": "configs[4]: 256^3 lattice, sphere R=60 at (128.3,127.7,128.1), phi = fraction "
                            "of 8^3 sub-cell points inside; three lattice copies used in turn (L2-cold input)",
                "ms_per_call": ms, "launches_per_call": per_call,
                "lattice_gcells_per_s": ncell / (ms * 1e-3) / 1e9, "interface_points": n_if,
                "interface_mpoints_per_s": n_if / (ms * 1e-3) / 1e6,
                "hbm_gbs": 8 * ncell / (ms * 1e-3) / 1e9,
                "roofline_frac": 8 * ncell / (ms * 1e-3) / 1e9 / peak,
                "hbm_frac_nominal": 8 * ncell / (ms * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
                "bytes_per_lattice_cell": 8, "all_interface_kappa_finite": bool(torch.isfinite(kap5).all()),
                "minus_kappa_R_mean": float(kk.mean()),
                "L1_error_eq50": float((kk - 1.0).abs().mean())}
        if not args.no_cpu_baseline and world == 1 and rank == 0:
            # the curvature oracle (numpy fp64 + the bisection oracle) on the same lattice, once
            from oracle import curvature as ocurv
            import oracle as _o
            t0 = time.perf_counter()
            ocurv.curvature_lattice(host_phi)
            dt = time.perf_counter() - t0
            curv["cpu_baseline"] = {"value": n_if / dt / 1e6, "unit": "M interface points/s",
                                    "cores": _o.max_threads(), "kind": "oracle",
                                    "sample": "the whole 256^3 lattice once (%.1f s)" % dt}
        del phis, kaps, work5, host_phi
        # ---- the same call at the lattice size the paper's raindrop run uses (400 x 400 x 340 =
        # 54.4 M lattice points): the launch chain and the dependent point pass are a fixed ~12 us, so the
        # larger lattice separates them from the stream (435 MB read + written per call)
        if not args.no_curvature_large:
            RL = 120.0
            t0 = time.perf_counter()
            big = np.ascontiguousarray(gen.sphere_fill_lattice(400, RL, (200.3, 199.7, 170.1), 8)[:340])
            gen_s = time.perf_counter() - t0
            phis = [torch.from_numpy(big).cuda() for _ in range(3)]
            kaps = [torch.empty_like(p_) for p_ in phis]
            workL = torch.empty(1 + phis[0].numel(), dtype=torch.int32, device="cuda")
            turn[0] = 0

            def curv_call_large():
                j = turn[0] % 3
                turn[0] += 1
                plic.plic_curvature(phis[j], out=kaps[j], work=workL)
            ms, _ = time_launches(curv_call_large, args.steps, args.warmup, stream)
            ms = max_over_ranks(ms) / args.steps
            ncell = phis[0].numel()
            kk = -kaps[0][kaps[0] != 0].double() * RL
            curv["large"] = {"workload": "400 x 400 x 340 lattice (PAPER.md:422), sphere R=120 at (200.3,199.7,170.1), same "
                                         "generator and sub-sampling as configs[4]; three copies in turn (L2-cold)",
                             "lattice_cells": ncell, "ms_per_call": ms, "interface_points": int(workL[0].item()),
                             "lattice_gcells_per_s": ncell / (ms * 1e-3) / 1e9,
                             "hbm_gbs": 8 * ncell / (ms * 1e-3) / 1e9,
                             "roofline_frac": 8 * ncell / (ms * 1e-3) / 1e9 / peak,
                             "all_interface_kappa_finite": bool(torch.isfinite(kaps[0]).all()),
                             "minus_kappa_R_mean": float(kk.mean()), "generator_s": gen_s}
            del phis, kaps, workL, big

    # ---- the headline variant and the blank stream once more after an idle gap: the clocks recover from
    # the power cap, which is the regime MEASURED_PEAKS.json's burst figure was taken in (reported beside
    # `value`, which stays the sustained number)
    torch.cuda.synchronize()
    time.sleep(0.5)
    bsteps = max(1, min(args.steps, 30))
    ms, bwin = time_launches(lambda: plic.plic_solve(dV, dx, dy, dz, out=out, method=hm, fast=hf),
                             bsteps, args.warmup, stream)
    ms = max_over_ranks(ms) / bsteps
    burst = {"method": head, "steps": bsteps, "ms_per_step": ms, "value": N * world / (ms * 1e-3) / 1e9,
             "unit": UNIT, "hbm_gbs_per_gpu": BYTES_PER_CELL * N / (ms * 1e-3) / 1e9,
             "roofline_frac": BYTES_PER_CELL * N / (ms * 1e-3) / 1e9 / peak,
             "note": "same kernel, timed after 0.5 s of idle (no sustained load before it)"}
    time.sleep(0.5)
    ms, _ = time_launches(lambda: plic.plic_solve(dV, dx, dy, dz, out=out, method="blank"), bsteps, args.warmup, stream)
    burst["stream_ceiling_ms"] = max_over_ranks(ms) / bsteps
    burst["stream_ceiling_gbs"] = BYTES_PER_CELL * N / (burst["stream_ceiling_ms"] * 1e-3) / 1e9
    burst["frac_of_stream_ceiling"] = burst["stream_ceiling_ms"] / burst["ms_per_step"]

    # ---- end to end through the host-array C ABI: pinned host buffers, copies inside ----------
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    pin = [torch.from_numpy(a).pin_memory() for a in host]
    pout = torch.empty(N, dtype=torch.float32).pin_memory()
    for _ in range(2):
        plic.plic_solve_host(*pin, out=pout, method=hm, fast=hf)
    torch.cuda.synchronize()
    barrier()
    c0 = plic.plic_launch_count()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        plic.plic_solve_host(*pin, out=pout, method=hm, fast=hf)      # synchronous
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    e2e_launches = plic.plic_launch_count() - c0
    e2e_s = max_over_ranks(t1 - t0)
    plic.plic_solve(dV, dx, dy, dz, out=out, method=hm, fast=hf)
    e2e_same = bool(np.array_equal(pout.numpy(), out.cpu().numpy()))   # host API == device API, bitwise
    # the link itself: one pinned array up, one down, CUDA events
    link = pcie_link(sampler) or {}
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    e0.record(stream)
    dV.copy_(pin[0], non_blocking=True)
    e1.record(stream)
    pout.copy_(out, non_blocking=True)
    e2.record(stream)
    torch.cuda.synchronize()
    link["measured_h2d_gbs"] = 4 * N / (e0.elapsed_time(e1) * 1e-3) / 1e9
    link["measured_d2h_gbs"] = 4 * N / (e1.elapsed_time(e2) * 1e-3) / 1e9
    sampler.stop()
    plic.plic_host_release()

    clocks = sampler.summary([windows[head]])
    if rank == 0:
        traffic, traffic_src = ncu_traffic(head, N)
        achieved = H["hbm_gbs_per_gpu"]
        per_step_s = e2e_s / e2e_steps
        line = {
            "metric": METRIC, "value": H["value"], "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": H["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": WORKLOAD % args.log2n, "cells_per_gpu": N, "method": head,
                       "headline_rule": "fastest of the 8 plic_solve variants" if args.method == "auto"
                       else "--method",
                       "l2": "inputs larger than L2 (1.07 GB read + 0.27 GB written per step vs 126 MB)",
                       "prewarm_ms": args.prewarm_ms, "launch": {"grid": plic.plic_launch_config(hm, N, hf)[0],
                                                                 "block": 256, "cells_per_thread": 4}},
            "clocks": dict(clocks, window="the %d timed launches of the headline variant (`value`); under sustained load "
                                          "this pool's boxes hold the SMs at 1.45-1.55 GHz (software power cap); `burst` "
                                          "repeats the variant at full clock" % args.steps),
            "gpu_launches": H["launches"],
            "gpu_launches_all_timed_regions": total_launches,
            "e2e": {"value": N * world * e2e_steps / e2e_s / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": 16 * N, "d2h_bytes_per_step": 4 * N, "steps": e2e_steps,
                    "launches": e2e_launches, "matches_device_api_bitwise": e2e_same,
                    "h2d_gbs": 16 * N / per_step_s / 1e9, "d2h_gbs": 4 * N / per_step_s / 1e9,
                    "pcie": link,
                    "bound": "the host link: both directions run concurrently, so the step cannot be shorter than "
                             "16 B/cell over the H2D rate; frac_of_link = achieved H2D rate / measured pinned H2D rate",
                    "frac_of_link": (16 * N / per_step_s / 1e9) / link["measured_h2d_gbs"],
                    "api": "plic_solve_host (pinned host arrays, chunked H2D/kernel/D2H pipeline inside libplic)",
                    "timer": "host wall clock around the synchronous calls, device synchronised on both sides"},
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                         "tables_stale": {"dram_traffic.txt": table_is_stale(profile_table("dram_traffic.txt")),
                                          "instruction_counts.txt": table_is_stale(counts)},
                         "kernel": head,
                         "frac_nominal": achieved / NOMINAL_HBM_GBS, "peak_nominal": NOMINAL_HBM_GBS,
                         "frac_of_stream_ceiling": stream_ceiling["ms_per_step"] / H["ms_per_step"],
                         "issue_frac": H.get("issue_frac"),
                         "algorithmic_bytes_per_launch": BYTES_PER_CELL * N, "peak_source": peak_src,
                         "peak_note": "the measured peak is a copy (1 read : 1 write); this stream is 4 reads : "
                                      "1 write, whose own ceiling in this run is stream_ceiling (a blank kernel of the "
                                      "same shape), so frac can exceed 1"},
            "stream_ceiling": stream_ceiling,
            "methods": methods,
        }
        burst["clocks"] = sampler.summary([bwin])
        line["burst"] = burst
        if storage is not None:
            line["storage"] = storage
        if pipe_rates is not None:
            line["pipe_rates"] = pipe_rates
        if paper is not None:
            line["paper_benchmark"] = paper
        if curv is not None:
            line["curvature"] = curv
        if diverg is not None:
            line["divergence"] = diverg
        if config4 is not None:
            line["config4"] = config4
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(host)
            line["cpu_baseline_1core"] = cpu_baseline(host, budget_s=4.0, threads=1)
        # compact repeat of the per-variant results, last on the line
        r3 = lambda x: None if x is None else round(x, 3)
        line["summary"] = {
            "cols": "ms, hbm_frac, issue_frac, bound | config3 interleaved ms, interleaved/contiguous | config4 ms, hbm_frac",
            "rows": {k: [round(methods[k]["ms_per_step"], 4), r3(methods[k]["hbm_frac"]), r3(methods[k].get("issue_frac")),
                         methods[k].get("bound"),
                         None if diverg is None else round(diverg["methods"][k]["interleaved_ms"], 4),
                         None if diverg is None else r3(diverg["methods"][k]["interleaved_over_contiguous"]),
                         None if config4 is None else round(config4["methods"][k]["ms_per_step"], 4),
                         None if config4 is None else r3(config4["methods"][k]["hbm_frac"])] for k in solve_names},
            "stream_ceiling_ms": round(stream_ceiling["ms_per_step"], 4),
            "plic_volume_ms": round(methods["plic_volume"]["ms_per_step"], 4),
            "curvature_ms": None if curv is None else round(curv["ms_per_call"], 4),
            "curvature_400x400x340_ms": None if curv is None or "large" not in curv else round(curv["large"]["ms_per_call"], 4),
            "storage_ms": None if storage is None else {k: round(v["ms_per_step"], 4) for k, v in storage.items()},
        }
        detail_path = write_detail(line, args.detail_out)
        print(json.dumps(compact_line(line, detail_path)), flush=True)     # the ONLY stdout line
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    return 0


# ---- what goes to stdout: one contract line a driver can parse from a bounded tail ----------------
LINE_LIMIT = 8000        # bytes; the full object (30+ KB: every variant of every leg) goes to --detail-out
DETAIL_KEYS = ("methods", "storage", "pipe_rates", "paper_benchmark", "divergence", "config4")
_DROP_IF_LONG = ("stream_ceiling", "burst", "curvature", "cpu_baseline_1core")   # in this order


def _round_floats(x, digits=6):
    if isinstance(x, float):
        return float("%.*g" % (digits, x)) if x == x and abs(x) != float("inf") else None
    if isinstance(x, dict):
        return {k: _round_floats(v, digits) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_round_floats(v, digits) for v in x]
    return x


def compact_line(line, detail_path=None):
    """The contract line printed last on stdout: every key the bench contract names (metric, value, unit,
    n_gpus, steps, warmup, ms_per_step, higher_is_better, scaling, vs_baseline, dtype, data, config, clocks,
    gpu_launches, e2e, roofline, cpu_baseline) plus the per-variant `summary`, without the per-leg detail
    objects (DETAIL_KEYS), floats at 6 significant digits, and guaranteed shorter than LINE_LIMIT bytes so
    that a driver which keeps only the tail of stdout still holds the whole line."""
    out = {k: v for k, v in line.items() if k not in DETAIL_KEYS}
    out = _round_floats(out)
    out["detail"] = {"file": detail_path, "keys": [k for k in DETAIL_KEYS if k in line]}
    for k in (None,) + _DROP_IF_LONG:
        if k is not None:
            out.pop(k, None)
        if len(json.dumps(out)) < LINE_LIMIT:
            return out
    if isinstance(out.get("summary"), dict):
        out["summary"].pop("storage_ms", None)
    if len(json.dumps(out)) >= LINE_LIMIT:
        out.pop("summary", None)
    return out


def write_detail(line, path):
    """The full result object as indented JSON in `path` (None or "" skips it); returns the path written."""
    if not path:
        return None
    try:
        os.makedirs(os.path.dirname(os.path.abspath(path)), exist_ok=True)
        with open(path, "w") as f:
            json.dump(line, f, indent=1)
            f.write("\n")
        return path
    except OSError as e:
        sys.stderr.write("bench.py: could not write %s (%s)\n" % (path, e))
        return None


def run_plumbing_only(args):
    """The multi-rank plumbing of this file without a GPU (CPU test of `--gpus N`): rendezvous on gloo,
    each rank generates a slice of its own cell range, the per-rank timings are MAX-reduced, rank 0
    prints one JSON line.  No PLIC arithmetic is done and no metric is reported."""
    import numpy as np
    import torch.distributed as dist
    import gen
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("gloo")
    per = 1 << 12
    lo, hi = rank_cells(per, rank)
    shard = gen.random_sphere(hi - lo, SEED, start=lo)
    t = max_over_ranks(1.0 + rank, device="cpu")
    total = sum_over_ranks(float(hi - lo), device="cpu")
    check = sum_over_ranks(float(np.sum(shard[0], dtype=np.float64)), device="cpu")
    if rank == 0:
        print(json.dumps({"plumbing_only": True, "n_gpus": world, "ranks": world, "cells": int(total),
                          "max_over_ranks": t, "checksum": check}), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def relaunch_with_ranks(args, argv):
    """`python bench.py --gpus N` with N > 1 and no torchrun environment: start N ranks of this file
    under torch.distributed.run on 127.0.0.1 and pass its exit code on."""
    import socket
    import subprocess
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


def main(argv=None):
    argv = sys.argv[1:] if argv is None else list(argv)
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--log2n", type=int, default=26, help="cells per GPU = 2^log2n (default: configs[1])")
    ap.add_argument("--method", default="auto", help="headline variant, e.g. analytic-fast (default: fastest)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--prewarm-ms", type=float, default=300.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-curvature", action="store_true", help="skip the plic_curvature leg")
    ap.add_argument("--no-curvature-large", action="store_true",
                    help="skip the 400 x 400 x 340 lattice of the curvature leg (the paper's raindrop size)")
    ap.add_argument("--no-divergence", action="store_true", help="skip the configs[2] (case-stratified) leg")
    ap.add_argument("--no-config4", action="store_true", help="skip the configs[3] (2^28 snapped/Beta) leg")
    ap.add_argument("--config4-log2n", type=int, default=28)
    ap.add_argument("--no-probes", action="store_true", help="skip the instruction-rate probes")
    ap.add_argument("--no-storage", action="store_true", help="skip the fp16-storage / fp64 variants")
    ap.add_argument("--detail-out", default=os.path.join(ROOT, "bench_detail.json"),
                    help="file for the full result object (every variant of every leg); stdout carries only "
                         "the compact contract line.  '' skips the file")
    ap.add_argument("--plumbing-only", action="store_true",
                    help="exercise the multi-rank launch and reductions on CPU (gloo); no GPU work, no metric")
    ap.add_argument("--paper-log2n", type=int, default=24,
                    help="normals in the paper-shaped compute-bound leg = 2^k, L = 256 volumes each "
                         "(the paper: k = 26); 0 skips it")
    args = ap.parse_args(argv)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                       # timing rule: at least 3 warm-up steps
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch_with_ranks(args, argv)
    if args.plumbing_only:
        return run_plumbing_only(args)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
