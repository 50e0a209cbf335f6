#!/usr/bin/env python
"""bench.py -- throughput of the SCMF Monte-Carlo step on B200 (BASELINE.json `metric`: attempted bead
moves/s and MC steps/s on 1 B200; % of HBM roofline).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config I] [--impl ours|reference]

A "step" is one whole MC step (rows a1-a5 of SURVEY.md section 8(a): both half-sweeps, re-binning,
omega) over the full synthetic system of BASELINE.json `configs[I]` (default I = 4, the 134 M-bead
diblock melt `north_star` quotes its target on).  Timed with CUDA events on the stream the library
launches on, K steps after W warm-up steps, positions resident in HBM (`value`); `e2e` is the
config's whole run through the C ABI from pinned HOST buffers back to HOST buffers.  N > 1: the path
does not shard (`north_star`: one GPU, no collectives) -- N independent replicas, one process per
GPU, barrier + max-over-ranks timing, `value` = all ranks' moves / that time ("replicas only").

`--impl reference`: the CPU oracle (oracle/), as it stands, timed on the host cores on a bounded
sample of the same workload; rank 0 only.
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

import numpy as np

# ncu counters of the dominant kernel (dram bytes, L2 sectors, ...) are NOT measured by bench.py: they come
# from the committed table profiles/ncu_counters.csv, one row per (kernel path, config, source hash of the
# kernels).  A row whose hash is not the hash of the sources this run was built from is stale and ignored.
NCU_TABLE = os.path.join(ROOT, "profiles", "ncu_counters.csv")
# soma_api.cu is in the key because the launch geometry of the captured kernel lives there (threads per block, chunk,
# carve-out, the thresholds that pick packed counters and the on-the-fly field)
KERNEL_SOURCES = ("soma_device.cuh", "soma_kernels.cuh", "soma_lean.cuh", "soma_api.cu")

METRIC = "attempted bead moves/s"
UNIT = "moves/s"


# --------------------------------------------------------------------------------------------------
# roofline bookkeeping
# --------------------------------------------------------------------------------------------------

def algorithmic_bytes(w) -> dict:
    """Bytes the method itself must move per MC step (perfect caching of anything touched twice
    inside a kernel): positions read once + written once; counts atomically written, read by omega,
    re-zeroed; omega written, read at least once by the moves."""
    B, TC = w.n_beads, w.n_types * w.n_cells
    return {
        "move_bin_kernel": 24 * B + 8 * TC,        # positions r+w, omega read once, counts written once
        "omega_kernel": 12 * TC,                   # counts read, omega written, other count buffer zeroed
        "step": 24 * B + 20 * TC,
    }


def kernel_source_hash() -> str:
    """First 12 hex digits of the sha256 over the kernel sources: the key that ties an ncu capture to a build."""
    import hashlib
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2606_09356_b200", "csrc", name), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:12]


def ncu_counters(path: int, config: int, table: str = NCU_TABLE):
    """Row of profiles/ncu_counters.csv for this (path, config) captured on the current kernel sources, or None."""
    import csv
    try:
        with open(table, newline="") as f:
            rows = [r for r in csv.DictReader(f)]
    except OSError:
        return None
    key = kernel_source_hash()
    for r in rows:
        if int(r["path"]) == path and int(r["config"]) == config and r["source_hash"] == key:
            return r
    return None


def cpu_info() -> dict:
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for ln in f:
                if ln.startswith("model name"):
                    model = ln.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return {"cpu_model": model, "logical_cores": os.cpu_count()}


def pin_to_one_core():
    """Pin this process to the core it runs on (the oracle leg is single-threaded
    and pinned).  Returns the core, or None where the platform has no affinity call."""
    try:
        allowed = sorted(os.sched_getaffinity(0))
        core = allowed[len(allowed) // 2]
        os.sched_setaffinity(0, {core})
        return core, allowed
    except (AttributeError, OSError):
        return None, None


def unpin(allowed):
    if allowed:
        try:
            os.sched_setaffinity(0, set(allowed))
        except OSError:
            pass


def measured_peaks() -> tuple[float, str]:
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written) or the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (measured copy bandwidth)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md; MEASURED_PEAKS.json absent)"


# --------------------------------------------------------------------------------------------------
# clocks during the timed region (NVML, sampled from a thread)
# --------------------------------------------------------------------------------------------------

_REASONS = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
            0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}


class ClockSampler:
    def __init__(self, cuda_index: int, period_s: float = 0.001):
        self.period, self.samples, self.mask, self.power = period_s, [], 0, []
        self.sm_max, self._stop, self._thread, self._h, self._nv = None, threading.Event(), None, None, None
        self._running = threading.Event()
        try:
            import pynvml as nv
            import torch
            nv.nvmlInit()
            uuid = "GPU-" + str(torch.cuda.get_device_properties(cuda_index).uuid)
            try:
                self._h = nv.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self._h = nv.nvmlDeviceGetHandleByIndex(cuda_index)
            self.sm_max = int(nv.nvmlDeviceGetMaxClockInfo(self._h, nv.NVML_CLOCK_SM))
            self._nv = nv
        except Exception as e:                       # no NVML: report that instead of inventing clocks
            self.error = repr(e)

    def _run(self):
        nv = self._nv
        self._running.set()
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
                except Exception:
                    self.mask |= int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self._nv is not None:
            self.samples, self.mask, self.power = [], 0, []
            self._stop.clear()
            self._running.clear()
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
            self._running.wait(1.0)          # the sampling loop is up before the timed region begins: a 20 ms window gets >= 5 samples

    def stop(self) -> dict:
        if self._nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": getattr(self, "error", "nvml unavailable")}
        self._stop.set()
        self._thread.join()
        reasons = [name for bit, name in _REASONS.items() if self.mask & bit and name != "gpu_idle"]
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.sm_max,
                "reasons": reasons, "samples": len(self.samples),
                "power_w_max": max(self.power) if self.power else None}


# --------------------------------------------------------------------------------------------------
# multi-GPU: replicas only.  Barrier, max-over-ranks time, sum-over-ranks work.
# --------------------------------------------------------------------------------------------------

def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def aggregate_over_ranks(local_ms: float, local_units: float, device=None):
    """(max over ranks of local_ms, sum over ranks of local_units).  Works on any torch.distributed
    backend (nccl on the GPUs, gloo in the CPU test); identity when no process group is up."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(local_ms), float(local_units)
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


# --------------------------------------------------------------------------------------------------
# the CPU oracle as a timed baseline (test infrastructure; never on the product path)
# --------------------------------------------------------------------------------------------------

def sample_workload(w, factor: int):
    """The same melt (beads per cell, cell size, fields, architecture) at 1/factor of the chains and
    cells; factor a power of two, grid axes halved in turn (x, y, z, x, ...)."""
    import scmf_inputs as si
    grid, d, f = list(w.grid), 0, factor
    while f > 1:
        if grid[d % 3] % 2 == 0 and grid[d % 3] > 1:
            grid[d % 3] //= 2
            f //= 2
        d += 1
    return si.scaled(w, w.n_chains // factor, tuple(grid))


ORACLE_SAMPLE_FACTOR = 8      # both arms time the oracle on 1/8 of the config (same beads per cell) unless a step count forces less


def oracle_sample(w, n_steps: int):
    """The bounded sample both arms time the oracle on: 1/ORACLE_SAMPLE_FACTOR of the workload at the same
    beads per cell (a power of two more if n_steps oracle steps of that would take longer than ~100 s at
    ~120 ns per attempted move).  Returns (sample workload, factor)."""
    factor = 1
    while factor < ORACLE_SAMPLE_FACTOR and w.n_chains // (factor * 2) >= 1024:
        factor *= 2
    while w.n_beads // factor * 120e-9 * max(1, n_steps) > 100.0 and w.n_chains // (factor * 2) >= 1024:
        factor *= 2
    return (sample_workload(w, factor) if factor > 1 else w), factor


def time_oracle(system, steps: int, warmup: int = 0, budget_s: float | None = None):
    """Oracle MC steps on `system`, single-threaded and pinned to one core, as it stands.
    Returns (seconds, steps timed, core)."""
    import oracle
    core, allowed = pin_to_one_core()
    try:
        o = oracle.Oracle.from_system(system)
        o.load_state(system.x, system.y, system.z)
        if warmup:
            o.mc_steps(warmup)
        done, t0 = 0, time.perf_counter()
        while done < steps:
            o.mc_steps(1)
            done += 1
            if budget_s is not None and time.perf_counter() - t0 >= budget_s:
                break
        dt = time.perf_counter() - t0
        o.close()
    finally:
        unpin(allowed)
    return dt, done, core


def sample_text(w, ws, factor: int) -> str:
    if factor == 1:
        return f"the whole of {w.name} ({w.n_beads} beads); every step is one oracle MC step"
    return (f"{ws.n_chains} chains x {ws.N} beads on a {ws.grid[0]}x{ws.grid[1]}x{ws.grid[2]} grid = 1/{factor} of "
            f"{w.name} at the same beads per cell; every step is one oracle MC step over that sample")


def run_reference(args):
    """`--impl reference`: the oracle on the host cores, on a bounded sample of the same workload."""
    import scmf_inputs as si
    rank, _, world = dist_env()
    if rank != 0:
        return
    w = si.config(args.config)
    ws, factor = oracle_sample(w, args.steps + args.warmup)
    s = si.make_system(ws)
    dt, done, core = time_oracle(s, args.steps, warmup=args.warmup)
    value = ws.n_beads * done / dt
    sample = sample_text(w, ws, factor)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": done,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / done, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "sample": sample, "mc_steps_per_s": done / dt},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "pinned_core": core, **cpu_info()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# --------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------

def run_dry(args):
    """`--dry`: the multi-rank plumbing of run_ours without a GPU (process group on `--backend`, barrier,
    max-over-ranks time, sum-over-ranks work, rank 0 prints the line) on made-up per-rank timings.  For the
    CPU tests of the launch path; the line says "dry": true and carries no measurement."""
    import torch.distributed as dist
    import scmf_inputs as si
    rank, _, world = dist_env()
    if world > 1:
        dist.init_process_group(args.backend)
    w = si.config(args.config)
    barrier()
    ms, moves = aggregate_over_ranks(10.0 + 5.0 * rank, float(w.n_beads) * args.steps)
    barrier()
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": moves / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms / args.steps, "dry": True, "scaling": "weak",
                          "config": {"workload": w.name, "parallelism": "replicas only" if world > 1 else "1 gpu"}}))
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2606_09356_b200 as soma
    import scmf_inputs as si

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group(args.backend, device_id=dev if args.backend == "nccl" else None)
    soma.load_library()                                 # raises if the CUDA library is missing

    w = si.config(args.config)
    s = si.make_system(w)                               # every rank: an independent replica of the config
    B = w.n_beads
    pinned = [torch.from_numpy(v).pin_memory() for v in (s.x, s.y, s.z)]
    out_pos = [torch.empty(B, dtype=torch.float32).pin_memory() for _ in range(3)]
    out_den = torch.empty((w.n_types, w.n_cells), dtype=torch.int32).pin_memory()
    stream = torch.cuda.current_stream()
    g = soma.Soma.from_system(s, smc_mobility=args.smc_mobility)
    if args.path:
        g.set_option("path", args.path)
    for kv in args.opt:
        k, v = kv.split("=")
        g.set_option(k, int(v))
    clocks = ClockSampler(local_rank)

    # ---- device-resident timing: K steps after W warm-up steps --------------------------------
    g.load_state(pinned[0], pinned[1], pinned[2])
    g.mc_steps(max(args.warmup, 0))
    g.set_option("kernel_timing", 1)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    barrier()
    c0 = g.counters()
    clocks.start()
    ev0.record(stream)
    g.mc_steps(args.steps)                              # asynchronous: no host sync inside
    ev1.record(stream)
    torch.cuda.synchronize()
    clk = clocks.stop()
    barrier()
    local_ms = ev0.elapsed_time(ev1)
    kt = g.kernel_times()
    g.set_option("kernel_timing", 0)
    c1 = g.counters()
    launches = c1["launches"] - c0["launches"]
    resorts_in_window = c1["resorts"] - c0["resorts"]
    g_path = c1["path"]
    otf = c1["omega_otf"]
    ms, moves = aggregate_over_ranks(local_ms, float(B) * args.steps, dev)
    value = moves / (ms * 1e-3)

    # ---- the chain re-ordering on its own (it runs every `interval` steps: K decides how many fall into the
    # window above, so the line also carries a per-step figure that does not depend on K) ---------------
    interval = 64 if w.n_chains >= 4096 else 0
    for kv in args.opt:
        if kv.startswith("resort_interval="):
            interval = int(kv.split("=")[1])
    resort_ms = 0.0
    if interval:
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g.set_option("resort_now", 0)
        torch.cuda.synchronize()
        r0.record(stream)
        for _ in range(3):
            g.set_option("resort_now", 0)
        r1.record(stream)
        torch.cuda.synchronize()
        resort_ms = r0.elapsed_time(r1) / 3
    steady_local = (local_ms - resorts_in_window * resort_ms) / args.steps + (resort_ms / interval if interval else 0.0)
    steady_ms, _ = aggregate_over_ranks(steady_local, 0.0, dev)

    # ---- one whole re-ordering cycle: the re-ordering and the interval_steps MC steps up to the next one, timed as one
    # region.  Unlike the window above this holds everything a long run pays per step: the re-ordering itself, the decay of
    # the memory locality between two re-orderings, and the clock the chip settles at under sustained load. ----
    cycle_ms, cycle = None, None
    if interval:
        clocks_c = ClockSampler(local_rank)
        q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        barrier()
        cc0 = g.counters()
        clocks_c.start()
        q0.record(stream)
        g.set_option("resort_now", 0)
        g.mc_steps(interval)
        q1.record(stream)
        torch.cuda.synchronize()
        clk_c = clocks_c.stop()
        barrier()
        cc1 = g.counters()
        cycle_ms, _ = aggregate_over_ranks(q0.elapsed_time(q1) / interval, 0.0, dev)
        cycle = {"steps": interval, "resorts": cc1["resorts"] - cc0["resorts"], "ms": cycle_ms * interval, "clocks": clk_c}
    sustained_ms = cycle_ms if cycle_ms else steady_ms

    # ---- end to end: the config's own run through the C ABI, host buffers in and out -----------
    S = w.steps
    torch.cuda.synchronize()
    barrier()
    t0 = time.perf_counter()
    g.load_state(pinned[0], pinned[1], pinned[2])       # H2D 12 B/bead
    g.mc_steps(S)
    soma.soma_get_density(g._h, out_den)                # D2H 4 T C
    soma.soma_get_positions(g._h, *out_pos)             # D2H 12 B/bead
    torch.cuda.synchronize()
    e2e_local = (time.perf_counter() - t0) * 1e3
    barrier()
    e2e_ms, e2e_moves = aggregate_over_ranks(e2e_local, float(B) * S, dev)
    assert int(out_den.sum()) == B, "density grids do not sum to the bead count"
    g.close()

    # ---- roofline of the dominant kernel (fused move + bin), from the live event times ---------
    peak, peak_src = measured_peaks()
    ab = algorithmic_bytes(w)
    n_t = max(1, kt["steps"])
    move_ms, omega_ms = kt["move_bin_ms"] / n_t, kt["omega_ms"] / n_t
    achieved = ab["move_bin_kernel"] / (move_ms * 1e-3) / 1e9
    kname = {1: "half_sweep_kernel x2 + bin_kernel (rows a1+a2+a3+a5)", 2: "lean_step_kernel (rows a1+a2+a3+a5)"}[g_path]
    if args.smc_mobility > 0 or (g_path == 2 and any(kv == "fused_lean=0" for kv in args.opt)):
        kname = kname.replace("lean_step_kernel", "fused_step_kernel")
    if otf:
        kname = "lean_step_kernel, omega computed on the fly from the packed counters (rows a1+a2+a3+a4+a5)"
    ncu = ncu_counters(g_path, args.config) if args.smc_mobility == 0 and not args.opt else None
    roofline = {"bound": "hbm", "kernel": kname,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": (float(ncu["dram_bytes_read"]) + float(ncu["dram_bytes_write"])) if ncu else None,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": ab["move_bin_kernel"],
                "kernel_ms": move_ms, "omega_kernel_ms": omega_ms,
                "omega_kernel_frac": ab["omega_kernel"] / (omega_ms * 1e-3) / 1e9 / peak if omega_ms > 0 and not otf else None,
                "row_a4": ("inside the move kernel: omega is computed from the previous step's packed counters where it is needed and never "
                           "stored; omega_kernel_ms is the memset of the next count buffer; `achieved` still counts SURVEY's algorithmic bytes "
                           "(omega written and read once), so the DRAM traffic is below them") if otf else "omega_kernel",
                "step_frac": ab["step"] / (sustained_ms * 1e-3) / 1e9 / peak,
                "step_frac_of_8TBps": ab["step"] / (sustained_ms * 1e-3) / 8e12,
                "step_frac_basis": "resort.ms_per_step_cycle" if cycle_ms else "resort.ms_per_step_steady",
                "target_step_frac_of_8TBps": 0.60, "target_met": ab["step"] / (sustained_ms * 1e-3) / 8e12 >= 0.60,
                "bytes_per_move": ab["step"] / B}
    if ncu:
        roofline["ncu"] = {"source": f"profiles/ncu_counters.csv ({ncu['capture']})", "source_hash": ncu["source_hash"],
                           "l2_sectors_per_launch": float(ncu["lts_sectors"]),
                           "warp_instructions_per_launch": float(ncu["inst_executed"]),
                           "l1tex_to_xbar_request_cycles_pct": float(ncu["l1tex2xbar_req_pct"]),
                           "lsu_wavefronts_pct": float(ncu["lsu_wavefronts_pct"]),
                           "issue_active_pct": float(ncu["issue_active_pct"]),
                           "limiter": ncu["limiter"]}
    else:
        roofline["ncu"] = None     # no capture of these kernel sources / this path and config: nothing is quoted

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "n_chains": w.n_chains, "beads_per_chain": w.N, "beads": B, "grid": list(w.grid),
                   "chiN": w.chiN, "kappaN": w.kappaN, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": f"inputs larger than L2: positions {12 * B / 1e6:.0f} MB + grids {12 * w.n_types * w.n_cells / 1e6:.0f} MB per step",
                   "mc_steps_per_s": world * args.steps / (ms * 1e-3),
                   **({"moves": f"bond-force-biased, A = {args.smc_mobility}"} if args.smc_mobility > 0 else {})},
        "resort": {"interval_steps": interval, "ms": resort_ms, "in_timed_window": int(resorts_in_window),
                   "ms_per_step_amortised": resort_ms / interval if interval else 0.0,
                   "ms_per_step_steady": steady_ms, "moves_per_s_steady": world * B / (steady_ms * 1e-3),
                   "ms_per_step_cycle": cycle_ms, "moves_per_s_cycle": world * B / (cycle_ms * 1e-3) if cycle_ms else None,
                   "cycle": cycle,
                   "what": "the chains are re-ordered in memory every interval_steps MC steps; ms_per_step_steady = the timed steps "
                           "without the re-orderings that fell into the window + one re-ordering per interval_steps, so it does not depend on K; "
                           "ms_per_step_cycle = one re-ordering + the interval_steps steps after it timed as one region (CUDA events), its own "
                           "clock record in `cycle`: the sustained figure, and the one roofline.step_frac* and target_met are computed from"},
        "clocks": clk, "gpu_launches": int(launches),
        "e2e": {"value": e2e_moves / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 12 * B / S,
                "d2h_bytes_per_step": (12 * B + 4 * w.n_types * w.n_cells) / S, "mc_steps": S, "ms": e2e_ms,
                "what": f"soma_load_state(pinned host) + soma_mc_steps({S}) + soma_get_density(host) + soma_get_positions(pinned host); "
                        f"the copies happen once per {S}-step run, bytes are per MC step"},
        "roofline": roofline,
    }

    # ---- the oracle on the host cores, rank 0 at N = 1 only ------------------------------------
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        ws, factor = oracle_sample(w, 4)
        ss = si.make_system(ws) if factor > 1 else s
        dt, done, core = time_oracle(ss, steps=4, budget_s=20.0)
        line["cpu_baseline"] = {"value": ws.n_beads * done / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": sample_text(w, ws, factor) + f"; {done} step(s), {dt:.1f} s",
                                "pinned_core": core, **cpu_info()}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def relaunch_under_torchrun(n: int) -> int:
    """`python bench.py --gpus N` without a launcher: start N ranks of this script with torch.distributed.run
    (one process per GPU, rendezvous on 127.0.0.1) and return its exit code."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index (default 4: 134 M beads)")
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--path", type=int, default=0, help="library kernel path: 0 auto, 1 generic, 2 fused")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=INT", help="soma_set_option(NAME, INT) before the run (tuning)")
    ap.add_argument("--smc-mobility", type=float, default=0.0,
                    help="A > 0: bond-force-biased moves (DESIGN.md R24) instead of the configs' uniform moves; not the headline metric")
    ap.add_argument("--backend", choices=["nccl", "gloo"], default="nccl", help="torch.distributed backend of the barrier / aggregation")
    ap.add_argument("--dry", action="store_true", help="multi-rank plumbing only, no GPU work (CPU tests)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                   # timing rule: at least 3 warm-up steps
    world_env = os.environ.get("WORLD_SIZE")
    if world_env is None and args.gpus > 1 and args.impl == "ours":
        raise SystemExit(relaunch_under_torchrun(args.gpus))       # one replica per GPU
    if world_env is not None and int(world_env) != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world_env}")
    if args.impl == "reference":
        run_reference(args)
    elif args.dry:
        run_dry(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
