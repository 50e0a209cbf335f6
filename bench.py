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
    def __init__(self, cuda_index: int, period_s: float = 0.004):
        self.period, self.samples, self.mask, self.power = period_s, [], 0, []
        self.sm_max, self._stop, self._thread, self._h, self._nv = None, threading.Event(), None, None, None
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
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

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
