"""Host-side helpers for bench.py: replica aggregation over torch.distributed and clock sampling.

The path does not shard inside one problem (BASELINE.json:north_star: one GPU, no collectives); with
N > 1 GPUs bench.py runs N independent replicas ("replicas only").  The only communication is
a barrier and a MAX/SUM reduction of the timing scalars, done here so that it can be tested with gloo."""
from __future__ import annotations

import os
import subprocess
import threading
import time


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def aggregate_throughput(units_local: float, elapsed_s_local: float, device=None):
    """(sum of units over ranks, max of elapsed over ranks).  Single process: passthrough."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(units_local), float(elapsed_s_local)
    t = torch.tensor([elapsed_s_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()), float(t.item())


def whole_job_value(units_local: float, elapsed_s_local: float, device=None) -> float:
    """Whole-job throughput = units all ranks processed / max-over-ranks time."""
    u, t = aggregate_throughput(units_local, elapsed_s_local, device)
    return u / t if t > 0 else 0.0


_REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
            0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}


class ClockSampler:
    """Samples SM clock and throttle reasons every `period` s on a background thread (NVML, else nvidia-smi)."""

    def __init__(self, index: int = 0, period: float = 0.1):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._nvml = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self._nvml = None

    def _sample_once(self):
        if self._nvml is not None:
            nv = self._nvml
            mhz = float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
            try:
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self._h))
            except Exception:
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h))
            self.samples.append(mhz)
            for bit, name in _REASONS.items():
                if mask & bit:
                    self.reasons.add(name)
        else:
            q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
                "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
            r = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=10)
            f = [x.strip() for x in r.stdout.strip().split(",")]
            self.samples.append(float(f[0]))
            self.max_mhz = float(f[1])
            for flag, name in zip(f[2:], ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]):
                if flag.lower().startswith("active"):
                    self.reasons.add(name)

    def _run(self):
        while not self._stop.is_set():
            try:
                self._sample_once()
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        self._thr = threading.Thread(target=self._run, daemon=True)
        self._thr.start()
        return self

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join(timeout=5)
        s = sorted(self.samples)
        med = s[len(s) // 2] if s else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(s)}
