"""Host-side helpers: replica aggregation over torch.distributed, clock sampling, and the chain-sharded
evaluation of Sigma^corr_mm.

bench.py: the timed path does not shard inside one problem (BASELINE.json:north_star: one GPU, no
collectives); with N > 1 GPUs it runs N independent replicas ("replicas only"), and the only
communication is a barrier and a MAX/SUM reduction of the timing scalars.

Chain sharding (sharded_sigma_state): the N_v + N_c Lanczos chains of one state m are independent (one per n,
PAPER.md:87, :155), so each rank takes a contiguous slice of n, runs them on its own GPU with its own replica
of Phi and V, and ONE all-reduce (SUM) of n_omega complex numbers does the sum of Eq. 10.
Nothing is exchanged inside the step loop.  Everything here works on gloo/CPU tensors too (tests)."""
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


def shard_range(n: int, rank: int, world: int, quantum: int = 1):
    """Contiguous slice [lo, hi) of n items for `rank` of `world`.
    quantum = 1: balanced to +-1 item (the first n % world ranks get one more).
    quantum = q > 1: whole tiles of q items are handed out, balanced to +-1 TILE, and the ragged last tile goes with its
    rank; every cut is a multiple of q.  This is the cut for Lanczos chains: a block of chains costs whole GEMM column
    tiles (q = 128 for the wide kernels), so 160 chains cost two tiles exactly like 256 do, and the
    step time of the job is the LARGEST tile count of any rank -- ceil(ceil(n/q) / world), which this cut attains.  Ranks
    beyond the tile count get an empty slice (they could only shorten the job by taking part of a tile, which costs a
    whole one)."""
    n, rank, world, q = int(n), int(rank), int(world), max(1, int(quantum))
    tiles = -(-n // q)
    base, rem = divmod(tiles, world)
    t_lo = rank * base + min(rank, rem)
    t_hi = t_lo + base + (1 if rank < rem else 0)
    return min(t_lo * q, n), min(t_hi * q, n)


def tile_efficiency(n: int, world: int, quantum: int) -> float:
    """Useful columns / columns paid for on the critical path: n / (world * quantum * max tiles of any rank)."""
    q = max(1, int(quantum))
    worst = max(-(-(hi - lo) // q) for lo, hi in (shard_range(n, r, world, q) for r in range(int(world))))
    return float(n) / float(world * q * worst) if worst else 1.0


def sharded_sigma_state(local_sigma_sum, n_orb: int, quantum: int = 1):
    """Sigma^corr_mm(omega) = sum over all n (Eq. 10) with the chains n partitioned over the ranks.
    local_sigma_sum(lo, hi) -> float64 tensor [n_omega, 2] holding the sum over n in [lo, hi) (zeros if empty),
    on the device of the process group's backend.  `quantum`: see shard_range (128 for the GPU path).
    Returns the all-reduced tensor (same on every rank)."""
    import torch.distributed as dist
    on = dist.is_available() and dist.is_initialized()
    rank = dist.get_rank() if on else 0
    world = dist.get_world_size() if on else 1
    lo, hi = shard_range(n_orb, rank, world, quantum)
    part = local_sigma_sum(lo, hi)
    if on and world > 1:
        dist.all_reduce(part, op=dist.ReduceOp.SUM)
    return part


def gwl_local_sigma_sum(ctx, m_idx: int, steps: int, block: int, reorth: int, omega_d, eta: float):
    """local_sigma_sum for sharded_sigma_state on a gwl.Context in device-pointer mode: chains (n, m) for n in
    [lo, hi) through gwl_set_chains / gwl_lanczos / gwl_selfenergy (sum only), result left on the GPU."""
    import numpy as np
    import torch

    def run(lo, hi):
        out = torch.zeros(omega_d.numel(), 2, dtype=torch.float64, device=omega_d.device)
        if hi > lo:
            n = np.arange(lo, hi, dtype=np.int32)
            ctx.set_chains(n, np.full_like(n, m_idx))
            ctx.lanczos(hi - lo, steps, block, reorth, out=None)
            ctx.selfenergy(omega_d, eta, out=(None, out))
        return out
    return run


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
