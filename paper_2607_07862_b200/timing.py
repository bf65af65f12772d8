"""Timing helpers shared by bench.py and the trace CLI: synthetic device inputs, the timed loop, the clock sampler.

No arithmetic of the method lives here, and nothing here touches `oracle/`.  `torch` is passed in by the caller so that
importing this module stays cheap.
"""
from __future__ import annotations

import os
import statistics
import time

N_WEIGHT_SETS = 3  # rotating weight sets: no step can reuse the previous step's weights from L2
L2_BYTES = 126e6


def weight_sets_for(cfg):
    """Rotating weight sets: at least 3, and enough of them that one full rotation is larger than twice the L2 (a small
    config such as cfg 0 would otherwise be served from L2 step after step)."""
    w_bytes = sum(2 * cfg.widths[l] * cfg.widths[l + 1] for l in range(cfg.n_layers))
    return int(min(64, max(N_WEIGHT_SETS, -(-int(2 * L2_BYTES) // w_bytes))))


class ClockSampler:
    """SM clock and throttle reasons DURING the timed region, polled through NVML in a thread (the timed
    region is only milliseconds long, too short for `nvidia-smi -lms`); same fields as the recipe's
    nvidia-smi clocks line in B200_PROFILING.md."""

    def __init__(self, device_index: int):
        self.idx = device_index
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._stop = False
        self._thr = None
        self._h = None

    def start(self):
        try:
            import threading

            import pynvml as nv
            nv.nvmlInit()
            self._nv = nv
            self._h = nv.nvmlDeviceGetHandleByIndex(self.idx)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(self._h, nv.NVML_CLOCK_SM))
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        except Exception:
            self._h = None

    def _loop(self):
        nv = self._nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self._stop:
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self._h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.001)

    def stop(self):
        self._stop = True
        if self._thr is not None:
            self._thr.join(timeout=2)
        out = {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}
        if self.samples:
            out["sm_mhz"] = statistics.median(self.samples)
        return out


def nvml_index_for(torch, dev: int) -> int:
    """NVML index of CUDA device `dev` (they differ under CUDA_VISIBLE_DEVICES)."""
    try:
        import pynvml as nv
        nv.nvmlInit()
        uuid = "GPU-" + str(torch.cuda.get_device_properties(dev).uuid)
        return nv.nvmlDeviceGetIndex(nv.nvmlDeviceGetHandleByUUID(uuid.encode() if isinstance(uuid, str) else uuid))
    except Exception:
        vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
        try:
            return int(vis.split(",")[dev]) if vis else dev
        except Exception:
            return dev


def device_inputs(torch, cfg, n_sets):
    """Synthetic inputs created on the device with the config's distribution (DESIGN.md input recipe):
    X ~ N(0,1) (or U[-1,1] for cfg 0), W_l ~ N(0, 1/fan_in); n_sets independent weight sets."""
    g = torch.Generator(device="cuda")
    g.manual_seed(cfg.seed)

    def draw(shape, scale):
        if cfg.dist == "uniform":
            t = torch.rand(shape, device="cuda", generator=g) * 2 - 1
        else:
            t = torch.randn(shape, device="cuda", generator=g)
        return (t * scale).to(torch.bfloat16)

    X = draw((cfg.M, cfg.widths[0]), 1.0)
    sets = [[draw((cfg.widths[l + 1], cfg.widths[l]), cfg.widths[l] ** -0.5) for l in range(cfg.n_layers)] for _ in range(n_sets)]
    return X, sets


def time_steps(torch, pipe, X, sets, Y, steps, warmup, sampler=None, dist=None):
    """W untimed warm-up steps, then EXACTLY `steps` steps bracketed by barrier + synchronize; per-step
    CUDA events on the launch stream give the latency distribution."""
    n = len(sets)
    for i in range(warmup):
        pipe.run(X, sets[i % n], Y)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    t_all0, t_all1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    if sampler is not None:
        sampler.start()
    torch.cuda._sleep(2_000_000)  # ~1 ms of queue head-room so launches are not host-bound
    t_all0.record()
    for i in range(steps):
        ev[i][0].record()
        pipe.run(X, sets[(warmup + i) % n], Y)
        ev[i][1].record()
    t_all1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    clocks = sampler.stop() if sampler is not None else None
    per = sorted(a.elapsed_time(b) * 1e3 for a, b in ev)
    total_ms = t_all0.elapsed_time(t_all1)
    q = lambda f: per[min(len(per) - 1, int(f * len(per)))]
    return {"median": q(0.5), "p10": q(0.1), "p90": q(0.9), "min": per[0], "mean": sum(per) / len(per),
            "ms_per_step": total_ms / steps}, clocks
