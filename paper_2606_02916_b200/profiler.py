"""Coefficient measurement for the analytical energy model, re-measured on
this box: the paper's profiler issues initiation probes (loops of single-node fetches) and payload
probes (a sweep over transfer sizes) against every remote owner and fits eps_payload(m, x)
linearly.  Here an owner is a pinned host range and a transfer is one cudaMemcpyAsync, so the
probes are pinned host -> HBM copies of 1 row .. 64 MB timed with CUDA events, and power comes
from NVML.  Measurement harness only (torch for memory / events, NVML for power): none of the
method's arithmetic lives here -- the model is evaluated by gg_simulate.
"""
from __future__ import annotations

import time
from typing import Dict, Optional

import numpy as np
import torch


def _nvml_handle(index: int):
    try:
        import pynvml
        pynvml.nvmlInit()
        return pynvml, pynvml.nvmlDeviceGetHandleByIndex(index)
    except Exception:
        return None, None


def _power_w(nv, h) -> Optional[float]:
    try:
        return nv.nvmlDeviceGetPowerUsage(h) / 1e3
    except Exception:
        return None


def measure_energy_model(device, row_bytes: int, num_parts: int, local_part: int = 0,
                         reps: int = 30) -> Dict:
    """Returns the dict Graph.simulate() takes: per-owner eps_init / eps_pay_* (J), lam_* (s),
    bw (bytes/s), p_idle (W), plus the raw probe table under "probes"."""
    dev = torch.device(device)
    nv, h = _nvml_handle(dev.index or 0)
    torch.cuda.synchronize(dev)
    # NVML power is a ~1 s moving average: let it settle before reading the quiescent baseline
    p_idle = None
    if nv:
        time.sleep(1.0)
        idle = []
        for _ in range(10):
            time.sleep(0.1)
            idle.append(_power_w(nv, h))
        idle = [x for x in idle if x]
        p_idle = float(min(idle)) if idle else None
    sizes = [row_bytes, 4096, 65536, 1 << 20, 1 << 22, 1 << 24, 1 << 26]
    src = torch.empty(max(sizes), dtype=torch.uint8, pin_memory=True)
    dst = torch.empty(max(sizes), dtype=torch.uint8, device=dev)
    probes = []
    for nbytes in sizes:
        best = []
        for _ in range(reps if nbytes < (1 << 24) else 8):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            dst[:nbytes].copy_(src[:nbytes], non_blocking=True)
            b.record()
            b.synchronize()
            best.append(a.elapsed_time(b) * 1e-3)
        probes.append((nbytes, float(np.median(best))))
    # payload probe under sustained load for the active power
    t_end = time.time() + 1.5
    p_act = []
    while time.time() < t_end:
        dst.copy_(src, non_blocking=True)
        torch.cuda.synchronize(dev)
        pw = _power_w(nv, h) if nv else None
        if pw:
            p_act.append(pw)
    p_active = float(np.median(p_act[len(p_act) // 2:])) if p_act else None
    x = np.array([p[0] for p in probes], dtype=np.float64)
    y = np.array([p[1] for p in probes], dtype=np.float64)
    lam_init = float(y[0])                                   # initiation probe: one row
    big = x >= (1 << 20)
    slope = float(np.polyfit(x[big], y[big], 1)[0])          # s per byte, payload-dominated regime
    bw = 1.0 / slope
    p_idle = p_idle if p_idle is not None else 140.0
    p_active = p_active if p_active is not None else p_idle + 60.0
    p_xfer = max(p_active - p_idle, 1.0)                     # power attributable to the transfer
    model = dict(eps_init=[0.0] * num_parts, eps_pay_a=[0.0] * num_parts, eps_pay_b=[0.0] * num_parts,
                 lam_init=[0.0] * num_parts, lam_pay_a=[0.0] * num_parts, lam_pay_b=[0.0] * num_parts,
                 bw=bw, p_idle=p_idle)
    for m in range(num_parts):
        if m == local_part:
            continue
        model["lam_init"][m] = lam_init
        model["lam_pay_b"][m] = slope * row_bytes
        model["eps_init"][m] = p_active * lam_init           # a transfer keeps the device awake for lam_init
        model["eps_pay_b"][m] = p_xfer * slope * row_bytes
    model["probes"] = probes
    model["p_active"] = p_active
    return model
