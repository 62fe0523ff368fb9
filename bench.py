#!/usr/bin/env python
"""bench.py -- DG DoF-updates/s per RK stage on one B200 (BASELINE.json metric), with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4|cfg5|cfg2|cfg3|cfg1] [--degree n]
    python bench.py --impl reference ...          # the CPU oracle, as it stands, on a bounded sample

A "step" is one full SSP-RK3 time step = 3 passes of the fused stage kernel (all rows of SURVEY.md 8(a)) over
the whole synthetic mesh, plus the Eq.-23 timestep kernel.  `value` = cells * M * V * 3 * K / t with the state
resident in HBM; `e2e` = the same through the C-ABI with HOST buffers (dg_set_state + dg_step + dg_get_state
inside the timed region).  The path does not shard ("replicas only"): with --gpus N every rank runs
an independent replica and `value` is the sum.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2208_11131_b200 import roofline as rl          # noqa: E402
from paper_2208_11131_b200 import workloads as wk         # noqa: E402

METRIC = "DG DoF-updates/sec (fp64, per RK stage)"
UNIT = "DoF-updates/s"


def pick_workload(name: str, degree):
    i = int(name[3])
    wl = wk.config(i, degree=degree)
    label = {1: "cfg1 2D advected wave 16x16 Euler", 2: "cfg2 2D Kelvin-Helmholtz 128x256 NS",
             3: "cfg3 2D Sod tube 1024x16 Euler+AV", 4: "cfg4 3D turbulence box 128^3 NS+AV",
             5: "cfg5 3D advected wave 64^3 Euler"}[i]
    return wl, "%s, degree %d (order %d, %d modes/cell)" % (label, wl.degree, wl.order, wl.modes)


def measured_peaks():
    """(hbm_gbs, which) from MEASURED_PEAKS.json, else the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index=0, period=0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10}
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def oracle_sample(wl, budget_cells=None):
    """Time the CPU oracle, as it stands, on a bounded sample of `wl`: the same problem (ICs, physics, degree)
    on a coarser mesh of the same domain, one full RK3 step.  Returns (dof_updates_per_s, cores, text)."""
    from oracle import dg_oracle as orc
    per_cell = wl.modes ** 2 * wl.nvar               # dense per-cell operators: cost ~ M^2 V
    if budget_cells is None:
        budget_cells = max(8, int(6.0e8 / per_cell))
    n1 = max(2, int(round(budget_cells ** (1.0 / wl.dim))))
    n1 = min(n1, wl.ncell[0])
    ncell = tuple(max(2, int(round(n1 * wl.ncell[a] / wl.ncell[0]))) for a in range(wl.dim))
    sub = wk.with_mesh(wl, ncell)
    w0 = wk.initial_modes(sub)
    o = orc.DGOracle(sub.dim, sub.ncell, sub.h, sub.order, sub.gamma, sub.nu, sub.chi,
                     orc.Options(f_cfl=sub.f_cfl, av_enable=sub.av))
    o.set_state(w0)
    o.step(1)                                          # warm-up (also the lagged AV sensor becomes non-trivial)
    c0, t0 = time.process_time(), time.perf_counter()
    nst = 2
    o.step(nst)
    wall = time.perf_counter() - t0
    cpu = time.process_time() - c0
    cores = max(1, int(round(cpu / wall)))
    dof = sub.ncells * sub.modes * sub.nvar * 3 * nst / wall
    text = "%d RK3 steps of the numpy oracle on %s cells (same ICs/physics/degree as the workload)" % (
        nst, "x".join(str(c) for c in sub.ncell))
    return dof, cores, text, wall
