#!/usr/bin/env python
"""bench.py -- overlap D[mu] psi applies/s on B200 (BASELINE.json metric), with roofline and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl native|reference] [--workload cfg3|cfg1] ...

One "step" = one application y = D[mu] psi of the whole hot path (deflation projection,
N fused Wilson/Chebyshev orders, deflation update + overlap assembly) on one lattice.  Default workload = BASELINE
config 3: 20^3 x 64, fp64, 18-real links, mu = 0.01, Chebyshev degree 400, 50 deflation vectors -- the HBM-bound
configuration north_star's 75 % target is quoted on.  The a9 row (D^dag, CG on D^dag D) and the dslash GB/s of the
metric are measured in the same run and reported under "extras" on the same JSON line.

N > 1 (torchrun): the path on one lattice does not shard without a halo exchange, so ranks
are independent replicas with their own right-hand side (propagator-style workload), no data-path collective:
"scaling": "weak"; value = N * applies / max-over-ranks device time.
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

from paper_1510_06897_b200 import inputs  # noqa: E402

WORKLOADS = {
    # name: dims, link eps, stout steps, mu, degree, nev, eps of the polynomial (lower spectral edge / lambda_max)
    "cfg3": dict(dims=(20, 20, 20, 64), link_eps=0.25, stout=3, mu=0.01, degree=400, nev=50, poly_eps=0.95 * 0.5 / 6.5,
                 desc="BASELINE config 3: 20^3x64, U=exp(0.25iH)+3 stout rho=0.1, mu=0.01, degree 400, 50 deflation vectors"),
    "cfg1": dict(dims=(8, 8, 8, 32), link_eps=0.3, stout=3, mu=0.01, degree=200, nev=20, poly_eps=0.95 * 0.505 / 6.5,
                 desc="BASELINE config 1: 8^3x32, U=exp(0.3iH)+3 stout rho=0.1, mu=0.01, degree 200, 20 deflation vectors"),
    "tiny": dict(dims=(4, 4, 4, 8), link_eps=0.3, stout=1, mu=0.01, degree=40, nev=4, poly_eps=0.09,
                 desc="4^3x8 smoke-sized workload (not a benchmark)"),
}
METRIC = "overlap D[mu]psi applies/s"
UNIT = "applies/s"


def make_inputs(w, seed_off=0, need_phi=True):
    """Seeded synthetic stand-ins for the paper's ensembles (DESIGN.md input recipe)."""
    dims = w["dims"]
    k = {"cfg3": 3, "cfg1": 1, "tiny": 9}.get(w.get("name", ""), 7)
    U = inputs.config_links(dims, w["link_eps"], inputs.SEED_BASE + k, stout_steps=w["stout"])
    psi = inputs.gaussian_spinor(dims, inputs.SEED_BASE + 100 + k + 1000 * seed_off)
    alpha = inputs.chebyshev_sign_coeffs(w["degree"], w["poly_eps"])
    nev = w["nev"]
    phi = inputs.phase_vectors(dims, nev, inputs.SEED_BASE + 200 + k) if (nev and need_phi) else None
    lam = 0.5 * np.where(np.arange(nev) % 2 == 0, 1.0, -1.0) * (1.0 + 0.002 * np.arange(nev))
    return U, psi, alpha, phi, lam


def poly_bytes(alpha, V, prec_bytes, recon):
    """Algorithmic (compulsory) HBM bytes of the polynomial loop, summed order by order:
    every order reads t_m (S) and the 4 links a site owns (4L); reads t_{m-1} (S) from the second order on; writes
    t_{m+1} (S) except in the last order; reads+writes the accumulator (2S) when alpha_{m+1} != 0 (write only in the
    first order)."""
    S = 24 * prec_bytes
    L = recon * prec_bytes
    last = max(1, max([m for m in range(1, len(alpha)) if alpha[m] != 0.0] or [1]))
    total = 0
    for m in range(last):  # order m produces t_{m+1}
        b = S + 4 * L
        if m >= 1:
            b += S
        if m + 1 < last:
            b += S
        if m == 0:
            b += S
        elif alpha[m + 1] != 0.0:
            b += 2 * S
        total += b
    return total * V, last


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML; nvidia-smi fallback)."""

    def __init__(self, index=0, period=0.02):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.index, self.period = index, period
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
                 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
                 0x10: "sync_boost"}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        if self.nv is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml_unavailable"]}
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"
