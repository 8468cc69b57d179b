#!/usr/bin/env python
"""bench.py — throughput of the P_N pseudospectral RTE time step on B200, one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfgX] [--impl ours|reference]

A "step" is one forward-Euler step of the whole hot path (per-axis pencil DFT -> i k ->
IDFT -> moment coupling, scattering diagonal, PML, source, integrator) over the full grid of the workload.
metric = coefficient-cell updates per second = C * G * K / time (BASELINE.json `metric`).

  value       device-resident: state, media and source already in HBM; K rte_step calls bracketed by CUDA events.
  e2e         the same job through the HOST-buffer C-ABI entry points: rte_set_state_host (pinned host -> device),
              K steps, rte_fluence_host (device -> host), all inside the timed region.
  roofline    per-kernel CUDA-event times (rte_step_profile, events on the context's stream) against the algorithmic
              bytes of DESIGN.md "Kernels" and the measured HBM copy bandwidth of MEASURED_PEAKS.json.
  cpu_baseline the fp64 oracle, as it stands, on the host cores, on a bounded sample of the same workload.

N > 1 (torchrun): the path is "replicas only": every rank advances an independent copy of
the workload, no data-path collective; value = units of all ranks / max-over-ranks time.

--impl reference times the oracle (oracle/) on the host cores on a bounded sample of the workload; that arm and the
cpu_baseline leg are the only places this file touches oracle/.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "coefficient-cell updates/s"
UNIT = "coefficient-cells/s"
DEFAULT_WORKLOAD = "cfg4"          # largest single-GPU configuration of BASELINE.json (384^3, P_7, 14.5 GB state)
DEFAULT_STEPS = {"cfg0": 2000, "cfg1": 400, "cfg2": 400, "cfg3": 60, "cfg4": 40}
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# bounded oracle sample per workload: (grid extent, PML width, steps) — ~10-30 s of CPU work on ~8-32 cores
ORACLE_SAMPLE = {"cfg0": (64, 0, 200), "cfg1": (256, 16, 6), "cfg2": (64, 8, 4), "cfg3": (64, 8, 2),
                 "cfg4": (64, 8, 1)}


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD, choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    a = ap.parse_args(argv)
    if a.steps is None:
        a.steps = DEFAULT_STEPS[a.workload]
    a.warmup = max(a.warmup, 3) if a.impl == "ours" else max(a.warmup, 0)
    return a


def hbm_peak():
    """(GB/s, 'measured'|'fallback') — the roofline denominator."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


# ---------------------------------------------------------------------------------------------------------------------
# algorithmic bytes: S = 4*C*G bytes is one fp32 state
# ---------------------------------------------------------------------------------------------------------------------
def algorithmic_bytes(cfg):
    """Bytes each per-axis kernel must move per launch, and per step.  x pass: read psi, write partial (2 S);
    middle pass (3-D y): read psi + partial, write partial (3 S); last pass: read psi + partial, write psi (3 S)
    plus the three per-cell coefficient maps (12 B/cell).  2-D has no middle pass."""
    S = 4 * cfg.C * cfg.G
    per_axis = [2 * S, 3 * S, 3 * S + 12 * cfg.G] if cfg.dim == 3 else [2 * S, 3 * S + 12 * cfg.G, 0]
    return per_axis, sum(per_axis)


# ---------------------------------------------------------------------------------------------------------------------
# clocks sampler (nvidia-smi during the timed region)
# ---------------------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.out = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.out,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        res = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return res
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            self.out.close()
            rows = [ln.strip().split(",") for ln in open(self.path) if ln.strip()]
            os.unlink(self.path)
        except Exception:
            return res
        sm, reasons, smax, pw = [], set(), None, []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                smax = float(r[1])
                pw.append(float(r[2]))
            except ValueError:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.strip().lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            sm.sort()
            res.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=smax, reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw) if pw else None)
        return res
