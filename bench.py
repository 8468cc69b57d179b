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
DEFAULT_STEPS = {"cfg0": 2000, "cfg1": 400, "cfg2": 400, "cfg3": 60, "cfg4": 40,
                 "paper_exp1": 400, "paper_exp2": 25000}       # the paper's own step counts
FALLBACK_HBM_GBS = 6650.0          # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# bounded oracle sample per workload: (grid extent, PML width, steps) — ~10-30 s of CPU work on ~8-32 cores
ORACLE_SAMPLE = {"cfg0": (64, 0, 200), "cfg1": (256, 16, 6), "cfg2": (64, 8, 4), "cfg3": (64, 8, 2),
                 "cfg4": (96, 8, 2), "paper_exp1": (32, 0, 3), "paper_exp2": (64, 9, 12)}
# the paper's wall-clock for its two runs on a Tesla K40 (context, not the target): seconds for all steps
PAPER_WALL_S = {"paper_exp1": (70.0, "PAPER.md:141"), "paper_exp2": (223.0, "PAPER.md:167")}


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD,
                    choices=["cfg0", "cfg1", "cfg2", "cfg3", "cfg4", "paper_exp1", "paper_exp2"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "cufft_literal"],
                    help="ours: the product; reference: the fp64 oracle on the host cores; cufft_literal: the paper's own "
                         "GPU structure (3-D cuFFT per complex field + eq.(10) k-space kernel + pointwise kernel) as a timed "
                         "reference point on the same box (SURVEY 8(f4), 3-D workloads)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    ap.add_argument("--no-others", action="store_true", help="skip the short cfg2/cfg3 side measurements")
    ap.add_argument("--oracle-full-size", action="store_true",
                    help="time the oracle leg (cpu_baseline / --impl reference) on the FULL workload for 2 steps instead of the "
                         "bounded sample (cfg2: seconds, cfg3: ~1 min on 16 cores; cfg4: ~90 GB of host RAM and ~5 min)")
    ap.add_argument("--krylov-plain", action="store_true",
                    help="with --steady-state: also run unpreconditioned GMRES(30) on L psi = q (minutes on cfg3)")
    ap.add_argument("--steady-state", action="store_true",
                    help="also run the workload to the steady-state criterion of configs[3] (DESIGN.md R17) with the "
                         "SSP-RK3 integrator at dt = 0.3 dx/c and report steps / seconds (constant-source workloads)")
    a = ap.parse_args(argv)
    global FULL_SIZE_ORACLE
    FULL_SIZE_ORACLE = bool(a.oracle_full_size)
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
def first_axis(cfg):
    """Axis of the FIRST pass (the one that stores the new buffer; the others add to it): x.  (FIRST on z, whose coupling
    has the smaller fan-in, was measured and rejected: DESIGN.md 6.)"""
    return 0


def algorithmic_bytes(cfg):
    """Bytes each per-axis kernel must move per launch, and per step.  FIRST pass: read psi and the three per-cell
    coefficient maps (12 B/cell), write the new buffer (2 S + 12 G); every other pass: read psi, read + write the new
    buffer (the reductions are read-modify-write in the L2: 3 S).  2-D has no z pass."""
    S = 4 * cfg.C * cfg.G
    per_axis = [3 * S, 3 * S, 3 * S if cfg.dim == 3 else 0]
    per_axis[first_axis(cfg)] = 2 * S + 12 * cfg.G
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


# ---------------------------------------------------------------------------------------------------------------------
# the oracle legs (the only code in this file that touches oracle/)
# ---------------------------------------------------------------------------------------------------------------------
FULL_SIZE_ORACLE = False


def oracle_sample_config(wl, cfg):
    n, W, steps = ORACLE_SAMPLE[cfg.name]
    if FULL_SIZE_ORACLE:      # cfg4: ~90 GB of host memory at the peak (three fp64 fields of 29 GB), ~2 min per step on 16 cores
        return cfg, 2, f"{cfg.name} at FULL size ({cfg.nx}^{cfg.dim}, C={cfg.C}), 2 steps"
    if n >= max(cfg.nx, cfg.ny, cfg.nz):
        return cfg, min(steps, cfg.steps), f"{cfg.name} at full size, {min(steps, cfg.steps)} step(s)"
    small = wl.reduced(cfg, n, pml_width=W)
    what = f"{cfg.name} structure (P_{cfg.N}, C={cfg.C}) on a {n}^{cfg.dim} grid, PML {small.pml[0]} cells, {steps} step(s)"
    return small, steps, what


def time_oracle(wl, cfg, repeats=1):
    """Seconds per oracle step on the bounded sample, units (coefficient-cells) per step, threads, description."""
    import numpy as np
    from oracle import rte_oracle as orc
    small, steps, what = oracle_sample_config(wl, cfg)
    if small.media == "lognormal":      # the CPU generator costs more than the timed steps; a seeded smooth stand-in
        rng = np.random.default_rng(small.seed)
        mu = (np.full(small.shape, small.background[0], np.float32),
              (small.background[1] * np.exp(0.3 * rng.standard_normal(small.shape))).astype(np.float32),
              np.full(small.shape, small.background[2], np.float32))
    else:
        mu = wl.media_maps(small)
    o = orc.Oracle(small.dim, small.nx, small.ny, small.nz, small.N, small.dx, small.dt, small.c, *mu, *small.pml)
    o.set_state(wl.random_state(small, seed=1))
    src = wl.source_term(small)
    if src is not None:
        o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    best = float("inf")
    for _ in range(repeats):
        t0 = time.perf_counter()
        o.step(steps)
        best = min(best, time.perf_counter() - t0)
    o.close()
    return best / steps, small.C * small.G, orc.num_threads(), what


def run_reference(args, wl, cfg):
    """--impl reference: the fp64 oracle on the host cores; one 'step' = one oracle step on the bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np
    from oracle import rte_oracle as orc
    small, _, what = oracle_sample_config(wl, cfg)
    mu = tuple(np.full(small.shape, v, np.float32) for v in small.background) if small.media == "lognormal" \
        else wl.media_maps(small)
    o = orc.Oracle(small.dim, small.nx, small.ny, small.nz, small.N, small.dx, small.dt, small.c, *mu, *small.pml)
    o.set_state(wl.random_state(small, seed=1))
    src = wl.source_term(small)
    if src is not None:
        o.set_source(src["w"], src["S"], src["origin"], src["extent"], src["kind"], src["t0"], src["sigma_t"])
    if args.warmup:
        o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    sec = time.perf_counter() - t0
    value = small.C * small.G * args.steps / sec
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sec / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg.name, "sample": what},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": what},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------------------
def device_media(rte, wl, cfg, torch, dev):
    """Media maps generated ON THE DEVICE by the geometry layer (north_star item (3)); scalars for homogeneous."""
    if cfg.media == "homogeneous":
        return cfg.background
    if cfg.media == "slab":         # the paper's sharp mu_s step (exp. 1): a tiny host-made map
        return tuple(torch.from_numpy(m).to(dev) for m in wl.media_maps(cfg))
    if cfg.media in ("disks", "ellipsoids"):
        a, s, g = (torch.empty(cfg.shape, dtype=torch.float32, device=dev) for _ in range(3))
        rte.rte_media_ellipsoids(cfg.grid, cfg.dx, cfg.background, wl.inclusion_list(cfg), a, s, g)
        return a, s, g
    if cfg.media == "lognormal":
        s = torch.empty(cfg.shape, dtype=torch.float32, device=dev)
        scratch = torch.empty_like(s)
        rte.rte_media_lognormal(cfg.grid, cfg.dx, cfg.seed, cfg.background[1], cfg.extra["sigma_log"],
                                cfg.extra["corr_len_mm"], s, scratch)
        torch.cuda.synchronize()
        del scratch
        return cfg.background[0], s, cfg.background[2]
    raise ValueError(cfg.media)


def make_context(rte, wl, cfg, torch, dev):
    mu_a, mu_s, g = device_media(rte, wl, cfg, torch, dev)
    ctx = rte.rte_create(cfg.grid, cfg.N, cfg.dx, cfg.dt, cfg.c, mu_a, mu_s, g, cfg.pml)
    src = wl.source_term(cfg)
    if src is not None:
        rte.rte_set_source(ctx, src["w"], torch.from_numpy(src["S"]).to(dev), src["origin"], src["extent"],
                           src["kind"], src["t0"], src["sigma_t"])
    return ctx


def device_initial_state(wl, cfg, torch, dev):
    """psi(0) [C,nz,ny,nx] on the device.  The pulse configs start from their delta / Gaussian initial radiance plus a
    weak seeded random background (1e-3 of the pulse scale) so that every cell carries non-trivial data; the fields'
    values do not change the work done."""
    psi = torch.zeros((cfg.C,) + cfg.shape, dtype=torch.float32, device=dev)
    gen = torch.Generator(device=dev)
    gen.manual_seed(cfg.seed)
    for c in range(cfg.C):
        psi[c].normal_(0.0, 1e-3, generator=gen)
    if cfg.source in ("gaussian_pulse_ic", "point_pulse_ic"):
        cz = cfg.nz // 2 if cfg.dim == 3 else 0
        if cfg.source == "point_pulse_ic":
            psi[0, cz, cfg.ny // 2, cfg.nx // 2] += 1.0
        else:
            S, org, ext = wl.gaussian_footprint(cfg, (cfg.nx // 2, cfg.ny // 2, cz), cfg.extra["sigma_mm"])
            psi[0, org[2]:org[2] + ext[2], org[1]:org[1] + ext[1], org[0]:org[0] + ext[0]] += \
                torch.from_numpy(S).to(dev) * (cfg.dx ** cfg.dim)
    return psi


def timed_steps(rte, ctx, torch, steps, dist=None):
    """K steps bracketed by barrier + synchronize on both sides; device time by CUDA events on the launch stream."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    rte.rte_step(ctx, steps)
    e1.record()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    return e0.elapsed_time(e1)


def measure_workload(rte, wl, cfg, torch, dev, steps, warmup, dist=None, sampler=None):
    """Device-resident throughput + per-axis kernel times for one workload.  Returns a dict."""
    ctx = make_context(rte, wl, cfg, torch, dev)
    psi0 = device_initial_state(wl, cfg, torch, dev)
    rte.rte_set_state(ctx, psi0)
    del psi0
    rte.rte_step(ctx, warmup)
    rte.rte_sync(ctx)
    l0 = rte.rte_launch_count(ctx)
    if sampler is not None:
        sampler.start()
    ms = timed_steps(rte, ctx, torch, steps, dist)
    clocks = sampler.stop() if sampler is not None else None
    launches = rte.rte_launch_count(ctx) - l0
    # per-kernel times, measured live with CUDA events on the context's stream (same launch configuration)
    nprof = max(3, min(steps, 20))
    ms_axis, n_axis = rte.rte_step_profile(ctx, nprof)
    phi = torch.empty(cfg.shape, dtype=torch.float32, device=dev)
    rte.rte_fluence(ctx, phi)
    rte.rte_sync(ctx)
    finite = bool(torch.isfinite(phi).all().item())
    return dict(ctx=ctx, ms=ms, launches=launches, clocks=clocks, finite=finite,
                ms_axis=[m / max(1, n) for m, n in zip(ms_axis, n_axis)], prof_steps=nprof)


def roofline_of(cfg, res, peak, peak_kind):
    per_axis, per_step = algorithmic_bytes(cfg)
    naxes = cfg.dim
    fa = first_axis(cfg)
    names = [f"pass_{'xyz'[a]} (" + ("first: coupling, DFT-ik-IDFT, sigma_l, PML, source -> stores the new buffer)" if a == fa
                                     else "coupling, DFT-ik-IDFT -> vector reductions into the new buffer)") for a in range(3)]
    dom = max(range(naxes), key=lambda a: res["ms_axis"][a])
    ach = per_axis[dom] / (res["ms_axis"][dom] * 1e-3) / 1e9
    kernels = []
    for a in range(naxes):
        gbs = per_axis[a] / (res["ms_axis"][a] * 1e-3) / 1e9
        kernels.append({"kernel": names[a], "ms": res["ms_axis"][a], "algorithmic_bytes": per_axis[a],
                        "achieved_gbs": gbs, "frac": gbs / peak})
    step_gbs = per_step / (1e-3 * sum(res["ms_axis"][:naxes])) / 1e9
    return {"bound": "hbm", "kernel": names[dom], "achieved": ach, "peak": peak, "peak_kind": peak_kind + " (burst copy)",
            "unit": "GB/s", "frac": ach / peak, "traffic": TRAFFIC_NCU.get(cfg.name, {}).get(dom),
            "bytes_per_coefficient_cell_step": per_step / (cfg.C * cfg.G),
            "whole_step": {"algorithmic_bytes": per_step, "achieved_gbs": step_gbs, "frac": step_gbs / peak,
                           "frac_of_nominal_8000": step_gbs / 8000.0},
            "kernels": kernels,
            "note": "fractions are of the HBM roofline; the FIRST (x) pass is limited by the SM load/store data path (ncu: 65-70 % "
                    "busy at 16 warps per SM, profiles/), the accumulating passes by HBM"}


# dram__bytes_read.sum + dram__bytes_write.sum per launch of each axis kernel, from the committed ncu --set full
# captures under profiles/ (filled in from the capture named there; None until one exists for that workload)
TRAFFIC_NCU = {"cfg4": {0: 29826771000, 1: 43432582000, 2: 43432402000},       # profiles/r2r_summary.md §3 (ncu --set full,
               "cfg3": {0: 5007557999, 1: 7193890000, 2: 7201423999},          # one launch per axis kernel)
               "cfg2": {0: 246775552, 1: 345737728, 2: 346095360}}


def max_over_ranks(ms, dist, device):
    """Device time of the job = the slowest rank's (replicas only: no data-path collective; this one scalar all-reduce
    is the only communication, outside the timed region)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(cfg, steps, world, ms):
    """Whole-job throughput: every rank advances its own replica of the workload (weak scaling)."""
    return cfg.C * cfg.G * steps * world / (ms * 1e-3)


def steady_state_run(rte, wl, cfg, torch, dev, max_steps=20000, tol=1e-6, plain_krylov=False):
    """configs[3]: "stepped to steady state (until relative change in l=0 fluence < 1e-6 per 100 steps)" (R17).  With the
    paper's forward Euler the stable dt of cfg3 (0.1 fs) makes that 1e5-1e6 steps; the SSP-RK3 step (not the
    paper's integrator) is stable at dt = 0.3 dx/c, hundreds of times larger, and gets there in seconds."""
    from dataclasses import replace
    dt = 0.3 * cfg.dx / cfg.c
    c2 = replace(cfg, dt=dt)
    ctx = make_context(rte, wl, c2, torch, dev)
    rte.rte_set_state(ctx, torch.zeros((cfg.C,) + cfg.shape, dtype=torch.float32, device=dev))
    rte.rte_fluence_change(ctx)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    steps, change, hist = 0, float("inf"), []
    while steps < max_steps:
        rte.rte_step_ssprk3(ctx, 100)
        steps += 100
        change = rte.rte_fluence_change(ctx)       # synchronises
        hist.append(change)
        if not math.isfinite(change) and steps > 100:
            break
        if change < tol:
            break
    sec = time.perf_counter() - t0
    rk = {"integrator": "ssprk3 (non-paper)", "dt_ps": dt, "euler_dt_ps": cfg.dt, "steps": steps, "seconds": sec,
          "operator_applications": 3 * steps,
          "simulated_ps": steps * dt, "criterion": f"relative L2 change of the fluence over Omega per 100 steps < {tol:g}",
          "final_change": change, "converged": bool(change < tol),
          "change_every_1000_steps": [hist[i] for i in range(9, len(hist), 10)][:20]}
    phi_rk = torch.empty(cfg.shape, dtype=torch.float32, device=dev)
    rte.rte_fluence(ctx, phi_rk)
    rte.rte_sync(ctx)
    ctx0 = ctx
    del ctx
    # SURVEY 8(f1) / PAPER.md:109,195: the same steady state by the device-resident Krylov solver, L psi = q
    out = {"ssprk3": rk}
    # the true residual ||q - L psi|| / ||q|| of the time-stepped state: a solve that stops before its first cycle
    _, rk["true_relative_residual_of_the_final_state"] = rte.rte_solve_steady(ctx0, restart=1, tol=1e-30, max_restarts=0)
    del ctx0
    torch.cuda.empty_cache()
    dtp = 0.3 * cfg.dx / cfg.c
    # restart 40 needs 46 state-sized fields of extra workspace (cfg3: 111 GB); smaller boards: restart 20 (26 fields, ~20 % slower)
    free_b, _ = torch.cuda.mem_get_info()
    field_b = 4 * cfg.G * (cfg.C + cfg.C % 2)
    restart = 40 if free_b > 50 * field_b else 20
    variants = [(f"gmres{restart}_rk3x8", dict(restart=restart, tol=1e-5, max_restarts=100, precond_steps=8, precond_dt_ps=dtp))]
    if plain_krylov:
        variants.append(("gmres30_plain", dict(restart=30, tol=1e-5, max_restarts=400)))
    for name, kw in variants:
        ctx = make_context(rte, wl, cfg, torch, dev)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        napp, rr = rte.rte_solve_steady(ctx, **kw)
        rte.rte_sync(ctx)
        ksec = time.perf_counter() - t0
        phi_k = torch.empty(cfg.shape, dtype=torch.float32, device=dev)
        rte.rte_fluence(ctx, phi_k)
        rte.rte_sync(ctx)
        diff = float((phi_k - phi_rk).norm() / phi_rk.norm())
        out[name] = {"solver": "rte_solve_steady: device-resident restarted GMRES" +
                               (" on (I - Phi^s) psi = Phi^s(0; q), Phi = SSP-RK3 step" if kw.get("precond_steps") else " on L psi = q"),
                     **{k: v for k, v in kw.items()}, "seconds": ksec, "operator_sweeps": napp,
                     "true_relative_residual": rr, "converged": bool(rr <= kw["tol"]),
                     "extra_workspace_fields": kw["restart"] + 3 + (3 if kw.get("precond_steps") else 0),
                     "fluence_rel_l2_difference_from_the_time_stepped_state": diff}
        del ctx, phi_k
        torch.cuda.empty_cache()
    return out


def run_cufft_literal(args, wl, cfg):
    """The paper's structure on this box: a reference point for DESIGN.md 7, not the product."""
    import torch
    if cfg.dim != 3:
        print(json.dumps({"impl": "cufft_literal", "unavailable": "the literal variant is 3-D only"}), flush=True)
        return 0
    import paper_1801_06364_b200 as rte
    from baseline import cufft_literal as cl
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    torch.cuda.set_device(0)
    dev = torch.device("cuda:0")
    peak, peak_kind = hbm_peak()
    mu_a, mu_s, g = device_media(rte, wl, cfg, torch, dev)
    full = lambda v: v if isinstance(v, torch.Tensor) else torch.full(cfg.shape, float(v), dtype=torch.float32, device=dev)
    mu_b = torch.empty(cfg.shape, dtype=torch.float32, device=dev)
    inside = torch.empty(cfg.shape, dtype=torch.uint8, device=dev)
    rte.rte_pml_profile(cfg.grid, cfg.pml, mu_b, inside)
    torch.cuda.synchronize()
    sa = torch.where(inside.bool(), full(mu_a), mu_b)
    ss = torch.where(inside.bool(), full(mu_s), torch.zeros_like(mu_b))
    gm = full(g).clone()
    del mu_b, inside, mu_a, mu_s, g
    sol = cl.Solver(cfg.nx, cfg.ny, cfg.nz, cfg.N, cfg.dx, cfg.dt, cfg.c, sa, ss, gm)
    psi = device_initial_state(wl, cfg, torch, dev)
    pc = cl.real_to_complex(psi)
    del psi
    sol.set_state(pc)
    del pc
    torch.cuda.empty_cache()
    sol.step(args.warmup)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    l0 = sol.own_kernel_launches()
    e0.record()
    sol.step(args.steps)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    finite = bool(torch.isfinite(torch.view_as_real(sol.get_state()[0])).all().item())
    S = 4 * cfg.C * cfg.G
    # its own minimal traffic on the same accounting (S = one REAL fp32 state; its fields are complex, 2 S per sweep):
    # forward 3-D FFT >= read + write (4 S), k-space kernel read + write (4 S), inverse FFT (4 S), pointwise read psi,
    # read T, write psi (6 S) = 18 S when every 3-D FFT makes ONE pass over its field (it makes more)
    line = {"impl": "cufft_literal", "metric": METRIC, "value": cfg.C * cfg.G * args.steps / (ms * 1e-3), "unit": UNIT,
            "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c64", "data": "synthetic",
            "config": {"workload": cfg.name, "structure": "PAPER.md:123-131: 3-D C2C cuFFT per complex field, eq.(10) in k-space, "
                       "inverse cuFFT, pointwise potential + eq.(11); no source term", "complex_fields": cfg.C,
                       "device_bytes": sol.device_bytes()},
            "gpu_launches": sol.own_kernel_launches() - l0, "cufft_execs_per_step": 2 * cfg.C, "finite": finite,
            "traffic_model_bytes_per_step_lower_bound": 18 * S,
            "effective_gbs_of_the_products_8S_model": (8 * S + 12 * cfg.G) / (ms / args.steps * 1e-3) / 1e9,
            "hbm_peak_gbs": peak, "peak_kind": peak_kind}
    print(json.dumps(line), flush=True)
    return 0


def run_ours(args, wl, cfg):
    import torch
    try:
        import paper_1801_06364_b200 as rte
    except ImportError as e:     # fail loudly: there is no fallback path
        print(f"bench.py: the CUDA library is not built: {e}", file=sys.stderr)
        return 2
    if not torch.cuda.is_available():
        print("bench.py: no CUDA device; this path has no CPU fallback", file=sys.stderr)
        return 2
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    torch.cuda.set_device(local)
    dev = torch.device(f"cuda:{local}")
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=dev)
        dist = dist_mod
    peak, peak_kind = hbm_peak()

    sampler = ClockSampler(local) if rank == 0 else None
    res = measure_workload(rte, wl, cfg, torch, dev, args.steps, args.warmup, dist, sampler)
    ms = max_over_ranks(res["ms"], dist, dev)
    units = cfg.C * cfg.G * args.steps * world
    value = job_value(cfg, args.steps, world, ms)
    ctx = res["ctx"]

    # ---- e2e: host buffers through the C ABI (pinned host -> device state, K steps, fluence device -> host) ----------
    e2e = None
    if not args.no_e2e:
        h_state = torch.empty((cfg.C,) + cfg.shape, dtype=torch.float32, pin_memory=True)
        rte.rte_get_state_host(ctx, h_state)            # a real state to upload
        h_phi = torch.empty(cfg.shape, dtype=torch.float32, pin_memory=True)
        rte.rte_set_state_host(ctx, h_state)            # warm the path once
        rte.rte_step(ctx, 1)
        rte.rte_fluence_host(ctx, h_phi)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        e0.record()
        rte.rte_set_state_host(ctx, h_state)
        rte.rte_step(ctx, args.steps)
        rte.rte_fluence_host(ctx, h_phi)                # synchronises the stream
        e1.record()
        torch.cuda.synchronize()
        wall_ms = 1e3 * (time.perf_counter() - t0)
        e_ms = max(e0.elapsed_time(e1), wall_ms)
        e_ms = max_over_ranks(e_ms, dist, dev)
        e2e = {"value": units / (e_ms * 1e-3), "unit": UNIT, "ms_total": e_ms,
               "h2d_bytes_per_step": h_state.numel() * 4 / args.steps, "d2h_bytes_per_step": h_phi.numel() * 4 / args.steps,
               "what": f"rte_set_state_host (pinned, {h_state.numel() * 4 / 1e9:.2f} GB) + {args.steps} x rte_step + rte_fluence_host, per rank"}
        del h_state, h_phi

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    roof = roofline_of(cfg, res, peak, peak_kind)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "grid": [cfg.nx, cfg.ny, cfg.nz][:cfg.dim], "P_N": cfg.N, "coefficients": cfg.C,
                       "cells": cfg.G, "state_bytes": 4 * cfg.C * cfg.G, "dx_mm": cfg.dx, "dt_ps": cfg.dt,
                       "pml_cells": cfg.pml[0], "media": cfg.media, "source": cfg.source,
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "state larger than L2 (no flush needed)" if 4 * cfg.C * cfg.G > 2 * 126e6
                             else "state comparable to / smaller than the 126 MB L2: DRAM fraction not meaningful"},
            "clocks": res["clocks"], "e2e": e2e, "gpu_launches": res["launches"], "finite": res["finite"],
            "roofline": roof,
            "paper_context": {"k40_updates_per_s_complex": [7.25e8, 1.88e9], "source": "PAPER.md:141,167 (Tesla K40; context only)"}}

    if cfg.name in PAPER_WALL_S:
        k40_s, where = PAPER_WALL_S[cfg.name]
        line["paper_run"] = {"steps": cfg.steps, "this_run_seconds_for_those_steps": ms / args.steps * cfg.steps * 1e-3,
                             "paper_seconds_tesla_k40": k40_s, "source": where,
                             "note": "the paper's own parameter set; its hardware, precision unstated: context only"}

    if not args.no_others and world == 1:
        # side measurement (not the paper's integrator): SSP-RK3 = 3 Euler updates, stage combinations fused in
        k = max(2, args.steps // 8)
        rte.rte_step_ssprk3(ctx, 1)                    # allocates the third state buffer, warms up
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        rte.rte_step_ssprk3(ctx, k)
        e1.record()
        torch.cuda.synchronize()
        rk_ms = e0.elapsed_time(e1) / k
        S = 4 * cfg.C * cfg.G
        rk_bytes = 3 * roof["whole_step"]["algorithmic_bytes"] + 2 * S      # stages 2, 3 also read u^n in their FIRST pass
        line["ssprk3"] = {"ms_per_step": rk_ms, "steps": k, "algorithmic_bytes_per_step": rk_bytes,
                          "frac_of_hbm_roofline": rk_bytes / (rk_ms * 1e-3) / 1e9 / peak,
                          "note": "non-paper integrator; stable up to dt ~ dx/c, i.e. tens of times the Euler dt"}
        rte.rte_set_extra_workspace(ctx, 0)
        torch.cuda.empty_cache()
        # side measurement: exponential Euler step, generic kernels, diagonal table in every pass
        rte.rte_step_exp(ctx, 1)
        torch.cuda.synchronize()
        e0.record()
        rte.rte_step_exp(ctx, k)
        e1.record()
        torch.cuda.synchronize()
        ex_ms = e0.elapsed_time(e1) / k
        S_ = 4 * cfg.C * cfg.G
        spec_grid = cfg.name in ("cfg0", "cfg1", "cfg2", "cfg3", "cfg4", "paper_exp2")
        # specialised grids: 3 passes for -c dt T (no maps) + one pointwise kernel (read psi, read + write the new buffer, 3 maps)
        ex_bytes = (roof["whole_step"]["algorithmic_bytes"] + 3 * S_) if spec_grid \
            else roof["whole_step"]["algorithmic_bytes"] + 2 * 12 * cfg.G * (cfg.dim - 1)
        line["exp_step"] = {"ms_per_step": ex_ms, "steps": k, "algorithmic_bytes_per_step": ex_bytes,
                            "frac_of_hbm_roofline": ex_bytes / (ex_ms * 1e-3) / 1e9 / peak,
                            "note": "rte_step_exp: exact diagonal exp(-c dt sigma_l); " +
                                    ("specialised passes for -c dt T + one pointwise exp/phi_1/source kernel" if spec_grid
                                     else "fused into the generic kernels")}

    if not args.no_others and world == 1 and cfg.name == DEFAULT_WORKLOAD:
        del res, ctx
        torch.cuda.empty_cache()
        others = {}
        for name in ("cfg2", "cfg3"):
            c2 = wl.CONFIGS[name]
            r2 = measure_workload(rte, wl, c2, torch, dev, DEFAULT_STEPS[name], max(3, args.warmup))
            rf = roofline_of(c2, r2, peak, peak_kind)
            others[name] = {"ms_per_step": r2["ms"] / DEFAULT_STEPS[name],
                            "value": c2.C * c2.G * DEFAULT_STEPS[name] / (r2["ms"] * 1e-3),
                            "whole_step_frac": rf["whole_step"]["frac"],
                            "whole_step_frac_of_nominal_8000": rf["whole_step"]["frac_of_nominal_8000"],
                            "dominant_kernel_frac": rf["frac"], "finite": r2["finite"]}
            del r2
            torch.cuda.empty_cache()
        line["other_3d_workloads"] = others

    if args.steady_state and world == 1:
        if wl.source_term(cfg) is None or wl.source_term(cfg)["kind"] != 1:
            line["steady_state"] = {"skipped": "workload has no constant source"}
        else:
            try:
                del res, ctx
            except NameError:
                pass
            torch.cuda.empty_cache()
            line["steady_state"] = steady_state_run(rte, wl, cfg, torch, dev, plain_krylov=args.krylov_plain)

    if not args.no_cpu_baseline:
        sec, units_small, cores, what = time_oracle(wl, cfg)
        line["cpu_baseline"] = {"value": units_small / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "ms_per_step": 1e3 * sec, "sample": what}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main(argv=None):
    args = parse_args(argv)
    import rte_workloads as wl
    cfg = wl.CONFIGS[args.workload] if args.workload in wl.CONFIGS else wl.PAPER_EXPERIMENTS[args.workload]
    if args.impl == "reference":
        return run_reference(args, wl, cfg)
    if args.impl == "cufft_literal":
        return run_cufft_literal(args, wl, cfg)
    return run_ours(args, wl, cfg)


if __name__ == "__main__":
    sys.exit(main())
