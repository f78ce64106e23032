#!/usr/bin/env python
"""bench.py -- GCUPS of one explicit Heun step of the AMR Euler hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" = compute_dt + advance = 2 x (ghost fill + fused stage kernel) over
every block of the BASELINE.json config (default: config 3, 3D uniform 512^3
in 16^3 blocks, fp64 -- the headline).  GCUPS = interior cells x 2 RK stages x
steps / time / 1e9.  Rank 0 prints ONE JSON line.

N > 1 (torchrun): the path does not shard in this build ("replicas only",
DESIGN.md): every rank runs the same workload independently; value = units of
all ranks / max-over-ranks time; no data-path collective.
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

from paper_2605_07612_b200 import workloads as W  # noqa: E402

METRIC = "GCUPS (fp64, 3D, 1 B200) and achieved fraction of HBM roofline; ghost-fill GB/s"
UNIT = "GCUPS"


def workload_name(cfg):
    d, n = cfg["dim"], cfg["block_n"]
    ext = [cfg["brick"][a] * 2 ** cfg["base_level"] for a in range(d)]
    return f"{cfg['name']}: {d}D {'x'.join(str(e * n) for e in ext)} cells, {n}^{d} blocks, " \
           f"{'uniform' if cfg['max_level'] == cfg['base_level'] else 'adaptive'}, Ng=2, fp64, Heun, CFL {cfg['cfl']}"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            with open(p) as f:
                d = json.load(f)
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", float(d.get("sm_max_mhz", 1965.0))
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)", 1965.0


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
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
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        tries = 0
        while not (self.stop_flag and (self.samples or tries > 3)):   # at least one sample, also for a very short timed region
            tries += 1
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.01)

    def result(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def fill_initial_state(cfg, lev, co, out, chunk=1024):
    """Seeded synthetic state written block-chunk by block-chunk into a (pinned) host array."""
    for b0 in range(0, len(lev), chunk):
        out[b0:b0 + chunk] = W.initial_state(cfg, lev[b0:b0 + chunk], co[b0:b0 + chunk])


def oracle_sample(cfg, target_updates=1.2e7, nthreads=1):
    """The oracle, as it stands, on a bounded sample of the same workload: same generator and block
    size, smaller uniform base level (or fewer extra levels); returns (GCUPS, cores, description).
    nthreads > 1: the block-parallel driver of the same routines (bit-identical results, tests/test_oracle_pins.py)."""
    from oracle import oracle as O
    n, d = cfg["block_n"], cfg["dim"]
    scfg = dict(cfg)
    if cfg["max_level"] == cfg["base_level"]:
        lvl = 0
        while True:
            cells = np.prod([cfg["brick"][a] * 2 ** (lvl + 1) * n for a in range(d)])
            if cells * 2 * 4 > target_updates or lvl + 1 > cfg["base_level"]:
                break
            lvl += 1
        scfg["base_level"] = scfg["max_level"] = lvl
    else:
        scfg["base_level"], scfg["max_level"] = 1, 1
    om = O.OracleMesh.from_config(scfg)
    W.apply_physics(scfg, om)
    lev, co = om.get_blocks()
    om.set_state(0, W.initial_state(scfg, lev, co))
    cells = len(lev) * n ** d
    steps = max(2, int(round(target_updates / (2.0 * cells))))
    nthreads = max(1, min(int(nthreads), len(lev)))

    def one():
        if nthreads == 1:
            om.advance(om.compute_dt(0, cfg["cfl"]))
        else:
            om.advance_mt(om.compute_dt_mt(0, cfg["cfl"], nthreads), nthreads)

    one()  # warm
    t0 = time.perf_counter()
    for _ in range(steps):
        one()
    el = time.perf_counter() - t0
    ext = [scfg["brick"][a] * 2 ** scfg["base_level"] * n for a in range(d)]
    desc = f"{'x'.join(map(str, ext))} cells ({len(lev)} blocks of {n}^{d}), {steps} Heun steps, same generator/seed"
    return cells * 2.0 * steps / el / 1e9, nthreads, desc, el, steps


def pattern_bytes(mesh, n, d):
    """Algorithmic bytes (read, written) of one full execution of the ghost pattern, from its records
    (SURVEY.md 8(a) rows a1-a4): SRL/BC copy Ng*N^(d-1)*Nvar doubles; an F2C record writes a
    1/2^(d-1) share of a coarse face and reads 2^d fine cells per ghost; a C2F record writes a fine face and
    reads the (Ng/2+2) x (N/2+2)^(d-1) coarse cells of its slope stencils."""
    rec, n1, n2 = mesh.pattern()
    nvar, ng = mesh.nvar, 2
    face = ng * n ** (d - 1) * nvar * 8
    ops = rec[:, 0]
    n_copy = int(np.sum((ops == 0) | (ops == 1)))
    n_f2c = int(np.sum(ops == 2))
    n_c2f = int(np.sum(ops == 3))
    rd = n_copy * face + n_f2c * face * 2 + n_c2f * (ng // 2 + 2) * (n // 2 + 2) ** (d - 1) * nvar * 8
    wr = n_copy * face + n_f2c * face // 2 ** (d - 1) + n_c2f * face
    return rd, wr, {"srl_bc": n_copy, "f2c": n_f2c, "c2f": n_c2f}


def adaptive_flags(cfg, mesh):
    """Reading A15: config 5's pressure-jump flags, computed on the device from state 0 (f4_refine_flags fills the
    ghosts and returns one int per block)."""
    from paper_2605_07612_b200 import f4
    if cfg.get("criterion", ("pjump",))[0] == "lohner":          # config 7: eq. (12)
        _, var, params = cfg["criterion"]
        return mesh.refine_flags(0, f4.CRIT_LOHNER, params, var)[0]
    return mesh.refine_flags(0, f4.CRIT_PJUMP, (0.1, 0.025))[0]


def adaptive_initial_mesh(cfg, mesh):
    """{set analytic state, fill ghosts, flag, adapt} up to (max_level - base_level) times, then the analytic state."""
    for _ in range(cfg["max_level"] - cfg["base_level"]):
        lev, co = mesh.get_blocks()
        mesh.set_state(0, W.initial_state(cfg, lev, co))
        if not mesh.adapt(adaptive_flags(cfg, mesh)):
            break
    lev, co = mesh.get_blocks()
    mesh.set_state(0, W.initial_state(cfg, lev, co))


def max_over_ranks(ms, dist, device):
    """Timing rule for N > 1: the step time of the job is the MAX over ranks of the device-timed region.
    `dist` is torch.distributed (or None for one process); works on any backend (nccl on GPUs, gloo in the CPU tests)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, updates_per_rank, ms):
    """Replicas only: every rank advances the same workload independently; value = cell
    updates of ALL ranks / max-over-ranks time, in GCUPS."""
    return world * updates_per_rank / (ms * 1e-3) / 1e9


def run_reference(args, cfg, rank):
    """--impl reference: this tier's reference arm is the CPU oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from oracle import oracle as O
    n, d = cfg["block_n"], cfg["dim"]
    scfg = dict(cfg)
    if cfg["max_level"] == cfg["base_level"]:
        lvl = min(cfg["base_level"], 2 if n <= 16 else 1)
        scfg["base_level"] = scfg["max_level"] = lvl
    else:
        scfg["base_level"], scfg["max_level"] = 1, 1
    om = O.OracleMesh.from_config(scfg)
    W.apply_physics(scfg, om)
    lev, co = om.get_blocks()
    om.set_state(0, W.initial_state(scfg, lev, co))
    cells = len(lev) * n ** d
    for _ in range(args.warmup):
        om.advance(om.compute_dt(0, cfg["cfl"]))
    t0 = time.perf_counter()
    for _ in range(args.steps):
        om.advance(om.compute_dt(0, cfg["cfl"]))
    el = time.perf_counter() - t0
    val = cells * 2.0 * args.steps / el / 1e9
    ext = [scfg["brick"][a] * 2 ** scfg["base_level"] * n for a in range(d)]
    sample = f"bounded sample of {cfg['name']}: {'x'.join(map(str, ext))} cells ({len(lev)} blocks of {n}^{d}) per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None,
                    help="timed steps (default: 20; config 5: the 100 steps BASELINE.json states, regrid every 10)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3,
                    help="1-5: BASELINE.json configs (3 = headline); 6: the paper's own Rayleigh-Taylor benchmark; "
                         "7: the same with AMR driven by the paper's criterion eq. (12); 8: the paper's 3D scalar "
                         "advection benchmark (eq. 13, 512^3 in 16^3 blocks)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--host-dt", action="store_true",
                    help="step = f4_compute_dt (dt read back) + f4_advance(dt) instead of f4_advance_cfl (dt stays on the device)")
    ap.add_argument("--sync-regrid", action="store_true",
                    help="adaptive configs: blocking f4_adapt before the step instead of f4_adapt_begin / f4_adapt_end "
                         "around it (host mesh work overlapped with the step, new mesh one step later)")
    ap.add_argument("--flux-fix", action="store_true",
                    help="adaptive configs: conservative flux fixing at refinement boundaries (PAPER.md:253-261)")
    ap.add_argument("--rk", default="heun", choices=["heun", "euler", "ssp33", "ssp43", "rk4"],
                    help="Runge-Kutta scheme of eq. (5) (default: Heun, the configs' scheme); GCUPS counts one cell "
                         "update per sub-step (PAPER.md:453)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    cfg = W.config(args.config)
    if args.steps is None:
        args.steps = 100 if args.config == 5 else 20

    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import torch
    from paper_2605_07612_b200 import f4
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the f4 path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device(dev))
        dist = dist_mod

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    adaptive = cfg["max_level"] > cfg["base_level"]
    rk = {"heun": f4.RK_HEUN, "euler": f4.RK_EULER, "ssp33": f4.RK_SSP33, "ssp43": f4.RK_SSP43, "rk4": f4.RK_RK4}[args.rk]
    nstages = f4.RK_STAGES[rk]
    mesh = f4.Mesh.from_config(cfg, n_states=f4.RK_STATES[rk], max_blocks=None if not adaptive else 40000)
    mesh.set_rk_scheme(rk)
    W.apply_physics(cfg, mesh)
    mesh.set_flux_fix(args.flux_fix)
    stream = torch.cuda.Stream(dev)
    mesh.bind_torch(dev, stream)
    n, d = cfg["block_n"], cfg["dim"]
    if adaptive:
        adaptive_initial_mesh(cfg, mesh)
        host = host_np = None
    else:
        lev, co = mesh.get_blocks()
        host = torch.empty(mesh._shape(False), dtype=torch.float64).pin_memory()
        host_np = host.numpy()
        fill_initial_state(cfg, lev, co, host_np)
        mesh.set_state(0, host_np)

    counters = {"step": 0, "updates": 0.0, "adapt_s": 0.0, "regrids": 0, "changed": 0}

    def step():
        # config 5: regrid on the host every cfg["regrid_every"] steps (rule A15), inside the timed region.  Default:
        # the flags of step s start the host part of the regrid on a worker thread (f4_adapt_begin), the device
        # advances step s on the current mesh meanwhile, and the new mesh takes over after that step (f4_adapt_end);
        # --sync-regrid: the blocking f4_adapt before the step
        pend = False
        if adaptive and counters["step"] and counters["step"] % cfg["regrid_every"] == 0:
            t0 = time.perf_counter()
            flags = adaptive_flags(cfg, mesh)
            if args.sync_regrid:
                counters["changed"] += int(mesh.adapt(flags))
            else:
                mesh.adapt_begin(flags)
                pend = True
            counters["regrids"] += 1
            counters["adapt_s"] += time.perf_counter() - t0
        if args.host_dt:
            dt = mesh.compute_dt(0, cfg["cfl"])      # reads the CFL maximum back: one host round trip per step
            mesh.advance(dt)
        else:
            mesh.advance_cfl(cfg["cfl"])             # the same two calls with dt kept on the device (no round trip)
        counters["step"] += 1
        counters["updates"] += float(nstages) * mesh.num_blocks * n ** d     # the blocks this step advanced
        if pend:
            t0 = time.perf_counter()
            counters["changed"] += int(mesh.adapt_end())
            counters["adapt_s"] += time.perf_counter() - t0

    for _ in range(max(args.warmup, 0)):
        step()
    mesh.profile_get(reset=True)
    mesh.profile_enable(True)
    l0 = mesh.launch_count()
    counters.update(updates=0.0, adapt_s=0.0, regrids=0, changed=0)
    sampler = ClockSampler(local_rank)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    ev0.record(stream)
    for _ in range(args.steps):
        step()
    ev1.record(stream)
    barrier()
    sampler.stop_flag = True
    sampler.join(timeout=1.0)
    ms = ev0.elapsed_time(ev1)
    launches = mesh.launch_count() - l0
    prof = mesh.profile_get(reset=True)
    mesh.profile_enable(False)
    updates = counters["updates"]
    adapt_info = dict(counters)
    totals_after = mesh.conserved_totals(0)
    ms = max_over_ranks(ms, dist, dev)
    value = whole_job_value(world, updates, ms)
    nb = mesh.num_blocks
    cells = nb * n ** d

    # ---- ghost-fill GB/s: the whole pattern (SRL included) executed standalone by f4_fill_ghosts, outside the step
    rd_b, wr_b, rec_counts = pattern_bytes(mesh, n, d)
    mesh.fill_ghosts(0)
    mesh.profile_get(reset=True)
    mesh.profile_enable(True)
    NFILL = 5
    for _ in range(NFILL):
        mesh.fill_ghosts(0)
    gprof = mesh.profile_get(reset=True)
    mesh.profile_enable(False)
    fill_ms = (gprof["ghost_r1"][0] + gprof["ghost_r2"][0]) / NFILL

    # ---- end to end through the C-ABI with HOST buffers: H2D of the state, the step, D2H of the result metric
    if adaptive:
        host = torch.empty(mesh._shape(False), dtype=torch.float64).pin_memory()
        host_np = host.numpy()
        mesh.get_state(0, out=host_np)
        counters["step"] = 1                 # no regrid inside the end-to-end loop
    else:
        fill_initial_state(cfg, lev, co, host_np)
    e2e_steps = max(1, args.e2e_steps)
    back = torch.empty(mesh._shape(False), dtype=torch.float64).pin_memory()
    back_np = back.numpy()

    def e2e_loop(full):
        """set_state from pinned host memory -> compute_dt + advance -> the result back on the host: the whole new
        state (full) or only its digest (per-block conserved sums)."""
        mesh.set_state(0, host_np)
        step()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(e2e_steps):
            mesh.set_state(0, host_np)          # pinned host -> device staging -> store
            if adaptive:
                counters["step"] = 1            # no regrid inside the end-to-end loop
            step()
            if full:
                mesh.get_state(0, out=back_np)  # device -> pinned host: the new state
            else:
                mesh.conserved_totals(0)        # device -> host: per-block sums
        b.record(stream)
        barrier()
        return max_over_ranks(a.elapsed_time(b), dist, dev)

    ms_e2e = e2e_loop(True)
    ms_dig = e2e_loop(False)
    e2e = {"value": whole_job_value(world, cells * float(nstages) * e2e_steps, ms_e2e), "unit": UNIT,
           "h2d_bytes_per_step": int(host_np.nbytes), "d2h_bytes_per_step": int(back_np.nbytes + 8),
           "steps": e2e_steps, "ms_per_step": ms_e2e / e2e_steps,
           "digest_only": {"value": whole_job_value(world, cells * float(nstages) * e2e_steps, ms_dig),
                           "d2h_bytes_per_step": int(nb * (d + 2) * 8 + 8),
                           "note": "same loop with the per-block conserved sums read back instead of the state"}}

    if rank != 0:
        return
    # ---- roofline of the dominant kernel (fused stage kernel), algorithmic bytes
    peak, peak_src, sm_max = peaks()
    # per cell update: read s_deriv interior + face halo (bpc*r: the y / z halo straight from the neighbours'
    # interiors), write s_out interior + the x face layers pushed into the neighbours' ghost cells
    # (bpc*(1 + 2*Ng/N)), extra s_prev reads (bpc/2 on average for Heun); the same-level ghost copy is fused into
    # the stage kernel, so on a uniform mesh there is no separate ghost-fill traffic.
    r = 1.0 + 2.0 * d * 2 / n
    bpc = 8 * mesh.nvar                                   # Euler: d + 2 variables; scalar advection: 1
    st_ms, st_n = prof["stage"]
    cells_per_launch = updates / max(st_n, 1)            # = cells on a static mesh; the average on an adaptive one
    # previous states other than s_deriv read per sub-step, averaged over the scheme's sub-steps (Heun: 0 and 1)
    extra_prev = {"heun": 0.5, "euler": 0.0, "ssp33": 2.0 / 3.0, "ssp43": 0.25, "rk4": 1.25}[args.rk]
    stage_bytes = cells_per_launch * (bpc * r + bpc * (1.0 + 2.0 * 2 / n) + extra_prev * bpc)
    g_n = prof["ghost_r1"][1] + prof["ghost_r2"][1]
    g_ms = prof["ghost_r1"][0] + prof["ghost_r2"][0]
    stage_gbs = stage_bytes / (st_ms / max(st_n, 1) * 1e-3) / 1e9 if st_ms > 0 else None
    ghost_gbs = ((rd_b + wr_b) / (fill_ms * 1e-3) / 1e9) if fill_ms > 0 else None
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")     # from the committed ncu --set full summary
    if os.path.exists(tp):
        try:
            import csv
            for row in csv.DictReader(open(tp)):
                if row["key"] == f"config{args.config}_stage_dram_bytes_per_launch":
                    traffic = float(row["dram_bytes_per_launch"])
        except Exception:
            traffic = None
    # fp64 issue bound of the stage kernel: 64 DFMA-class instr/clk/SM x 148 SM x clock
    clocks = sampler.result()
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
        # BASELINE.md holds a paper number only for the paper's own workload (config 6 at full size, Heun):
        # 1.35 GCUPS on one H100, PAPER.md:496 -- another machine's: context, not the target
        # (config 6) and 10.89 GCUPS for its 3D scalar advection row (config 8)
        "vs_baseline": (value / 1.35) if (args.config == 6 and args.rk == "heun") else
                       ((value / 10.89) if (args.config == 8 and args.rk == "heun") else None),
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "physics": cfg.get("physics", "euler"), "blocks": nb, "cells": cells,
                   "l2": "state (2 x %.1f GB) is larger than L2; no flush needed" % (mesh.storage_bytes() / 2e9),
                   "parallelism": "replicas only" if world > 1 else "1 GPU", "rk": args.rk,
                   "step": "f4_compute_dt + f4_advance(dt)" if args.host_dt else "f4_advance_cfl (compute_dt + advance, dt on the device)",
                   "flux_fix": bool(args.flux_fix)},
        "roofline": {"bound": "hbm", "achieved": stage_gbs, "peak": peak, "unit": "GB/s",
                     "frac": (stage_gbs / peak) if stage_gbs else None, "traffic": traffic,
                     "kernel": ("advect2_kernel" if d == 3 else "advect_kernel") if cfg.get("physics") == "advection" else "stage_kernel",
                     "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": stage_bytes, "avg_launch_ms": st_ms / max(st_n, 1)},
        "ghost_fill": {"GBps": ghost_gbs, "frac_of_hbm_peak": (ghost_gbs / peak) if ghost_gbs else None,
                       "ms_per_fill": fill_ms, "bytes_read": int(rd_b), "bytes_written": int(wr_b),
                       "records": rec_counts, "launches_per_fill": (gprof["ghost_r1"][1] + gprof["ghost_r2"][1]) // NFILL,
                       "in_step_executor_launches": int(g_n), "in_step_executor_ms_per_step": g_ms / args.steps,
                       "note": "GBps: f4_fill_ghosts (whole pattern: same-level copies by source block, then the "
                               "BC/F2C/C2F records) timed standalone after the step "
                               "loop; inside advance the same-level copies are pushed by the stage kernel and the "
                               "executor runs only BC/F2C/C2F records (none on a uniform periodic mesh)"},
        "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()},
        "step_algorithmic_GBps": (nstages * stage_bytes) / (ms / args.steps * 1e-3) / 1e9,
        "adaptive": ({"regrids": adapt_info["regrids"], "mesh_changed": adapt_info["changed"],
                      "adapt_ms_total": 1e3 * adapt_info["adapt_s"], "blocks_at_end": nb,
                      "regrid_mode": "blocking f4_adapt before the step" if args.sync_regrid else
                                     "f4_adapt_begin before / f4_adapt_end after the step (host part overlapped)",
                      # host wall time inside the regrid calls; with f4_advance_cfl the host runs ahead of the device,
                      # so this includes waiting for queued steps: only with --host-dt --sync-regrid is
                      # (time - adapt time) the time of the steps alone
                      "value_excluding_adapt": (world * updates / max(ms * 1e-3 - adapt_info["adapt_s"], 1e-9) / 1e9)
                      if (args.host_dt and args.sync_regrid) else None}
                     if adaptive else None),
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "totals": [float(x) for x in totals_after],
    }
    if world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on one core (its definition), and the block-parallel driver of the same routines on
        # all host cores (SURVEY 8(d) "Timing the oracle beside it"); both on bounded samples of the workload
        v, cores, desc, el, cs = oracle_sample(cfg)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                               "seconds": el}
        ncores = os.cpu_count() or 1
        if ncores > 1:
            va, ca, desca, ela, _ = oracle_sample(cfg, target_updates=1.2e7 * min(ncores, 16), nthreads=ncores)
            out["cpu_baseline"]["all_cores"] = {"value": va, "unit": UNIT, "cores": ca, "kind": "oracle",
                                                "sample": desca, "seconds": ela,
                                                "note": "block-parallel driver of the same routines, bit-identical"}
    print(json.dumps(out))
    mesh.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
