#!/usr/bin/env python
"""bench.py — Riccati trajectory-step updates/s of one self-consistent iteration (sweep + A-solve + mixing).

  python bench.py --gpus N --steps K --warmup W [--impl reference] [--cfg C]

A step = one `sc_iterate` (Algorithm 1 :203-205) over one synthetic grain: rotate-in, march
(gamma-tilde down, gamma up, node products, energy reduction), rotate-back + finalise, FFT vector-potential
solve, Barzilai-Borwein mixing.  Workload at N=1: BASELINE.json configs[4] (s-wave disc R = 40 xi0,
1600x1600 grid, 256 angles, 512 Matsubara energies, kappa = 2, 20 vortices), the config the metric's FP64
target is quoted on.  Inputs are seeded synthetic fields (workloads/), resident in HBM for `value`; `e2e`
repeats the measurement with pinned HOST buffers copied in and out every step.
With --gpus N > 1 (torchrun) the Matsubara energies are sharded across ranks (the march, the specular
boundary condition and the boundary stores never couple energies) and the partial Delta_new, j, I fields are
summed with one NCCL all-reduce per sweep; per-rank work shrinks as N grows -> "strong" scaling.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "riccati_trajectory_step_updates_per_s"
UNIT = "updates/s"
# FP64-pipe instructions the closed-form path needs per unit = (piece, energy, angle pair) = 4 logical updates
# (gamma and gamma-tilde for angles k and k+N/2): DESIGN.md §6 tally of the kernel's own algorithm.
#   "recompute" rounds (every piece inside the radius of the per-energy Taylor table of T): T twice 2 x 15, two Moebius
#       steps 2 x 27, node products 26 (28 with non-unit weights; the bench's Matsubara table has unit weights and the
#       kernel variant with the weights compiled out runs), energy reduction 8 = 118, + half a Moebius step 13.5 because
#       only every second gamma-tilde is spilled and the other is re-stepped in pass 2 = 131.5; scratch traffic 8 B
#       written + 8 B read = 16 B
#   "recompute_pole" rounds (|a| beyond that table but inside the pole-subtracted one): T twice 2 x 24 (degree 5 + the
#       pole term with one reciprocal), 54, 26, 8, 13.5 = 149.5; 16 B per unit
#   "stored-T" rounds (strong vector potential): T once from the pole-subtracted table 36, 54, 26, 8 = 124; 64 B per unit
# Evaluating T from its definition (sqrt, exp, sin/cos) would be 86 per evaluation — reported as context only.
ALGO_FP64_INSTR_PER_UNIT = {"recompute": 131.5, "recompute_pole": 149.5, "stored": 124.0}
# the least FP64 work any of these layouts could do per unit if nothing were evaluated twice: T once 15, two steps 54,
# node products 26, reduction 8 — reported beside the roofline so that recomputation is not mistaken for useful work
MIN_WORK_FP64_INSTR_PER_UNIT = 103.0
ALGO_HBM_BYTES_PER_UNIT = {"recompute": 16.0, "recompute_pole": 16.0, "stored": 64.0}
TEXTBOOK_FP64_INSTR_PER_UNIT = 184.0
ALGO_FP64_INSTR_PER_UNIT_MIDPOINT = 2 * 66.0 + 28.0 + 8.0     # the mid-point kernels keep the weights
# dram__bytes_read.sum + dram__bytes_write.sum of ONE march launch at configs[4], fp64, closed-form stepper, all rounds in
# "recompute" mode (--sweep-only: A = A_ext), from the `ncu --set full` capture summarised in profiles/
# (profiles/r1_march_fp64_cfg4_ncu_full.md: 1.518 TB read + 1.255 TB written)
NCU_TRAFFIC_BYTES = {(4, 64, 0): 2.773331e12}
NCU_PIPE_FP64_ACTIVE_PCT = {(4, 64, 0): 74.3}


class ClockSampler(threading.Thread):
    def __init__(self, index=0, period=0.2):
        super().__init__(daemon=True)
        self.index, self.period, self.rows, self._halt = index, period, [], threading.Event()

    def run(self):
        q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._halt.wait(self.period)

    def stop(self):
        self._halt.set()
        self.join(timeout=5)
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cfg", type=int, default=4)
    ap.add_argument("--pts-per-xi", type=float, default=None)
    ap.add_argument("--n-angles", type=int, default=None)
    ap.add_argument("--n-energies", type=int, default=None)
    ap.add_argument("--size-scale", type=float, default=1.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep-only", action="store_true", help="time sc_riccati_sweep alone (profiling aid)")
    ap.add_argument("--stepper", type=int, default=0, help="0 closed-form step (north_star), 1 the paper's implicit mid-point rule")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32], help="arithmetic of the march (ABI buffers stay fp64)")
    ap.add_argument("--no-fp32-leg", action="store_true", help="skip the extra FP32-mode timing that configs[4] asks for")
    return ap.parse_args()


def workload_from_args(a):
    kw = {}
    if a.pts_per_xi: kw["pts_per_xi"] = a.pts_per_xi
    if a.n_angles: kw["n_angles"] = a.n_angles
    if a.n_energies: kw["n_energies"] = a.n_energies
    if a.size_scale != 1.0: kw["size_scale"] = a.size_scale
    return workloads.make_workload(a.cfg, **kw)


def config_of(wl, a, extra=None):
    c = {"workload": f"BASELINE.json configs[{wl.cfg}]: {wl.name}", "grid": f"{wl.nx}x{wl.ny}", "n_in": wl.n_in,
         "n_angles": wl.n_angles, "n_energies": wl.n_energies, "t": wl.t, "kappa": wl.kappa,
         "step": "one self-consistent iteration (sweep + A-solve + BB mixing)",
         "l2": "inputs larger than L2 (march scratch and partial sums are GBs per step); no flush needed"}
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------------
def oracle_sample(wl, cores):
    """One bounded sample of the workload on the oracle: a subset of angles (one per core, evenly spaced) and
    the lowest Matsubara energies, sized to ~10-30 s.  Returns (updates, seconds, description)."""
    import oracle
    os.environ.setdefault("OMP_NUM_THREADS", str(cores))
    o = oracle.Oracle.from_workload(wl)
    per_angle_nodes = wl.n_in
    target = 1.2e8                                  # updates per core at ~130 ns each -> ~15 s
    ne = int(max(1, min(wl.n_energies, target // (2 * per_angle_nodes))))
    nang = min(cores, wl.n_angles)
    angles = [int(round(i * wl.n_angles / nang)) % wl.n_angles for i in range(nang)]
    z, w = o.matsubara(ne)
    Ax, Ay = (wl.Aext_x, wl.Aext_y) if np.any(wl.Aext_x) else (None, None)
    stores = o.reset_stores(wl.delta0, Ax, Ay, z)
    t0 = time.perf_counter()
    r = o.raw_sweep(wl.delta0, Ax, Ay, z, w, stores, angle_list=angles)
    dt = time.perf_counter() - t0
    return r["stats"]["n_updates"], dt, f"{nang} of {wl.n_angles} angles x {ne} of {wl.n_energies} energies, all trajectories, 1 sweep"


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = workload_from_args(a)
    cores = os.cpu_count() or 1
    for _ in range(min(a.warmup, 1)):
        pass                                        # the oracle has no warm-up state worth timing away
    tot_u, tot_t, desc = 0, 0.0, ""
    for _ in range(a.steps):
        u, t, desc = oracle_sample(wl, cores)
        tot_u += u; tot_t += t
    val = tot_u / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": 1e3 * tot_t / a.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_of(wl, a),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# CUDA path
# ------------------------------------------------------------------------------------------------
def run_ours(a):
    import torch
    import paper_2205_15000_b200 as sc

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    import torch.distributed as dist
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    devname = f"cuda:{local}"
    wl = workload_from_args(a)
    ctx = sc.ScContext.from_workload(wl, device=local, stepper=a.stepper, precision=a.precision)
    if world > 1:
        # energy sharding: this rank marches its slice of the Matsubara table; one NCCL all-reduce of the
        # five accumulator fields per sweep; A-solve and mixing are replicated (deterministic, identical on all ranks)
        from paper_2205_15000_b200 import sharding
        sharding.attach(ctx, wl.t, wl.n_energies)
    dev = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=devname)
    ng = wl.nx * wl.ny
    delta = dev(wl.delta0.astype(np.complex128))
    aix = torch.zeros((wl.ny, wl.nx), dtype=torch.float64, device=devname); aiy = torch.zeros_like(aix)
    ctx.sc_set_external_field(dev(wl.Aext_x), dev(wl.Aext_y))
    acc = wl.accelerator
    dn = torch.zeros_like(delta); jx = torch.zeros_like(aix); jy = torch.zeros_like(aix); fe = torch.zeros_like(aix)

    def step():
        if a.sweep_only:
            ctx.sc_set_fields(delta, dev_ax, dev_ay)
            ctx.sc_riccati_sweep(dn, jx, jy, fe)
        else:
            ctx.sc_iterate(acc, 1.0, False, delta, aix, aiy)

    dev_ax, dev_ay = dev(wl.Aext_x), dev(wl.Aext_y)

    for _ in range(max(a.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local); sampler.start()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ctx.sc_debug_march_time()                       # reset: count only the march launches of the timed steps
    ctx.sc_debug_march_units()
    ctx.sc_debug_launch_count()
    e0.record()
    for _ in range(a.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    gpu_launches = ctx.sc_debug_launch_count()      # kernels of the library launched by the timed steps (counted at the launch sites)
    timed_kernel = ctx.sc_debug_last_march_variant()
    march_total_ms, march_launches = ctx.sc_debug_march_time()      # CUDA events around each march launch of the timed region
    units_timed, units_timed_stored, units_timed_pole = ctx.sc_debug_march_units()     # units of those launches, by mode
    if world > 1:                                   # device time of the slowest rank
        tmax = torch.tensor([ms], dtype=torch.float64, device=devname)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        ms = float(tmax.item())

    # unit counts of one sweep (one extra sweep with stats, outside the timed region)
    ctx.sc_set_fields(delta, dev_ax + aix, dev_ay + aiy)
    st = ctx.sc_riccati_sweep(dn, jx, jy, fe, want_stats=True)
    units = st.n_updates / 4.0                    # this rank's (node, energy, angle-pair) units incl. the boundary pieces
    n_updates, n_exec = st.n_updates, st.n_updates_executed
    if world > 1:                                 # whole-job updates = sum over the energy shards
        tot = torch.tensor([n_updates, n_exec], dtype=torch.float64, device=devname)
        dist.all_reduce(tot)
        n_updates, n_exec = int(tot[0].item()), int(tot[1].item())
    peak_dfma, clk = ctx.sc_debug_fp64_peak()
    mk_ms = march_total_ms / max(march_launches, 1)
    full_size = world == 1 and not (a.pts_per_xi or a.n_angles or a.n_energies or a.size_scale != 1.0)
    # algorithmic work of ONE average march launch of the timed region (units counted by the library, by mode)
    nl = max(march_launches, 1)
    u_all = units_timed / nl; u_st = units_timed_stored / nl; u_pl = units_timed_pole / nl; u_rec = u_all - u_st - u_pl
    if a.stepper == 0:
        instr = sum(ALGO_FP64_INSTR_PER_UNIT[k] * u for k, u in (("recompute", u_rec), ("recompute_pole", u_pl), ("stored", u_st)))
        hbm = sum(ALGO_HBM_BYTES_PER_UNIT[k] * u for k, u in (("recompute", u_rec), ("recompute_pole", u_pl), ("stored", u_st)))
    else:
        instr = ALGO_FP64_INSTR_PER_UNIT_MIDPOINT * u_all
        hbm = 32.0 * u_all
    if a.precision == 32:
        hbm *= 0.5
    achieved = 2.0 * instr / (mk_ms * 1e-3) / 1e12
    peak_burst = 2.0 * peak_dfma / 1e12
    peak_sustained = 2.0 * ctx.sc_debug_fp64_peak_sustained(2.0) / 1e12
    peak = max(peak_burst, peak_sustained)
    peak_kind = "measured register-resident DFMA rate (fp64 pipe)"
    if a.precision == 32:
        # the fp32 march runs the same instruction stream on the FP32 pipe: 128 FMA lanes per SM (twice the fp64 lanes);
        # no measured fp32 figure exists here, so the peak is nominal (unit count x maximum SM clock)
        peak = 2.0 * 148 * 128 * (clocks.get("sm_max_mhz") or 1965.0) * 1e6 / 1e12
        peak_kind = "nominal fp32 pipe: 148 SMs x 128 FMA lanes x max SM clock"
    key = (wl.cfg, a.precision, a.stepper)
    roofline = {"bound": "alu", "kernel": "sck::" + timed_kernel,
                "launches_timed": march_launches, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak,
                "traffic": NCU_TRAFFIC_BYTES.get(key) if full_size else None,
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum, profiles/) of a launch with ALL rounds in recompute mode (16 B algorithmic per unit = 2.11e12, + 0.39e12 running sums + 0.3e12 coefficient records); stored-T rounds move 64 B per unit",
                "algorithmic_bytes_per_launch": hbm,
                "ncu_pipe_fp64_cycles_active_pct": NCU_PIPE_FP64_ACTIVE_PCT.get(key) if full_size else None,
                "note": "fp64 pipe: flops = 2 x FP64-pipe instructions; achieved = algorithmic count (DESIGN.md §6) x units / "
                        "march duration (CUDA events around the march launches of the timed steps); peak = register-resident "
                        "DFMA rate measured in this process: the larger of a best-of-3 burst (11 ms) and a 2 s sustained run",
                "peak_kind": peak_kind, "peak_burst": peak_burst, "peak_sustained": peak_sustained,
                "min_work_context": {"fp64_instr_per_unit": MIN_WORK_FP64_INSTR_PER_UNIT,
                                     "tflops": 2.0 * MIN_WORK_FP64_INSTR_PER_UNIT * u_all / (mk_ms * 1e-3) / 1e12,
                                     "frac": 2.0 * MIN_WORK_FP64_INSTR_PER_UNIT * u_all / (mk_ms * 1e-3) / 1e12 / peak,
                                     "note": "FP64 instructions if T and every gamma-tilde were evaluated once; the kernel re-evaluates "
                                             "them on purpose (bytes cost more watts than instructions under the 1 kW cap)"},
                "textbook_count_context": {"fp64_instr_per_unit": TEXTBOOK_FP64_INSTR_PER_UNIT,
                                           "tflops": 2.0 * TEXTBOOK_FP64_INSTR_PER_UNIT * u_all / (mk_ms * 1e-3) / 1e12},
                "march_ms": mk_ms, "march_share_of_step": mk_ms / (ms / a.steps),
                "algo_fp64_instr_per_unit": instr / max(u_all, 1.0), "units_per_launch": u_all,
                "units_share_stored_T": u_st / max(u_all, 1.0), "units_share_recompute_pole_table": u_pl / max(u_all, 1.0),
                "hbm_bytes_per_unit_algorithmic": hbm / max(u_all, 1.0),
                "hbm_gbs_algorithmic": hbm / (mk_ms * 1e-3) / 1e9}

    # end to end through the C ABI with HOST buffers: H2D of Delta, A_ind; iterate; D2H of Delta, A_ind + stats
    hd = torch.empty((wl.ny, wl.nx), dtype=torch.complex128).pin_memory(); hd.copy_(delta)
    hax = torch.zeros((wl.ny, wl.nx), dtype=torch.float64).pin_memory(); hay = torch.zeros_like(hax).pin_memory()
    hax.copy_(aix); hay.copy_(aiy)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(a.steps):
        delta.copy_(hd, non_blocking=True); aix.copy_(hax, non_blocking=True); aiy.copy_(hay, non_blocking=True)
        st2 = ctx.sc_iterate(acc, 1.0, False, delta, aix, aiy, want_stats=True)
        hd.copy_(delta, non_blocking=True); hax.copy_(aix, non_blocking=True); hay.copy_(aiy, non_blocking=True)
        torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / a.steps
    if world > 1:
        tmax = torch.tensor([e2e_s], dtype=torch.float64, device=devname)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        e2e_s = float(tmax.item())
    bytes_io = ng * 16 + 2 * ng * 8

    # configs[4]: "... FP64, with an FP32 mode also timed": the same step with opts.precision = 32 (same inputs, same
    # warm-up and step counts), reported beside the FP64 headline, never instead of it
    fp32_leg = None
    if a.precision == 64 and wl.cfg == 4 and not a.no_fp32_leg and not a.sweep_only:
        ctx.close(); del ctx
        torch.cuda.empty_cache()
        c32 = sc.ScContext.from_workload(wl, device=local, stepper=a.stepper, precision=32)
        if world > 1:
            from paper_2205_15000_b200 import sharding
            sharding.attach(c32, wl.t, wl.n_energies)
        c32.sc_set_external_field(dev_ax, dev_ay)
        d32 = dev(wl.delta0.astype(np.complex128)); ax32 = torch.zeros_like(aix); ay32 = torch.zeros_like(aix)
        for _ in range(max(a.warmup, 3)):
            c32.sc_iterate(acc, 1.0, False, d32, ax32, ay32)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        f0 = torch.cuda.Event(enable_timing=True); f1 = torch.cuda.Event(enable_timing=True)
        c32.sc_debug_march_time()
        f0.record()
        for _ in range(a.steps):
            c32.sc_iterate(acc, 1.0, False, d32, ax32, ay32)
        f1.record(); torch.cuda.synchronize()
        ms32 = f0.elapsed_time(f1)
        if world > 1:
            tmax = torch.tensor([ms32], dtype=torch.float64, device=devname)
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
            ms32 = float(tmax.item())
        fp32_leg = {"dtype": "f32", "value": n_updates * a.steps / (ms32 * 1e-3), "unit": UNIT, "ms_per_step": ms32 / a.steps,
                    "march_ms": c32.sc_debug_march_time()[0] / a.steps}
        c32.close()

    value = n_updates * a.steps / (ms * 1e-3)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": max(a.warmup, 3),
            "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64" if a.precision == 64 else "f32",
            "data": "synthetic", "config": config_of(wl, a, {"seconds_per_self_consistent_iteration": ms / a.steps / 1e3,
                                                             "updates_per_step": n_updates, "updates_executed_per_step": n_exec,
                                                             "stepper": "closed-form" if a.stepper == 0 else "implicit mid-point",
                                                             "parallelism": f"energy-sharded x{world}, 1 all-reduce/sweep" if world > 1 else "single GPU"}),
            "clocks": clocks,
            "e2e": {"value": n_updates / e2e_s, "unit": UNIT, "h2d_bytes_per_step": bytes_io, "d2h_bytes_per_step": bytes_io + 64,
                    "res_delta_last": st2.res_delta,
                    "note": "the e2e steps continue the same self-consistency run (iterations after the timed ones): as the "
                            "Barzilai-Borwein transient of A_ind decays more rounds take the cheaper table tiers, so a step here "
                            "can be faster than a timed one although it also pays the host copies"},
            "gpu_launches": gpu_launches, "roofline": roofline}
    if fp32_leg:
        line["config"]["fp32_mode"] = fp32_leg
    if not a.no_cpu_baseline and rank == 0:
        cores = os.cpu_count() or 1
        u, t, desc = oracle_sample(wl, cores)
        line["cpu_baseline"] = {"value": u / t, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)
