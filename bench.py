#!/usr/bin/env python
"""bench.py — Riccati trajectory-step updates/s of one self-consistent iteration (sweep + A-solve + mixing).

  python bench.py --gpus N --steps K --warmup W [--impl reference] [--cfg C]

A step = one `sc_iterate` (Algorithm 1 :203-205) over one synthetic grain: rotate-in, march
(gamma-tilde down, gamma up, node products, energy reduction), rotate-back + finalise, FFT vector-potential
solve, Barzilai-Borwein mixing.  Workload at N=1: BASELINE.json configs[4] (s-wave disc R = 40 xi0,
1600x1600 grid, 256 angles, 512 Matsubara energies, kappa = 2, 20 vortices), the config the metric's FP64
target is quoted on.  Inputs are seeded synthetic fields (workloads/), resident in HBM for `value`; `e2e`
repeats the measurement with pinned HOST buffers copied in and out every step.

The timed state.  The first Barzilai-Borwein iterations at kappa = 2 overshoot the induced vector potential
(|A| up to 6 A0), which sends march rounds to dearer table tiers; from iteration ~10 on the cost of an iteration
is constant to 0.3 % (profiles/r2_transient.md).  The run therefore first does `--burnin` untimed iterations,
then W warm-up steps, then the K timed steps, then the K end-to-end steps: all legs sit on the same stationary
part of the run, so `value` does not depend on --steps and e2e = value + the host copies.  The cost of the very
first iterations is reported beside it (`config.transient`).

With --gpus N > 1 (torchrun) the Matsubara energies are sharded across ranks (the march, the specular
boundary condition and the boundary stores never couple energies) and the partial Delta_new, j, I fields are
summed with one NCCL all-reduce per sweep; per-rank work shrinks as N grows -> "strong" scaling.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import hashlib
import json
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

# ---- FP64-pipe instruction tallies per unit = (piece, energy, angle pair) = 4 logical updates (gamma and gamma-tilde
# for angles k and k + N/2; the kernel marches two of them, Eq. 13 gives the other two).  FMA = one instruction = 2 flops.
# Each stage is derived in DESIGN.md §6; the EXECUTED tally is checked against the ncu instruction counters
# (profiles/r2_march_ncu.json, read below when it belongs to the kernel sources in the tree).
STAGE_FP64 = {
    "T_table_deg5": 15.0,       # dw 1, |dw|^2 2, real-coefficient degree-5 polynomial at complex dw 10, remainder 2
    "T_table_deg3": 11.0,       # FP32 mode: degree 3 (truncation 2e-8 relative at the edge of its radius)
    "T_pole_table": 24.0,       # pole term (one reciprocal) + degree-5 remainder
    "T_pole_table_deg8": 36.0,  # stored-T rounds: degree 8, warp vote
    "moebius_step": 27.0,       # z g + De 4, N 4, z + conj(De) g 4, Q 4, |Q|^2 2, reciprocal 3, N conj(Q) / |Q|^2 6
    "node_products": 25.0,      # one energy per lane: P 4, 1+P 1, |.|^2 2, reciprocal 3, 1/(1+P) 2, SF 4, X2 4, SG 1 (weight), SI 4
    "node_products_pairs": 24.0,  # two energies per lane, per unit: the same without the SG instruction; the second energy's terms are
                                  # accumulated onto the first's by the last FMA of each term (no separate additions)
    "energy_reduction": 8.0,    # one energy per lane: column sums of the transpose stage + running sum
    "energy_reduction_pairs": 4.5,  # two energies per lane: SG addition 0.5 + half the column sums and running sum 4
}
ROUND1_LEAST_WORK = 103.0       # the count round 1's fraction (0.556) was quoted on: kept beside `frac` for comparison


def stage_counts(precision):
    """(least work per unit, executed per unit by round type) for the closed-form stepper"""
    T = STAGE_FP64["T_table_deg5" if precision == 64 else "T_table_deg3"]
    # least work: nothing evaluated twice — T once, gamma and gamma-tilde stepped once, products, reduction (two energies per lane)
    least = T + 2 * STAGE_FP64["moebius_step"] + STAGE_FP64["node_products_pairs"] + STAGE_FP64["energy_reduction_pairs"]
    # what the kernel executes: T in both passes, and every second gamma-tilde re-stepped in pass 2 instead of spilled;
    # stored-T rounds run one energy per lane
    one = least + (STAGE_FP64["node_products"] - STAGE_FP64["node_products_pairs"]) + (STAGE_FP64["energy_reduction"] - STAGE_FP64["energy_reduction_pairs"])
    executed = {"recompute": least + T + 0.5 * STAGE_FP64["moebius_step"],
                "recompute_pole": least - T + 2 * STAGE_FP64["T_pole_table"] + 0.5 * STAGE_FP64["moebius_step"],
                "stored": one - T + STAGE_FP64["T_pole_table_deg8"]}
    return least, executed


LEAST_WORK_FP64, EXECUTED_FP64 = stage_counts(64)
EXECUTED_FP64_MIDPOINT = 2 * 66.0 + 28.0 + 8.0
ALGO_HBM_BYTES_PER_UNIT = {"recompute": 16.0, "recompute_pole": 16.0, "stored": 64.0}   # scratch out + back


def source_hash():
    """sha256 over the kernel sources: ncu figures in profiles/ are only quoted for the code they were captured from"""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2205_15000_b200", "csrc")
    for f in ("sc_kernels.cuh", "sc_math.cuh"):            # the files the march kernel is compiled from
        h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()


def ncu_capture(key):
    """figures of the committed ncu capture `key`, or None when the kernel sources have changed since"""
    p = os.path.join(ROOT, "profiles", "r2_march_ncu.json")
    if not os.path.exists(p):
        return None
    j = json.load(open(p))
    c = j.get("captures", {}).get(key)
    if not c or c.get("source_sha256") != source_hash():
        return None
    return c


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
        pw = [float(r[2]) for r in self.rows if r[2].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w": float(np.median(pw)) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


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
    ap.add_argument("--burnin", type=int, default=None, help="untimed self-consistent iterations before the warm-up (default 12 with an induced A, else 0)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep-only", action="store_true", help="time sc_riccati_sweep alone at the initial fields (profiling aid)")
    ap.add_argument("--stepper", type=int, default=0, help="0 closed-form step (north_star), 1 the paper's implicit mid-point rule")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32], help="arithmetic of the march (ABI buffers stay fp64)")
    ap.add_argument("--no-fp32-leg", action="store_true", help="skip the extra FP32-mode timing that configs[4] asks for")
    ap.add_argument("--no-ldos-leg", action="store_true", help="skip the sc_ldos timing on configs[3]")
    ap.add_argument("--ldos-only", action="store_true", help="time sc_ldos on configs[3] alone (profiling aid)")
    ap.add_argument("--issue-probe", action="store_true", help="print the DFMA rate next to integer / shared-memory instructions (DESIGN.md §6) and exit")
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


CPU_NOTE = ("the parity checker as it stands (g++ -O2, std::complex, library sqrt/exp, no Eq. 13 symmetry, every logical update "
            "executed): a reported baseline, not a tuned CPU implementation")


def textbook_count():
    """real flops of one trajectory-step update as the oracle states the closed-form step, counted by running the
    oracle's own statements on an operation-counting scalar (oracle.step_opcount)"""
    import oracle
    c = oracle.step_opcount(0)
    ops = {k: c[k] for k in ("mul", "add", "div", "sqrt", "exp", "sincos")}
    return {"per_update": ops, "flops_per_update": sum(ops.values()), "flops_per_unit": 4 * sum(ops.values()),
            "note": "textbook complex arithmetic, each division / square root / exponential / sin-cos pair counted as ONE flop; "
                    "4 logical updates per unit"}


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = workload_from_args(a)
    cores = os.cpu_count() or 1
    tot_u, tot_t, desc = 0, 0.0, ""
    for _ in range(a.steps):
        u, t, desc = oracle_sample(wl, cores)
        tot_u += u; tot_t += t
    val = tot_u / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": 1e3 * tot_t / a.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config_of(wl, a),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "note": CPU_NOTE},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# CUDA path
# ------------------------------------------------------------------------------------------------
def time_iterations(ctx, torch, dist, world, devname, nsteps, step_fn):
    """K steps between barriers + synchronize, CUDA events on the stream the library launches on; returns
    (ms of the slowest rank, march ms per launch, launches, units (all, stored-T, pole table), kernels launched)"""
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ctx.sc_debug_march_time(); ctx.sc_debug_march_units(); ctx.sc_debug_launch_count()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(nsteps):
        step_fn()
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    launches = ctx.sc_debug_launch_count()
    mms, nl = ctx.sc_debug_march_time()
    units = ctx.sc_debug_march_units()
    if world > 1:
        tmax = torch.tensor([ms], dtype=torch.float64, device=devname)
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        ms = float(tmax.item())
    return ms, mms / max(nl, 1), nl, units, launches


def march_roofline(a, wl, ctx, kernel, mk_ms, nl, units, step_ms, precision, full_size, clocks):
    """roofline object of the march kernel for one timed leg"""
    u_all, u_st, u_pl = (v / max(nl, 1) for v in units)
    u_rec = u_all - u_st - u_pl
    least_pu, exec_pu = stage_counts(precision)
    if a.stepper == 0:
        executed = sum(exec_pu[k] * u for k, u in (("recompute", u_rec), ("recompute_pole", u_pl), ("stored", u_st)))
        hbm = sum(ALGO_HBM_BYTES_PER_UNIT[k] * u for k, u in (("recompute", u_rec), ("recompute_pole", u_pl), ("stored", u_st)))
        least = least_pu * u_all
    else:
        executed = EXECUTED_FP64_MIDPOINT * u_all; hbm = 32.0 * u_all; least = executed; least_pu = EXECUTED_FP64_MIDPOINT
    if precision == 32:
        hbm *= 0.5
    sec = mk_ms * 1e-3
    if precision == 64:
        burst = 2.0 * ctx.sc_debug_fp64_peak()[0] / 1e12
        sustained = 2.0 * ctx.sc_debug_fp64_peak_sustained(2.0) / 1e12
        peak_kind = "measured register-resident DFMA rate (fp64 pipe): larger of a best-of-3 11 ms burst and a 2 s sustained run"
    else:
        burst = sustained = 2.0 * ctx.sc_debug_pipe_peak(1, 2.0) / 1e12
        peak_kind = "measured register-resident FFMA rate (fp32 pipe), 2 s sustained run"
    peak = max(burst, sustained)
    cap = ncu_capture(f"cfg{wl.cfg}_f{precision}_stepper{a.stepper}") if full_size else None
    achieved = 2.0 * least / sec / 1e12
    r = {"bound": "alu", "kernel": "sck::" + kernel, "launches_timed": nl,
         "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
         "frac_basis": f"least-work count: {least_pu:.1f} fp{precision}-pipe instructions per unit (T once, two Moebius steps, node "
                       "products, energy reduction with two energies per lane; nothing evaluated twice) x units / march time (CUDA events around the march "
                       "launches of the timed steps) / measured peak",
         "frac_on_round1_count": 2.0 * ROUND1_LEAST_WORK * u_all / sec / 1e12 / peak if (precision == 64 and a.stepper == 0) else None,
         "traffic": cap["dram_bytes"] if cap else None,
         "algorithmic_bytes_per_launch": hbm,
         "peak_kind": peak_kind, "peak_burst": burst, "peak_sustained": sustained,
         "pipe_utilisation": {"instr_per_unit_tally": executed / max(u_all, 1.0),
                              "tflops": 2.0 * executed / sec / 1e12, "frac": 2.0 * executed / sec / 1e12 / peak,
                              "note": "what the kernel executes on purpose: T evaluated in both passes and every second gamma-tilde "
                                      "re-stepped instead of spilled (DESIGN.md §6)"},
         "march_ms": mk_ms, "march_share_of_step": mk_ms / step_ms,
         "units_per_launch": u_all, "units_share_stored_T": u_st / max(u_all, 1.0), "units_share_recompute_pole_table": u_pl / max(u_all, 1.0),
         "hbm_bytes_per_unit_algorithmic": hbm / max(u_all, 1.0), "hbm_gbs_algorithmic": hbm / sec / 1e9}
    if cap:     # figures of the committed ncu capture of THIS source tree (profiles/r2_march_ncu.json)
        r["ncu"] = {k: cap[k] for k in cap if k != "source_sha256"}
        if "fp_pipe_warp_instr_per_unit" in cap:
            r["pipe_utilisation"]["instr_per_unit_ncu"] = cap["fp_pipe_warp_instr_per_unit"]
    else:
        r["ncu"] = None
    if precision == 32:
        mufu = ctx.sc_debug_pipe_peak(2, 1.0)
        r["sfu"] = {"mufu_peak_per_s": mufu, "mufu_per_unit_tally": 3.5,
                    "mufu_issue_frac": 3.5 * u_all / sec / mufu,
                    "note": "MUFU.RCP seeds of the reciprocals: one per Moebius step and node product (3.5 per unit with the re-stepped "
                            "gamma-tilde) against the measured MUFU issue rate"}
        r["issue_note"] = ("the fp32 pipe issues one warp instruction per cycle per scheduler, like every other pipe: the fp32 march is bound "
                           "by instruction issue (ncu: issue_active_pct of the capture below), not by the fp32 lanes")
    else:
        mufu = ctx.sc_debug_pipe_peak(3, 1.0)
        r["sfu"] = {"mufu_peak_per_s": mufu, "mufu_per_unit_tally": 3.5, "mufu_issue_frac": 3.5 * u_all / sec / mufu,
                    "note": "MUFU.RCP64H seeds (3.5 per unit) against the measured MUFU.RCP64H issue rate"}
    return r


def run_leg(a, sc, torch, dist, wl, local, world, precision, burnin, full_size):
    """burn-in, warm-up, K device-resident steps, K end-to-end steps for one arithmetic precision"""
    devname = f"cuda:{local}"
    dev = lambda x: torch.as_tensor(np.ascontiguousarray(x), device=devname)
    ctx = sc.ScContext.from_workload(wl, device=local, stepper=a.stepper, precision=precision)
    if world > 1:
        from paper_2205_15000_b200 import sharding
        sharding.attach(ctx, wl.t, wl.n_energies)
    ng = wl.nx * wl.ny
    delta = dev(wl.delta0.astype(np.complex128))
    aix = torch.zeros((wl.ny, wl.nx), dtype=torch.float64, device=devname); aiy = torch.zeros_like(aix)
    dev_ax, dev_ay = dev(wl.Aext_x), dev(wl.Aext_y)
    ctx.sc_set_external_field(dev_ax, dev_ay)
    acc = wl.accelerator
    dn = torch.zeros_like(delta); jx = torch.zeros_like(aix); jy = torch.zeros_like(aix); fe = torch.zeros_like(aix)

    def step():
        if a.sweep_only:
            ctx.sc_set_fields(delta, dev_ax, dev_ay)
            ctx.sc_riccati_sweep(dn, jx, jy, fe)
        else:
            ctx.sc_iterate(acc, 1.0, False, delta, aix, aiy)

    # the first iterations: their cost (context for `transient`), and the burn-in that takes the run past them
    transient = []
    for it in range(burnin):
        ctx.sc_debug_march_time(); ctx.sc_debug_march_units()
        t0 = time.perf_counter(); step(); torch.cuda.synchronize(); dt = time.perf_counter() - t0
        u = ctx.sc_debug_march_units()
        transient.append({"iteration": it, "s": round(dt, 4), "march_ms": round(ctx.sc_debug_march_time()[0], 1),
                          "stored_T": round(u[1] / max(u[0], 1), 4), "pole_table": round(u[2] / max(u[0], 1), 4)})
    for _ in range(max(a.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(local); sampler.start()
    ms, mk_ms, nl, units, launches = time_iterations(ctx, torch, dist, world, devname, a.steps, step)
    clocks = sampler.stop()
    kernel = ctx.sc_debug_last_march_variant()

    # end to end through the C ABI with HOST buffers, continuing on the same stationary part of the run: every step copies
    # Delta and A_ind from pinned host memory, iterates, and copies Delta, A_ind and the residuals back
    hd = torch.empty((wl.ny, wl.nx), dtype=torch.complex128).pin_memory(); hd.copy_(delta)
    hax = torch.zeros((wl.ny, wl.nx), dtype=torch.float64).pin_memory(); hay = torch.zeros_like(hax).pin_memory()
    hax.copy_(aix); hay.copy_(aiy)
    torch.cuda.synchronize()
    e2e = None
    if not a.sweep_only:
        if world > 1:
            dist.barrier()
        ctx.sc_debug_march_units()
        t0 = time.perf_counter()
        for _ in range(a.steps):
            delta.copy_(hd, non_blocking=True); aix.copy_(hax, non_blocking=True); aiy.copy_(hay, non_blocking=True)
            st2 = ctx.sc_iterate(acc, 1.0, False, delta, aix, aiy, want_stats=True)
            hd.copy_(delta, non_blocking=True); hax.copy_(aix, non_blocking=True); hay.copy_(aiy, non_blocking=True)
            torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / a.steps
        ue = ctx.sc_debug_march_units()
        if world > 1:
            tmax = torch.tensor([e2e_s], dtype=torch.float64, device=devname)
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
            e2e_s = float(tmax.item())
        e2e = {"s_per_step": e2e_s, "res_delta_last": st2.res_delta, "bytes": ng * 16 + 2 * ng * 8,
               "units_share_stored_T": ue[1] / max(ue[0], 1), "units_share_recompute_pole_table": ue[2] / max(ue[0], 1)}

    # logical / executed update counts of one sweep (one extra sweep with stats, outside the timed regions)
    ctx.sc_set_fields(delta, dev_ax + aix, dev_ay + aiy)
    st = ctx.sc_riccati_sweep(dn, jx, jy, fe, want_stats=True)
    n_updates, n_exec = st.n_updates, st.n_updates_executed
    if world > 1:
        tot = torch.tensor([n_updates, n_exec], dtype=torch.float64, device=devname)
        dist.all_reduce(tot)
        n_updates, n_exec = int(tot[0].item()), int(tot[1].item())
    roof = march_roofline(a, wl, ctx, kernel, mk_ms, nl, units, ms / a.steps, precision, full_size, clocks)
    ctx.close()
    del ctx
    torch.cuda.empty_cache()
    return dict(ms=ms, clocks=clocks, launches=launches, roofline=roof, e2e=e2e, n_updates=n_updates, n_exec=n_exec, transient=transient)


def ldos_leg(sc, torch, local, steps):
    """sc_ldos on configs[3] (d-wave [110] square, 512 real energies, 128 angles): 8 boundary sweeps + the LDOS sweep"""
    wl = workloads.make_workload(3)
    devname = f"cuda:{local}"
    ctx = sc.ScContext.from_workload(wl, device=local)
    ctx.sc_set_fields(torch.as_tensor(np.ascontiguousarray(wl.delta0.astype(np.complex128)), device=devname))
    out = torch.zeros((len(wl.ldos_energies), wl.ny, wl.nx), dtype=torch.float64, device=devname)
    iters = 8
    st = ctx.sc_ldos(wl.ldos_energies, wl.ldos_broadening, iters, out, want_stats=True)        # warm-up (allocations, tables)
    torch.cuda.synchronize()
    ctx.sc_debug_march_time(); ctx.sc_debug_launch_count()
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        ctx.sc_ldos(wl.ldos_energies, wl.ldos_broadening, iters, out)
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    mms, nl = ctx.sc_debug_march_time()
    launches = ctx.sc_debug_launch_count()
    kernel = ctx.sc_debug_last_march_variant()
    ok = bool(torch.isfinite(out).all().item()) and bool((out[:, torch.as_tensor(wl.mask > 0, device=devname)] > 0).all().item())
    ctx.close()
    return {"workload": f"BASELINE.json configs[3]: {wl.name}", "grid": f"{wl.nx}x{wl.ny}", "n_angles": wl.n_angles,
            "n_energies": len(wl.ldos_energies), "boundary_sweeps": iters, "dtype": "f64",
            "value": st.n_updates / (ms * 1e-3), "unit": UNIT, "s_per_call": ms * 1e-3, "updates_per_call": st.n_updates,
            "march_ms_per_call": mms / steps, "march_launches_per_call": nl / steps, "gpu_launches_per_call": launches / steps,
            "last_march_kernel": "sck::" + kernel, "ldos_positive_and_finite": ok,
            "note": "general (off-axis) energies: complex Taylor table of T (Horner, 4 instructions per term); boundary sweeps "
                    "march for the end values only (MODE 2), the last sweep writes Re g per (node, energy) and is rotated back per energy"}


def run_ours(a):
    import torch
    import torch.distributed as dist
    import paper_2205_15000_b200 as sc

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    if a.ldos_only:
        print(json.dumps({"metric": METRIC, "ldos": ldos_leg(sc, torch, local, a.steps)}))
        return
    if a.issue_probe:
        ctx = sc.ScContext.from_workload(workloads.make_workload(0), device=local)
        names = {10: "DFMA only", 11: "+ 0.5 integer per DFMA", 12: "+ 1 integer per DFMA", 13: "+ 0.125 LDS (and its DADD) per DFMA",
                 14: "+ 0.375 integer + 0.125 LDS (and its DADD) per DFMA", 15: "DFMA only, three different changing register operands"}
        base = ctx.sc_debug_pipe_peak(10, 1.0)
        print(json.dumps({"issue_probe": {names[k]: {"dfma_tflops": 2e-12 * v, "of_dfma_only": v / base}
                                          for k, v in ((k, ctx.sc_debug_pipe_peak(k, 1.0)) for k in names)}}))
        return
    wl = workload_from_args(a)
    full_size = world == 1 and not (a.pts_per_xi or a.n_angles or a.n_energies or a.size_scale != 1.0)
    burnin = a.burnin if a.burnin is not None else (12 if (wl.kappa > 0 and not a.sweep_only) else 0)
    L = run_leg(a, sc, torch, dist, wl, local, world, a.precision, burnin, full_size)

    # configs[4]: "... FP64, with an FP32 mode also timed": the same legs with opts.precision = 32, beside the headline
    fp32 = None
    if a.precision == 64 and wl.cfg == 4 and not a.no_fp32_leg and not a.sweep_only:
        F = run_leg(a, sc, torch, dist, wl, local, world, 32, burnin, full_size)
        fp32 = {"dtype": "f32", "value": F["n_updates"] * a.steps / (F["ms"] * 1e-3), "unit": UNIT, "ms_per_step": F["ms"] / a.steps,
                "e2e_value": F["n_updates"] / F["e2e"]["s_per_step"], "clocks": F["clocks"], "roofline": F["roofline"]}
    ldos = None
    if full_size and wl.cfg == 4 and a.precision == 64 and not a.no_ldos_leg and not a.sweep_only and rank == 0:
        ldos = ldos_leg(sc, torch, local, max(1, min(a.steps, 2)))

    ms, n_updates = L["ms"], L["n_updates"]
    value = n_updates * a.steps / (ms * 1e-3)
    cfg = config_of(wl, a, {"seconds_per_self_consistent_iteration": ms / a.steps / 1e3,
                            "updates_per_step": n_updates, "updates_executed_per_step": L["n_exec"],
                            "updates_counted": "LOGICAL updates (gamma and gamma-tilde, every angle, every energy, every piece: the metric's "
                                               "unit and what the CPU oracle executes); the kernel executes half of them, Eq. 13 gives the rest",
                            "value_executed_updates_per_s": L["n_exec"] * a.steps / (ms * 1e-3),
                            "stepper": "closed-form" if a.stepper == 0 else "implicit mid-point",
                            "parallelism": f"energy-sharded x{world}, 1 all-reduce/sweep" if world > 1 else "single GPU",
                            "burnin_iterations": burnin,
                            "timed_state": "iterations after the Barzilai-Borwein transient of A_ind (stationary cost per iteration); "
                                           "the e2e steps follow the timed ones on the same part of the run",
                            "transient": L["transient"]})
    if a.sweep_only:
        cfg["step"] = "one sc_riccati_sweep at the initial fields (A = A_ext)"
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": max(a.warmup, 3),
            "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64" if a.precision == 64 else "f32", "data": "synthetic", "config": cfg, "clocks": L["clocks"],
            "gpu_launches": L["launches"], "roofline": L["roofline"]}
    if L["e2e"]:
        e = L["e2e"]
        line["e2e"] = {"value": n_updates / e["s_per_step"], "unit": UNIT, "h2d_bytes_per_step": e["bytes"], "d2h_bytes_per_step": e["bytes"] + 64,
                       "s_per_step": e["s_per_step"], "res_delta_last": e["res_delta_last"],
                       "units_share_stored_T": e["units_share_stored_T"], "units_share_recompute_pole_table": e["units_share_recompute_pole_table"]}
    if fp32:
        line["config"]["fp32_mode"] = fp32
    if ldos:
        line["config"]["ldos"] = ldos
    if rank == 0:
        try:
            line["roofline"]["textbook_count_context"] = textbook_count()
        except Exception as ex:       # the oracle is test infrastructure: its absence must not break the bench
            line["roofline"]["textbook_count_context"] = {"unavailable": str(ex)}
    if not a.no_cpu_baseline and rank == 0:
        cores = os.cpu_count() or 1
        u, t, desc = oracle_sample(wl, cores)
        line["cpu_baseline"] = {"value": u / t, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "note": CPU_NOTE}
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
