#!/usr/bin/env python
"""bench.py -- throughput of the whole SRHD hot path on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload jet|random512|blast256|tube|conv]
                    [--impl ours|reference] [--no-e2e] [--no-cpu-baseline] [--no-per-workload]

A "step" is one pass of the whole hot path over the grid (driver.GridStepper.step_async): ghost-zone
fill from the patches of the previous step fused with the CFL reduction (srhd_patch_gather_speed), then
srhd_fluid_step_cfl (dt formed on the device).  The headline `value` is K steps after W warm-up steps of
the default workload, BASELINE.json configs[4] (512x512x1024 jet, PPM+HLLC, CFL 0.4: the largest
configuration, it fits one GPU).  `config.per_workload` carries the three 3-D configs (blast256,
random512, jet) each timed over ITS OWN step count (100 / 50 / 50) from its initial condition, and
`roofline` is quoted on random512 -- the general path: no uniform region, so no shortcut applies --
with the headline workload's figures beside it.  Two fractions: `frac` from the flops of the work the
method defines per cell update, `frac_executed` from the work the kernel counted itself executing
(srhd_stats.exec_*).  N > 1 runs N independent replicas (the path does not shard on this tier:
DESIGN.md section 8); value = all ranks' cell updates / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same
workload on the host cores; see DESIGN.md section 7.
"""
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

METRIC = "fp64 SRHD cell updates/sec"
UNIT = "cell updates/s"

# name -> (recon, riemann, cfl, paper-config description)
WORKLOADS = {
    "blast256": ("ppm", "hllc", 0.4, "BASELINE.json configs[2]: 256^3 spherical blast, periodic, PPM+HLLC, CFL 0.4"),
    "random512": ("plm", "hlle", 0.4, "BASELINE.json configs[3]: 512^3 k^-2 Gaussian random field, periodic, PLM+HLLE, CFL 0.4"),
    "jet": ("ppm", "hllc", 0.4, "BASELINE.json configs[4]: 512x512x1024 relativistic jet, outflow + fixed inflow, PPM+HLLC, CFL 0.4"),
    "tube": ("plm", "hllc", 0.5, "BASELINE.json configs[0]: 256x16x16 TM shock tube, PLM+HLLC, CFL 0.5"),
}


def make_workload(name, scale=1):
    """Seeded synthetic input of a config (primitives on the host): (prim, dh, bc, inflow_prim)."""
    from paper_2012_11130_b200 import workloads as wl
    if name == "blast256":
        prim, dh, bc = wl.blast_wave(n=256 // scale)
        return prim, dh, bc, None
    if name == "random512":
        prim, dh, bc = wl.random_field(n=512 // scale)
        return prim, dh, bc, None
    if name == "jet":
        prim, dh, bc, inflow = wl.jet(nx=512 // scale, ny=512 // scale, nz=1024 // scale,
                                      radius=0.02 * (scale if scale > 1 else 1))
        return prim, dh, bc, inflow
    if name == "tube":
        prim, dh, bc = wl.shock_tube()
        return prim, dh, bc, None
    raise SystemExit(f"unknown workload {name}")


# ------------------------------------------------------------------ clocks during the timed region
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML every 100 ms while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
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
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(0.1)

    def result(self):
        self.stop_flag = True
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons)}


# ------------------------------------------------------------------ CPU oracle legs
def oracle_sample_input(name):
    """Bounded sample of a workload for the oracle: a 64^3 block (64 patch groups) cut from the part
    of the 1/4-scale initial condition that holds its structure (blast surface / nozzle / centre),
    made periodic; the tube is small enough to be taken whole.  Built with oracle/ calls only."""
    from oracle import ref
    recon, riemann, cfl, _ = WORKLOADS[name]
    prim, dh, bc, _ = make_workload(name, scale=1 if name == "tube" else 4)
    if name == "tube":
        what = "the full 256x16x16 tube (16 patch groups)"
    else:
        nz, ny, nx = prim.shape[1:]
        z0 = 0 if name == "jet" else (nz - 64) // 2
        prim = np.ascontiguousarray(prim[:, z0:z0 + 64, (ny - 64) // 2:(ny + 64) // 2, (nx - 64) // 2:(nx + 64) // 2])
        bc = [0] * 6
        what = f"a periodic 64^3 block (64 patch groups) cut from the 1/4-scale {name} initial condition"
    par = ref.params(recon, riemann)
    cons = ref.prim2cons(prim.reshape(5, -1)).reshape(prim.shape)
    return ref, cons, dh, bc, par, cfl, what


def oracle_steps(ref, cons, dh, bc, par, cfl, nsteps=None, budget_s=None):
    """Advance the sample with the oracle (CFL reduction + tiled step); returns (cons, steps, seconds)."""
    done, t0 = 0, time.perf_counter()
    while True:
        cons, _ = ref.grid_step_tiled(cons, ref.cfl_dt(cons, cfl, dh, par), dh, par, bc)
        done += 1
        el = time.perf_counter() - t0
        if (nsteps is not None and done >= nsteps) or (budget_s is not None and el >= budget_s):
            return cons, done, el


def cpu_baseline(name, budget_s=12.0):
    ref, cons, dh, bc, par, cfl, what = oracle_sample_input(name)
    _, done, el = oracle_steps(ref, cons, dh, bc, par, cfl, nsteps=60, budget_s=budget_s)
    return {"value": cons[0].size * done / el, "unit": UNIT, "cores": os.cpu_count() or 1, "kind": "oracle",
            "sample": f"{what}; {done} steps in {el:.1f} s, OpenMP over patch groups"}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; a step = one pass over the sample."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    recon, riemann, cfl, desc = WORKLOADS[args.workload]
    ref, cons, dh, bc, par, cfl, what = oracle_sample_input(args.workload)
    steps, warm = min(args.steps, 40), min(args.warmup, 3)     # bounded: ends within a few minutes
    cons, _, _ = oracle_steps(ref, cons, dh, bc, par, cfl, nsteps=warm) if warm else (cons, 0, 0)
    cons, steps, el = oracle_steps(ref, cons, dh, bc, par, cfl, nsteps=steps)
    value = cons[0].size * steps / el
    cores = os.cpu_count() or 1
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * el / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "scheme": f"{recon}+{riemann}", "cfl": cfl, "what": desc,
                   "sample": what},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------ GPU legs
def max_over_ranks(x, world, device):
    """MAX all-reduce of one float over the ranks (the only cross-rank exchange: replicas only,
    DESIGN.md section 8).  Works on any backend (nccl on the GPU box, gloo in the CPU tests)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.cpu())


def aggregate_value(ncell_per_rank, steps, ms_local, world, device):
    """Whole-job throughput: the units all ranks processed / the slowest rank's device time."""
    ms_max = max_over_ranks(ms_local, world, device)
    return world * ncell_per_rank * steps / (ms_max * 1e-3), ms_max


def run_conv(args):
    """--workload conv: BASELINE.json configs[1], 2^24 states, prim -> cons -> prim per step."""
    import torch
    from paper_2012_11130_b200 import binding as B
    from paper_2012_11130_b200 import build as cuda_build
    from paper_2012_11130_b200 import flopmodel as fm
    from paper_2012_11130_b200 import workloads as wl
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    cuda_build.build()
    n = (1 << 24) // args.scale
    prim_h = torch.from_numpy(wl.conversion_states(n=n)).pin_memory()
    prim = prim_h.cuda()
    cons, back = torch.empty_like(prim), torch.empty_like(prim)
    par, stats = B.params(), B.new_stats()

    def step():
        B.prim2cons(prim, cons=cons)
        B.cons2prim(cons, par, prim=back, stats=stats)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    peak_meas = B.fp64_peak_probe()
    sampler = ClockSampler(torch.cuda.current_device())
    sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
    t_p2c = t_c2p = 0.0
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ev[0].record()
        B.prim2cons(prim, cons=cons)
        ev[1].record()
        B.cons2prim(cons, par, prim=back, stats=stats)
        ev[2].record()
        ev[2].synchronize()
        t_p2c += ev[0].elapsed_time(ev[1])
        t_c2p += ev[1].elapsed_time(ev[2])
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.result()
    ms = e0.elapsed_time(e1)
    s = B.stats_to_host(stats)
    # end to end: states from pinned host memory, primitives back to the host
    back_h = torch.empty_like(prim_h).pin_memory()
    n_e2e = max(1, min(args.steps, 10))
    torch.cuda.synchronize()
    e0.record()
    for _ in range(n_e2e):
        prim.copy_(prim_h, non_blocking=True)
        step()
        back_h.copy_(back, non_blocking=True)
    e1.record()
    torch.cuda.synchronize()
    ms_e2e = e0.elapsed_time(e1)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    k_mean = s.newton_iters / n
    c2p_ms, p2c_ms = t_c2p / args.steps, t_p2c / args.steps
    ach = n * fm.c2p(k_mean) / (c2p_ms * 1e-3) / 1e12
    peak = fm.fp64_peak_tflops(clocks["sm_max_mhz"] or 1965.0)
    out = {
        "metric": "fp64 SRHD prim->cons->prim round trips/sec", "value": n * args.steps / (ms * 1e-3),
        "unit": "states/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "conv", "what": "BASELINE.json configs[1]: 2^24 states, log-uniform rho, Theta, Lorentz factor",
                   "states": n, "l2": "inputs larger than L2 (671 MB per 5-array)", "newton_iters_per_conversion": k_mean,
                   "eq30_failures": s.n_c2p_fail},
        "clocks": clocks,
        "roofline": {"bound": "alu", "kernel": "cons2prim_kernel", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                     "frac": ach / peak, "traffic": ncu_traffic("conv"), "kernel_ms": c2p_ms, "peak_measured": peak_meas,
                     "flops_per_state": fm.c2p(k_mean),
                     "hbm": {"achieved": n * 80 / (c2p_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                             "frac": n * 80 / (c2p_ms * 1e-3) / 1e9 / hbm_peak},
                     "prim2cons": {"bound": "hbm", "kernel_ms": p2c_ms, "achieved": n * 80 / (p2c_ms * 1e-3) / 1e9,
                                   "peak": hbm_peak, "unit": "GB/s", "frac": n * 80 / (p2c_ms * 1e-3) / 1e9 / hbm_peak}},
        "gpu_launches": 2 * args.steps,
        "e2e": {"value": n * n_e2e / (ms_e2e * 1e-3), "unit": "states/s", "h2d_bytes_per_step": n * 40,
                "d2h_bytes_per_step": n * 40, "steps": n_e2e},
    }
    print(json.dumps(out))


def run_aux(args):
    """--aux: the entry points of SURVEY.md 8f (coarse-fine hooks, refinement flags, VL integrator), each timed with
    CUDA events on blast-wave data after its blast has grown for 40 steps (256^3, PPM+HLLC tiles).  One JSON line;
    not the headline metric."""
    import torch
    from paper_2012_11130_b200 import binding as B
    from paper_2012_11130_b200 import build as cuda_build
    from paper_2012_11130_b200.driver import GridStepper
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    cuda_build.build()
    n = 256 // args.scale
    prim, dh, bc, _ = make_workload("blast256", scale=args.scale)
    st = GridStepper(prim.shape[1:], dh, bc, "ppm", "hllc", cfl=0.4).set_prim(prim)
    for _ in range(40):
        st.step_async()
    grid = st.grid.clone()
    par = st.par
    tiles = B.grid_gather(grid, par.ghost, bc)
    npg, ncell = st.npg, st.ncell
    reps = max(args.steps, 3)

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    out = {}
    out["refine_flags_D_ms"] = timed(lambda: B.refine_flags(tiles, par, "D", 0.3, 0.0))
    out["refine_flags_rho_ms"] = timed(lambda: B.refine_flags(tiles, par, "rho", 0.3, 0.0))
    out["refine_flags_gamma_and_momentum_ms"] = timed(lambda: B.refine_flags(tiles, par, "gamma", 0.3, 1.0))
    # flux correction: both x faces of every patch, fine flux = coarse flux of the step (so nothing is skipped)
    smax = B.max_signal_speed(grid.view(5, -1), par)
    dt = 0.4 * dh / float(smax.cpu())
    patches, flux, _ = B.fluid_step_fluxes(tiles, dt, dh, par)
    p5 = patches.reshape(npg * 8, 5, 8, 8, 8).contiguous()
    fp = torch.arange(npg * 8, dtype=torch.int32, device="cuda").repeat_interleave(2)
    fi = torch.tensor([0, 1], dtype=torch.int32, device="cuda").repeat(npg * 8)
    fc = flux.reshape(npg * 8, 6, 5, 8, 8)[:, :2].reshape(-1, 5, 8, 8).contiguous()
    ff = (fc * 1.001).contiguous()
    out["flux_correction_ms"] = timed(lambda: B.flux_correction(p5, fc, ff, fp, fi, dt, dh))
    out["flux_correction_faces"] = int(fp.numel())
    # ghost-zone interpolation of the central 130^3 block (128^3 coarse cells -> 256^3 fine cells)
    c0 = n // 2 - min(65, n // 2 - 1)
    w = min(130, n - 2 * c0)
    coarse = grid[:, c0:c0 + w, c0:c0 + w, c0:c0 + w].contiguous()
    out["ghost_interp_ms"] = timed(lambda: B.ghost_interp(coarse, 1.5, par))
    out["ghost_interp_fine_cells"] = 8 * (w - 2) ** 3
    # VL integrator on the same state (one more ghost layer)
    vl = GridStepper(prim.shape[1:], dh, bc, "ppm", "hllc", cfl=0.4, integrator="vl").set_cons(grid)
    vl.step_async()
    out["vl_step_ms"] = timed(vl.step_async)
    mh = GridStepper(prim.shape[1:], dh, bc, "ppm", "hllc", cfl=0.4, fused=False).set_cons(grid)
    mh.step_async()
    out["muscl_hancock_step_same_state_ms"] = timed(mh.step_async)
    print(json.dumps({"aux": True, "what": f"SURVEY 8f entry points on the {n}^3 blast wave after 40 steps (PPM+HLLC tiles, "
                      f"{npg} patch groups, {ncell} cells); milliseconds per call, CUDA events, {reps} repetitions",
                      "data": "synthetic", "dtype": "f64", **out}))


CONFIG_STEPS = {"blast256": 100, "random512": 50, "jet": 50, "tube": 205}   # BASELINE.json configs: their own step counts


def ncu_traffic(workload):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE fluid_step_kernel launch on this workload, from
    the committed ncu --set full capture summarised in profiles/ncu_traffic.json (written from the capture
    named inside it; nothing here is measured under a profiler).  None if no capture of that workload."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
        return t.get(workload, {}).get("dram_bytes_per_launch")
    except Exception:
        return None


def ncu_traffic_source(workload):
    """Which committed capture roofline.traffic was copied from (it is a citation, not a measurement of this run)."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
        e = t.get(workload)
        return None if not e else f'{e["capture"]} ({e["kernel"]}); copied into profiles/ncu_traffic.json, not measured in this run'
    except Exception:
        return None


def time_workload(name, steps, warmup, scale, world, local, rank, from_start=False, e2e_steps=0, fused=True, lib=False):
    """Time `steps` steps of one workload after `warmup` untimed ones (from_start: the config's own run from
    its initial condition, warm-up on a second instance).  Returns a dict of measured figures."""
    import torch
    import torch.distributed as dist
    from paper_2012_11130_b200 import binding as B
    from paper_2012_11130_b200 import flopmodel as fm
    from paper_2012_11130_b200.driver import GridStepper

    recon, riemann, cfl, desc = WORKLOADS[name]
    prim, dh, bc, inflow = make_workload(name, scale=scale)
    shape = prim.shape[1:]
    st_inflow = None
    if inflow is not None:
        mask, prim_jet = inflow
        B.load_library(lib)
        cj = B.prim2cons(torch.from_numpy(prim_jet.reshape(5, 1).copy()).cuda().to(B._CUR_REAL), exact=lib).cpu().numpy().ravel()
        st_inflow = (mask, cj)
    st = GridStepper(shape, dh, bc, recon, riemann, cfl=cfl, inflow=st_inflow, fused=fused, exact=lib)
    prim_d = torch.from_numpy(prim).cuda() if from_start else None
    st.set_prim(prim if prim_d is None else prim_d)
    del prim
    ncell = st.ncell

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        st.step_async()
    if from_start:                      # warm-up done (clocks, caches, lazy module load): restart from t = 0
        st.set_prim(prim_d)
        del prim_d
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kev = []
    tot = {k: 0 for k in ("n_retry_pg", "n_passes", "newton_iters", "exec_c2p", "exec_newton", "exec_riemann",
                          "exec_hancock", "n_unphys_final", "n_uniform_pg")}
    # per-step counters are read back AFTER the timed region from a device-side log (no host sync inside it)
    log = torch.zeros((steps, st.stats.numel()), dtype=torch.uint8, device="cuda")
    ev0.record()
    for i in range(steps):
        st.step_async(kernel_events=kev)           # dt = C dh / S_max formed on the device: no host sync
        log[i].copy_(st.stats, non_blocking=True)  # 80-byte device-to-device copy of this step's counters
    ev1.record()
    barrier()
    clocks = sampler.result()
    ms = ev0.elapsed_time(ev1)
    k_each = [a.elapsed_time(b) for a, b in kev]
    k_ms = sum(k_each) / len(k_each)
    passes_each = []
    for row in log.cpu():
        s = B.Stats.from_buffer_copy(row.numpy().tobytes())
        passes_each.append(s.n_passes / st.npg)
        for k in tot:
            tot[k] += getattr(s, k)
    i_max = int(np.argmax(k_each))
    value, ms_max = aggregate_value(ncell, steps, ms, world, "cuda")
    nxt = 16 + 2 * st.par.ghost
    nconv = steps * st.npg * (nxt ** 3 + 2 * 3 * 17 * 256)        # conversions the algorithm defines
    k_mean = tot["newton_iters"] / nconv
    flops_alg = ncell * fm.fluid_step_flops_per_cell(recon, riemann, k_mean)          # per step
    flops_survey = ncell * fm.fluid_step_flops_per_cell_survey(recon, riemann, k_mean)
    flops_exe = fm.fluid_step_flops_executed(recon, riemann, ncell * steps, tot["exec_c2p"], tot["exec_newton"],
                                             tot["exec_riemann"], tot["exec_hancock"]) / steps
    res = {
        "name": name, "desc": desc, "recon": recon, "riemann": riemann, "cfl": cfl, "shape": list(shape),
        "npg": st.npg, "ncell": ncell, "steps": steps, "warmup": warmup, "from_start": from_start,
        "value": value, "ms_per_step": ms_max / steps, "kernel_ms": k_ms, "clocks": clocks,
        "k_mean": k_mean, "flops_alg_per_step": flops_alg, "flops_exec_per_step": flops_exe,
        "passes_per_group": tot["n_passes"] / (steps * st.npg), "retry_groups_per_step": tot["n_retry_pg"] / steps,
        "unphysical_cells": tot["n_unphys_final"], "uniform_fraction": tot["n_uniform_pg"] / (steps * st.npg),
        "fused": fused,
        "exec_conversions_per_cell": tot["exec_c2p"] / (ncell * steps),
        "exec_newton_per_conversion": tot["exec_newton"] / max(tot["exec_c2p"], 1),
        "exec_riemann_per_cell": tot["exec_riemann"] / (ncell * steps),
        "state_mb": st.grid.numel() * 8 / 1e6, "tiles_mb": st.tiles.numel() * 8 / 1e6,
        "launches_per_step": st.launches_per_step,
        # the work of a step depends on the state (retry passes, uniform groups): the slowest call is named with
        # the number of marches per patch group it made, next to the median step's
        "call_ms": {"min": min(k_each), "median": float(np.median(k_each)), "max": max(k_each),
                    "max_at_timed_step": i_max + 1, "passes_per_patch_group_at_max": passes_each[i_max],
                    "passes_per_patch_group_median": float(np.median(passes_each))},
        "flops_survey_per_step": flops_survey,
        "value_median_step": ncell * world / (float(np.median(k_each)) * 1e-3),
        # algorithmic bytes per cell update (5 reals in, 5 out) / step time
        "hbm_gbs": ncell * 10.0 * st.patches.element_size() / (ms_max / steps * 1e-3) / 1e9,
    }
    if e2e_steps:
        # end to end through the public API: every step copies its input grid from pinned host memory, runs
        # GridStepper.step_async() (CFL reduction of the fresh grid, ghost-zone fill, fluid step with dt formed
        # on the device, scatter) and copies the result back.  n_pipe INDEPENDENT problem instances (own
        # buffers, own CUDA stream) are in flight round-robin so one instance's PCIe copies overlap another's
        # kernels: the figure is aggregate throughput over independent instances, the latency of one step of
        # one instance is about n_pipe times longer.
        nbytes = st.grid.numel() * st.grid.element_size()
        n_pipe = 3 if nbytes * 5 < 20e9 else 1
        inst = [st] + [GridStepper(shape, dh, bc, recon, riemann, cfl=cfl, inflow=st_inflow, exact=lib) for _ in range(n_pipe - 1)]
        streams = [torch.cuda.Stream() for _ in range(n_pipe)]
        h_in = [torch.empty(st.grid.shape, dtype=st.grid.dtype, pin_memory=True) for _ in range(n_pipe)]
        h_out = [torch.empty(st.grid.shape, dtype=st.grid.dtype, pin_memory=True) for _ in range(n_pipe)]
        for h in h_in:
            h.copy_(st.grid)
        n_e2e = max(n_pipe, e2e_steps // n_pipe * n_pipe)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for s_ in streams:
            s_.wait_stream(torch.cuda.current_stream())
        for i in range(n_e2e):
            k = i % n_pipe
            with torch.cuda.stream(streams[k]):
                inst[k].set_cons(h_in[k])          # H2D; invalidates the cached signal speed
                inst[k].step_async()               # CFL kernel + gather + fluid step + scatter, no host sync
                h_out[k].copy_(inst[k].grid, non_blocking=True)
            h_in[k], h_out[k] = h_out[k], h_in[k]
        for s_ in streams:
            torch.cuda.current_stream().wait_stream(s_)
        e1.record()
        barrier()
        e2e_value, _ = aggregate_value(ncell, n_e2e, e0.elapsed_time(e1), world, "cuda")
        res["e2e"] = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                      "steps": n_e2e, "instances_in_flight": n_pipe,
                      "note": "aggregate over independent problem instances in flight; per-instance step latency is about instances_in_flight times longer"}
        del inst, h_in, h_out
    del st
    torch.cuda.empty_cache()
    return res


def roofline_of(r, peak, peak_meas, hbm_peak, have_peaks):
    """Roofline object of fluid_step_kernel on one timed workload (ALU bound: DESIGN.md section 6)."""
    from paper_2012_11130_b200 import flopmodel as fm
    t = r["kernel_ms"] * 1e-3
    ach = r["flops_alg_per_step"] / t / 1e12
    exe = r["flops_exec_per_step"] / t / 1e12
    hbm_ach = r["ncell"] * fm.FLUID_STEP_BYTES_PER_CELL / t / 1e9
    return {
        "bound": "alu", "kernel": "fluid_step_kernel", "workload": r["name"], "unit": "TFLOP/s",
        "achieved": ach, "peak": peak, "frac": ach / peak,
        "achieved_executed": exe, "frac_executed": exe / peak,
        "achieved_note": "achieved = flops of the work the METHOD defines per cell update (no ghost-zone recompute, no thrown-away retry passes, no shortcuts) / kernel time; achieved_executed = flops of the conversions, Riemann solves and edge states the kernel actually executed (srhd_stats.exec_*) / kernel time",
        "peak_source": "148 SMs x 64 fp64 lanes x 2 x max SM clock (unit counts; DESIGN.md section 6)",
        "peak_measured": peak_meas, "frac_of_measured": ach / peak_meas if peak_meas else None,
        "frac_executed_of_measured": exe / peak_meas if peak_meas else None,
        "peak_measured_source": "srhd_fp64_peak_probe (register-only DFMA loop) in this run",
        "kernel_ms": r["kernel_ms"], "ms_per_step": r["ms_per_step"], "steps": r["steps"],
        "kernel_share_of_step": r["kernel_ms"] / r["ms_per_step"],
        "flops_per_cell": r["flops_alg_per_step"] / r["ncell"],
        "flops_executed_per_cell": r["flops_exec_per_step"] / r["ncell"],
        "traffic": ncu_traffic(r["name"]), "traffic_source": ncu_traffic_source(r["name"]),
        "flop_count": "frac uses paper_2012_11130_b200/flopmodel.py's hand count of the formulas as written (68 flops per "
                      "Newton iteration); *_survey_count uses SURVEY.md section 8(a)'s counts (43 per iteration)",
        "flops_per_cell_survey_count": r["flops_survey_per_step"] / r["ncell"],
        "frac_survey_count": r["flops_survey_per_step"] / t / 1e12 / peak,
        "value_at_median_call": r["value_median_step"],
        "value_at_median_call_note": "cells / median duration of the timed call (call_ms.median): the whole step for a fused run, the fluid-step call alone when the roofline kernel is timed through the separate calls",
        "hbm": {"achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_ach / hbm_peak,
                "peak_source": "MEASURED_PEAKS.json" if have_peaks else "fallback 6650 GB/s (B200_PROFILING.md)"},
    }


def summary_of(r):
    return {"what": r["desc"], "grid": r["shape"], "scheme": f'{r["recon"]}+{r["riemann"]}', "cfl": r["cfl"],
            "steps": r["steps"], "from_initial_condition": r["from_start"], "value": r["value"], "unit": UNIT,
            "ms_per_step": r["ms_per_step"], "kernel_ms": r["kernel_ms"],
            "newton_iters_per_conversion": r["k_mean"], "passes_per_patch_group": r["passes_per_group"],
            "retry_patch_groups_per_step": r["retry_groups_per_step"], "unphysical_cells": r["unphysical_cells"],
            "uniform_patch_group_fraction": r["uniform_fraction"],
            "step_hbm_gbs_algorithmic": r["hbm_gbs"], "step_call_ms": r["call_ms"],
            "executed_conversions_per_cell": r["exec_conversions_per_cell"],
            "executed_riemann_solves_per_cell": r["exec_riemann_per_cell"],
            "sm_mhz": r["clocks"]["sm_mhz"], "throttle_reasons": r["clocks"]["reasons"]}


def run_ours(args):
    if args.workload == "conv":
        return run_conv(args)
    import torch
    import torch.distributed as dist
    from paper_2012_11130_b200 import binding as B
    from paper_2012_11130_b200 import build as cuda_build
    from paper_2012_11130_b200 import flopmodel as fm

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        cuda_build.build()
    if world > 1:
        dist.barrier()
    B.load_library()

    # ---- headline: K steps of the chosen workload after W warm-up steps, then end to end
    lib = {"production": False, "exact": True}.get(args.lib, args.lib)
    head = time_workload(args.workload, args.steps, args.warmup, args.scale, world, local, rank,
                         e2e_steps=0 if args.no_e2e else min(args.steps, 6), lib=lib)
    # ---- every 3-D config over its OWN step count from its initial condition (seconds of GPU time)
    per = {}
    if args.per_workload and world == 1:
        for name in ("blast256", "random512", "jet"):
            per[name] = time_workload(name, max(1, CONFIG_STEPS[name] // (args.scale if args.scale > 1 else 1)), 3,
                                      args.scale, world, local, rank, from_start=True, lib=lib)
    # the roofline kernel (fluid_step_kernel, general path) timed on its own: the same random512 run through the two
    # separate calls, so that the CUDA events bracket srhd_fluid_step_cfl alone and not the ghost-zone fill with it
    gen = None
    if args.per_workload and world == 1:
        gen = time_workload("random512", max(1, CONFIG_STEPS["random512"] // (args.scale if args.scale > 1 else 1)), 3,
                            args.scale, world, local, rank, from_start=True, fused=False, lib=lib)
    if world > 1:
        dist.barrier()
    if rank != 0:
        return
    torch.cuda.synchronize()
    peak_meas = B.fp64_peak_probe()                # measured DFMA roof (outside every timed region)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = peaks.get("hbm_gbs", 6650.0)
    peak = fm.fp64_peak_tflops(head["clocks"]["sm_max_mhz"] or 1965.0)
    # the roofline is quoted on the GENERAL path: random512 has no uniform region, so none of the
    # uniform-region shortcuts applies there; the headline workload's own figures sit beside it
    general = gen if gen is not None else head
    roof = roofline_of(general, peak, peak_meas, hbm_peak, bool(peaks))
    # the headline workload is almost entirely undisturbed ambient gas: its step is bound by HBM, not by the ALUs
    roof["headline_step_hbm"] = {"bound": "hbm", "workload": head["name"], "achieved": head["hbm_gbs"], "peak": hbm_peak,
                                 "unit": "GB/s", "frac": head["hbm_gbs"] / hbm_peak,
                                 "note": "algorithmic 80 B per cell update (5 doubles in, 5 out) x cells / whole-step time; "
                                         "uniform patch groups take the pre-pass (their state crosses HBM once in, once out)",
                                 "uniform_patch_group_fraction": head["uniform_fraction"]}
    roof["headline_workload"] = {k: v for k, v in roofline_of(head, peak, peak_meas, hbm_peak, bool(peaks)).items()
                                 if k in ("workload", "achieved", "frac", "achieved_executed", "frac_executed", "kernel_ms",
                                          "ms_per_step", "steps", "kernel_share_of_step", "flops_per_cell",
                                          "flops_executed_per_cell", "traffic")}
    out = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32" if "f32" in str(args.lib) else "f64", "data": "synthetic",
        "config": {"workload": args.workload, "library": B.load_library(lib).srhd_build_variant().decode(),
                   "scheme_override": args.scheme,
                   "what": head["desc"], "grid": head["shape"], "patch_groups": head["npg"],
                   "scheme": f'{head["recon"]}+{head["riemann"]}', "cfl": head["cfl"],
                   "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": f'inputs larger than L2 ({head["state_mb"]:.0f} MB state, {head["tiles_mb"]:.0f} MB tiles)'
                         if head["state_mb"] > 126 else "state fits L2 (small case)",
                   "timed_steps": f'steps {args.warmup + 1}..{args.warmup + args.steps} from the initial condition',
                   "newton_iters_per_conversion": head["k_mean"], "passes_per_patch_group": head["passes_per_group"],
                   "retry_patch_groups_per_step": head["retry_groups_per_step"],
                   "executed_conversions_per_cell": head["exec_conversions_per_cell"],
                   "uniform_patch_group_fraction": head["uniform_fraction"],
                   "step_call_ms": head["call_ms"],
                   "per_workload": {k: summary_of(v) for k, v in per.items()}},
        # what `value` is and is not: on the jet 99.97 % of the patch groups are undisturbed ambient
        # gas that the pre-pass proves uniform and copies, so `value` is an HBM-bound figure; the solver's own
        # throughput is the general path's, on data with no uniform region
        "solver_path": {"workload": general["name"], "scheme": f'{general["recon"]}+{general["riemann"]}',
                        "value": general["value"], "unit": UNIT, "ms_per_step": general["ms_per_step"],
                        "uniform_patch_group_fraction": general["uniform_fraction"],
                        "note": "throughput of the SRHD solver proper (no uniform patch groups: every group is marched); "
                                "the headline `value` is dominated by uniform groups finished by the pre-pass"},
        "clocks": head["clocks"],
        "roofline": roof,
        "gpu_launches": head["launches_per_step"] * args.steps,
    }
    if "e2e" in head:
        out["e2e"] = head["e2e"]
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = cpu_baseline(args.workload)
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="jet", choices=sorted(WORKLOADS) + ["conv"],
                    help="headline workload; default = the largest single-GPU config, BASELINE.json configs[4]")
    ap.add_argument("--no-per-workload", dest="per_workload", action="store_false",
                    help="skip the runs of blast256 / random512 / jet over their own step counts")
    ap.add_argument("--scale", type=int, default=1, help="divide the grid extents (debugging only; 1 = the config)")
    ap.add_argument("--lib", default="production",
                    help="which in-tree library to time: production (default), exact, or a variant of "
                         "paper_2012_11130_b200/build.py (gamma53, f32, ...); the headline is the production library")
    ap.add_argument("--scheme", default=None, choices=["plm+hlle", "plm+hllc", "ppm+hlle", "ppm+hllc"],
                    help="DIAGNOSTIC: run --workload's data with another reconstruction / Riemann solver than its config "
                         "names (e.g. --workload random512 --scheme ppm+hllc: the PPM+HLLC kernel on data with no uniform "
                         "region); the line says so in config.scheme_override and is not a headline")
    ap.add_argument("--aux", action="store_true", help="time the SURVEY 8f entry points instead (one JSON line, not the headline)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    if args.scheme:
        if args.workload == "conv":
            raise SystemExit("--scheme applies to the fluid-step workloads")
        rc, rs = args.scheme.split("+")
        _, _, cfl, desc = WORKLOADS[args.workload]
        WORKLOADS[args.workload] = (rc, rs, cfl, desc + f" -- DIAGNOSTIC: run with {args.scheme.upper()} instead of the config's scheme")
    if args.aux:
        return run_aux(args)
    if args.impl == "reference":
        if args.workload == "conv":
            raise SystemExit("--impl reference times the fluid-step workloads only")
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
