#!/usr/bin/env python
"""bench.py -- cell-updates/sec of the patch-group MHD update on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--scheme vl|ctu] [--prec f32|f64]

Workload (config.workload): BASELINE.json configs[1] -- a batch of 512 patch groups of 16^3 cells (+3 ghost cells,
VL+PLM+HLLD+CT; flux_out and emf_out requested), seeded synthetic state of paper_1804_03479_b200.inputs.config2_batch
(DESIGN.md "Input recipe").  One "step" = one pass of the whole hot path over the batch: mhd_advance_dt = S0-S8 with the
CFL reduction (S9) of the new state fused into the final update (bit-identical to mhd_advance + mhd_dt_reduce).  The headline line is FP32 (the paper's headline precision); the same run measures
FP64 and reports it under "fp64".  The batch (177 MB FP32 / 355 MB FP64 of input) is larger than the 126 MB L2, so
no explicit L2 flush is needed between iterations (config.l2: "inputs larger than L2").

N > 1 (torchrun): every rank advances its own 512-group batch (weak scaling, no data-path collective; the only
communication is the barrier around the timed region and the max-over-ranks of the device time).

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores, on the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

N_PS2, NGROUPS = 16, 512
PAPER_P100 = {"f32": 1.2e8, "f64": 5.5e7}       # PAPER.md:12, :465-467 (Tesla P100, VL+PLM+Roe) -- context only
# algorithmic work per Riemann solve and per group, DESIGN.md "Roofline arithmetic"
# exact operation counts of the oracle instantiated with a counting scalar (oracle/count_ops.cpp; add/sub/mul/div/sqrt = 1)
FLOP_PER_SOLVE = {"hlld": 381, "roe": 1107, "hlle": 361}
FLOP_PER_CELL_UPDATE = {("vl", "hlld"): 6263.5, ("vl", "roe"): 15289.0, ("ctu", "hlld"): 26067.6, ("ctu", "roe"): 35160.4}   # whole step
FLOP_PLM_PER_FACE = 140     # two MC-limited primitive slopes + the two face states (VL pass 2)
# dram__bytes_read.sum + dram__bytes_write.sum of each stage's launches of one 512-group step (two slices of 256), VL+PLM+HLLD, from the
# ncu --set full captures summarised in profiles/r01h_full_top_kernels.md and r01h_f64_full_top_kernels.md (MB)
NCU_TRAFFIC_MB = {"f32": {"pass1_fused": 968.0, "emf_pass1": 351.3, "half_step": 856.6, "flux_pass2": 609.4,
                          "emf_pass2": 229.2, "final_update": 418.6},
                  "f64": {"pass1_fused": 1756.3, "emf_pass1": 691.7, "half_step": 1631.1, "flux_pass2": 1058.2,
                          "emf_pass2": 438.1, "final_update": 831.7}}
NOMINAL_TFLOPS = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scheme", default="vl", choices=["vl", "ctu"])
    ap.add_argument("--riemann", default="hlld", choices=["hlle", "hlld", "roe"])
    ap.add_argument("--prec", default="f32", choices=["f32", "f64"], help="precision of the headline value")
    ap.add_argument("--groups", type=int, default=NGROUPS)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--config5", type=int, default=0, metavar="POOL", help="instead of the batch: BASELINE config 5, 262144 "
                    "group-updates (= 1024^3 cells) in FP32 streamed from a pinned pool of POOL groups (a multiple of 512, e.g. 4096), "
                    "VL+PLM and CTU+PPM, with and without transfers")
    ap.add_argument("--sweep", action="store_true", help="instead of the batch: throughput against the number of patch groups per "
                    "call (8 ... 4096; the axis of the paper's Fig. 18), FP32 and FP64, device-resident")
    ap.add_argument("--grid", type=int, default=0, help="instead of the batch: a periodic n^3 ABC grid (BASELINE config 3 "
                    "state) kept on the device; step = mhd_grid_advance_dt (pack + scheme with fused dt + unpack)")
    return ap.parse_args()


def scheme_params(args):
    from paper_1804_03479_b200 import mhd
    if args.scheme == "vl":
        return dict(scheme=mhd.VL, recon=mhd.PLM, g=3, name="VL+PLM")
    return dict(scheme=mhd.CTU, recon=mhd.PPM, g=4, name="CTU+PPM")


def faces_per_group(g, scheme):
    """Riemann solves per group in pass 1 and pass 2 (index ranges of DESIGN.md 'Index ranges')."""
    N, T = N_PS2, N_PS2 + 2 * g
    if scheme == "vl":
        return 3 * (T - 1) * T * T, 3 * (N + 1) * (N + 2) ** 2
    r = 2
    return 3 * (T - 2 * r - 1) * T * T, 3 * (N + 1) * (N + 2) ** 2


class ClockSampler(threading.Thread):
    """SM clock + throttle reasons sampled through NVML while the timed region runs."""

    def __init__(self, index, period=0.004):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.stop_flag, self.max_mhz = [], set(), False, None
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
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def result(self):
        self.stop_flag = True
        if self.is_alive():
            self.join(timeout=2)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


def hbm_peak():
    """measured copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the guide's fallback"""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def make_batch(G, g, npdt):
    """config-2 batch: a pool of 16 distinct seeded groups tiled to G (the kernels' work does not depend on values)."""
    import numpy as np
    from paper_1804_03479_b200 import inputs
    pool = min(G, 16)
    U, B, dh = inputs.config2_batch(pool, N=N_PS2, g=g, dtype=npdt)
    reps = (G + pool - 1) // pool
    return np.tile(U, (reps, 1))[:G].copy(), np.tile(B, (reps, 1))[:G].copy(), dh


def measure(args, prec_name, rank, world, dist):
    """Time K steps of mhd_advance_dt on device-resident data, then the per-stage profile, then e2e."""
    import numpy as np
    import torch
    from paper_1804_03479_b200 import mhd, shard
    sp = scheme_params(args)
    g, G = sp["g"], args.groups
    prec = mhd.FP32 if prec_name == "f32" else mhd.FP64
    npdt = np.float32 if prec_name == "f32" else np.float64
    esz = 4 if prec_name == "f32" else 8
    riem = {"hlle": mhd.HLLE, "hlld": mhd.HLLD, "roe": mhd.ROE}[args.riemann]
    dev = torch.device("cuda", torch.cuda.current_device())
    solver = mhd.Solver(mhd.make_config(N=N_PS2, g=g, scheme=sp["scheme"], recon=sp["recon"], riemann=riem, prec=prec,
                                        max_groups=G, device=dev.index))
    hU, hB, dh = make_batch(G, g, npdt)
    dU, dB = torch.from_numpy(hU).to(dev), torch.from_numpy(hB).to(dev)
    out = solver.alloc_outputs(G, planes=True, device=dev)
    stream = torch.cuda.current_stream()
    dt0, _ = solver.dt_reduce(dU, dB, G, g, dh, 0.3)

    def step():
        # S0-S8 + S9 as one call: the final update also reduces the CFL speed of the state it writes (bit-identical to
        # mhd_advance followed by mhd_dt_reduce on U_out / B_out, tests/test_gpu_api.py)
        return solver.advance_dt(dU, dB, out["U"], out["B"], out["flux"], out["emf"], G, dt0, dh, 0.3, stream)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(dev.index)
    l0 = solver.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    clocks = sampler.result()
    ms = e0.elapsed_time(e1)
    launches = solver.launch_count() - l0
    ms = shard.max_over_ranks(ms, dist, dev)          # job time = slowest rank's device time
    cells = G * N_PS2 ** 3 * args.steps * world
    res = dict(value=cells / (ms * 1e-3), ms_per_step=ms / args.steps, launches=launches, clocks=clocks)

    # per-stage device time over K more steps (events around every stage launch on the launching stream)
    solver.set_profiling(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    p0.record(stream)
    for _ in range(args.steps):
        step()
    p1.record(stream)
    torch.cuda.synchronize()
    prof = solver.get_profile()
    solver.set_profiling(False)
    prof_ms = p0.elapsed_time(p1)
    stages = {k: {"ms_per_step": v[0] / args.steps, "launches_per_step": v[1] / args.steps} for k, v in prof.items() if v[1]}
    f1, f2 = faces_per_group(g, args.scheme)
    fl = FLOP_PER_SOLVE[args.riemann]
    top = max(stages, key=lambda k: stages[k]["ms_per_step"])
    flops_stage = {"flux_pass1": fl * f1 * G, "flux_pass2": (fl + (FLOP_PLM_PER_FACE if args.scheme == "vl" else 0)) * f2 * G}
    if args.scheme == "vl":
        # S0-S2 in one kernel: the pass-1 Riemann solves + con->prim and the reference EMFs of the T^3 cells (27 + 9 flops each)
        flops_stage["pass1_fused"] = (fl * f1 + 36 * (N_PS2 + 2 * g) ** 3) * G
    roof = None
    if top in flops_stage:
        n_launch = stages[top]["launches_per_step"]
        dur = stages[top]["ms_per_step"] / n_launch * 1e-3            # average launch duration
        ach = flops_stage[top] / n_launch / dur / 1e12
        peak = NOMINAL_TFLOPS[prec_name]
        roof = {"bound": "alu", "kernel": top, "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "peak_source": "nominal: 148 SMs x %d FMA lanes x 2 x 1.965 GHz (DESIGN.md)" % (128 if prec_name == "f32" else 64),
                "peak_fma_measured": mhd.measure_fma_peak(dev.index, prec),
                "traffic": (NCU_TRAFFIC_MB[prec_name][top] * 1e6 / n_launch if (args.scheme == "vl" and args.riemann == "hlld" and G == NGROUPS
                                                                                   and top in NCU_TRAFFIC_MB[prec_name]) else None),
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum of the stage's launches of one step, "
                                "profiles/r01h_*, / launches per step)",
                "avg_launch_ms": dur * 1e3, "launches_per_step": n_launch,
                "share_of_step": stages[top]["ms_per_step"] / (prof_ms / args.steps)}
    # HBM view of the whole step: algorithmic bytes = read the ghost-zoned tile once, write the results once (the CFL
    # reduction is fused into the final update: no second read of the new state)
    sz = solver.sizes()
    bytes_step = (sz["n_U_in"] + sz["n_B_in"] + sz["n_U_out"] + sz["n_B_out"] + sz["n_flux"] + sz["n_emf"]) * esz * G
    if args.scheme == "vl" and args.riemann == "hlld" and G == NGROUPS and set(stages) == set(NCU_TRAFFIC_MB[prec_name]):
        tot = sum(NCU_TRAFFIC_MB[prec_name].values()) * 1e6
        res["dram_traffic"] = {"bytes_per_step_ncu": tot, "GBs": tot / 1e9 / (res["ms_per_step"] * 1e-3),
                               "frac_of_hbm_peak": tot / 1e9 / (res["ms_per_step"] * 1e-3) / hbm_peak()[0],
                               "note": "all stage kernels of one step; the intermediates between stages go through HBM"}
    fpc = FLOP_PER_CELL_UPDATE.get((args.scheme, args.riemann))
    if fpc:
        tf = fpc * res["value"] / world / 1e12
        res["alu_whole_step"] = {"flops_per_cell_update": fpc, "achieved_TFLOPs": tf, "frac_of_nominal_peak": tf / NOMINAL_TFLOPS[prec_name],
                                 "note": "oracle's exact operation count on its maximal index ranges (oracle/count_ops.cpp) x measured cell-updates/s"}
    res.update(stages=stages, roofline=roof, profiled_ms_per_step=prof_ms / args.steps,
               hbm={"algorithmic_GB_per_step": bytes_step / 1e9, "achieved_GBs": bytes_step / 1e9 / (res["ms_per_step"] * 1e-3),
                    "peak_GBs": hbm_peak()[0], "peak_source": hbm_peak()[1],
                    "frac": bytes_step / 1e9 / (res["ms_per_step"] * 1e-3) / hbm_peak()[0]})

    # end to end through mhd_advance_host_dt (the same step S0-S9 as the device-resident line): pinned host buffers, H2D + kernels + D2H inside the timed region
    pin = lambda a: torch.from_numpy(a).pin_memory()
    pU, pB = pin(hU), pin(hB)
    hout = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.items()}
    chunk, nstr = max(1, min(G, 32)), 4          # measured best of chunk x streams on this box: PCIe-bound (69 GB/s H2D+D2H)
    for _ in range(2):
        solver.advance_host_dt(pU, pB, hout["U"], hout["B"], hout["flux"], hout["emf"], G, dt0, dh, chunk, nstr, 0.3)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        solver.advance_host_dt(pU, pB, hout["U"], hout["B"], hout["flux"], hout["emf"], G, dt0, dh, chunk, nstr, 0.3)
    torch.cuda.synchronize()
    te = time.perf_counter() - t0
    te = shard.max_over_ranks(te, dist, dev)
    h2d = (sz["n_U_in"] + sz["n_B_in"]) * esz * G
    d2h = (sz["n_U_out"] + sz["n_B_out"] + sz["n_flux"] + sz["n_emf"]) * esz * G
    res["e2e"] = {"value": cells / te, "unit": "cell-updates/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                  "api": "mhd_advance_host_dt(chunk_groups=%d, nstreams=%d): S0-S9 through pinned host memory" % (chunk, nstr),
                  "h2d_plus_d2h_GBs": (h2d + d2h) * world / 1e9 / (te / args.steps)}
    res["stats"] = solver.get_stats()
    solver.destroy()
    return res


def measure_config5(args, scheme_name):
    """BASELINE config 5: 1024^3 cells = 262144 patch groups of the ABC state (config 3), FP32, one step, streamed as
    16^3 patch-group batches from a pinned host pool (the full set would be 91-118 GB in / 52 GB out):
    the pool = the patch groups of a 256^3 ABC grid, cycled.  With transfers: mhd_advance_host (H2D, kernels and D2H of
    successive chunks overlapped on CUDA streams), host wall clock.  Without: the same pool resident on
    the device, mhd_advance per 512-group batch, CUDA events."""
    import numpy as np
    import torch
    from paper_1804_03479_b200 import inputs, mhd
    P, total, batch = args.config5, (1024 // N_PS2) ** 3, 512
    a2 = argparse.Namespace(**{**vars(args), "scheme": scheme_name})
    sp = scheme_params(a2)
    g = sp["g"]
    riem = {"hlle": mhd.HLLE, "hlld": mhd.HLLD, "roe": mhd.ROE}[args.riemann]
    solver = mhd.Solver(mhd.make_config(N=N_PS2, g=g, scheme=sp["scheme"], recon=sp["recon"], riemann=riem, prec=mhd.FP32, max_groups=P))
    U, bx, by, bz, dh = inputs.abc_grid(256, seed=1805, p0=0.15, vamp=1e-2)
    hU, hB = inputs.pack_groups(U, bx, by, bz, N_PS2, g, np.float32)
    reps = (P + hU.shape[0] - 1) // hU.shape[0]
    hU, hB = np.tile(hU, (reps, 1))[:P].copy(), np.tile(hB, (reps, 1))[:P].copy()
    dt0 = 0.3 * dh / 6.0                                         # well below the CFL limit of the state (max speed ~ 2.5)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    pU, pB = pin(hU), pin(hB)
    out = solver.alloc_outputs(P, planes=True)
    hout = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.items()}
    passes = total // P
    chunk, nstr = 32, 4
    solver.advance_host(pU, pB, hout["U"], hout["B"], hout["flux"], hout["emf"], P, dt0, dh, chunk, nstr)
    sampler = ClockSampler(torch.cuda.current_device())
    torch.cuda.synchronize()
    sampler.start()
    t0 = time.perf_counter()
    for _ in range(passes):
        solver.advance_host(pU, pB, hout["U"], hout["B"], hout["flux"], hout["emf"], P, dt0, dh, chunk, nstr)
    torch.cuda.synchronize()
    te = time.perf_counter() - t0
    clocks = sampler.result()
    sz = solver.sizes()
    h2d = (sz["n_U_in"] + sz["n_B_in"]) * 4 * total
    d2h = (sz["n_U_out"] + sz["n_B_out"] + sz["n_flux"] + sz["n_emf"]) * 4 * total
    # device-resident pool, 512-group batches
    dU, dB = pU.cuda(), pB.cuda()
    stream = torch.cuda.current_stream()
    views = lambda t, b: t[b * batch:(b + 1) * batch]
    l0 = solver.launch_count()

    def one_pass():
        for b in range(P // batch):
            solver.advance(views(dU, b), views(dB, b), views(out["U"], b), views(out["B"], b), views(out["flux"], b), views(out["emf"], b),
                           batch, dt0, dh, stream)
    one_pass()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(passes):
        one_pass()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    cells = total * N_PS2 ** 3
    res = {"scheme": sp["name"], "with_transfers": {"value": cells / te, "unit": "cell-updates/s", "seconds": te, "h2d_bytes": h2d, "d2h_bytes": d2h,
                                                     "h2d_plus_d2h_GBs": (h2d + d2h) / 1e9 / te,
                                                     "api": "mhd_advance_host(chunk_groups=%d, nstreams=%d), pinned pool of %d groups x %d passes" % (chunk, nstr, P, passes)},
           "without_transfers": {"value": cells / (ms * 1e-3), "unit": "cell-updates/s", "seconds": ms * 1e-3,
                                 "api": "mhd_advance, %d-group batches of the device-resident pool" % batch},
           "clocks": clocks, "gpu_launches": solver.launch_count() - l0, "stats": solver.get_stats()}
    solver.destroy()
    return res


def measure_sweep(args, prec_name):
    """Cell-updates/s of mhd_advance_dt against the number of patch groups per call (the saturation curve of PAPER.md:467, Fig. 18)."""
    import numpy as np
    import torch
    from paper_1804_03479_b200 import mhd
    sp = scheme_params(args)
    g = sp["g"]
    prec = mhd.FP32 if prec_name == "f32" else mhd.FP64
    npdt = np.float32 if prec_name == "f32" else np.float64
    riem = {"hlle": mhd.HLLE, "hlld": mhd.HLLD, "roe": mhd.ROE}[args.riemann]
    stream = torch.cuda.current_stream()
    curve = []
    for G in (8, 16, 32, 64, 128, 256, 512, 1024, 2048, 4096):
        solver = mhd.Solver(mhd.make_config(N=N_PS2, g=g, scheme=sp["scheme"], recon=sp["recon"], riemann=riem, prec=prec, max_groups=G))
        hU, hB, dh = make_batch(G, g, npdt)
        dU, dB = torch.from_numpy(hU).cuda(), torch.from_numpy(hB).cuda()
        out = solver.alloc_outputs(G, planes=True)
        dt0, _ = solver.dt_reduce(dU, dB, G, g, dh, 0.3)
        steps = max(args.steps, min(400, 8192 // G))          # short calls: more repetitions
        for _ in range(args.warmup):
            solver.advance_dt(dU, dB, out["U"], out["B"], out["flux"], out["emf"], G, dt0, dh, 0.3, stream)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(steps):
            solver.advance_dt(dU, dB, out["U"], out["B"], out["flux"], out["emf"], G, dt0, dh, 0.3, stream)
        e1.record(stream)
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        curve.append({"groups": G, "cells": G * N_PS2 ** 3, "ms_per_step": ms, "value": G * N_PS2 ** 3 / (ms * 1e-3)})
        solver.destroy()
        del dU, dB, out
        torch.cuda.empty_cache()
    return curve


def measure_grid(args, prec_name):
    """Uniform periodic grid resident on the device (NEXT-1): K steps of mhd_grid_advance_dt."""
    import numpy as np
    import torch
    from paper_1804_03479_b200 import inputs, mhd
    sp = scheme_params(args)
    n, g = args.grid, sp["g"]
    prec = mhd.FP32 if prec_name == "f32" else mhd.FP64
    npdt = np.float32 if prec_name == "f32" else np.float64
    riem = {"hlle": mhd.HLLE, "hlld": mhd.HLLD, "roe": mhd.ROE}[args.riemann]
    G = (n // N_PS2) ** 3
    solver = mhd.Solver(mhd.make_config(N=N_PS2, g=g, scheme=sp["scheme"], recon=sp["recon"], riemann=riem, prec=prec, max_groups=G))
    U, bx, by, bz, dh = inputs.abc_grid(n, seed=1805, p0=0.15, vamp=1e-2)
    grid = [torch.from_numpy(np.ascontiguousarray(a, dtype=npdt)).cuda() for a in (U, bx, by, bz)]
    shape = (n, n, n)
    stream = torch.cuda.current_stream()

    dt_next = [solver.grid_dt(*grid, shape, dh, 0.3, stream)[0]]

    def step():
        # pack + S0-S8 + unpack; the final update also reduces the CFL speed of the new state (the next step's dt)
        dt_next[0], _ = solver.grid_advance_dt(*grid, shape, dt_next[0], dh, 0.3, stream)

    for _ in range(args.warmup):
        step()
    sampler = ClockSampler(torch.cuda.current_device())
    l0 = solver.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    sampler.start()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    res = dict(value=n ** 3 * args.steps / (ms * 1e-3), ms_per_step=ms / args.steps, launches=solver.launch_count() - l0,
               clocks=sampler.result(), stats=solver.get_stats(), dtype=prec_name)
    solver.destroy()
    return res


def cpu_baseline(args, groups, reps=None, target_seconds=12.0):
    """The oracle, as it stands, on the host cores: `reps` passes (default: as many as fill ~target_seconds of CPU
    work) over `groups` groups of the workload, one pass = advance + dt; value from the mean pass time."""
    import numpy as np
    from oracle import mhdref
    mhdref.build()
    sp = scheme_params(args)
    U, B, dh = make_batch(groups, sp["g"], np.float64)
    riem = {"hlle": mhdref.HLLE, "hlld": mhdref.HLLD, "roe": mhdref.ROE}[args.riemann]
    cfg = mhdref.make_config(N=N_PS2, g=sp["g"], scheme=sp["scheme"], recon=sp["recon"], riemann=riem)
    dt, _ = mhdref.dt_reduce(cfg, U, B, sp["g"], dh, 0.3)

    def one_pass():
        t0 = time.perf_counter()
        o = mhdref.advance(cfg, U, B, dt, dh)
        mhdref.dt_reduce(cfg, o["U"], o["B"], 0, dh, 0.3)
        return time.perf_counter() - t0

    first = one_pass()                                   # also the warm-up
    if reps is None:
        reps = max(1, min(200, int(round(target_seconds / max(first, 1e-3)))))
    times = [one_pass() for _ in range(reps)]
    mean = sum(times) / len(times)
    return {"value": groups * N_PS2 ** 3 / mean, "unit": "cell-updates/s", "cores": os.cpu_count(), "kind": "oracle",
            "sample": "%d of the workload's patch groups x %d passes (advance + dt each), mean pass time, FP64, OpenMP "
                      "over groups" % (groups, reps), "seconds": sum(times), "best_pass_value": groups * N_PS2 ** 3 / min(times),
            "_one_pass": one_pass}


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    sp_name = "VL+PLM" if args.scheme == "vl" else "CTU+PPM"
    g = 3 if args.scheme == "vl" else 4
    config = {"workload": "BASELINE.json configs[1]: batch of %d patch groups of 16^3 cells + %d ghost cells, %s+%s+CT, "
                          "flux_out and emf_out requested; per rank" % (args.groups, g, sp_name, args.riemann.upper()),
              "groups_per_rank": args.groups, "ps2": N_PS2, "nghost": g, "scheme": sp_name, "riemann": args.riemann,
              "step": "mhd_advance_dt: S0-S8 with the CFL reduction S9 fused into the final update", "l2": "inputs larger than L2 (no flush needed)",
              "parallelism": "independent batches per GPU (no collective)" if world > 1 else "single GPU"}

    if args.impl == "reference":
        if rank != 0:
            return 0
        # the oracle on the host cores; each step = one pass over a bounded sample of the workload
        sample = min(args.groups, 256)
        cb = cpu_baseline(args, sample, reps=max(1, args.warmup))          # builds the oracle, warms up
        one_pass = cb.pop("_one_pass")
        t0 = time.perf_counter()
        for _ in range(args.steps):
            one_pass()
        t = time.perf_counter() - t0
        val = sample * N_PS2 ** 3 * args.steps / t
        cb.update(value=val, seconds=t, sample="%d of the %d patch groups per step (advance + dt), FP64 oracle, OpenMP over "
                                                 "groups" % (sample, args.groups))
        cb.pop("best_pass_value", None)
        config = dict(config, step="the same step on the oracle: mhdref advance (S0-S8) + dt_reduce (S9) of its output")
        line = {"impl": "reference", "metric": "cell-updates/sec", "value": val, "unit": "cell-updates/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
                "cpu_baseline": cb,
                "e2e": {"value": val, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    from paper_1804_03479_b200 import build
    build.build()
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    if args.config5:
        r = [measure_config5(args, "vl"), measure_config5(args, "ctu")]
        config.update(workload="BASELINE.json configs[4]: 1024^3 cells = 262144 patch groups of 16^3 of the config-3 ABC state, FP32, one step, "
                               "streamed from a pinned pool of %d groups (the patch groups of a 256^3 ABC grid, cycled)" % args.config5,
                      step="mhd_advance_host over the whole stream (with transfers) / mhd_advance per 512-group batch (without)",
                      groups_per_rank=262144, scheme="VL+PLM and CTU+PPM")
        print(json.dumps({"metric": "cell-updates/sec", "value": r[0]["without_transfers"]["value"], "unit": "cell-updates/s", "n_gpus": 1,
                          "steps": 1, "warmup": 1, "ms_per_step": r[0]["without_transfers"]["seconds"] * 1e3, "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config,
                          "clocks": r[0]["clocks"], "gpu_launches": r[0]["gpu_launches"],
                          "e2e": {"value": r[0]["with_transfers"]["value"], "unit": "cell-updates/s", "h2d_bytes_per_step": r[0]["with_transfers"]["h2d_bytes"],
                                  "d2h_bytes_per_step": r[0]["with_transfers"]["d2h_bytes"]},
                          "vl_plm": r[0], "ctu_ppm": r[1]}))
        return 0
    if args.sweep:
        sampler = ClockSampler(torch.cuda.current_device())
        sampler.start()
        c32, c64 = measure_sweep(args, "f32"), measure_sweep(args, "f64")
        clocks = sampler.result()
        config.update(workload="BASELINE.json configs[1] state, 8 ... 4096 patch groups of 16^3 per call (the axis of the paper's Fig. 18, "
                               "PAPER.md:467), %s+%s+CT, device-resident" % (sp_name, args.riemann.upper()),
                      step="mhd_advance_dt", groups_per_rank=[c["groups"] for c in c32])
        top = max(c32, key=lambda c: c["value"])
        print(json.dumps({"metric": "cell-updates/sec", "value": top["value"], "unit": "cell-updates/s", "n_gpus": 1, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": top["ms_per_step"], "higher_is_better": True, "scaling": "weak",
                          "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config, "clocks": clocks,
                          "curve_f32": c32, "curve_f64": c64,
                          "paper_context": "P100: throughput saturates above ~2e6 cells per call (PAPER.md:467)"}))
        return 0
    if args.grid:
        a, b = measure_grid(args, args.prec), measure_grid(args, "f64" if args.prec == "f32" else "f32")
        config.update(workload="BASELINE.json config 3 state: periodic %d^3 ABC grid (beta 0.1) resident on the device, cut "
                               "into %d patch groups of 16^3 every step, %s+%s+CT" % (args.grid, (args.grid // N_PS2) ** 3, sp_name, args.riemann.upper()),
                      step="mhd_grid_advance_dt (device-side pack, S0-S8 with the CFL reduction S9 fused into the final update, unpack)", groups_per_rank=(args.grid // N_PS2) ** 3)
        print(json.dumps({"metric": "cell-updates/sec", "value": a["value"], "unit": "cell-updates/s", "n_gpus": 1,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": a["ms_per_step"], "higher_is_better": True,
                          "scaling": "weak", "vs_baseline": None, "dtype": a["dtype"], "data": "synthetic", "config": config,
                          "clocks": a["clocks"], "gpu_launches": a["launches"], "stats": a["stats"],
                          ("fp64" if b["dtype"] == "f64" else "fp32"): b}))
        return 0
    main_prec = args.prec
    other = "f64" if main_prec == "f32" else "f32"
    r_main = measure(args, main_prec, rank, world, dist)
    r_other = measure(args, other, rank, world, dist)
    if rank == 0:
        cb = None
        if not args.no_cpu_baseline and world == 1:
            cb = cpu_baseline(args, args.groups)
            cb.pop("_one_pass")

        def sub(r, prec):
            return {"value": r["value"], "unit": "cell-updates/s", "ms_per_step": r["ms_per_step"], "dtype": prec,
                    "roofline": r["roofline"], "hbm": r["hbm"], "stages_ms_per_step": {k: round(v["ms_per_step"], 4) for k, v in r["stages"].items()},
                    "profiled_ms_per_step": r["profiled_ms_per_step"], "e2e": r["e2e"], "clocks": r["clocks"],
                    "stats": r["stats"], "paper_p100_context": PAPER_P100[prec]}

        line = {"metric": "cell-updates/sec", "value": r_main["value"], "unit": "cell-updates/s", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": r_main["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": main_prec, "data": "synthetic", "config": config,
                "clocks": r_main["clocks"], "e2e": r_main["e2e"], "gpu_launches": r_main["launches"],
                "roofline": r_main["roofline"], "cpu_baseline": cb, "dram_traffic": r_main.get("dram_traffic"), "alu_whole_step": r_main.get("alu_whole_step"),
                "hbm": r_main["hbm"], "stages_ms_per_step": {k: round(v["ms_per_step"], 4) for k, v in r_main["stages"].items()},
                "profiled_ms_per_step": r_main["profiled_ms_per_step"],
                "paper_p100_context": {"value": PAPER_P100[main_prec], "note": "Tesla P100, VL+PLM+Roe, PAPER.md:12,:465 -- context, not a target"},
                {"f32": "fp32", "f64": "fp64"}[other]: sub(r_other, other)}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
