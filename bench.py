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
# Algorithmic work: exact operation counts of the oracle instantiated with a counting scalar
# (oracle/count_ops.cpp; add / sub / mul / div / sqrt = 1 each), pinned to that tool's output by tests/test_op_counts.py.
FLOP_PER_SOLVE = {"hlld": 381, "roe": 1107, "hlle": 361}
# whole step per interior cell-update: "max" = on the oracle's maximal index ranges, "min" = every stage only where the final update
# needs it (mhdref_config.minimal_ranges; the device's ranges): the work the method itself requires
FLOP_PER_CELL_UPDATE = {("vl", "hlld"): {"max": 6127.4, "min": 5586.4}, ("vl", "roe"): {"max": 15153.0, "min": 13924.0},
                        ("ctu", "hlld"): {"max": 25945.8, "min": 18657.6}, ("ctu", "roe"): {"max": 35038.5, "min": 25627.7}}
# flops per patch group of the seven steps of the update on the minimal ranges: con->prim, pass-1 fluxes (CTU: + reconstruction),
# EMF-1, half step, pass-2 states + fluxes, EMF-2, full update
FLOP_PER_GROUP_STEPS = {("vl", "hlld"): [276848, 11617452, 1230060, 654004, 8236384, 638118, 229122],
                        ("vl", "roe"): [276848, 33754644, 1230060, 654004, 20249952, 638118, 229122],
                        ("ctu", "hlld"): [359426, 64502472, 896730, 477254, 9318565, 638118, 229122],
                        ("ctu", "roe"): [359426, 81055272, 896730, 477254, 21314989, 638118, 229122]}
# which steps each profiled stage (mhd_set_profiling) covers; stages that share a step are timed together
STAGE_STEPS = {"march_pass1": (1, 2, 3, 4), "march_pass2": (5, 6, 7), "emf_pass1": (3,), "half_step": (4,), "flux_pass2": (5,), "emf_pass2": (6,),
               "final_update": (7,)}
NOMINAL_TFLOPS = {"f32": 148 * 128 * 2 * 1.965e9 / 1e12, "f64": 148 * 64 * 2 * 1.965e9 / 1e12}
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")
# host path: groups per chunk and streams, the measured best of 16 ... 256 x 2 ... 8 on this box (PCIe-bound; CTU's longer kernels want
# the shorter pipeline fill of smaller chunks)
E2E_CHUNK, E2E_STREAMS = {"vl": 64, "ctu": 32}, 4


def ncu_traffic():
    """profiles/r02_dram_traffic.csv (written from ncu --set full captures, command in profiles/r02_dram_traffic.md):
    {(scheme, riemann, prec): {stage: (launches per 512-group step, MB read + written per launch)}}; {} if the file is missing"""
    out = {}
    try:
        import csv
        for r in csv.DictReader(open(TRAFFIC_CSV)):
            key = (r["scheme"], r["riemann"], r["prec"])
            out.setdefault(key, {})[r["stage"]] = (float(r["launches_per_step"]), float(r["dram_read_MB"]) + float(r["dram_write_MB"]))
    except Exception:
        pass
    return out


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
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--main-only", action="store_true", help="only the headline arm and its other precision (no ctu / roe / config5 sub-records)")
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


_BATCH_CACHE = {}


def make_batch(G, g, npdt):
    """config-2 batch (BASELINE.json configs[1]): G DISTINCT seeded patch groups (seed 3479 + group id): the branch pattern of
    the Riemann solver, the floors and the upwind ramp depend on the values"""
    import numpy as np
    from paper_1804_03479_b200 import inputs
    key = (G, g)
    if key not in _BATCH_CACHE:
        _BATCH_CACHE[key] = inputs.config2_batch(G, N=N_PS2, g=g, dtype=np.float64)
    U, B, dh = _BATCH_CACHE[key]
    return U.astype(npdt), B.astype(npdt), dh


def pcie_peaks(dev, nbytes=256 << 20):
    """pinned host <-> device copy bandwidth of this box, measured in the same run: H2D alone, D2H alone, both at once (GB/s)"""
    import torch
    h1, h2 = torch.empty(nbytes, dtype=torch.uint8).pin_memory(), torch.empty(nbytes, dtype=torch.uint8).pin_memory()
    d1, d2 = torch.empty(nbytes, dtype=torch.uint8, device=dev), torch.empty(nbytes, dtype=torch.uint8, device=dev)
    s1, s2 = torch.cuda.Stream(dev), torch.cuda.Stream(dev)

    def run(h2d, d2h, reps=4):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(reps):
            if h2d:
                with torch.cuda.stream(s1):
                    d1.copy_(h1, non_blocking=True)
            if d2h:
                with torch.cuda.stream(s2):
                    h2.copy_(d2, non_blocking=True)
        torch.cuda.synchronize()
        return (int(h2d) + int(d2h)) * nbytes * reps / (time.perf_counter() - t0) / 1e9
    run(True, True, 1)
    return {"h2d_GBs": run(True, False), "d2h_GBs": run(False, True), "bidirectional_GBs": run(True, True)}


def merge_stages(stages):
    """profiled stages -> roofline units: the stages that share steps 1-2 of the update (tile staging / con->prim, reconstruction,
    pass-1 Riemann solves) are timed together; returns {unit: {ms_per_step, launches_per_step, steps}}"""
    out = {k: dict(v, steps=STAGE_STEPS.get(k)) for k, v in stages.items()}
    parts = [k for k in ("load_prim", "recon_ctu", "flux_pass1", "pass1_fused") if k in out]
    if parts:
        ms = sum(out[k]["ms_per_step"] for k in parts)
        nl = max(out[k]["launches_per_step"] for k in parts)
        for k in parts:
            del out[k]
        out["+".join(parts)] = {"ms_per_step": ms, "launches_per_step": nl, "steps": (1, 2)}
    return out


def measure(args, prec_name, rank, world, dist, scheme=None, riemann=None, steps=None, e2e=True, pcie=None):
    """Time K steps of mhd_advance_dt on device-resident data, then the per-stage profile, then e2e."""
    import numpy as np
    import torch
    from paper_1804_03479_b200 import mhd, shard
    a2 = argparse.Namespace(**{**vars(args), "scheme": scheme or args.scheme, "riemann": riemann or args.riemann})
    sp = scheme_params(a2)
    steps = steps or args.steps
    g, G = sp["g"], args.groups
    prec = mhd.FP32 if prec_name == "f32" else mhd.FP64
    npdt = np.float32 if prec_name == "f32" else np.float64
    esz = 4 if prec_name == "f32" else 8
    riem = {"hlle": mhd.HLLE, "hlld": mhd.HLLD, "roe": mhd.ROE}[a2.riemann]
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
    for _ in range(steps):
        step()
    e1.record(stream)
    barrier()
    clocks = sampler.result()
    ms = e0.elapsed_time(e1)
    launches = solver.launch_count() - l0
    ms = shard.max_over_ranks(ms, dist, dev)          # job time = slowest rank's device time
    cells = G * N_PS2 ** 3 * steps * world
    res = dict(value=cells / (ms * 1e-3), ms_per_step=ms / steps, launches=launches, clocks=clocks, steps=steps,
               variant="%s+%s" % (sp["name"], a2.riemann.upper()))

    # per-stage device time over K more steps (events around every stage launch on the launching stream; the slices of a
    # step then run one after the other, so the stage times add up to a little more than the overlapped step)
    solver.set_profiling(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    p0.record(stream)
    for _ in range(steps):
        step()
    p1.record(stream)
    torch.cuda.synchronize()
    prof = solver.get_profile()
    solver.set_profiling(False)
    prof_ms = p0.elapsed_time(p1)
    stages = {k: {"ms_per_step": v[0] / steps, "launches_per_step": v[1] / steps} for k, v in prof.items() if v[1]}
    key = (a2.scheme, a2.riemann)
    units = merge_stages(stages)
    roof = None
    step_flops = FLOP_PER_GROUP_STEPS.get(key)
    traffic = ncu_traffic().get((a2.scheme, a2.riemann, prec_name), {}) if G == NGROUPS else {}
    if step_flops:
        top = max(units, key=lambda k: units[k]["ms_per_step"])
        if units[top]["steps"]:
            n_launch = units[top]["launches_per_step"]
            dur = units[top]["ms_per_step"] / n_launch * 1e-3            # average launch duration
            fl = sum(step_flops[i - 1] for i in units[top]["steps"]) * G   # algorithmic flops of the steps this kernel covers, per step
            ach = fl / n_launch / dur / 1e12
            peak = NOMINAL_TFLOPS[prec_name]
            trs = [traffic[k] for k in top.split("+") if k in traffic]
            tr = (n_launch, sum(a * b for a, b in trs) / n_launch) if len(trs) == len(top.split("+")) else None
            roof = {"bound": "alu", "kernel": top, "steps_covered": list(units[top]["steps"]), "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                    "frac": ach / peak, "flops_per_launch": fl / n_launch,
                    "peak_source": "nominal: 148 SMs x %d FMA lanes x 2 x 1.965 GHz (DESIGN.md)" % (128 if prec_name == "f32" else 64),
                    "peak_fma_measured": mhd.measure_fma_peak(dev.index, prec),
                    "traffic": (tr[1] * 1e6 if tr else None),
                    "traffic_unit": "bytes per launch: ncu dram__bytes_read.sum + dram__bytes_write.sum, read at run time from "
                                    "profiles/r02_dram_traffic.csv (a %d-group launch)" % int(round(G / max(n_launch, 1))),
                    "avg_launch_ms": dur * 1e3, "launches_per_step": n_launch,
                    "share_of_step": units[top]["ms_per_step"] / (prof_ms / steps),
                    # the same arithmetic for every kernel of the step (the dominant one is the headline of this object)
                    "all_kernels": {k: {"steps_covered": list(u["steps"]), "ms_per_step": u["ms_per_step"],
                                        "achieved": sum(step_flops[i - 1] for i in u["steps"]) * G / (u["ms_per_step"] * 1e-3) / 1e12,
                                        "frac": sum(step_flops[i - 1] for i in u["steps"]) * G / (u["ms_per_step"] * 1e-3) / 1e12 / peak}
                                    for k, u in units.items() if u["steps"]}}
    # HBM view of the whole step: algorithmic bytes = read the ghost-zoned tile once, write the results once (the CFL
    # reduction is fused into the final update: no second read of the new state)
    sz = solver.sizes()
    bytes_step = (sz["n_U_in"] + sz["n_B_in"] + sz["n_U_out"] + sz["n_B_out"] + sz["n_flux"] + sz["n_emf"]) * esz * G
    if traffic and all(k in traffic for k in stages):
        tot = sum(traffic[k][0] * traffic[k][1] for k in stages) * 1e6
        res["dram_traffic"] = {"bytes_per_step_ncu": tot, "over_algorithmic": tot / bytes_step, "GBs": tot / 1e9 / (res["ms_per_step"] * 1e-3),
                               "frac_of_hbm_peak": tot / 1e9 / (res["ms_per_step"] * 1e-3) / hbm_peak()[0],
                               "source": "profiles/r02_dram_traffic.csv, all stage kernels of one 512-group step"}
    fpc = FLOP_PER_CELL_UPDATE.get(key)
    if fpc:
        tf = {k: v * res["value"] / world / 1e12 for k, v in fpc.items()}
        res["alu_whole_step"] = {"flops_per_cell_update_minimal_ranges": fpc["min"], "flops_per_cell_update_oracle_ranges": fpc["max"],
                                 "achieved_TFLOPs": tf["min"], "frac_of_nominal_peak": tf["min"] / NOMINAL_TFLOPS[prec_name],
                                 "achieved_TFLOPs_oracle_ranges": tf["max"],
                                 "note": "exact operation count of the oracle (oracle/count_ops.cpp) on the minimal index ranges (the work the "
                                         "method requires = the device's ranges) x measured cell-updates/s; the maximal-range count beside it"}
    res.update(stages=stages, roofline=roof, profiled_ms_per_step=prof_ms / steps,
               hbm={"algorithmic_GB_per_step": bytes_step / 1e9, "achieved_GBs": bytes_step / 1e9 / (res["ms_per_step"] * 1e-3),
                    "peak_GBs": hbm_peak()[0], "peak_source": hbm_peak()[1],
                    "frac": bytes_step / 1e9 / (res["ms_per_step"] * 1e-3) / hbm_peak()[0]})
    if e2e and not args.no_e2e:
        # end to end through mhd_advance_host_dt (the same step S0-S9 as the device-resident line): pinned host buffers, H2D +
        # kernels + D2H inside the timed region
        pin = lambda a: torch.from_numpy(a).pin_memory()
        pU, pB = pin(hU), pin(hB)
        hout = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.items()}
        chunk, nstr = max(1, min(G, E2E_CHUNK[a2.scheme])), E2E_STREAMS
        ksteps = max(3, steps // 4)
        for _ in range(2):
            solver.advance_host_dt(pU, pB, hout["U"], hout["B"], hout["flux"], hout["emf"], G, dt0, dh, chunk, nstr, 0.3)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ksteps):
            solver.advance_host_dt(pU, pB, hout["U"], hout["B"], hout["flux"], hout["emf"], G, dt0, dh, chunk, nstr, 0.3)
        torch.cuda.synchronize()
        te = time.perf_counter() - t0
        te = shard.max_over_ranks(te, dist, dev)
        h2d = (sz["n_U_in"] + sz["n_B_in"]) * esz * G
        d2h = (sz["n_U_out"] + sz["n_B_out"] + sz["n_flux"] + sz["n_emf"]) * esz * G
        gbs = (h2d + d2h) / 1e9 / (te / ksteps)
        res["e2e"] = {"value": G * N_PS2 ** 3 * ksteps * world / te, "unit": "cell-updates/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                      "steps": ksteps, "api": "mhd_advance_host_dt(chunk_groups=%d, nstreams=%d): S0-S9 through pinned host memory" % (chunk, nstr),
                      "h2d_plus_d2h_GBs": gbs}
        if pcie:
            # the copies of a step at the measured one-direction rates, overlapped perfectly: the PCIe-bound time of the step
            t_pcie = max(h2d / pcie["h2d_GBs"], d2h / pcie["d2h_GBs"], (h2d + d2h) / pcie["bidirectional_GBs"]) / 1e9
            res["e2e"].update(pcie_peak_GBs=pcie, pcie_bound_value=G * N_PS2 ** 3 / t_pcie, frac=(te / ksteps and t_pcie / (te / ksteps)))
    res["stats"] = solver.get_stats()
    solver.destroy()
    return res


def measure_config5(args, scheme_name, pool=None):
    """BASELINE config 5: 1024^3 cells = 262144 patch groups of the ABC state (config 3), FP32, one step, streamed as
    16^3 patch-group batches from a pinned host pool (the full set would be 91-118 GB in / 52 GB out):
    the pool = the first POOL patch groups of the 1024^3 grid itself (inputs.abc_groups, dh = 1/1024), cycled.  With transfers: mhd_advance_host (H2D, kernels and D2H of
    successive chunks overlapped on CUDA streams), host wall clock.  Without: the same pool resident on
    the device, mhd_advance per 512-group batch, CUDA events."""
    import numpy as np
    import torch
    from paper_1804_03479_b200 import inputs, mhd
    P, total, batch = pool or args.config5, (1024 // N_PS2) ** 3, 512
    a2 = argparse.Namespace(**{**vars(args), "scheme": scheme_name})
    sp = scheme_params(a2)
    g = sp["g"]
    riem = {"hlle": mhd.HLLE, "hlld": mhd.HLLD, "roe": mhd.ROE}[args.riemann]
    solver = mhd.Solver(mhd.make_config(N=N_PS2, g=g, scheme=sp["scheme"], recon=sp["recon"], riemann=riem, prec=mhd.FP32, max_groups=P))
    # the first P patch groups of the 1024^3 grid (dh = 1/1024), generated group by group
    hU, hB, dh = inputs.abc_groups(1024, 0, P, N_PS2, g, dtype=np.float32)
    dt0 = 0.3 * dh / 6.0                                         # well below the CFL limit of the state (max speed ~ 2.5)
    pin = lambda a: torch.from_numpy(a).pin_memory()
    pU, pB = pin(hU), pin(hB)
    out = solver.alloc_outputs(P, planes=True)
    hout = {k: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k, v in out.items()}
    passes = total // P
    chunk, nstr = E2E_CHUNK[scheme_name], E2E_STREAMS
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


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def cpu_baseline(args, groups, reps=None, target_seconds=12.0):
    """The oracle, as it stands, on the host cores: `reps` passes (default: as many as fill ~target_seconds of CPU
    work) over `groups` groups of the workload, one pass = advance + dt; value from the mean pass time.  Beside it the
    same on ONE thread (a bounded sample of 8 groups, best of 3), SURVEY 8(d)."""
    import numpy as np
    from oracle import mhdref
    mhdref.build()
    sp = scheme_params(args)
    U, B, dh = make_batch(groups, sp["g"], np.float64)
    riem = {"hlle": mhdref.HLLE, "hlld": mhdref.HLLD, "roe": mhdref.ROE}[args.riemann]
    cfg = mhdref.make_config(N=N_PS2, g=sp["g"], scheme=sp["scheme"], recon=sp["recon"], riemann=riem)
    dt, _ = mhdref.dt_reduce(cfg, U, B, sp["g"], dh, 0.3)

    def one_pass(Ux=U, Bx=B):
        t0 = time.perf_counter()
        o = mhdref.advance(cfg, Ux, Bx, dt, dh)
        mhdref.dt_reduce(cfg, o["U"], o["B"], 0, dh, 0.3)
        return time.perf_counter() - t0

    first = one_pass()                                   # also the warm-up
    if reps is None:
        reps = max(1, min(200, int(round(target_seconds / max(first, 1e-3)))))
    times = [one_pass() for _ in range(reps)]
    mean = sum(times) / len(times)
    # one thread: the OpenMP loop over groups with a single group per call has nothing to share out
    n1 = min(groups, 8)
    t1 = min(sum(one_pass(U[q:q + 1], B[q:q + 1]) for q in range(n1)) for _ in range(3))
    return {"value": groups * N_PS2 ** 3 / mean, "unit": "cell-updates/s", "cores": os.cpu_count(), "kind": "oracle",
            "sample": "%d of the workload's patch groups x %d passes (advance + dt each), mean pass time, FP64, OpenMP "
                      "over groups" % (groups, reps), "seconds": sum(times), "best_pass_value": groups * N_PS2 ** 3 / min(times),
            "one_thread": {"value": n1 * N_PS2 ** 3 / t1, "unit": "cell-updates/s", "sample": "%d groups, one group per call (one thread), best of 3" % n1},
            "cpu_model": cpu_model(), "_one_pass": one_pass}


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    sp_name = "VL+PLM" if args.scheme == "vl" else "CTU+PPM"
    g = 3 if args.scheme == "vl" else 4
    config = {"workload": "BASELINE.json configs[1]: batch of %d DISTINCT seeded patch groups (seed 3479 + group id) of 16^3 cells + %d ghost "
                          "cells, %s+%s+CT, flux_out and emf_out requested; per rank" % (args.groups, g, sp_name, args.riemann.upper()),
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
        # config is the same object as in our arm (the driver compares them); what the oracle runs for that step is said beside it
        line = {"impl": "reference", "metric": "cell-updates/sec", "value": val, "unit": "cell-updates/s", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
                "cpu_baseline": cb, "reference_step": "the same step on the oracle: mhdref advance (S0-S8) + dt_reduce (S9) of its output",
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
                               "streamed from a pinned pool of %d groups (the first groups of the 1024^3 grid, dh = 1/1024, cycled)" % args.config5,
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
    pcie = pcie_peaks(torch.device("cuda", local))
    r_main = measure(args, main_prec, rank, world, dist, pcie=pcie)
    r_other = measure(args, other, rank, world, dist, pcie=pcie)
    extra = {}
    if not args.main_only and world == 1:
        # the other variants the paper names, in the driver's line (fewer steps each: they are sub-records, not the headline)
        k2 = max(10, args.steps // 4)
        if (args.scheme, args.riemann) != ("ctu", "hlld"):      # CTU+PPM+HLLD: BASELINE configs 3-5
            extra["ctu_ppm_hlld"] = {pr: measure(args, pr, rank, world, dist, scheme="ctu", riemann="hlld", steps=k2, e2e=(pr == "f32"), pcie=pcie) for pr in ("f32", "f64")}
        if (args.scheme, args.riemann) != ("vl", "roe"):        # VL+PLM+Roe: the combination of the paper's Fig. 18
            extra["vl_plm_roe"] = {pr: measure(args, pr, rank, world, dist, scheme="vl", riemann="roe", steps=k2, e2e=False) for pr in ("f32", "f64")}
        # BASELINE configs[4]: 1024^3 cells streamed as 16^3 patch-group batches, with and without transfers
        extra["config5"] = {"workload": "BASELINE.json configs[4]: 262144 group-updates (= 1024^3 cells) of the 1024^3 ABC state, FP32, streamed from a "
                                        "pinned pool of 1024 groups (the first groups of that grid, dh = 1/1024), HLLD",
                            "vl_plm": measure_config5(args, "vl", pool=1024), "ctu_ppm": measure_config5(args, "ctu", pool=1024)}
    if rank == 0:
        cb = None
        if not args.no_cpu_baseline and world == 1:
            cb = cpu_baseline(args, args.groups)
            cb.pop("_one_pass")

        def sub(r, prec):
            d = {"variant": r["variant"], "value": r["value"], "unit": "cell-updates/s", "ms_per_step": r["ms_per_step"], "steps": r["steps"], "dtype": prec,
                 "roofline": r["roofline"], "alu_whole_step": r.get("alu_whole_step"), "dram_traffic": r.get("dram_traffic"), "hbm": r["hbm"],
                 "stages_ms_per_step": {k: round(v["ms_per_step"], 4) for k, v in r["stages"].items()},
                 "profiled_ms_per_step": r["profiled_ms_per_step"], "gpu_launches": r["launches"], "clocks": r["clocks"],
                 "stats": r["stats"], "paper_p100_context": PAPER_P100[prec]}
            if "e2e" in r:
                d["e2e"] = r["e2e"]
            return d

        line = {"metric": "cell-updates/sec", "value": r_main["value"], "unit": "cell-updates/s", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": r_main["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": main_prec, "data": "synthetic", "config": config,
                "clocks": r_main["clocks"], "e2e": r_main.get("e2e"), "gpu_launches": r_main["launches"],
                "roofline": r_main["roofline"], "cpu_baseline": cb, "dram_traffic": r_main.get("dram_traffic"), "alu_whole_step": r_main.get("alu_whole_step"),
                "hbm": r_main["hbm"], "stages_ms_per_step": {k: round(v["ms_per_step"], 4) for k, v in r_main["stages"].items()},
                "profiled_ms_per_step": r_main["profiled_ms_per_step"],
                "paper_p100_context": {"value": PAPER_P100[main_prec], "note": "Tesla P100, VL+PLM+Roe, PAPER.md:12,:465 -- context, not a target"},
                {"f32": "fp32", "f64": "fp64"}[other]: sub(r_other, other)}
        for name, recs in extra.items():
            line[name] = recs if name == "config5" else {pr: sub(r, pr) for pr, r in recs.items()}
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
