"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star; R14): per field max|gpu-oracle|/max|oracle|
<= 1e-11 in FP64 and <= 1e-4 in FP32 after 10 steps; the FP32 path is compared with the FP64 oracle started from
the FP32-rounded inputs and fed the oracle's dt sequence."""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import gpu_util as GU
import parity_cases as PC

pytestmark = pytest.mark.gpu

TOL = {1: 1e-11, 0: 1e-4}
TOL_ONE_STEP = {1: 2e-13, 0: 1e-4}
SCHEMES = [("vl_plm", 0, 0, 3), ("ctu_plm", 1, 0, 3), ("ctu_ppm", 1, 1, 4)]


EMF_TIE = PC.EMF_TIE   # DESIGN.md R10a: the tie width is part of the method and follows the working precision


def oracle_fn(oracle, N, g, scheme, recon, riemann, limvar, prec=1):
    cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann, limvar=limvar, emf_tie=EMF_TIE[prec])
    return cfg, (lambda Ui, Bi, dt, dh: oracle.advance(cfg, Ui, Bi, dt, dh))


def assert_fields(errs, tol, what):
    bad = {k: v for k, v in errs.items() if not (v <= tol)}
    assert not bad, f"{what}: fields over tolerance {tol:g}: {bad}; all: {errs}"


# ---------------------------------------------------------------------------------------------------------------
# one step, every scheme x Riemann solver x limiter variable x precision, config-2 type groups, planes included
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,scheme,recon,g", SCHEMES)
@pytest.mark.parametrize("riemann", [0, 1, 2])
@pytest.mark.parametrize("limvar", [0, 1])
@pytest.mark.parametrize("prec", [1, 0])
def test_one_step_every_variant(oracle, name, scheme, recon, g, riemann, limvar, prec):
    N, G = 16, 5
    dtp = GU.np_dtype(prec)
    U_in, B_in, dh = inputs.config2_batch(G, N=N, g=g, dtype=dtp)
    U64, B64 = U_in.astype(np.float64), B_in.astype(np.float64)
    cfg, adv = oracle_fn(oracle, N, g, scheme, recon, riemann, limvar, prec)
    dt, _ = oracle.dt_reduce(cfg, U64, B64, g, dh, 0.3)
    ref = adv(U64, B64, dt, dh)
    gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann, limvar=limvar, prec=prec, max_groups=G)
    out = gpu(U_in, B_in, dt, dh)
    assert_fields(GU.field_errors(out, ref, N), TOL_ONE_STEP[prec], f"{name} riemann={riemann} limvar={limvar}")
    if prec == 1:
        # the kernels evaluate pass 2 only where the final update needs it, the oracle on its maximal index ranges:
        # every floor / fallback event of the device is one of the oracle's
        assert all(a <= b for a, b in zip(gpu.stats(), ref["stats"]))


# ---------------------------------------------------------------------------------------------------------------
# config 1: 32^3 periodic ABC grid, VL+PLM+CT, FP64, 10 steps at CFL 0.3 (8 groups of 16^3, g = 3)
# ---------------------------------------------------------------------------------------------------------------
def run_grid(adv, U, bx, by, bz, dts, dh, N, g, dtype=np.float64):
    out = None
    for dt in dts:
        U, bx, by, bz, out, mism = H.step_grid(adv, U, bx, by, bz, dt, dh, N, g, dtype)
        assert mism == 0.0, "faces shared by two groups must be bitwise equal"
    return U, bx, by, bz, out


def oracle_dt_sequence(oracle, adv, U, bx, by, bz, dh, N, g, nsteps, cfl=0.3):
    """advance the oracle nsteps with its own CFL dt; returns (dts, final state, last output)."""
    n = U.shape[-1]
    c0 = oracle.make_config(N=n, g=3)
    dts, out = [], None
    for _ in range(nsteps):
        Ui, Bi = inputs.pack_groups(U, bx, by, bz, n, 0)
        dt, _ = oracle.dt_reduce(c0, Ui, Bi, 0, dh, cfl)
        dts.append(dt)
        U, bx, by, bz, out, _ = H.step_grid(adv, U, bx, by, bz, dt, dh, N, g)
    return dts, (U, bx, by, bz), out


def grid_errors(a, b):
    names = ["rho", "Mx", "My", "Mz", "e"]
    errs = {nm: H.field_err(a[0][v], b[0][v]) for v, nm in enumerate(names)}
    errs.update(Bx=H.field_err(a[1], b[1]), By=H.field_err(a[2], b[2]), Bz=H.field_err(a[3], b[3]))
    return errs


def test_config1_abc32_vl_plm_fp64_10_steps(oracle):
    n, N, g = 32, 16, 3
    U, bx, by, bz, dh = inputs.abc_grid(n, seed=1804, p0=1.0, vamp=1e-3)
    cfg, adv = oracle_fn(oracle, N, g, 0, 0, 1, 0)
    dts, ref, ref_out = oracle_dt_sequence(oracle, adv, U, bx, by, bz, dh, N, g, 10)
    gpu = GU.GpuRunner(N=N, g=g, scheme=0, recon=0, riemann=1, prec=1, max_groups=8)
    res = run_grid(gpu, U, bx, by, bz, dts, dh, N, g)
    assert_fields(grid_errors(res, ref), TOL[1], "config 1 state")
    assert_fields(GU.field_errors(res[4], ref_out, N), TOL[1], "config 1 planes of step 10")
    assert H.rel_divb(res[1], res[2], res[3], dh) < 1e-13
    t0, t1 = H.totals(U), H.totals(res[0])
    assert abs(t1[0] - t0[0]) / t0[0] < 1e-13 and abs(t1[4] - t0[4]) / t0[4] < 1e-13


# ---------------------------------------------------------------------------------------------------------------
# config 2: batch of independent 16^3 boxes (each its own periodic domain), VL+PLM+CT, FP64 and FP32, 10 steps
# ---------------------------------------------------------------------------------------------------------------
def _fp32_reference(oracle, cfg):
    """the oracle instantiated in single precision (oracle/mhd_oracle_f32.cpp): its distance from the FP64 oracle is the
    error inherent to the plain algorithm in IEEE single precision and sets the FP32 gate (R14b)"""
    return lambda Ui, Bi, dt, dh: oracle.advance32(cfg, Ui, Bi, dt, dh)


@pytest.mark.parametrize("prec", [1, 0])
def test_config2_batch_vl_plm_10_steps(oracle, prec):
    N, g, G = 16, 3, 24
    dtp = GU.np_dtype(prec)
    boxes0, dh = PC.config2_boxes(G, N, prec)
    cfg, adv = oracle_fn(oracle, N, g, 0, 0, 1, 0, prec)
    dts, ref_boxes, ref_out, _ = PC.run_boxes_oracle(oracle, cfg, boxes0, dh, N, g)
    gpu = GU.GpuRunner(N=N, g=g, scheme=0, recon=0, riemann=1, prec=prec, max_groups=G)
    gpu_boxes, gpu_out = PC.run_boxes(gpu, boxes0, dts, dh, N, g, dtp)
    errs = PC.boxes_errors(gpu_boxes, ref_boxes)
    errs.update({k: v for k, v in GU.field_errors(gpu_out, ref_out, N).items() if k.startswith(("flux", "emf"))})
    if prec == 1:
        assert_fields(errs, TOL[1], "config 2 FP64, state and planes of step 10")
    else:
        # every field of every group -- also the planes of the groups whose pressure floor fires (floors fire in 7 of the
        # 24 groups from step 6 on) -- at the north-star 1e-4, or 2 x the FP32 oracle's own error where that is larger
        # (it is not on this config: measured <= 3.3e-5, profiles/r02_fp32_controls.md)
        b32, o32 = PC.run_boxes(_fp32_reference(oracle, cfg), boxes0, dts, dh, N, g, np.float32)
        e32 = PC.boxes_errors(b32, ref_boxes)
        e32.update({k: v for k, v in GU.field_errors(o32, ref_out, N).items() if k.startswith(("flux", "emf"))})
        gate = PC.fp32_gate(e32)
        assert max(gate.values()) <= 1e-4 + 1e-12, gate       # the inherent FP32 error itself stays below 5e-5 here
        bad = {k: (v, gate[k]) for k, v in errs.items() if not v <= gate[k]}
        assert not bad, f"config 2 FP32 over the gate (R14b): {bad}; all {errs}; oracle-FP32 {e32}"
        assert ref_out["stats"][1] > 0                       # the floors did fire: that path is inside the gate
    for q in range(G):
        bx, by, bz = (np.asarray(a, dtype=np.float64) for a in gpu_boxes[q][1:])
        assert H.rel_divb(bx, by, bz, dh) < (1e-13 if prec == 1 else 2e-5)


# ---------------------------------------------------------------------------------------------------------------
# configs 3 and 4 at oracle-sized grids (64^3 -> 64 groups, g = 4): CTU+PPM+CT, 10 steps
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [1, 0])
def test_config3_abc_ctu_ppm_10_steps(oracle, prec):
    n, N, g = 64, 16, 4
    dtp = GU.np_dtype(prec)
    state0, dh = PC.config3_grid(n, prec)
    cfg, adv = oracle_fn(oracle, N, g, 1, 1, 1, 1, prec)
    dts, ref, ref_out = PC.run_grid_oracle(oracle, adv, state0, dh, N, g)
    gpu = GU.GpuRunner(N=N, g=g, scheme=1, recon=1, riemann=1, limvar=1, prec=prec, max_groups=64)
    res, gpu_out = PC.run_grid(gpu, state0, dts, dh, N, g, dtype=dtp)
    errs = PC.grid_errors(res, ref)
    errs.update({k: v for k, v in GU.field_errors(gpu_out, ref_out, N).items() if k.startswith(("flux", "emf"))})
    if prec == 1:
        assert_fields(errs, TOL[1], "config 3 FP64")
    else:
        # R14b: |M| <= 1.2e-2 here while the momentum flux is O(pT) = 3.2, so the plain algorithm in
        # IEEE single precision (the FP32 oracle) is itself 2.4e-4 .. 8.8e-4 of max|M| away from the FP64 oracle after 10
        # steps, and 2.6e-4 / 1.9e-4 / 5.5e-4 in the mass flux, energy flux and EMF planes.  Gate per field:
        # max(1e-4, 2 x that); measured GPU / gate <= 0.4 (profiles/r02_fp32_controls.md).  rho, e, B, momentum fluxes: 1e-4.
        s32, o32 = PC.run_grid(_fp32_reference(oracle, cfg), state0, dts, dh, N, g, dtype=np.float32)
        e32 = PC.grid_errors(s32, ref)
        e32.update({k: v for k, v in GU.field_errors(o32, ref_out, N).items() if k.startswith(("flux", "emf"))})
        gate = PC.fp32_gate(e32)
        for k in ("rho", "e", "Bx", "By", "Bz", "flux_Mx", "flux_My", "flux_Mz"):
            assert gate[k] == 1e-4, (k, gate[k])
        bad = {k: (v, gate[k]) for k, v in errs.items() if not v <= gate[k]}
        assert not bad, f"config 3 FP32 over the gate (R14b): {bad}; all {errs}; oracle-FP32 {e32}"
    assert H.rel_divb(*(np.asarray(a, dtype=np.float64) for a in res[1:4]), dh) < (1e-13 if prec == 1 else 2e-5)
    assert gpu.stats() == (0, 0, 0)


def test_config4_blast_ctu_ppm_fp64_10_steps(oracle):
    n, N, g = 64, 16, 4
    U, bx, by, bz, dh = inputs.blast_grid(n)
    cfg, adv = oracle_fn(oracle, N, g, 1, 1, 1, 1)
    dts, ref, ref_out = oracle_dt_sequence(oracle, adv, U, bx, by, bz, dh, N, g, 10)
    gpu = GU.GpuRunner(N=N, g=g, scheme=1, recon=1, riemann=1, limvar=1, prec=1, max_groups=64)
    res = run_grid(gpu, U, bx, by, bz, dts, dh, N, g)
    assert_fields(grid_errors(res, ref), TOL[1], "config 4")
    assert H.rel_divb(res[1], res[2], res[3], dh) < 1e-13
    t0, t1 = H.totals(U), H.totals(res[0])
    assert abs(t1[4] - t0[4]) / t0[4] < 1e-13


# ---------------------------------------------------------------------------------------------------------------
# degenerate states through the plane-marching VL kernels: B = 0 (HLLD's double-star state collapses, every EMF is zero), the
# static blast (zero velocity: every mass flux sits inside the dead zone of the CT switch; strong shock; floors)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [1, 0])
@pytest.mark.parametrize("which", ["hydro", "blast"])
def test_vl_march_on_degenerate_states(oracle, which, prec):
    n, N, g = 32, 16, 3
    dtp = GU.np_dtype(prec)
    if which == "hydro":
        U, bx, by, bz, dh = inputs.random_group_grid(n, 99)
        bx, by, bz = np.zeros_like(bx), np.zeros_like(by), np.zeros_like(bz)
        rho = U[0]
        v = U[1:4] / rho
        U = inputs.conserved(rho, v[0], v[1], v[2], 0.6 + 0.0 * rho, bx, by, bz)
    else:
        U, bx, by, bz, dh = inputs.blast_grid(n)
    state0 = tuple(a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz))
    cfg, adv = oracle_fn(oracle, N, g, 0, 0, 1, 0, prec)
    dts, ref, ref_out = PC.run_grid_oracle(oracle, adv, state0, dh, N, g)
    gpu = GU.GpuRunner(N=N, g=g, scheme=0, recon=0, riemann=1, prec=prec, max_groups=8)
    res, gpu_out = PC.run_grid(gpu, state0, dts, dh, N, g, dtype=dtp)
    errs = PC.grid_errors(res, ref)
    if which == "hydro":
        for k in ("Bx", "By", "Bz"):
            assert errs.pop(k) == 0.0 and not np.any(res[1:][("Bx", "By", "Bz").index(k)])      # B stays exactly zero
    if prec == 1:
        assert_fields(errs, TOL[1], f"{which} FP64")
    else:
        s32, _ = PC.run_grid(_fp32_reference(oracle, cfg), state0, dts, dh, N, g, dtype=np.float32)
        e32 = PC.grid_errors(s32, ref)
        gate = PC.fp32_gate({k: e32[k] for k in errs})
        bad = {k: (v, gate[k]) for k, v in errs.items() if not v <= gate[k]}
        assert not bad, f"{which} FP32 over the gate (R14b): {bad}; oracle-FP32 {e32}"
    t0, t1 = H.totals(state0[0]), H.totals(res[0].astype(np.float64))
    assert abs(t1[0] - t0[0]) / t0[0] < (1e-13 if prec == 1 else 2e-6) and abs(t1[4] - t0[4]) / t0[4] < (1e-13 if prec == 1 else 2e-6)
