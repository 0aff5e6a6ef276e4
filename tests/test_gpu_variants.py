"""-m gpu parity tests of the NEXT-4 variants: minmod / van Leer slope limiters and VL + PPM, the CUDA
path through the C ABI against the oracle on the same seeded inputs.  Tolerances as tests/test_gpu_parity.py."""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import gpu_util as GU

pytestmark = pytest.mark.gpu

TOL = {1: 1e-11, 0: 1e-4}
TOL_ONE_STEP = {1: 2e-13, 0: 1e-4}
EMF_TIE = {1: 1e-12, 0: 1e-5}

# name, scheme, recon, g, limiter
VARIANTS = [("vl_ppm", 0, 1, 4, 0), ("vl_ppm_minmod", 0, 1, 4, 1), ("vl_ppm_vanleer", 0, 1, 4, 2), ("vl_plm_minmod", 0, 0, 3, 1),
            ("vl_plm_vanleer", 0, 0, 3, 2), ("ctu_plm_minmod", 1, 0, 3, 1), ("ctu_plm_vanleer", 1, 0, 3, 2), ("ctu_ppm_minmod", 1, 1, 4, 1),
            ("ctu_ppm_vanleer", 1, 1, 4, 2)]


def bad_fields(errs, tol):
    return {k: v for k, v in errs.items() if not (v <= tol)}


@pytest.mark.parametrize("name,scheme,recon,g,limiter", VARIANTS)
@pytest.mark.parametrize("limvar", [0, 1])
@pytest.mark.parametrize("prec", [1, 0])
def test_one_step_every_variant(oracle, name, scheme, recon, g, limiter, limvar, prec):
    N, G = 16, 5
    dtp = GU.np_dtype(prec)
    U_in, B_in, dh = inputs.config2_batch(G, N=N, g=g, dtype=dtp)
    U64, B64 = U_in.astype(np.float64), B_in.astype(np.float64)
    for riemann in (1, 2):
        cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann, limvar=limvar, limiter=limiter, emf_tie=EMF_TIE[prec])
        dt, _ = oracle.dt_reduce(cfg, U64, B64, g, dh, 0.3)
        ref = oracle.advance(cfg, U64, B64, dt, dh)
        gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann, limvar=limvar, prec=prec, max_groups=G, limiter=limiter)
        out = gpu(U_in, B_in, dt, dh)
        errs = GU.field_errors(out, ref, N)
        assert not bad_fields(errs, TOL_ONE_STEP[prec]), (name, riemann, limvar, errs)


@pytest.mark.parametrize("prec", [1, 0])
def test_vl_ppm_ten_steps_on_a_periodic_grid(oracle, prec):
    """config-1 type run (32^3 periodic ABC grid cut into 8 groups, 10 steps at CFL 0.3) with VL + PPM, g = 4: per-field
    parity at step 10, div B and shared faces on the device side"""
    n, N, g = 32, 16, 4
    dtp = GU.np_dtype(prec)
    U, bx, by, bz, dh = inputs.abc_grid(n, seed=1804, p0=1.0, vamp=1e-3)
    cfg = oracle.make_config(N=N, g=g, scheme=0, recon=1, emf_tie=EMF_TIE[prec])
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    gpu = GU.GpuRunner(N=N, g=g, scheme=0, recon=1, prec=prec, max_groups=8)
    ref = [a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz)]
    dev = [a.astype(dtp) for a in (U, bx, by, bz)]
    for _ in range(10):
        Ui, Bi = inputs.pack_groups(*ref, n, 0)
        dt, _ = oracle.dt_reduce(oracle.make_config(N=n, g=3), Ui, Bi, 0, dh, 0.3)
        ref = list(H.step_grid(adv, *ref, dt, dh, N, g)[:4])
        r = H.step_grid(gpu, *dev, dt, dh, N, g, dtype=dtp)
        dev = list(r[:4])
        assert r[5] == 0.0                                       # faces shared by two groups: bitwise equal
    assert H.rel_divb(*[a.astype(np.float64) for a in dev[1:]], dh) < (1e-13 if prec == 1 else 2e-5)
    names = ["rho", "Mx", "My", "Mz", "e"]
    errs = {names[v]: H.field_err(dev[0][v], ref[0][v]) for v in (0, 4)}
    mom = max(np.abs(ref[0][v]).max() for v in (1, 2, 3))        # the three momentum components share one scale
    for v in (1, 2, 3):
        errs[names[v]] = float(np.abs(dev[0][v] - ref[0][v]).max() / mom)
    for k, a, b in (("Bx", dev[1], ref[1]), ("By", dev[2], ref[2]), ("Bz", dev[3], ref[3])):
        errs[k] = H.field_err(a, b)
    assert not bad_fields(errs, TOL[prec]), errs


@pytest.mark.parametrize("name", ["rj2a", "torrilhon"])
@pytest.mark.parametrize("prec", [1, 0])
def test_shock_tubes_ctu_ppm_roe(oracle, name, prec):
    """the paper's 1-D Riemann problems (Table 1) with its own combination CTU + PPM + Roe, patch
    groups of 8^3 along the tube: 20 steps on the device against the oracle with the oracle's dt sequence"""
    import tubes
    n, g = 64, 4
    dtp = GU.np_dtype(prec)
    cfg = oracle.make_config(N=tubes.NT, g=g, scheme=1, recon=1, riemann=2, emf_tie=EMF_TIE[prec])
    adv = lambda Ui, Bi, dt, dh: oracle.advance(cfg, Ui, Bi, dt, dh)
    c0 = oracle.make_config(N=tubes.NT, g=3)

    def dt_fn(U, bx, by, bz, dh):
        Ui, Bi = inputs.pack_groups(U, bx, by, bz, tubes.NT, 0)
        return oracle.dt_reduce(c0, Ui.astype(np.float64), Bi.astype(np.float64), 0, dh, 0.3)[0]
    ref, dh, dts = tubes.run_tube(adv, dt_fn, name, n, max_steps=20, g=g)
    if prec == 0:       # the FP64 oracle started from the FP32-rounded state (the tube states are not FP32 numbers)
        U, bx, by, bz, _ = inputs.shock_tube(name, n, 0, tubes.NT)
        ref = [a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz)]
        for dt in dts:
            ref = list(H.step_grid(adv, *ref, dt, dh, tubes.NT, g)[:4])
    gpu = GU.GpuRunner(N=tubes.NT, g=g, scheme=1, recon=1, riemann=2, prec=prec, max_groups=2 * n // tubes.NT)
    it = iter(dts)
    dev, _, _ = tubes.run_tube(gpu, lambda *a: next(it), name, n, t_end=sum(dts), dtype=dtp, g=g)
    Pd, Pr = tubes.profile(dev, 2 * n), tubes.profile(ref, 2 * n)
    mom = np.abs(Pr[1:4]).max()
    errs = {}
    for v, nm in enumerate(["rho", "Mn", "Mt1", "Mt2", "e", "Bt1", "Bt2"]):
        den = mom if v in (1, 2, 3) else np.abs(Pr[v]).max()
        errs[nm] = float(np.abs(Pd[v] - Pr[v]).max() / den)
    assert not bad_fields(errs, TOL[prec]), errs
    assert np.array_equal(dev[1], np.full_like(dev[1], dtp(inputs.RIEMANN_PROBLEMS[name]["Bn"])))      # B_n untouched
