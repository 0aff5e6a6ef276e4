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


# ---------------------------------------------------------------------------------------------------------------
# Roe solver with H-correction (R19): device path for VL + PLM (the combination of the paper's Fig. 18)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("limvar", [0, 1])
@pytest.mark.parametrize("prec", [1, 0])
def test_h_correction_one_step_and_ten_steps(oracle, limvar, prec):
    N, G, g = 16, 5, 4
    dtp = GU.np_dtype(prec)
    U_in, B_in, dh = inputs.config2_batch(G, N=N, g=g, dtype=dtp)
    U64, B64 = U_in.astype(np.float64), B_in.astype(np.float64)
    cfg = oracle.make_config(N=N, g=g, scheme=0, recon=0, riemann=2, limvar=limvar, emf_tie=EMF_TIE[prec], hcorr=1)
    dt, _ = oracle.dt_reduce(cfg, U64, B64, g, dh, 0.3)
    ref = oracle.advance(cfg, U64, B64, dt, dh)
    gpu = GU.GpuRunner(N=N, g=g, scheme=0, recon=0, riemann=2, limvar=limvar, prec=prec, max_groups=8, hcorr=1)
    out = gpu(U_in, B_in, dt, dh)
    errs = GU.field_errors(out, ref, N)
    assert not bad_fields(errs, TOL_ONE_STEP[prec]), errs
    # and it is the H-correction that was compared: the plain Roe solver differs on this transonic state
    plain = oracle.advance(oracle.make_config(N=N, g=g, scheme=0, recon=0, riemann=2, limvar=limvar, emf_tie=EMF_TIE[prec]), U64, B64, dt, dh)
    assert np.abs(plain["U"] - ref["U"]).max() > 1e-6
    assert all(a <= b for a, b in zip(gpu.stats(), ref["stats"]))
    # ten steps on a periodic 32^3 grid: shared faces bitwise, div B, parity
    n = 32
    U, bx, by, bz, dh = inputs.random_group_grid(n, 77)
    adv = lambda Ui, Bi, dt_, dh_: oracle.advance(cfg, Ui, Bi, dt_, dh_)
    r = [a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz)]
    d = [a.astype(dtp) for a in (U, bx, by, bz)]
    for _ in range(10):
        Ui, Bi = inputs.pack_groups(*r, n, 0)
        dt, _ = oracle.dt_reduce(oracle.make_config(N=n, g=3), Ui, Bi, 0, dh, 0.3)
        r = list(H.step_grid(adv, *r, dt, dh, N, g)[:4])
        o = H.step_grid(gpu, *d, dt, dh, N, g, dtype=dtp)
        assert o[5] == 0.0
        d = list(o[:4])
    for a, b in zip(d, r):
        assert H.field_err(a, b) <= TOL[prec]
    assert H.rel_divb(*(np.asarray(a, dtype=np.float64) for a in d[1:]), dh) < (1e-13 if prec == 1 else 2e-5)


def test_expansion_shock_dissolves_on_the_device(oracle):
    """the textbook failure of the plain Roe flux (tests/test_oracle_hcorr.py) through the CUDA path: 8^3 patch groups along the tube"""
    from test_oracle_hcorr import _tube_with_expansion_shock, _expansion_shock, GAM
    res = {}
    for hc in (0, 1):
        U, bx, by, bz, dh, xc = _tube_with_expansion_shock(64)
        U, bx, by, bz = (np.tile(a, (1, 2, 2, 1)) if a.ndim == 4 else a for a in (U, bx, by, bz))     # 8 cells across for 8^3 groups
        bx = np.zeros((8, 8, 129)); by = np.zeros((8, 9, 128)); bz = np.zeros((9, 8, 128))
        gpu = GU.GpuRunner(N=8, g=3 + hc, scheme=0, recon=0, riemann=2, prec=1, max_groups=16, hcorr=hc, gamma=GAM)
        ref_cfg = oracle.make_config(N=8, g=3 + hc, gamma=GAM, scheme=0, recon=0, riemann=2, hcorr=hc)
        Ur, br = U.copy(), (bx.copy(), by.copy(), bz.copy())
        for _ in range(40):
            U, bx, by, bz, _, _ = H.step_grid(gpu, U, bx, by, bz, 0.3 * dh / 3.6, dh, 8, 3 + hc)
            Ur, b0, b1, b2, _, _ = H.step_grid(lambda a, b, c, d_: oracle.advance(ref_cfg, a, b, c, d_), Ur, *br, 0.3 * dh / 3.6, dh, 8, 3 + hc)
            br = (b0, b1, b2)
        w = np.abs(xc - 0.5) < 0.2
        res[hc] = np.abs(np.diff(U[0][0, 0, :][w])).max()
        assert H.field_err(U[0], Ur[0]) < 1e-11, hc
    jump = _expansion_shock()[0][0] - _expansion_shock()[1][0]
    assert res[0] > 0.95 * jump and res[1] < 0.5 * jump, res


@pytest.mark.parametrize("scheme,recon,g", [(1, 1, 5), (1, 0, 4), (0, 1, 5)])
@pytest.mark.parametrize("prec", [1, 0])
def test_h_correction_ctu_and_ppm_one_step_and_ten_steps(oracle, scheme, recon, g, prec):
    """the other schemes (the paper's own test combination CTU + PPM + Roe; CTU + PLM; VL + PPM): eta of the corrected /
    parabola states, one more ghost cell, against the oracle"""
    N, G = 16, 4
    dtp = GU.np_dtype(prec)
    limvar = 1 if scheme == 1 else 0
    U_in, B_in, dh = inputs.config2_batch(G, N=N, g=g, dtype=dtp)
    U64, B64 = U_in.astype(np.float64), B_in.astype(np.float64)
    kw = dict(N=N, g=g, scheme=scheme, recon=recon, riemann=2, limvar=limvar)
    cfg = oracle.make_config(emf_tie=EMF_TIE[prec], hcorr=1, **kw)
    dt, _ = oracle.dt_reduce(cfg, U64, B64, g, dh, 0.3)
    ref = oracle.advance(cfg, U64, B64, dt, dh)
    gpu = GU.GpuRunner(prec=prec, max_groups=8, hcorr=1, **kw)
    out = gpu(U_in, B_in, dt, dh)
    errs = GU.field_errors(out, ref, N)
    assert not bad_fields(errs, TOL_ONE_STEP[prec]), errs
    plain = oracle.advance(oracle.make_config(emf_tie=EMF_TIE[prec], **kw), U64, B64, dt, dh)
    assert np.abs(plain["U"] - ref["U"]).max() > 1e-6               # it is the corrected solver that was compared
    assert all(a <= b for a, b in zip(gpu.stats(), ref["stats"]))
    n = 32
    U, bx, by, bz, dh = inputs.random_group_grid(n, 78)
    adv = lambda Ui, Bi, dt_, dh_: oracle.advance(cfg, Ui, Bi, dt_, dh_)
    r = [a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz)]
    d = [a.astype(dtp) for a in (U, bx, by, bz)]
    for _ in range(10):
        Ui, Bi = inputs.pack_groups(*r, n, 0)
        dt, _ = oracle.dt_reduce(oracle.make_config(N=n, g=3), Ui, Bi, 0, dh, 0.3)
        r = list(H.step_grid(adv, *r, dt, dh, N, g)[:4])
        o = H.step_grid(gpu, *d, dt, dh, N, g, dtype=dtp)
        assert o[5] == 0.0                                            # shared faces of neighbouring groups bitwise equal
        d = list(o[:4])
    for a, b in zip(d, r):
        assert H.field_err(a, b) <= TOL[prec]
    assert H.rel_divb(*(np.asarray(a, dtype=np.float64) for a in d[1:]), dh) < (1e-13 if prec == 1 else 2e-5)


def test_h_correction_argument_checks():
    from paper_1804_03479_b200 import mhd
    for kw in (dict(riemann=mhd.HLLD, g=4), dict(riemann=mhd.ROE, g=3), dict(riemann=mhd.ROE, g=4, scheme=mhd.CTU, recon=mhd.PPM),
               dict(riemann=mhd.ROE, g=4, scheme=mhd.VL, recon=mhd.PPM), dict(riemann=mhd.ROE, g=3, scheme=mhd.CTU, recon=mhd.PLM),
               dict(riemann=mhd.HLLE, g=5, scheme=mhd.CTU, recon=mhd.PPM)):
        with pytest.raises(mhd.MHDError) as ei:
            mhd.Solver(mhd.make_config(hcorr=1, max_groups=2, **kw))
        assert ei.value.code == mhd.EINVAL
