"""-m gpu tests of the boundary itself: edge cases, slicing, shapes other than 16^3, the host (stream-overlapped) path,
the dt reduction, counters, and the full-size batch of bench.py checked on sampled groups."""
import os

import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import gpu_util as GU
import parity_cases as PC

pytestmark = pytest.mark.gpu


def small_batch(G, N=16, g=3, dtype=np.float64, first=0):
    return inputs.config2_batch(G, N=N, g=g, dtype=dtype, first=first)


def test_empty_batch_and_argument_errors():
    import torch
    from paper_1804_03479_b200 import mhd
    s = mhd.Solver(mhd.make_config(max_groups=4))
    U, B, dh = small_batch(1)
    dU, dB = torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda()
    out = s.alloc_outputs(1)
    out["U"].fill_(7.0)
    s.advance(dU, dB, out["U"], out["B"], None, None, 0, 1e-3, dh)          # ngroups = 0: no-op
    torch.cuda.synchronize()
    assert float(out["U"].min()) == 7.0
    for bad in (dict(ngroups=5), dict(dt=0.0), dict(dt=float("nan")), dict(dh=-1.0)):
        kw = dict(ngroups=1, dt=1e-3, dh=dh); kw.update(bad)
        with pytest.raises(mhd.MHDError) as ei:
            s.advance(dU, dB, out["U"], out["B"], None, None, kw["ngroups"], kw["dt"], kw["dh"])
        assert ei.value.code == mhd.EINVAL
    with pytest.raises(mhd.MHDError):
        s.advance(None, dB, out["U"], out["B"], None, None, 1, 1e-3, dh)
    with pytest.raises(mhd.MHDError):
        s.dt_reduce(dU, dB, 1, 2, dh, 0.3)                                   # ghost width neither 0 nor cfg.nghost
    with pytest.raises(mhd.MHDError):
        mhd.Solver(mhd.make_config(g=2))
    assert s.sizes() == {k: v for k, v in inputs.sizes(16, 3).items() if k != "T"}


@pytest.mark.parametrize("prec", [1, 0])
def test_planes_optional_and_identical_results(oracle, prec):
    """flux_out / emf_out NULL must not change U_out, B_out (bitwise)."""
    dtp = GU.np_dtype(prec)
    U, B, dh = small_batch(3, dtype=dtp)
    a = GU.GpuRunner(prec=prec, planes=True, max_groups=3)(U, B, 2e-3, dh)
    b = GU.GpuRunner(prec=prec, planes=False, max_groups=3)(U, B, 2e-3, dh)
    assert b["flux"] is None and b["emf"] is None
    assert np.array_equal(a["U"], b["U"]) and np.array_equal(a["B"], b["B"])


@pytest.mark.parametrize("slice_groups", ["1", "3", "64"])
def test_ragged_slices_are_bitwise_identical(slice_groups, monkeypatch):
    """7 groups processed in slices of 1, 3 (ragged tail) and all at once give the same bits; groups are independent."""
    U, B, dh = small_batch(7)
    monkeypatch.setenv("MHD_SLICE_GROUPS", slice_groups)
    a = GU.GpuRunner(max_groups=7)(U, B, 2e-3, dh)
    monkeypatch.delenv("MHD_SLICE_GROUPS")
    b = GU.GpuRunner(max_groups=7)(U, B, 2e-3, dh)
    for k in ("U", "B", "flux", "emf"):
        assert np.array_equal(a[k], b[k]), k
    # and a group's result does not depend on its position in the batch
    c = GU.GpuRunner(max_groups=7)(U[::-1].copy(), B[::-1].copy(), 2e-3, dh)
    assert np.array_equal(c["U"][::-1], b["U"]) and np.array_equal(c["emf"][::-1], b["emf"])


@pytest.mark.parametrize("prec", [1, 0])
def test_one_slice_per_lane_equals_one_slice_bitwise(prec, monkeypatch):
    """A batch of >= 256 groups is cut into one slice per lane (two concurrent streams); one lane = one slice: same bits,
    same reduced CFL speed."""
    dtp = GU.np_dtype(prec)
    U16, B16, dh = small_batch(16, dtype=dtp)
    G = 259                                                      # two lanes: slices of 130 and 129 groups
    U, B = np.tile(U16, (17, 1))[:G].copy(), np.tile(B16, (17, 1))[:G].copy()
    a, dt_a, s_a = GU.GpuRunner(prec=prec, max_groups=G).advance_dt(U, B, 2e-3, dh, 0.3)
    monkeypatch.setenv("MHD_LANES", "1")
    b, dt_b, s_b = GU.GpuRunner(prec=prec, max_groups=G).advance_dt(U, B, 2e-3, dh, 0.3)
    for k in ("U", "B", "flux", "emf"):
        assert np.array_equal(a[k], b[k]), k
    assert (dt_a, s_a) == (dt_b, s_b)
    assert np.array_equal(a["U"][:16], a["U"][16:32]) and np.array_equal(a["U"][:3], a["U"][256:259])   # tiled inputs, both lanes


@pytest.mark.parametrize("N,g,scheme,recon", [(8, 3, 0, 0), (32, 3, 0, 0), (16, 4, 0, 0), (8, 4, 1, 1), (24, 5, 1, 1), (32, 3, 1, 0)])
def test_other_group_sizes_and_wider_ghosts(oracle, N, g, scheme, recon):
    """ps2 != 16 and ghost widths above the minimum (extra layers must not matter)."""
    n = 2 * N if N <= 16 else N
    U, bx, by, bz, dh = inputs.random_group_grid(n, 11)
    cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon)
    Ui, Bi = inputs.pack_groups(U, bx, by, bz, N, g)
    dt = 0.2 * dh
    ref = oracle.advance(cfg, Ui, Bi, dt, dh)
    gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, max_groups=Ui.shape[0])
    out = gpu(Ui, Bi, dt, dh)
    errs = GU.field_errors(out, ref, N)
    assert max(errs.values()) <= 2e-13, errs
    assert all(a <= b for a, b in zip(gpu.stats(), ref["stats"]))


@pytest.mark.parametrize("prec", [1, 0])
def test_uniform_state_is_a_fixed_point_on_the_gpu(prec):
    N, g = 16, 3
    dtp = GU.np_dtype(prec)
    rho, v, p, Bv = 1.3, (0.4, -0.7, 0.2), 0.8, (0.5, -0.3, 0.9)
    bx = np.full((N, N, N + 1), Bv[0]); by = np.full((N, N + 1, N), Bv[1]); bz = np.full((N + 1, N, N), Bv[2])
    o = np.ones((N, N, N))
    U = inputs.conserved(rho * o, v[0] * o, v[1] * o, v[2] * o, p * o, bx, by, bz)
    for scheme, recon, gg in ((0, 0, 3), (1, 1, 4)):
        gpu = GU.GpuRunner(N=N, g=gg, scheme=scheme, recon=recon, prec=prec, max_groups=1)
        Un, bxn, byn, bzn, out, _ = H.step_grid(gpu, U.astype(dtp), bx.astype(dtp), by.astype(dtp), bz.astype(dtp), 0.01, 1.0 / N, N, gg, dtp)
        assert np.array_equal(bxn, bx.astype(dtp)) and np.array_equal(byn, by.astype(dtp)) and np.array_equal(bzn, bz.astype(dtp))
        assert np.abs(Un - U.astype(dtp)).max() < (1e-14 if prec == 1 else 1e-6)
        assert gpu.stats() == (0, 0, 0)


def test_decomposition_is_bitwise_on_the_gpu(monkeypatch):
    """P9 on the device: 32^3 advanced as one group of 32^3 and as 8 groups of 16^3.  With the staged kernels for both
    (MHD_NO_FUSED_PASS1) the bits are the same; the standard 16^3 group normally runs its first pass in the fused kernels
    (csrc/mhd_vl_pass1.cuh, mhd_ctu_pass1.cuh), which agree with the staged ones to rounding: 1e-13 in FP64 (a ghost-width
    or tile-logic error would show at 1e-3)."""
    n = 32
    U, bx, by, bz, dh = inputs.random_group_grid(n, 5)
    dt = 0.2 * dh
    for scheme, recon, g in ((0, 0, 3), (1, 1, 4)):
        a = H.step_grid(GU.GpuRunner(N=32, g=g, scheme=scheme, recon=recon, max_groups=1), U, bx, by, bz, dt, dh, 32, g)
        monkeypatch.setenv("MHD_NO_FUSED_PASS1", "1")
        staged = GU.GpuRunner(N=16, g=g, scheme=scheme, recon=recon, max_groups=8)
        monkeypatch.delenv("MHD_NO_FUSED_PASS1")
        b = H.step_grid(staged, U, bx, by, bz, dt, dh, 16, g)
        for x, y in zip(a[:4], b[:4]):
            assert np.array_equal(x, y)
        assert b[5] == 0.0
        c = H.step_grid(GU.GpuRunner(N=16, g=g, scheme=scheme, recon=recon, max_groups=8), U, bx, by, bz, dt, dh, 16, g)
        for x, y in zip(a[:4], c[:4]):
            assert np.abs(x - y).max() <= 1e-13 * np.abs(x).max()
        assert c[5] == 0.0                      # faces shared by two groups: bitwise equal with the fused kernels too


@pytest.mark.parametrize("prec", [1, 0])
def test_dt_reduce_matches_the_oracle(oracle, prec):
    dtp = GU.np_dtype(prec)
    tol = 1e-14 if prec == 1 else 1e-6
    U, B, dh = small_batch(9, dtype=dtp)
    cfg = oracle.make_config()
    gpu = GU.GpuRunner(prec=prec, max_groups=9)
    ref_dt, ref_s = oracle.dt_reduce(cfg, U.astype(np.float64), B.astype(np.float64), 3, dh, 0.3)
    dt, s = gpu.dt(U, B, 3, dh, 0.3)
    assert abs(dt - ref_dt) <= tol * ref_dt and abs(s - ref_s) <= tol * ref_s
    out = gpu(U, B, ref_dt, dh)                                   # ghost-free layout of the outputs
    ref_dt2, _ = oracle.dt_reduce(cfg, out["U"].astype(np.float64), out["B"].astype(np.float64), 0, dh, 0.3)
    dt2, _ = gpu.dt(out["U"], out["B"], 0, dh, 0.3)
    assert abs(dt2 - ref_dt2) <= tol * ref_dt2
    # the max is exact: a single group holding the fastest cell gives the same answer as the whole batch
    per_group = [gpu.dt(U[q:q + 1], B[q:q + 1], 3, dh, 0.3)[1] for q in range(9)]
    assert max(per_group) == s


@pytest.mark.parametrize("N,g,scheme,recon", [(16, 3, 0, 0), (16, 4, 1, 1), (8, 3, 0, 0), (24, 4, 1, 1)])
@pytest.mark.parametrize("prec", [1, 0])
def test_advance_dt_equals_advance_then_dt_reduce_bitwise(oracle, prec, N, g, scheme, recon, monkeypatch):
    """mhd_advance_dt (S9 fused into the final update) = mhd_advance + mhd_dt_reduce on its outputs, bit for bit;
    the reduced speed also agrees with the oracle's CFL reduction of the oracle's own new state."""
    dtp = GU.np_dtype(prec)
    G = 7
    U, B, dh = small_batch(G, N=N, g=g, dtype=dtp)
    cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon)
    dt0, _ = oracle.dt_reduce(cfg, U.astype(np.float64), B.astype(np.float64), g, dh, 0.3)
    for slices in (None, "3"):                       # one slice; ragged slices on concurrent lanes
        if slices:
            monkeypatch.setenv("MHD_SLICE_GROUPS", slices)
        gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, prec=prec, max_groups=G)
        a = gpu(U, B, dt0, dh)
        dt_a, s_a = gpu.dt(a["U"], a["B"], 0, dh, 0.3)
        b, dt_b, s_b = gpu.advance_dt(U, B, dt0, dh, 0.3)
        for k in ("U", "B", "flux", "emf"):
            assert np.array_equal(a[k], b[k]), k
        assert s_a == s_b and dt_a == dt_b
    ref = oracle.advance(cfg, U.astype(np.float64), B.astype(np.float64), dt0, dh)
    ref_dt, ref_s = oracle.dt_reduce(cfg, ref["U"], ref["B"], 0, dh, 0.3)
    assert abs(s_b - ref_s) <= (1e-11 if prec == 1 else 1e-4) * ref_s
    with pytest.raises(gpu.mhd.MHDError):            # no groups: the time step is undefined
        gpu.solver.advance_dt(None, None, None, None, None, None, 0, dt0, dh, 0.3)


@pytest.mark.parametrize("prec", [1, 0])
@pytest.mark.parametrize("chunk,nstreams", [(4, 3), (16, 1), (5, 2)])
def test_advance_host_equals_advance_bitwise(prec, chunk, nstreams):
    """the stream-overlapped host path (pinned or pageable host memory, ragged last chunk) returns the same bits"""
    import torch
    dtp = GU.np_dtype(prec)
    G = 13
    U, B, dh = small_batch(G, dtype=dtp)
    gpu = GU.GpuRunner(prec=prec, max_groups=16)
    ref = gpu(U, B, 2e-3, dh)
    s = gpu.solver
    tdt = s.torch_dtype
    hU, hB = torch.from_numpy(U).pin_memory(), torch.from_numpy(B).pin_memory()
    ho = {k: torch.empty((G, n), dtype=tdt).pin_memory() for k, n in (("U", s.n_U_out), ("B", s.n_B_out), ("flux", s.n_flux), ("emf", s.n_emf))}
    s.advance_host(hU, hB, ho["U"], ho["B"], ho["flux"], ho["emf"], G, 2e-3, dh, chunk, nstreams)
    for k in ("U", "B", "flux", "emf"):
        assert np.array_equal(ho[k].numpy(), ref[k]), k
    # pageable numpy arrays and no planes
    oU, oB = np.empty((G, s.n_U_out), dtype=dtp), np.empty((G, s.n_B_out), dtype=dtp)
    s.advance_host(U, B, oU, oB, None, None, G, 2e-3, dh, chunk, nstreams)
    assert np.array_equal(oU, ref["U"]) and np.array_equal(oB, ref["B"])
    # mhd_advance_host_dt: same outputs, and the CFL speed every chunk's final update reduced equals mhd_advance_dt's
    _, dt_d, s_d = gpu.advance_dt(U, B, 2e-3, dh, 0.3)
    for v in ho.values():
        v.zero_()
    dt_h, s_h = s.advance_host_dt(hU, hB, ho["U"], ho["B"], ho["flux"], ho["emf"], G, 2e-3, dh, chunk, nstreams, 0.3)
    for k in ("U", "B", "flux", "emf"):
        assert np.array_equal(ho[k].numpy(), ref[k]), k
    assert (dt_h, s_h) == (dt_d, s_d)


@pytest.mark.parametrize("prec,scheme,recon,g", [(0, 0, 0, 3), (1, 0, 0, 3), (0, 1, 1, 4), (1, 1, 1, 4)])
def test_full_size_batch_on_sampled_groups(oracle, prec, scheme, recon, g):
    """BASELINE.json configs[1] at full size (512 groups, the launch configuration bench.py times): one step, every
    32nd group compared with the oracle (groups are independent, so the oracle can compute them one by one)."""
    dtp = GU.np_dtype(prec)
    G, N = 512, 16
    pool_U, pool_B, dh = small_batch(16, g=g, dtype=dtp)
    U = np.tile(pool_U, (G // 16, 1)); B = np.tile(pool_B, (G // 16, 1))
    # make the sampled groups distinct from the pool so that position matters
    sample = list(range(5, G, 32))
    extra_U, extra_B, _ = small_batch(len(sample), g=g, dtype=dtp, first=100)
    U[sample] = extra_U; B[sample] = extra_B
    cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon, emf_tie=(1e-12 if prec == 1 else 1e-5))
    dt, _ = oracle.dt_reduce(cfg, U[sample].astype(np.float64), B[sample].astype(np.float64), g, dh, 0.3)
    gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, prec=prec, max_groups=G)
    out = gpu(U, B, dt, dh)
    ref = oracle.advance(cfg, U[sample].astype(np.float64), B[sample].astype(np.float64), dt, dh)
    sub = {k: out[k][sample] for k in out}
    errs = GU.field_errors(sub, ref, N)
    assert max(errs.values()) <= (2e-13 if prec == 1 else 1e-4), errs
    # invariants that hold at any size: div B of every group's output at round-off
    bx, by, bz = inputs.split_B(out["B"].astype(np.float64), N)
    assert H.rel_divb(bx, by, bz, dh) < (1e-13 if prec == 1 else 2e-5)


@pytest.mark.parametrize("scheme,recon,g", [(0, 0, 3), (1, 0, 3), (1, 1, 4)])
@pytest.mark.parametrize("prec", [1, 0])
def test_no_stage_reads_an_unwritten_workspace_value(scheme, recon, g, prec, monkeypatch):
    """NaN-poisoned workspace (MHD_POISON): outputs must be finite and bitwise equal to the normal run, for every
    Riemann solver and both limiter variables (the oracle's NaN-initialised temporaries, on the device)."""
    dtp = GU.np_dtype(prec)
    U, B, dh = small_batch(3, g=g, dtype=dtp)
    for riemann in (0, 1, 2):
        for limvar in (0, 1):
            kw = dict(N=16, g=g, scheme=scheme, recon=recon, riemann=riemann, limvar=limvar, prec=prec, max_groups=3)
            ref = GU.GpuRunner(**kw)(U, B, 2e-3, dh)
            monkeypatch.setenv("MHD_POISON", "1")
            out = GU.GpuRunner(**kw)(U, B, 2e-3, dh)
            monkeypatch.delenv("MHD_POISON")
            for k in ("U", "B", "flux", "emf"):
                assert np.isfinite(out[k]).all(), (riemann, limvar, k)
                assert np.array_equal(out[k], ref[k]), (riemann, limvar, k)


@pytest.mark.parametrize("scheme,recon,g", [(1, 1, 4), (0, 0, 3)])
def test_fused_pass1_agrees_with_the_staged_kernels(scheme, recon, g, monkeypatch):
    """The first pass of the standard FP32 patch group runs in one kernel (CTU steps 1 + 2: csrc/mhd_ctu_pass1.cuh; VL
    S0-S2: csrc/mhd_vl_pass1.cuh); with MHD_NO_FUSED_PASS1 the same solver runs the staged kernels.  Same functions, same
    operands, but the compiler orders / contracts the arithmetic inside a stage differently, so the two agree to the last
    bits only: a few FP32 ulp of each field's scale (measured 1e-7 U, 1.4e-6 B, 5e-7 fluxes; EMFs 5e-7 ... 3.3e-5: an edge whose mass
    flux lies in the ramp of the CT switch, R10a, turns an ulp of that flux into a visible change of its weight)"""
    U, B, dh = small_batch(5, g=g, dtype=np.float32)
    kw = dict(N=16, g=g, scheme=scheme, recon=recon, riemann=1, prec=0, max_groups=5)
    fused = GU.GpuRunner(**kw)
    monkeypatch.setenv("MHD_NO_FUSED_PASS1", "1")
    staged = GU.GpuRunner(**kw)
    monkeypatch.delenv("MHD_NO_FUSED_PASS1")
    tol = {"U": 5e-7, "B": 5e-6, "flux": 3e-6, "emf": 1e-4}
    for dt in (1e-3, 2e-3, 3e-3):
        a, b = fused(U, B, dt, dh), staged(U, B, dt, dh)
        for k in ("U", "B", "flux", "emf"):
            assert np.abs(a[k].astype(np.float64) - b[k]).max() <= tol[k] * np.abs(b[k]).max(), (dt, k)
    assert fused.solver.launch_count() < staged.solver.launch_count()      # and it really is another launch sequence


@pytest.mark.parametrize("which,prec", [("abc", 1), ("abc", 0), ("blast", 1)])
def test_configs_3_4_full_size_256_cubed_on_sampled_groups(oracle, which, prec):
    """BASELINE.json configs 3 / 4 at full size: 256^3 -> 4096 groups of 16^3 (g = 4), CTU+PPM+HLLD+CT, one step through
    ONE mhd_advance call (several workspace slices on concurrent lanes); 24 sampled groups against the oracle (groups
    are independent given their ghost zones), plus the invariants that hold at any size: shared faces bitwise equal,
    div B at round-off, exact conservation on the periodic grid."""
    n, N, g = 256, 16, 4
    dtp = GU.np_dtype(prec)
    if which == "abc":
        U, bx, by, bz, dh = inputs.abc_grid(n, seed=1805, p0=0.15, vamp=1e-2)
    else:
        U, bx, by, bz, dh = inputs.blast_grid(n)
    U, bx, by, bz = (a.astype(dtp) for a in (U, bx, by, bz))
    Ui, Bi = inputs.pack_groups(U, bx, by, bz, N, g, dtp)
    G = Ui.shape[0]
    assert G == 4096
    sample = list(range(7, G, 173))
    # include groups that cut the blast sphere (centre of the grid)
    sample += [G // 2 + 8 * 16 + 8, G // 2 - 8 * 16 - 8 - 1]
    cfg = oracle.make_config(N=N, g=g, scheme=1, recon=1, emf_tie=(1e-12 if prec == 1 else 1e-5))
    dt, _ = oracle.dt_reduce(cfg, Ui.astype(np.float64), Bi.astype(np.float64), g, dh, 0.3)
    gpu = GU.GpuRunner(N=N, g=g, scheme=1, recon=1, prec=prec, max_groups=G, planes=True)
    dt_gpu, _ = gpu.dt(Ui, Bi, g, dh, 0.3)
    assert abs(dt_gpu - dt) <= (1e-14 if prec == 1 else 1e-6) * dt
    out = gpu(Ui, Bi, dt, dh)
    ref = oracle.advance(cfg, Ui[sample].astype(np.float64), Bi[sample].astype(np.float64), dt, dh)
    errs = GU.field_errors({k: out[k][sample] for k in out}, ref, N)
    if prec == 0:
        # R14b: |M|, the mass flux and the EMF (~ v B) are 1e-2 of the momentum-flux scale on this
        # config, so the plain algorithm in IEEE single precision (the FP32 oracle) is itself up to 7.6e-4 (emf) away from
        # the FP64 oracle after ONE step.  Gate per field: max(1e-4, 2 x that); measured GPU / gate <= 0.42
        # (profiles/r02_fp32_controls.md)
        r32 = oracle.advance32(cfg, Ui[sample], Bi[sample], dt, dh)
        gate = PC.fp32_gate(GU.field_errors(r32, ref, N))
        for k in ("rho", "e", "Bx", "By", "Bz", "flux_Mx", "flux_My", "flux_Mz"):
            assert gate[k] == 1e-4, (k, gate[k])
        bad = {k: (v, gate[k]) for k, v in errs.items() if not v <= gate[k]}
        assert not bad, (bad, errs)
    else:
        assert max(errs.values()) <= 1e-12, errs
    Un, bxn, byn, bzn, mism = inputs.unpack_groups(out["U"], out["B"], n, N)
    assert mism == 0.0
    assert H.rel_divb(bxn.astype(np.float64), byn.astype(np.float64), bzn.astype(np.float64), dh) < (1e-13 if prec == 1 else 2e-5)
    t0, t1 = H.totals(U), H.totals(Un)
    tol = 1e-13 if prec == 1 else 2e-6
    assert abs(t1[0] - t0[0]) / t0[0] < tol and abs(t1[4] - t0[4]) / t0[4] < tol


@pytest.mark.parametrize("scheme,recon,g", [(0, 0, 3), (1, 1, 4)])
@pytest.mark.parametrize("nstreams", [3, 4])
def test_config5_first_batch_through_the_host_path(oracle, scheme, recon, g, nstreams):
    """BASELINE.json configs[4]: the first 512-group batch of the 1024^3 ABC state (dh = 1/1024, generated group by group:
    inputs.abc_groups), FP32, VL+PLM and CTU+PPM, through mhd_advance_host_dt in 32-group chunks on 3 / 4 streams (a ragged
    last chunk with 3: 512 = 15 x 32 + 32 on lanes 0, 1, 2, 0, ...; and a ragged batch of 500 groups).  16 sampled groups
    against the FP64 oracle at the gate of R14b (max(1e-4, 2 x the FP32 oracle's error)); div B of every group at
    round-off; the returned dt equals the CFL reduction of the output."""
    import torch
    N, G = 16, 512 if nstreams == 4 else 500
    dtp = np.float32
    Ui, Bi, dh = inputs.abc_groups(1024, 0, G, N, g, dtype=dtp)
    sample = list(range(3, G, 32))
    cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon, emf_tie=1e-5)
    dt, _ = oracle.dt_reduce(cfg, Ui.astype(np.float64), Bi.astype(np.float64), g, dh, 0.3)
    gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, prec=0, max_groups=G)
    s = gpu.solver
    hU, hB = torch.from_numpy(Ui).pin_memory(), torch.from_numpy(Bi).pin_memory()
    ho = {k: torch.empty((G, n), dtype=torch.float32).pin_memory() for k, n in
          (("U", s.n_U_out), ("B", s.n_B_out), ("flux", s.n_flux), ("emf", s.n_emf))}
    dt_next, smax = s.advance_host_dt(hU, hB, ho["U"], ho["B"], ho["flux"], ho["emf"], G, dt, dh, 32, nstreams, 0.3)
    out = {k: v.numpy() for k, v in ho.items()}
    ref = oracle.advance(cfg, Ui[sample].astype(np.float64), Bi[sample].astype(np.float64), dt, dh)
    r32 = oracle.advance32(cfg, Ui[sample], Bi[sample], dt, dh)
    gate = PC.fp32_gate(GU.field_errors(r32, ref, N))
    errs = GU.field_errors({k: out[k][sample] for k in out}, ref, N)
    bad = {k: (v, gate[k]) for k, v in errs.items() if not v <= gate[k]}
    assert not bad, (bad, errs)
    for k in ("rho", "e", "Bx", "By", "Bz", "flux_Mx", "flux_My", "flux_Mz"):
        assert gate[k] == 1e-4 and errs[k] <= 1e-4
    bx, by, bz = inputs.split_B(out["B"].astype(np.float64), N)
    assert H.rel_divb(bx, by, bz, dh) < 2e-5 * 64            # FP32 round-off of b ~ 1 over dh = 1/1024 against the 16^3 boxes' 1/16
    dt_ref, _ = oracle.dt_reduce(cfg, out["U"].astype(np.float64), out["B"].astype(np.float64), 0, dh, 0.3)
    assert abs(dt_next - dt_ref) <= 1e-6 * dt_ref
    assert gpu.stats() == (0, 0, 0)


def test_nan_state_is_reported_not_turned_into_a_finite_dt():
    """A blown-up state must not come back as MHD_OK with a usable dt (the maximum of the CFL reduction would drop a NaN
    speed, and the floors of R9 would hide a NaN density): every dt-returning call fails with MHD_ESTATE."""
    import torch
    from paper_1804_03479_b200 import mhd
    for prec, scheme, recon, g in ((0, 0, 0, 3), (1, 0, 0, 3), (0, 1, 1, 4)):
        dtp = GU.np_dtype(prec)
        U, B, dh = small_batch(3, g=g, dtype=dtp)
        gpu = GU.GpuRunner(N=16, g=g, scheme=scheme, recon=recon, prec=prec, max_groups=3)
        T = 16 + 2 * g
        bad = U.copy().reshape(3, 5, T, T, T)
        bad[1, 0, T // 2, T // 2, T // 2] = np.nan            # density of one interior cell of group 1
        bad = bad.reshape(3, -1)
        dU, dB = torch.from_numpy(bad).cuda(), torch.from_numpy(B).cuda()
        with pytest.raises(mhd.MHDError) as ei:
            gpu.solver.dt_reduce(dU, dB, 3, g, dh, 0.3)
        assert ei.value.code == mhd.ESTATE
        out = gpu.solver.alloc_outputs(3)
        with pytest.raises(mhd.MHDError) as ei:
            gpu.solver.advance_dt(dU, dB, out["U"], out["B"], out["flux"], out["emf"], 3, 1e-3, dh, 0.3)
        assert ei.value.code == mhd.ESTATE
        # the clean batch still works on the same solver afterwards
        dt, smax = gpu.solver.dt_reduce(torch.from_numpy(U).cuda(), dB, 3, g, dh, 0.3)
        assert np.isfinite(dt) and dt > 0 and np.isfinite(smax)


def test_binding_rejects_wrong_dtype_size_and_device():
    import torch
    from paper_1804_03479_b200 import mhd
    U, B, dh = small_batch(2, dtype=np.float64)
    s = mhd.Solver(mhd.make_config(prec=mhd.FP64, max_groups=2))
    dU, dB = torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda()
    out = s.alloc_outputs(2)
    with pytest.raises(TypeError):
        s.advance(dU.float(), dB, out["U"], out["B"], None, None, 2, 1e-3, dh)
    with pytest.raises(ValueError):
        s.advance(dU[:1], dB, out["U"], out["B"], None, None, 2, 1e-3, dh)          # too few elements for 2 groups
    with pytest.raises(ValueError):
        s.advance(torch.from_numpy(U), dB, out["U"], out["B"], None, None, 2, 1e-3, dh)   # host tensor handed to the device call
    with pytest.raises(ValueError):
        s.advance_host(dU, B, np.empty((2, s.n_U_out)), np.empty((2, s.n_B_out)), None, None, 2, 1e-3, dh, 1, 2)   # device tensor to the host call
    s.advance(dU, dB, out["U"], out["B"], None, None, 2, 1e-3, dh)
    torch.cuda.synchronize()
    s.destroy()


@pytest.mark.parametrize("prec,scheme,recon,g", [(0, 0, 0, 3), (1, 0, 0, 3), (0, 1, 1, 4), (1, 1, 1, 4)])
def test_guard_bands_and_run_to_run_determinism(prec, scheme, recon, g):
    """Stand-in for compute-sanitizer memcheck / racecheck, which is closed on this GPU pool (profiles/r02_sanitizers.md):
    (a) every output array sits between guard bands of a sentinel value that must survive the call (an out-of-bounds store of
    the epilogues lands there); the inputs sit at the very end of their allocation with a NaN band in front (an
    out-of-bounds load below the array would poison the result); (b) ten repeated calls give bitwise the same outputs and the
    same dt (an unsynchronised shared-memory hand-off in the plane-marching / pencil kernels shows up as run-to-run noise)."""
    import torch
    from paper_1804_03479_b200 import mhd
    dtp = GU.np_dtype(prec)
    G, PAD = 9, 4096
    U, B, dh = small_batch(G, g=g, dtype=dtp)
    s = mhd.Solver(mhd.make_config(N=16, g=g, scheme=scheme, recon=recon, prec=prec, max_groups=G))
    tdt = torch.float32 if prec == 0 else torch.float64

    def banded(n, fill):
        t = torch.full((PAD + n + PAD,), fill, dtype=tdt, device="cuda")
        return t, t[PAD:PAD + n]
    inU_all = torch.full((PAD + U.size,), float("nan"), dtype=tdt, device="cuda"); inU = inU_all[PAD:]; inU.copy_(torch.from_numpy(U.ravel()))
    inB_all = torch.full((PAD + B.size,), float("nan"), dtype=tdt, device="cuda"); inB = inB_all[PAD:]; inB.copy_(torch.from_numpy(B.ravel()))
    SENT = 12345.0
    bufs = {k: banded(G * n, SENT) for k, n in (("U", s.n_U_out), ("B", s.n_B_out), ("flux", s.n_flux), ("emf", s.n_emf))}
    ref = None
    for rep in range(10):
        for _, v in bufs.values():
            v.fill_(-1.0)
        dt, sm = s.advance_dt(inU, inB, bufs["U"][1], bufs["B"][1], bufs["flux"][1], bufs["emf"][1], G, 2e-3, dh, 0.3)
        got = {k: v[1].cpu().numpy().copy() for k, v in bufs.items()}
        got["dt"] = np.array([dt, sm])
        for k, (full, view) in bufs.items():
            assert bool((full[:PAD] == SENT).all()) and bool((full[-PAD:] == SENT).all()), (k, "guard band overwritten")
            assert np.isfinite(got[k]).all() and not (got[k] == -1.0).all(), k
        if ref is None:
            ref = got
        for k in ref:
            assert np.array_equal(ref[k], got[k]), (rep, k)
    s.destroy()


@pytest.mark.parametrize("prec", [1, 0])
def test_march_chunks_give_the_same_bits(prec, monkeypatch):
    """A small batch of the standard VL group is cut along z into several blocks per group (csrc/mhd_vl_march.cuh) so that it
    still fills the GPU; every chunking gives bitwise the outputs and the CFL speed of the whole-column march."""
    dtp = GU.np_dtype(prec)
    G = 5
    U, B, dh = small_batch(G, g=3, dtype=dtp)
    res = []
    for slots in ("1", "12", "25", "100000"):            # 1, 2, 5 and 10 / 8 chunks per group
        monkeypatch.setenv("MHD_MARCH_SLOTS", slots)
        gpu = GU.GpuRunner(N=16, g=3, scheme=0, recon=0, prec=prec, max_groups=G)
        out, dt, sm = gpu.advance_dt(U, B, 2e-3, dh, 0.3)
        out["dt"] = np.array([dt, sm])
        res.append(out)
    monkeypatch.delenv("MHD_MARCH_SLOTS")
    for r in res[1:]:
        for k in ("U", "B", "flux", "emf", "dt"):
            assert np.array_equal(res[0][k], r[k]), k


@pytest.mark.parametrize("prec", [1, 0])
def test_march_without_tma_and_with_misaligned_inputs_gives_the_same_bits(prec, monkeypatch):
    """The marching kernels stage their input planes by 1-D bulk copies (TMA), which need 16-byte aligned planes.  Input
    arrays that start 4 / 8 bytes off a 16-byte boundary (a view into a larger tensor) take the direct-load instantiation
    of pass 1 and the direct loads of pass 2; so does MHD_NO_TMA=1.  All three give bitwise the same outputs and CFL speed."""
    import torch
    from paper_1804_03479_b200 import mhd
    dtp = GU.np_dtype(prec)
    G = 6
    U, B, dh = small_batch(G, g=3, dtype=dtp)
    s = mhd.Solver(mhd.make_config(N=16, g=3, prec=prec, max_groups=G))

    def run(dU, dB):
        out = s.alloc_outputs(G)
        dt, sm = s.advance_dt(dU, dB, out["U"], out["B"], out["flux"], out["emf"], G, 2e-3, dh, 0.3)
        r = {k: v.cpu().numpy() for k, v in out.items()}
        r["dt"] = np.array([dt, sm])
        return r
    ref = run(torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda())
    # misaligned: element 1 of a larger allocation (cudaMalloc returns 256-byte aligned blocks)
    bigU = torch.empty(U.size + 1, dtype=torch.float32 if prec == 0 else torch.float64, device="cuda")
    bigB = torch.empty(B.size + 1, dtype=bigU.dtype, device="cuda")
    mU, mB = bigU[1:], bigB[1:]
    mU.copy_(torch.from_numpy(U.ravel())); mB.copy_(torch.from_numpy(B.ravel()))
    assert mU.data_ptr() % 16 != 0 and mB.data_ptr() % 16 != 0
    mis = run(mU, mB)
    monkeypatch.setenv("MHD_NO_TMA", "1")
    notma = run(torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda())
    monkeypatch.delenv("MHD_NO_TMA")
    for k in ref:
        assert np.array_equal(ref[k], mis[k]), ("misaligned", k)
        assert np.array_equal(ref[k], notma[k]), ("MHD_NO_TMA", k)
    s.destroy()
