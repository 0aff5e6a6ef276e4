"""-m gpu tests of the device-side preparation / closing steps for a uniform periodic grid and of
multi-step runs that stay on the device (BASELINE configs 1, 3, 4: parity at step 10, invariants at steps 100 / 200)."""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import gpu_util as GU

pytestmark = pytest.mark.gpu


def to_dev(arrs, dtp):
    import torch
    return [torch.from_numpy(np.ascontiguousarray(a, dtype=dtp)).cuda() for a in arrs]


def random_grid(shape, seed, dtp):
    """generic (not divergence-free: pure data movement test) fields on an (nz, ny, nx) periodic grid"""
    nz, ny, nx = shape
    rng = np.random.default_rng(seed)
    U = rng.normal(size=(5, nz, ny, nx))
    bx = rng.normal(size=(nz, ny, nx + 1)); bx[:, :, nx] = bx[:, :, 0]
    by = rng.normal(size=(nz, ny + 1, nx)); by[:, ny, :] = by[:, 0, :]
    bz = rng.normal(size=(nz + 1, ny, nx)); bz[nz, :, :] = bz[0, :, :]
    return [a.astype(dtp) for a in (U, bx, by, bz)]


@pytest.mark.parametrize("prec", [1, 0])
@pytest.mark.parametrize("N,g,shape", [(16, 3, (16, 48, 32)), (16, 4, (32, 16, 16)), (8, 4, (24, 8, 16))])
def test_pack_and_unpack_are_bitwise_the_host_preparation(prec, N, g, shape):
    import torch
    dtp = GU.np_dtype(prec)
    U, bx, by, bz = random_grid(shape, 7, dtp)
    Ui_ref, Bi_ref = inputs.pack_groups(U, bx, by, bz, N, g, dtp)
    G = Ui_ref.shape[0]
    gpu = GU.GpuRunner(N=N, g=g, scheme=(1 if g == 4 else 0), recon=(1 if g == 4 else 0), prec=prec, max_groups=G)
    s = gpu.solver
    dU, dbx, dby, dbz = to_dev((U, bx, by, bz), dtp)
    Ui = torch.empty((G, s.n_U_in), dtype=s.torch_dtype, device="cuda")
    Bi = torch.empty((G, s.n_B_in), dtype=s.torch_dtype, device="cuda")
    s.grid_pack(dU, dbx, dby, dbz, shape, Ui, Bi)
    torch.cuda.synchronize()
    assert np.array_equal(Ui.cpu().numpy(), Ui_ref) and np.array_equal(Bi.cpu().numpy(), Bi_ref)
    # closing: scatter synthetic "outputs" back and compare with the host routine
    rng = np.random.default_rng(3)
    Uo = rng.normal(size=(G, s.n_U_out)).astype(dtp)
    Bo = rng.normal(size=(G, s.n_B_out)).astype(dtp)
    Un, bxn, byn, bzn, _ = inputs.unpack_groups(Uo, Bo, shape, N)
    out = [torch.full_like(t, 9.0) for t in (dU, dbx, dby, dbz)]
    s.grid_unpack(torch.from_numpy(Uo).cuda(), torch.from_numpy(Bo).cuda(), shape, *out)
    torch.cuda.synchronize()
    for a, b in zip(out, (Un, bxn, byn, bzn)):
        assert np.array_equal(a.cpu().numpy(), b)
    with pytest.raises(gpu.mhd.MHDError):
        s.grid_pack(dU, dbx, dby, dbz, (shape[0] + 1, shape[1], shape[2]), Ui, Bi)      # not a multiple of ps2


def device_run(gpu, grid, shape, dh, nsteps, cfl=0.3, dts=None):
    """nsteps of mhd_grid_dt + mhd_grid_advance entirely on the device; returns the dt sequence used"""
    used = []
    for n in range(nsteps):
        dt = dts[n] if dts is not None else gpu.solver.grid_dt(*grid, shape, dh, cfl)[0]
        gpu.solver.grid_advance(*grid, shape, dt, dh)
        used.append(dt)
    gpu.torch.cuda.synchronize()
    return used


@pytest.mark.parametrize("prec", [1, 0])
@pytest.mark.parametrize("N,g,scheme,recon", [(16, 3, 0, 0), (8, 4, 1, 1)])
def test_grid_advance_dt_is_the_two_calls_bitwise(prec, N, g, scheme, recon):
    """mhd_grid_advance_dt: the dt of the next step comes out of the final update; same bits as mhd_grid_advance + mhd_grid_dt"""
    n = 2 * N
    dtp = GU.np_dtype(prec)
    U, bx, by, bz, dh = inputs.abc_grid(n, seed=1806, p0=0.15, vamp=1e-2)
    gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, prec=prec, max_groups=8)
    a, b = to_dev((U, bx, by, bz), dtp), to_dev((U, bx, by, bz), dtp)
    shape = (n, n, n)
    dt = gpu.solver.grid_dt(*a, shape, dh, 0.3)[0]
    for _ in range(5):
        gpu.solver.grid_advance(*a, shape, dt, dh)
        dt_a, s_a = gpu.solver.grid_dt(*a, shape, dh, 0.3)
        dt_b, s_b = gpu.solver.grid_advance_dt(*b, shape, dt, dh, 0.3)
        assert (dt_a, s_a) == (dt_b, s_b)
        dt = dt_b
    for x, y in zip(a, b):
        assert gpu.torch.equal(x, y)


def test_config1_on_the_device_equals_the_host_prepared_path_and_the_oracle(oracle):
    n, N, g = 32, 16, 3
    U, bx, by, bz, dh = inputs.abc_grid(n, seed=1804, p0=1.0, vamp=1e-3)
    cfg = oracle.make_config(N=N, g=g)
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    c0 = oracle.make_config(N=n, g=3)
    ref, dts = (U, bx, by, bz), []
    for _ in range(10):
        Ui, Bi = inputs.pack_groups(*ref, n, 0)
        dt, _ = oracle.dt_reduce(c0, Ui, Bi, 0, dh, 0.3)
        dts.append(dt)
        ref = H.step_grid(adv, *ref, dt, dh, N, g)[:4]
    gpu = GU.GpuRunner(N=N, g=g, max_groups=8)
    grid = to_dev((U, bx, by, bz), np.float64)
    dt_dev = device_run(gpu, grid, (n, n, n), dh, 10)                    # the device's own CFL steps
    assert np.allclose(dt_dev, dts, rtol=1e-12, atol=0)
    res = [t.cpu().numpy() for t in grid]
    errs = {k: H.field_err(a, b) for k, a, b in zip(("U", "bx", "by", "bz"), res, ref)}
    assert max(errs.values()) <= 1e-11, errs
    # bitwise equal to the same kernels fed by the host preparation (numpy pack / unpack), same dt sequence
    host = (U, bx, by, bz)
    for dt in dt_dev:
        host = H.step_grid(gpu, *host, dt, dh, N, g)[:4]
    for a, b in zip(res, host):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("which,nsteps", [("abc", 100), ("blast", 200)])
def test_configs_3_4_long_runs_keep_the_invariants(which, nsteps):
    """CTU+PPM+HLLD+CT, FP64, 64^3 (what a test can afford), 100 / 200 steps at CFL 0.3 on the device: mass and energy
    conserved and div B at round-off at the END of the run (Eq. 16), density positive."""
    n, N, g = 64, 16, 4
    if which == "abc":
        U, bx, by, bz, dh = inputs.abc_grid(n, seed=1805, p0=0.15, vamp=1e-2)
    else:
        U, bx, by, bz, dh = inputs.blast_grid(n)
    gpu = GU.GpuRunner(N=N, g=g, scheme=1, recon=1, max_groups=64)
    grid = to_dev((U, bx, by, bz), np.float64)
    dts = device_run(gpu, grid, (n, n, n), dh, nsteps)
    Un, bxn, byn, bzn = [t.cpu().numpy() for t in grid]
    assert np.all(np.isfinite(Un)) and Un[0].min() > 0
    t0, t1 = H.totals(U), H.totals(Un)
    assert abs(t1[0] - t0[0]) / t0[0] < 1e-12 and abs(t1[4] - t0[4]) / t0[4] < 1e-12
    scale = np.abs(Un[1:4]).sum()
    assert np.all(np.abs(t1[1:4] - t0[1:4]) / scale < 1e-12)
    assert H.rel_divb(bxn, byn, bzn, dh) < 1e-13
    assert np.array_equal(bxn[:, :, n], bxn[:, :, 0]) and np.array_equal(bzn[n], bzn[0])
    assert min(dts) > 0 and sum(dts) > 0
    if which == "abc":
        assert gpu.stats() == (0, 0, 0)                  # no floor events expected on config 3 (R9)
        eb0 = 0.5 * sum(np.mean(a ** 2) for a in (bx[:, :, :n], by[:, :n, :], bz[:n]))
        eb1 = 0.5 * sum(np.mean(a ** 2) for a in (bxn[:, :, :n], byn[:, :n, :], bzn[:n]))
        assert 0.9 * eb0 < eb1 <= eb0 * (1 + 1e-12)      # the force-free field only relaxes: magnetic energy decays slowly
