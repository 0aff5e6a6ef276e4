"""mhd_dt_reduce_noalloc (include/mhd.h): the CFL reduction for callers that cannot allocate -- scratch in a fixed array of the
library's device image, no solver object, result left on the device.  Compared with the existing path (mhd_dt_reduce, solver-owned
scratch) on two calls in a row: maxima are exact, so dt and maxspeed must have the same bits.  This file is collected last on
purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the other GPU tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GAMMA, MIN_DENS, MIN_PRES = 5.0 / 3.0, 1e-10, 1e-10


def _batch(G, N, g, seed, vamp, dtype):
    """G groups in the U_in / B_in layout (g ghost cells): positive density and pressure, velocities of scale vamp"""
    rng = np.random.default_rng(seed)
    T = N + 2 * g
    rho = rng.uniform(0.5, 2.0, (G, T, T, T))
    v = vamp * rng.standard_normal((G, 3, T, T, T))
    bx = rng.standard_normal((G, T, T, T + 1)) * 0.5
    by = rng.standard_normal((G, T, T + 1, T)) * 0.5
    bz = rng.standard_normal((G, T + 1, T, T)) * 0.5
    bc2 = (0.5 * (bx[..., 1:] + bx[..., :-1])) ** 2 + (0.5 * (by[:, :, 1:] + by[:, :, :-1])) ** 2 + (0.5 * (bz[:, 1:] + bz[:, :-1])) ** 2
    e = rng.uniform(0.3, 1.5, rho.shape) / (GAMMA - 1.0) + 0.5 * rho * (v ** 2).sum(1) + 0.5 * bc2
    U = np.stack([rho, rho * v[:, 0], rho * v[:, 1], rho * v[:, 2], e], axis=1)
    B = np.concatenate([bx.reshape(G, -1), by.reshape(G, -1), bz.reshape(G, -1)], axis=1)
    return np.ascontiguousarray(U.reshape(G, -1), dtype=dtype), np.ascontiguousarray(B, dtype=dtype)


@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("N,g", [(16, 3), (16, 0), (8, 4)])
def test_noalloc_dt_has_the_bits_of_mhd_dt_reduce_on_two_calls_in_a_row(prec, N, g):
    import torch
    from paper_1804_03479_b200 import mhd
    dtype = np.float32 if prec == 0 else np.float64
    # the existing path needs a solver (any scheme: the reduction does not depend on it); its arrays have 0 or the solver's ghost width
    solver = mhd.Solver(mhd.make_config(N=N, g=g if g else 3, prec=prec, gamma=GAMMA, min_dens=MIN_DENS, min_pres=MIN_PRES, max_groups=64))
    dh, cfl = 1.0 / 128, 0.3
    out = torch.full((2,), -7.0, dtype=torch.float64, device="cuda")
    # the second call has FEWER blocks and SMALLER speeds than the first: anything left in the shared scratch by the first call
    # (its slots, its counter) would show up as the first call's larger maximum
    results = []
    for G, seed, vamp in ((37, 11, 3.0), (5, 12, 0.05)):
        U, B = _batch(G, N, g, seed, vamp, dtype)
        dU, dB = torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda()
        ref_dt, ref_speed = solver.dt_reduce(dU, dB, G, g, dh, cfl)
        out.fill_(-7.0)
        mhd.dt_reduce_noalloc(prec, dU, dB, G, N, g, GAMMA, MIN_DENS, MIN_PRES, dh, cfl, out)
        got = out.cpu().numpy()
        assert np.isfinite(ref_speed) and ref_speed > 0
        assert got[1] == ref_speed and got[0] == ref_dt, (G, got, ref_dt, ref_speed)      # bit for bit
        results.append(ref_speed)
    assert results[1] < 0.5 * results[0]                       # the sequence really is "large, then small"
    # and the same call repeated gives the same answer (the counter is cleared per call)
    out.fill_(-7.0)
    mhd.dt_reduce_noalloc(prec, dU, dB, 5, N, g, GAMMA, MIN_DENS, MIN_PRES, dh, cfl, out)
    assert out.cpu().numpy()[1] == results[1]


def test_noalloc_rejects_sizes_beyond_the_fixed_scratch_and_bad_arguments():
    import torch
    from paper_1804_03479_b200 import mhd
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    U, B = _batch(1, 16, 0, 3, 0.1, np.float32)
    dU, dB = torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda()
    args = (GAMMA, MIN_DENS, MIN_PRES, 0.01, 0.3, out)
    assert mhd.NOALLOC_MAX_BLOCKS == 65536
    for G in (mhd.NOALLOC_MAX_BLOCKS // 16 + 1, 70000):      # 16 blocks per group of 16^3: 4097 groups need 65552 slots
        with pytest.raises(mhd.MHDError) as ei:
            mhd.dt_reduce_noalloc(0, dU, dB, G, 16, 0, *args)
        assert ei.value.code == mhd.ELIMIT and "MHD_NOALLOC_MAX_BLOCKS" in str(ei.value)
    raw = mhd.lib().mhd_dt_reduce_noalloc                      # past the binding's size checks: the library's own argument checks
    pU, pB, pO = dU.data_ptr(), dB.data_ptr(), out.data_ptr()
    for bad in (dict(ngroups=0), dict(ps2=7), dict(ps2=66), dict(nghost=9), dict(nghost=-1), dict(prec=2), dict(U=None), dict(out=None)):
        rc = raw(bad.get("prec", 0), bad.get("U", pU), pB, bad.get("ngroups", 1), bad.get("ps2", 16), bad.get("nghost", 0), GAMMA, MIN_DENS,
                 MIN_PRES, 0.01, 0.3, bad.get("out", pO), None)
        assert rc == mhd.EINVAL, bad
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0                       # nothing was launched
    # the largest size that fits: 4096 groups of 16^3 (65536 blocks), uniform state -> every slot holds the same speed
    G = mhd.NOALLOC_MAX_BLOCKS // 16
    dU4, dB4 = dU.repeat(G, 1), dB.repeat(G, 1)
    mhd.dt_reduce_noalloc(0, dU4, dB4, G, 16, 0, *args)
    one = torch.zeros(2, dtype=torch.float64, device="cuda")
    mhd.dt_reduce_noalloc(0, dU, dB, 1, 16, 0, GAMMA, MIN_DENS, MIN_PRES, 0.01, 0.3, one)
    assert torch.equal(out, one) and float(one[1]) > 0


def test_noalloc_nan_state_reports_an_infinite_speed_and_zero_dt():
    import torch
    from paper_1804_03479_b200 import mhd
    U, B = _batch(3, 16, 3, 5, 0.1, np.float64)
    U[1, 12345] = np.nan
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    mhd.dt_reduce_noalloc(1, torch.from_numpy(U).cuda(), torch.from_numpy(B).cuda(), 3, 16, 3, GAMMA, MIN_DENS, MIN_PRES, 0.01, 0.3, out)
    got = out.cpu().numpy()
    assert np.isinf(got[1]) and got[0] == 0.0
