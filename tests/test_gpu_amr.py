"""-m gpu tests of the AMR correction operation: the device restriction / flux
fix-up / EMF fix-up against the numpy oracle (oracle/amr_ref.py) on the same inputs, and the invariants the operation
exists for (composite conservation, div B) with both levels advanced on the device."""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import amr_harness as A
import gpu_util as GU
from oracle import amr_ref

pytestmark = pytest.mark.gpu


class DeviceOps:
    """amr_ref-compatible wrapper (restrict / fixup in place on numpy grids) around the C-ABI calls"""

    def __init__(self, gpu, dtp):
        self.gpu, self.dtp = gpu, dtp

    def _dev(self, a):
        return self.gpu.torch.from_numpy(np.ascontiguousarray(a, dtype=self.dtp)).cuda()

    def _back(self, dev, hosts):
        self.gpu.torch.cuda.synchronize()
        for d, h in zip(dev, hosts):
            h[...] = d.cpu().numpy()

    def restrict(self, U_f, B_f, lo, hi, N, Uc, bxc, byc, bzc):
        dev = [self._dev(a) for a in (Uc, bxc, byc, bzc)]
        self.gpu.solver.amr_restrict(self._dev(U_f), self._dev(B_f), lo, hi, *dev, Uc.shape[1:])
        self._back(dev, (Uc, bxc, byc, bzc))

    def fixup(self, flux_c, emf_c, flux_f, emf_f, lo, hi, N, dt, dh_c, Uc, bxc, byc, bzc, w_c=1.0, w_f=1.0):
        dev = [self._dev(a) for a in (Uc, bxc, byc, bzc)]
        self.gpu.solver.amr_fixup(self._dev(flux_c), self._dev(emf_c), self._dev(flux_f), self._dev(emf_f), lo, hi, dt, dh_c,
                                  *dev, Uc.shape[1:], w_c=w_c, w_f=w_f)
        self._back(dev, (Uc, bxc, byc, bzc))


@pytest.mark.parametrize("prec", [1, 0])
@pytest.mark.parametrize("lo,hi", [((8, 8, 8), (24, 24, 24)), ((8, 16, 8), (16, 24, 24))])
def test_device_correction_matches_the_oracle(prec, lo, hi):
    """restriction and fix-ups on synthetic plane data: element by element against oracle/amr_ref.py"""
    n, N = 32, 16
    dtp = GU.np_dtype(prec)
    rng = np.random.default_rng(5)
    gpu = GU.GpuRunner(N=N, g=3, prec=prec, max_groups=8)
    s = gpu.solver
    nfine = int(np.prod([(hi[d] - lo[d]) // (N // 2) for d in range(3)]))
    grid0 = [rng.normal(size=sh).astype(dtp) for sh in ((5, n, n, n), (n, n, n + 1), (n, n + 1, n), (n + 1, n, n))]
    U_f, B_f = rng.normal(size=(nfine, s.n_U_out)).astype(dtp), rng.normal(size=(nfine, s.n_B_out)).astype(dtp)
    fc, ec = rng.normal(size=(8, s.n_flux)).astype(dtp), rng.normal(size=(8, s.n_emf)).astype(dtp)
    ff, ef = rng.normal(size=(nfine, s.n_flux)).astype(dtp), rng.normal(size=(nfine, s.n_emf)).astype(dtp)
    ref = [a.astype(np.float64) for a in grid0]
    amr_ref.fixup(fc.astype(np.float64), ec.astype(np.float64), ff.astype(np.float64), ef.astype(np.float64), lo, hi, N, 0.01, 1.0 / n,
                  *ref, w_c=0.7, w_f=1.3)
    amr_ref.restrict(U_f.astype(np.float64), B_f.astype(np.float64), lo, hi, N, *ref)
    dev = [a.copy() for a in grid0]
    ops = DeviceOps(gpu, dtp)
    ops.fixup(fc, ec, ff, ef, lo, hi, N, 0.01, 1.0 / n, *dev, w_c=0.7, w_f=1.3)
    ops.restrict(U_f, B_f, lo, hi, N, *dev)
    tol = 1e-14 if prec == 1 else 2e-6
    for a, b in zip(dev, ref):
        assert np.abs(a - b).max() <= tol * max(1.0, np.abs(b).max())
    # cells and faces away from the box and its one-cell neighbourhood are untouched (bitwise)
    far = np.ones((n, n, n), dtype=bool)
    far[lo[2] - 1:hi[2] + 1, lo[1] - 1:hi[1] + 1, lo[0] - 1:hi[0] + 1] = False
    assert np.array_equal(dev[0][:, far], grid0[0][:, far])
    with pytest.raises(gpu.mhd.MHDError):
        ops.restrict(U_f, B_f, (4, 8, 8), hi, N, *dev)                 # not patch-aligned


@pytest.mark.parametrize("scheme,recon,g", [(0, 0, 3), (1, 1, 4)])
def test_two_level_step_on_the_device_conserves_and_stays_divergence_free(scheme, recon, g):
    n, N = 32, 16
    U, bx, by, bz, dh = inputs.random_group_grid(n, 21)
    lo, hi = (8, 8, 8), (24, 24, 24)
    gpu = GU.GpuRunner(N=N, g=g, scheme=scheme, recon=recon, max_groups=8)
    Ui = gpu.torch.from_numpy(U).cuda()
    dt, _ = gpu.solver.grid_dt(Ui, *(gpu.torch.from_numpy(a).cuda() for a in (bx, by, bz)), (n, n, n), 0.5 * dh, 0.3)
    Uf0 = amr_ref.inject(U, bx, by, bz)[0]
    mask = np.ones((n, n, n), dtype=bool); mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = False
    box0 = Uf0[:, 2 * lo[2]:2 * hi[2], 2 * lo[1]:2 * hi[1], 2 * lo[0]:2 * hi[0]]
    tot0 = np.array([U[v][mask].sum() for v in range(5)]) * dh ** 3 + box0.reshape(5, -1).sum(axis=1) * (0.5 * dh) ** 3
    mom = np.abs(U[1:4]).sum() * dh ** 3
    scale = np.array([tot0[0], mom, mom, mom, tot0[4]])
    grid, out_c, out_f, _ = A.two_level_step(gpu, gpu, U, bx, by, bz, lo, hi, N, g, dt, dh, ops=DeviceOps(gpu, np.float64))
    tot1 = A.composite_totals(grid[0], out_f["U"], lo, hi, N, dh)
    assert np.all(np.abs(tot1 - tot0) / scale < 1e-13), (tot1 - tot0) / scale
    assert H.rel_divb(grid[1], grid[2], grid[3], dh) < 1e-13


@pytest.mark.parametrize("prec", [1, 0])
@pytest.mark.parametrize("lo,hi", [((2, 3, 4), (8, 7, 10)), ((0, 0, 0), (16, 16, 16)), ((13, 0, 5), (16, 2, 6))])
def test_device_prolongation_matches_the_oracle(prec, lo, hi):
    """NEXT-3: new fine grids on the device (closed-form coefficients) against oracle/amr_ref.prolong
    (numerical solve of the interface + divergence conditions), element by element; the box may touch the periodic rim"""
    n = 16
    dtp = GU.np_dtype(prec)
    U, bx, by, bz, dh = inputs.random_group_grid(n, 4)
    coarse = [np.ascontiguousarray(a, dtype=dtp) for a in (U, bx, by, bz)]
    ref = amr_ref.prolong(*[a.astype(np.float64) for a in coarse], lo, hi)
    assert ref[4] < 1e-12 if prec == 1 else True        # FP32-rounded coarse faces are divergence-free to 1e-7 only
    gpu = GU.GpuRunner(N=16, g=3, prec=prec, max_groups=1)
    t = gpu.torch
    out = [t.full(a.shape, float("nan"), dtype=t.float64 if prec == 1 else t.float32, device="cuda") for a in ref[:4]]
    gpu.solver.amr_prolong(*[t.from_numpy(a).cuda() for a in coarse], (n, n, n), lo, hi, *out)
    t.cuda.synchronize()
    out = [o.cpu().numpy().astype(np.float64) for o in out]
    tol = 1e-13 if prec == 1 else 2e-6
    for a, b in zip(out, ref[:4]):
        assert not np.isnan(a).any()
        assert np.abs(a - b).max() <= tol * np.abs(b).max()
    div = (out[1][:, :, 1:] - out[1][:, :, :-1]) + (out[2][:, 1:, :] - out[2][:, :-1, :]) + (out[3][1:] - out[3][:-1])
    assert np.abs(div).max() < (1e-13 if prec == 1 else 2e-5) * np.abs(bx).max() * n
    with pytest.raises(gpu.mhd.MHDError):
        gpu.solver.amr_prolong(*[t.from_numpy(a).cuda() for a in coarse], (n, n, n), (0, 0, 0), (17, 4, 4), *out)


def test_prolongation_then_restriction_returns_the_coarse_data():
    """the two AMR operators are consistent: restricting freshly prolonged data gives back the coarse cells and faces"""
    n, N = 32, 16
    lo, hi = (8, 8, 8), (24, 16, 24)
    U, bx, by, bz, dh = inputs.random_group_grid(n, 9)
    gpu = GU.GpuRunner(N=N, g=3, prec=1, max_groups=8)
    t = gpu.torch
    nb = [hi[d] - lo[d] for d in range(3)]
    shapes = [(5, 2 * nb[2], 2 * nb[1], 2 * nb[0]), (2 * nb[2], 2 * nb[1], 2 * nb[0] + 1), (2 * nb[2], 2 * nb[1] + 1, 2 * nb[0]),
              (2 * nb[2] + 1, 2 * nb[1], 2 * nb[0])]
    fine = [t.empty(s, dtype=t.float64, device="cuda") for s in shapes]
    dev = [t.from_numpy(a).cuda() for a in (U, bx, by, bz)]
    gpu.solver.amr_prolong(*dev, (n, n, n), lo, hi, *fine)
    t.cuda.synchronize()
    Uf, bxf, byf, bzf = [f.cpu().numpy() for f in fine]
    # cut the fine box into patch groups (z outermost, x fastest) in the U_out / B_out layout
    mf = [2 * nb[d] // N for d in range(3)]
    U_f, B_f = [], []
    for gz in range(mf[2]):
        for gy in range(mf[1]):
            for gx in range(mf[0]):
                sz, sy, sx = slice(gz * N, gz * N + N), slice(gy * N, gy * N + N), slice(gx * N, gx * N + N)
                U_f.append(Uf[:, sz, sy, sx].ravel())
                B_f.append(np.concatenate([bxf[sz, sy, gx * N:gx * N + N + 1].ravel(), byf[sz, gy * N:gy * N + N + 1, sx].ravel(),
                                           bzf[gz * N:gz * N + N + 1, sy, sx].ravel()]))
    scr = [t.from_numpy(np.full_like(a, 7.0)).cuda() for a in (U, bx, by, bz)]
    gpu.solver.amr_restrict(t.from_numpy(np.array(U_f)).cuda(), t.from_numpy(np.array(B_f)).cuda(), lo, hi, *scr, (n, n, n))
    t.cuda.synchronize()
    box = (slice(lo[2], hi[2]), slice(lo[1], hi[1]), slice(lo[0], hi[0]))
    assert np.abs(scr[0].cpu().numpy()[(slice(None),) + box] - U[(slice(None),) + box]).max() < 1e-14 * np.abs(U).max()
    assert np.abs(scr[1].cpu().numpy()[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0] + 1] - bx[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0] + 1]).max() < 1e-14
    assert np.abs(scr[3].cpu().numpy()[lo[2]:hi[2] + 1, lo[1]:hi[1], lo[0]:hi[0]] - bz[lo[2]:hi[2] + 1, lo[1]:hi[1], lo[0]:hi[0]]).max() < 1e-14
