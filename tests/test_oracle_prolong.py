"""Pins of the prolongation oracle (oracle/amr_ref.prolong): what the paper states the interpolation
does -- "maintain a divergence-free magnetic field", "the average of fine magnetic field values is the same as the coarse
value", conservative for the conserved variables -- plus exactness on affine fields, the paper's own 2-D system (Eq. 17,
10 coefficients) as the z-invariant special case, and covariance under a cyclic permutation of the axes."""
import numpy as np

from paper_1804_03479_b200 import inputs
from oracle import amr_ref


def fine_div(bxf, byf, bzf):
    return (bxf[:, :, 1:] - bxf[:, :, :-1]) + (byf[:, 1:, :] - byf[:, :-1, :]) + (bzf[1:] - bzf[:-1])


def test_fine_field_is_divergence_free_and_averages_to_the_coarse_one():
    U, bx, by, bz, dh = inputs.random_group_grid(16, 4)
    lo, hi = (2, 3, 4), (8, 7, 10)
    Uf, bxf, byf, bzf, res = amr_ref.prolong(U, bx, by, bz, lo, hi)
    assert res < 1e-12                                              # the 22 equations are consistent: 21 independent
    assert not any(np.isnan(a).any() for a in (Uf, bxf, byf, bzf))  # every fine face is set
    assert np.abs(fine_div(bxf, byf, bzf)).max() < 1e-13 * np.abs(bx).max() * 16
    # area average of the four fine faces on a coarse face = the coarse face value
    ax = 0.25 * (bxf[0::2, 0::2, 0::2] + bxf[1::2, 0::2, 0::2] + bxf[0::2, 1::2, 0::2] + bxf[1::2, 1::2, 0::2])
    assert np.abs(ax - bx[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0] + 1]).max() < 1e-14
    ay = 0.25 * (byf[0::2, 0::2, 0::2] + byf[1::2, 0::2, 0::2] + byf[0::2, 0::2, 1::2] + byf[1::2, 0::2, 1::2])
    assert np.abs(ay - by[lo[2]:hi[2], lo[1]:hi[1] + 1, lo[0]:hi[0]]).max() < 1e-14
    az = 0.25 * (bzf[0::2, 0::2, 0::2] + bzf[0::2, 1::2, 0::2] + bzf[0::2, 0::2, 1::2] + bzf[0::2, 1::2, 1::2])
    assert np.abs(az - bz[lo[2]:hi[2] + 1, lo[1]:hi[1], lo[0]:hi[0]]).max() < 1e-14
    # conservative: the mean of the eight fine cells = the coarse cell
    m = sum(Uf[:, dz::2, dy::2, dx::2] for dz in (0, 1) for dy in (0, 1) for dx in (0, 1)) / 8
    assert np.abs(m - U[:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]]).max() < 1e-14
    # the interpolation does interpolate: fine values differ from plain injection
    assert np.abs(bxf[:, :, 1::2] - 0.5 * (bxf[:, :, 0:-1:2] + bxf[:, :, 2::2])).max() > 1e-3


def test_affine_divergence_free_field_is_reproduced_exactly():
    n = 12
    c = (np.arange(n) + 0.5)
    f = np.arange(n + 1) * 1.0
    # B = B0 + G r with trace(G) = 0, coordinates in coarse cells
    B0 = np.array([0.3, -0.7, 1.1])
    G = np.array([[0.05, 0.02, -0.03], [0.01, -0.08, 0.04], [-0.02, 0.06, 0.03]])
    Z, Y, X = np.meshgrid(c, c, f, indexing="ij"); bx = B0[0] + G[0, 0] * X + G[0, 1] * Y + G[0, 2] * Z
    Z, Y, X = np.meshgrid(c, f, c, indexing="ij"); by = B0[1] + G[1, 0] * X + G[1, 1] * Y + G[1, 2] * Z
    Z, Y, X = np.meshgrid(f, c, c, indexing="ij"); bz = B0[2] + G[2, 0] * X + G[2, 1] * Y + G[2, 2] * Z
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    U = np.stack([2.0 + 0.1 * X - 0.05 * Y + 0.02 * Z] * 5)
    lo, hi = (3, 4, 2), (7, 8, 9)                                   # two cells away from the (non-periodic) rim
    Uf, bxf, byf, bzf, res = amr_ref.prolong(U, bx, by, bz, lo, hi)
    cf = lambda l, m: l + (np.arange(2 * m) + 0.5) * 0.5            # fine cell centres / face positions in coarse units
    ff = lambda l, m: l + np.arange(2 * m + 1) * 0.5
    nb = [hi[d] - lo[d] for d in range(3)]
    Z, Y, X = np.meshgrid(cf(lo[2], nb[2]), cf(lo[1], nb[1]), ff(lo[0], nb[0]), indexing="ij")
    assert np.abs(bxf - (B0[0] + G[0, 0] * X + G[0, 1] * Y + G[0, 2] * Z)).max() < 1e-13
    Z, Y, X = np.meshgrid(cf(lo[2], nb[2]), ff(lo[1], nb[1]), cf(lo[0], nb[0]), indexing="ij")
    assert np.abs(byf - (B0[1] + G[1, 0] * X + G[1, 1] * Y + G[1, 2] * Z)).max() < 1e-13
    Z, Y, X = np.meshgrid(ff(lo[2], nb[2]), cf(lo[1], nb[1]), cf(lo[0], nb[0]), indexing="ij")
    assert np.abs(bzf - (B0[2] + G[2, 0] * X + G[2, 1] * Y + G[2, 2] * Z)).max() < 1e-13
    Z, Y, X = np.meshgrid(cf(lo[2], nb[2]), cf(lo[1], nb[1]), cf(lo[0], nb[0]), indexing="ij")
    assert np.abs(Uf[0] - (2.0 + 0.1 * X - 0.05 * Y + 0.02 * Z)).max() < 1e-13


def paper_2d_interior(bxm, bxp, sxm, sxp, bym, byp, sym, syp):
    """PAPER.md:213-219 literally: the 10 coefficients of Eq. 17 from the eight interface conditions (values and in-face
    slopes of Bx at x = -+1/2 and of By at y = -+1/2) and the three divergence conditions; returns the four interior
    values (9)-(12): Bx(0, -+1/4) and By(-+1/4, 0)."""
    # unknowns: a0 ax ay axx axy b0 bx by byy bxy
    rows, rhs = [], []
    for x, val, sl in ((-0.5, bxm, sxm), (0.5, bxp, sxp)):
        rows.append([1, x, 0, x * x, 0, 0, 0, 0, 0, 0]); rhs.append(val)          # Bx(x, 0)
        rows.append([0, 0, 1, 0, x, 0, 0, 0, 0, 0]); rhs.append(sl)               # dBx/dy (x, 0)
    for y, val, sl in ((-0.5, bym, sym), (0.5, byp, syp)):
        rows.append([0, 0, 0, 0, 0, 1, 0, y, y * y, 0]); rhs.append(val)          # By(0, y)
        rows.append([0, 0, 0, 0, 0, 0, 1, 0, 0, y]); rhs.append(sl)               # dBy/dx (0, y)
    rows.append([0, 1, 0, 0, 0, 0, 0, 1, 0, 0]); rhs.append(0.0)                  # ax + by = 0
    rows.append([0, 0, 0, 2, 0, 0, 0, 0, 0, 1]); rhs.append(0.0)                  # 2 axx + bxy = 0
    rows.append([0, 0, 0, 0, 1, 0, 0, 0, 2, 0]); rhs.append(0.0)                  # axy + 2 byy = 0
    q, *_ = np.linalg.lstsq(np.array(rows, dtype=float), np.array(rhs), rcond=None)
    a0, ax, ay, axx, axy, b0, bx, by, byy, bxy = q
    return [a0 + ay * y for y in (-0.25, 0.25)], [b0 + bx * x for x in (-0.25, 0.25)]


def test_z_invariant_field_reduces_to_the_papers_2d_system():
    n = 8
    rng = np.random.default_rng(3)
    # 2-D divergence-free face field from a vector potential Az(x, y) on the coarse nodes, replicated along z
    Az = rng.normal(size=(n, n))
    bx2 = np.roll(Az, -1, axis=0) - Az                               # Bx(i, j) =  dAz/dy   [j][i]
    by2 = -(np.roll(Az, -1, axis=1) - Az)                            # By(i, j) = -dAz/dx
    bx = np.empty((n, n, n + 1)); bx[:, :, :n] = bx2[None]; bx[:, :, n] = bx2[None, :, 0]
    by = np.empty((n, n + 1, n)); by[:, :n, :] = by2[None]; by[:, n, :] = by2[None, 0, :]
    bz = np.full((n + 1, n, n), 0.4)
    U = np.ones((5, n, n, n))
    lo, hi = (2, 2, 2), (6, 6, 4)
    Uf, bxf, byf, bzf, res = amr_ref.prolong(U, bx, by, bz, lo, hi)
    assert np.abs(bzf - 0.4).max() < 1e-14 and np.abs(bxf[0] - bxf[-1]).max() < 1e-14
    P = lambda a, i, j: a[j % n, i % n]
    worst = 0.0
    for j in range(lo[1], hi[1]):
        for i in range(lo[0], hi[0]):
            sx = [amr_ref.mc(P(bx2, ii, j + 1) - P(bx2, ii, j), P(bx2, ii, j) - P(bx2, ii, j - 1)) for ii in (i, i + 1)]
            sy = [amr_ref.mc(P(by2, i + 1, jj) - P(by2, i, jj), P(by2, i, jj) - P(by2, i - 1, jj)) for jj in (j, j + 1)]
            ix, iy = paper_2d_interior(P(bx2, i, j), P(bx2, i + 1, j), sx[0], sx[1], P(by2, i, j), P(by2, i, j + 1), sy[0], sy[1])
            fi, fj = 2 * (i - lo[0]), 2 * (j - lo[1])
            worst = max(worst, abs(bxf[0, fj, fi + 1] - ix[0]), abs(bxf[0, fj + 1, fi + 1] - ix[1]),
                        abs(byf[0, fj + 1, fi] - iy[0]), abs(byf[0, fj + 1, fi + 1] - iy[1]))
    assert worst < 1e-13


def test_cyclic_permutation_of_the_axes():
    """relabelling (x, y, z) -> (y, z, x) of the input relabels the output"""
    U, bx, by, bz, dh = inputs.random_group_grid(8, 11)
    lo, hi = (1, 2, 3), (4, 6, 5)
    Uf, bxf, byf, bzf, _ = amr_ref.prolong(U, bx, by, bz, lo, hi)
    # new axes (x', y', z') = (y, z, x): arrays are [z][y][x] -> [z'][y'][x'] = [x][z][y]
    T = lambda a: np.ascontiguousarray(a.transpose(2, 0, 1))
    U2 = np.stack([T(U[0]), T(U[2]), T(U[3]), T(U[1]), T(U[4])])
    lo2, hi2 = (lo[1], lo[2], lo[0]), (hi[1], hi[2], hi[0])
    Vf, cxf, cyf, czf, _ = amr_ref.prolong(U2, T(by), T(bz), T(bx), lo2, hi2)
    assert np.abs(cxf - T(byf)).max() < 1e-13 and np.abs(cyf - T(bzf)).max() < 1e-13 and np.abs(czf - T(bxf)).max() < 1e-13
    assert np.abs(Vf[0] - T(Uf[0])).max() < 1e-14 and np.abs(Vf[1] - T(Uf[2])).max() < 1e-14
