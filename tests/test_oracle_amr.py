"""Pins of the correction-operation oracle (oracle/amr_ref.py) against what the paper says the operation is FOR
(PAPER.md:207): "These corrections are necessary to preserve the conservation law of conserved variables and the
divergence-free constraint on the magnetic field."  Static two-level mesh, CPU oracle solver on both levels."""
import numpy as np
import pytest

from paper_1804_03479_b200 import inputs
import harness as H
import amr_harness as A
from oracle import amr_ref


def setup(oracle, scheme, recon, g, seed=21, lo=(8, 8, 8), hi=(24, 24, 24)):
    n, N = 32, 16
    U, bx, by, bz, dh = inputs.random_group_grid(n, seed)
    cfg = oracle.make_config(N=N, g=g, scheme=scheme, recon=recon)
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    # refined box lo..hi: patch-aligned, interior of the periodic domain
    Ui, Bi = inputs.pack_groups(U, bx, by, bz, n, 0)
    dt, _ = oracle.dt_reduce(oracle.make_config(N=n, g=3), Ui, Bi, 0, 0.5 * dh, 0.3)       # CFL of the fine level
    return n, N, U, bx, by, bz, dh, adv, lo, hi, dt


def test_injection_is_divergence_free_and_conservative():
    U, bx, by, bz, dh = inputs.random_group_grid(16, 4)
    Uf, bxf, byf, bzf = amr_ref.inject(U, bx, by, bz)
    assert H.rel_divb(bxf, byf, bzf, 0.5 * dh) < 1e-13
    assert np.allclose(Uf.reshape(5, -1).sum(axis=1) / 8, U.reshape(5, -1).sum(axis=1), rtol=1e-14)
    assert np.array_equal(bxf[:, :, ::2][::2, ::2], bx)          # fine faces on coarse faces carry the coarse value


@pytest.mark.parametrize("scheme,recon,g,lo,hi", [(0, 0, 3, (8, 8, 8), (24, 24, 24)), (1, 1, 4, (8, 8, 8), (24, 24, 24)),
                                                  (0, 0, 3, (8, 16, 8), (16, 24, 24))])      # last: 1 x 1 x 2 fine groups
def test_correction_restores_conservation_and_div_b(oracle, scheme, recon, g, lo, hi):
    n, N, U, bx, by, bz, dh, adv, lo, hi, dt = setup(oracle, scheme, recon, g, lo=lo, hi=hi)
    Uf0 = amr_ref.inject(U, bx, by, bz)[0]
    box0 = Uf0[:, 2 * lo[2]:2 * hi[2], 2 * lo[1]:2 * hi[1], 2 * lo[0]:2 * hi[0]]
    mask = np.ones((n, n, n), dtype=bool); mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = False
    tot0 = np.array([U[v][mask].sum() for v in range(5)]) * dh ** 3 + box0.reshape(5, -1).sum(axis=1) * (0.5 * dh) ** 3
    scale = np.array([tot0[0], np.abs(U[1:4]).sum() * dh ** 3, np.abs(U[1:4]).sum() * dh ** 3, np.abs(U[1:4]).sum() * dh ** 3, tot0[4]])
    # with the correction: composite totals conserved, coarse div B at round-off everywhere
    grid, out_c, out_f, _ = A.two_level_step(adv, adv, U, bx, by, bz, lo, hi, N, g, dt, dh, correct=True)
    tot1 = A.composite_totals(grid[0], out_f["U"], lo, hi, N, dh)
    assert np.all(np.abs(tot1 - tot0) / scale < 1e-13), (tot1 - tot0) / scale
    assert H.rel_divb(grid[1], grid[2], grid[3], dh) < 1e-13
    # restriction: the covered coarse cells are the volume average of the fine ones
    fineU = np.asarray(out_f["U"]).reshape(-1, 5, N ** 3).sum(axis=(0, 2)) / 8
    assert np.allclose(grid[0][:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]].reshape(5, -1).sum(axis=1), fineU, rtol=1e-13)
    # the test has teeth: restriction alone (no flux / EMF fix-up) breaks both
    g2, oc2, of2, _ = A.two_level_step(adv, adv, U, bx, by, bz, lo, hi, N, g, dt, dh, correct=False)
    amr_ref.restrict(np.asarray(of2["U"]), np.asarray(of2["B"]), lo, hi, N, *g2)
    bad = A.composite_totals(g2[0], of2["U"], lo, hi, N, dh)
    assert np.max(np.abs(bad - tot0) / scale) > 1e-9
    assert H.rel_divb(g2[1], g2[2], g2[3], dh) > 1e-9


def test_uniform_state_needs_no_correction(oracle):
    n, N, g = 32, 16, 3
    o = np.ones((n, n, n))
    bx = np.full((n, n, n + 1), 0.5); by = np.full((n, n + 1, n), -0.3); bz = np.full((n + 1, n, n), 0.9)
    U = inputs.conserved(1.3 * o, 0.4 * o, -0.7 * o, 0.2 * o, 0.8 * o, bx, by, bz)
    cfg = oracle.make_config(N=N, g=g)
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    grid, *_ = A.two_level_step(adv, adv, U, bx, by, bz, (8, 8, 8), (24, 24, 24), N, g, 0.004, 1.0 / n)
    assert np.abs(grid[0] - U).max() < 1e-13 and np.abs(grid[1] - bx).max() < 1e-14


def test_weights_enter_linearly():
    """DESIGN.md section 11 A5 (sub-cycling weights): the fine planes of two sub-steps with weights 0.4 and 0.6 and the coarse
    planes once equal one call with w_c = w_f = 1 on the same planes"""
    n, N = 32, 16
    lo, hi = (8, 16, 8), (16, 24, 24)
    rng = np.random.default_rng(9)
    nfl, nem = 9 * 5 * N * N, 9 * 2 * (N + 1) * N
    fc, ec, ff, ef = rng.normal(size=(8, nfl)), rng.normal(size=(8, nem)), rng.normal(size=(2, nfl)), rng.normal(size=(2, nem))
    grid0 = [rng.normal(size=sh) for sh in ((5, n, n, n), (n, n, n + 1), (n, n + 1, n), (n + 1, n, n))]
    one = [a.copy() for a in grid0]
    amr_ref.fixup(fc, ec, ff, ef, lo, hi, N, 0.01, 1.0 / n, *one)
    two = [a.copy() for a in grid0]
    amr_ref.fixup(fc, ec, ff, ef, lo, hi, N, 0.01, 1.0 / n, *two, w_c=1.0, w_f=0.4)
    amr_ref.fixup(fc, ec, ff, ef, lo, hi, N, 0.01, 1.0 / n, *two, w_c=0.0, w_f=0.6)
    for a, b, c in zip(one, two, grid0):
        assert np.abs(a - b).max() < 1e-13 and np.abs(a - c).max() > 1e-3
    # cells of the box itself are never touched by the fix-up (they belong to the restriction)
    assert np.array_equal(one[0][:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]], grid0[0][:, lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]])
