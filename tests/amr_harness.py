"""Static two-level mesh harness for the correction operation: a periodic coarse grid with one refined
box, both levels advanced by the same dt with any group solver (oracle or CUDA binding).  Numpy only."""
from __future__ import annotations

import numpy as np

from paper_1804_03479_b200 import inputs
from oracle import amr_ref


def fine_groups_of_box(Ufine, bxf, byf, bzf, lo, hi, N, g, dtype=np.float64):
    """ghost-zoned fine groups covering the refined box (coarse indices lo..hi), cut from a fine periodic grid"""
    Ui, Bi = inputs.pack_groups(Ufine, bxf, byf, bzf, N, g, dtype)
    nf = Ufine.shape[-1] // N
    sel = []
    for gz in range(2 * lo[2] // N, 2 * hi[2] // N):
        for gy in range(2 * lo[1] // N, 2 * hi[1] // N):
            for gx in range(2 * lo[0] // N, 2 * hi[0] // N):
                sel.append((gz * nf + gy) * nf + gx)
    return Ui[sel], Bi[sel]


def composite_totals(Uc, U_f, lo, hi, N, dh_c):
    """sum of conserved variables over the leaf cells of the two-level mesh (coarse outside the box, fine inside)"""
    mask = np.ones(Uc.shape[1:], dtype=bool)
    mask[lo[2]:hi[2], lo[1]:hi[1], lo[0]:hi[0]] = False
    coarse = np.array([Uc[v][mask].sum() for v in range(5)]) * dh_c ** 3
    fine = np.asarray(U_f, dtype=np.float64).reshape(-1, 5, N ** 3).sum(axis=(0, 2)) * (0.5 * dh_c) ** 3
    return coarse + fine


def two_level_step(adv_c, adv_f, Uc, bxc, byc, bzc, lo, hi, N, g, dt, dh_c, correct=True, dtype=np.float64, ops=amr_ref):
    """one synchronised step of both levels + correction.  Returns the corrected coarse grid and the fine outputs."""
    n = Uc.shape[-1]
    Uf0, bxf0, byf0, bzf0 = amr_ref.inject(Uc, bxc, byc, bzc)
    Ui_c, Bi_c = inputs.pack_groups(Uc, bxc, byc, bzc, N, g, dtype)
    out_c = adv_c(Ui_c, Bi_c, dt, dh_c)
    Un, bxn, byn, bzn, _ = inputs.unpack_groups(np.asarray(out_c["U"]), np.asarray(out_c["B"]), n, N)
    Ui_f, Bi_f = fine_groups_of_box(Uf0, bxf0, byf0, bzf0, lo, hi, N, g, dtype)
    out_f = adv_f(Ui_f, Bi_f, dt, 0.5 * dh_c)
    grid = [np.array(a, dtype=np.float64) for a in (Un, bxn, byn, bzn)]
    if correct:
        ops.fixup(out_c["flux"], out_c["emf"], out_f["flux"], out_f["emf"], lo, hi, N, dt, dh_c, *grid)
        ops.restrict(np.asarray(out_f["U"], dtype=np.float64), np.asarray(out_f["B"], dtype=np.float64), lo, hi, N, *grid)
    # periodic duplicates of the face arrays (the box is away from the boundary, so only consistency)
    grid[1][:, :, n] = grid[1][:, :, 0]; grid[2][:, n, :] = grid[2][:, 0, :]; grid[3][n] = grid[3][0]
    return grid, out_c, out_f, (Uf0, bxf0, byf0, bzf0)
