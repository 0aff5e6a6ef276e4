"""Shock-tube runs shared by the oracle pin and the GPU parity test."""
from __future__ import annotations

import numpy as np

from paper_1804_03479_b200 import inputs
import harness as H

NT = 8          # cells across the tube = patch-group size of the runs


def run_tube(advance_fn, dt_fn, name, n, axis=0, t_end=None, max_steps=None, dtype=np.float64, g=3):
    """advance the doubled periodic tube (inputs.shock_tube) to t_end at CFL 0.3; returns grid arrays, dh, dt list"""
    U, bx, by, bz, dh = inputs.shock_tube(name, n, axis, NT)
    U, bx, by, bz = (a.astype(dtype) for a in (U, bx, by, bz))
    t_end = inputs.RIEMANN_PROBLEMS[name]["t_end"] if t_end is None else t_end
    t, dts = 0.0, []
    while t < t_end - 1e-12 and (max_steps is None or len(dts) < max_steps):
        dt = min(dt_fn(U, bx, by, bz, dh), t_end - t)
        U, bx, by, bz, out, mism = H.step_grid(advance_fn, U, bx, by, bz, dt, dh, NT, g, dtype)
        assert mism == 0.0
        t += dt; dts.append(dt)
    return (U, bx, by, bz), dh, dts


def profile(grid, n, axis=0):
    """the seven 1-D variables (rho, Mn, Mt1, Mt2, e, Bt1, Bt2) on the first tube, cells 0..n-1 along `axis`"""
    U, bx, by, bz = grid
    t1, t2 = (axis + 1) % 3, (axis + 2) % 3
    line = [0, 0, 0]; line[2 - axis] = slice(0, n)
    line = tuple(line)
    b = (bx, by, bz)
    return np.stack([U[0][line], U[1 + axis][line], U[1 + t1][line], U[1 + t2][line], U[4][line], b[t1][line], b[t2][line]]).astype(np.float64)
