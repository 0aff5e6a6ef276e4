"""Linear-wave set-up shared by the oracle pin (P5) and the GPU parity test.

Background and eigenvectors: tests/golden/linear_wave_modes.txt (PAPER.md:256-264 describes the test).
"""
from __future__ import annotations

import os

import numpy as np

from paper_1804_03479_b200 import inputs
import harness as H

GAMMA = 5.0 / 3.0
_G = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "linear_wave_modes.txt")


def load_modes():
    """-> dict(background=W0[8] (rho, vn, vt1, vt2, P, Bn, Bt1, Bt2), fast=(speed, R[7]), alfven=..., slow=...)"""
    out = {}
    for line in open(_G):
        line = line.split("#")[0].strip()
        if not line:
            continue
        name, vals = line.split(":")
        v = [eval(x, {"sqrt": np.sqrt}) for x in vals.split(",")]
        out[name.strip()] = np.array(v, dtype=np.float64)
    return out


def axis_wave(N, axis, mode, amp=1e-6, NT=16):
    """Wave along `axis` on a grid with N cells along it and NT along the others.  Returns U, bx, by, bz, dh, speed."""
    m = load_modes()
    W0 = m["background"]; spd = m[mode][0]; Rv = m[mode][1:]
    n, t1, t2 = axis, (axis + 1) % 3, (axis + 2) % 3
    shape = [NT, NT, NT]; shape[2 - axis] = N          # (nz, ny, nx)
    nz, ny, nx = shape
    dh = 1.0 / N
    xc = (np.arange(N) + 0.5) * dh
    ph = np.cos(2 * np.pi * xc)
    bshape = [1, 1, 1]; bshape[2 - axis] = N
    ph = ph.reshape(bshape)
    e0 = W0[4] / (GAMMA - 1) + 0.5 * (W0[5] ** 2 + W0[6] ** 2 + W0[7] ** 2)
    U = np.empty((5, nz, ny, nx))
    U[0] = W0[0] + amp * Rv[0] * ph
    U[1 + n] = amp * Rv[1] * ph
    U[1 + t1] = amp * Rv[2] * ph
    U[1 + t2] = amp * Rv[3] * ph
    U[4] = e0 + amp * Rv[4] * ph
    fs = [(nz, ny, nx + 1), (nz, ny + 1, nx), (nz + 1, ny, nx)]
    b = [None, None, None]
    b[n] = np.full(fs[n], W0[5])
    # transverse components live on their own faces, at the cell-centre coordinate along `axis`
    b[t1] = W0[6] + amp * Rv[5] * ph + np.zeros(fs[t1])
    b[t2] = W0[7] + amp * Rv[6] * ph + np.zeros(fs[t2])
    return U, b[0], b[1], b[2], dh, spd


def diagonal_wave(N, mode, amp=1e-6):
    """Wave along the body diagonal of [0,1)^3, k = 2*pi*(1,1,1); B perturbation from an edge vector potential."""
    m = load_modes()
    W0 = m["background"]; spd = m[mode][0]; Rv = m[mode][1:]
    e1 = np.array([1.0, 1.0, 1.0]) / np.sqrt(3.0)          # wave normal
    e2 = np.array([1.0, -1.0, 0.0]) / np.sqrt(2.0)
    e3 = np.cross(e1, e2)
    kw = 2 * np.pi * np.sqrt(3.0)                          # |k|; phase = kw * (e1 . x)
    dh = 1.0 / N
    c, f = (np.arange(N) + 0.5) * dh, np.arange(N + 1) * dh

    def vec(a1, a2, a3):
        return a1 * e1 + a2 * e2 + a3 * e3

    B0 = vec(W0[5], W0[6], W0[7])
    # dB(xi) = amp (R5 e2 + R6 e3) cos(kw xi)  =  curl of  A = amp/kw * (R6 e2 - R5 e3) sin(kw xi) ... sign fixed below
    # curl(g(xi) a) = g'(xi) e1 x a ; e1 x e2 = e3, e1 x e3 = -e2  => a = (-R5 e3 ... ) solve: e1 x a = R5 e2 + R6 e3
    # with a = alpha e2 + beta e3: e1 x a = alpha e3 - beta e2 => alpha = R6, beta = -R5
    avec = Rv[6] * e2 - Rv[5] * e3

    def pot(X, Y, Z):
        xi = e1[0] * X + e1[1] * Y + e1[2] * Z
        # uniform part B0 = curl(1/2 B0 x r) ; add linear potential A0 = 1/2 B0 x r (not periodic -> add B0 to faces instead)
        return amp / kw * np.sin(kw * xi)

    Zc, Yc, Xc = np.meshgrid(f, f, c, indexing="ij"); Ax = avec[0] * pot(Xc, Yc, Zc)
    Zc, Yc, Xc = np.meshgrid(f, c, f, indexing="ij"); Ay = avec[1] * pot(Xc, Yc, Zc)
    Zc, Yc, Xc = np.meshgrid(c, f, f, indexing="ij"); Az = avec[2] * pot(Xc, Yc, Zc)
    bx, by, bz = inputs.faces_from_potential(Ax, Ay, Az, dh)
    bx += B0[0]; by += B0[1]; bz += B0[2]
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    ph = np.cos(kw * (e1[0] * X + e1[1] * Y + e1[2] * Z))
    rho = W0[0] + amp * Rv[0] * ph
    M = [amp * (Rv[1] * e1[d] + Rv[2] * e2[d] + Rv[3] * e3[d]) * ph for d in range(3)]
    e0 = W0[4] / (GAMMA - 1) + 0.5 * (W0[5] ** 2 + W0[6] ** 2 + W0[7] ** 2)
    e = e0 + amp * Rv[4] * ph
    U = np.stack([rho, M[0], M[1], M[2], e])
    return U, bx, by, bz, dh, spd, 1.0 / np.sqrt(3.0)       # wavelength


def run_period(advance_fn, dt_fn, U, bx, by, bz, dh, period, N, g, cfl=0.3):
    """Advance to t = period with dt = cfl*dh/maxspeed (last step shortened)."""
    U0, b0 = U.copy(), (bx.copy(), by.copy(), bz.copy())
    t = 0.0
    nstep = 0
    while t < period * (1 - 1e-12):
        dt = min(dt_fn(U, bx, by, bz, dh, cfl), period - t)
        U, bx, by, bz, _, _ = H.step_grid(advance_fn, U, bx, by, bz, dt, dh, N, g)
        t += dt; nstep += 1
    errs = [np.mean(np.abs(U[v] - U0[v])) for v in range(5)]
    errs += [np.mean(np.abs(a - a0)) for a, a0 in zip((bx, by, bz), b0)]
    return float(np.sqrt(np.sum(np.square(errs)))), nstep, (U, bx, by, bz)
