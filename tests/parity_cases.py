"""The multi-step parity cases of BASELINE.json configs 2 and 3 as functions, shared by the -m gpu tests and by the FP32
control experiment (tests/fp32_controls.py): seeded initial states, the oracle's dt sequence, and a runner that takes any
`advance_fn` (FP64 oracle, FP32 oracle, CUDA path).  No solver arithmetic here."""
from __future__ import annotations

import numpy as np

from paper_1804_03479_b200 import inputs
import harness as H

EMF_TIE = {1: 1e-12, 0: 1e-5}   # DESIGN.md R10a: the tie width is part of the method and follows the working precision
MOM = ("Mx", "My", "Mz")


def config2_boxes(G=24, N=16, prec=1):
    """G independent periodic N^3 boxes of the config-2 state (seed 3479 + q); FP32 runs start from the FP32-rounded state
    on both sides (R14).  Returns (boxes [(U, bx, by, bz)] in float64, dh)."""
    dtp = np.float32 if prec == 0 else np.float64
    boxes, dh = [], None
    for q in range(G):
        U, bx, by, bz, dh = inputs.random_group_grid(N, 3479 + q)
        boxes.append(tuple(a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz)))
    return boxes, dh


def run_boxes_oracle(oracle, cfg, boxes, dh, N, g, nsteps=10, cfl=0.3):
    """advance with the FP64 oracle and its own CFL dt; returns (dts, final boxes, last output, packed input of the last step)"""
    adv = lambda Ui, Bi, dt, dh_: oracle.advance(cfg, Ui, Bi, dt, dh_)
    dts, out, last_in = [], None, None
    for _ in range(nsteps):
        Ui, Bi = H.pack_boxes(boxes, N, g)
        dt, _ = oracle.dt_reduce(cfg, Ui, Bi, g, dh, cfl)
        dts.append(dt)
        last_in = (Ui, Bi)
        boxes, out = H.step_boxes(adv, boxes, dt, dh, N, g)
    return dts, boxes, out, last_in


def run_boxes(adv, boxes, dts, dh, N, g, dtype):
    boxes = [tuple(np.asarray(a).astype(dtype) for a in b) for b in boxes]
    out = None
    for dt in dts:
        boxes, out = H.step_boxes(adv, boxes, dt, dh, N, g, dtype=dtype)
    return boxes, out


def config3_grid(n=64, prec=1):
    dtp = np.float32 if prec == 0 else np.float64
    U, bx, by, bz, dh = inputs.abc_grid(n, seed=1805, p0=0.15, vamp=1e-2)
    return tuple(a.astype(dtp).astype(np.float64) for a in (U, bx, by, bz)), dh


def run_grid_oracle(oracle, adv, state, dh, N, g, nsteps=10, cfl=0.3):
    """advance the FP64 oracle nsteps with its own CFL dt; returns (dts, final state, last output)"""
    U, bx, by, bz = state
    n = U.shape[-1]
    c0 = oracle.make_config(N=n, g=3)
    dts, out = [], None
    for _ in range(nsteps):
        Ui, Bi = inputs.pack_groups(U, bx, by, bz, n, 0)
        dt, _ = oracle.dt_reduce(c0, Ui, Bi, 0, dh, cfl)
        dts.append(dt)
        U, bx, by, bz, out, _ = H.step_grid(adv, U, bx, by, bz, dt, dh, N, g)
    return dts, (U, bx, by, bz), out


def run_grid(adv, state, dts, dh, N, g, dtype=np.float64):
    U, bx, by, bz = (np.asarray(a).astype(dtype) for a in state)
    out = None
    for dt in dts:
        U, bx, by, bz, out, mism = H.step_grid(adv, U, bx, by, bz, dt, dh, N, g, dtype)
        assert mism == 0.0, "faces shared by two groups must be bitwise equal"
    return (U, bx, by, bz), out


def grid_errors(a, b):
    """per-field err_f (R14) of a grid state (U, bx, by, bz) against the reference b"""
    names = ["rho", "Mx", "My", "Mz", "e"]
    errs = {nm: H.field_err(a[0][v], b[0][v]) for v, nm in enumerate(names)}
    errs.update(Bx=H.field_err(a[1], b[1]), By=H.field_err(a[2], b[2]), Bz=H.field_err(a[3], b[3]))
    return errs


def boxes_errors(a, b):
    """per-field err_f over a batch of boxes: max over the batch of |a-b| / max over the batch of |b|"""
    names = ["rho", "Mx", "My", "Mz", "e"]
    errs = {}
    for v, nm in enumerate(names):
        errs[nm] = H.field_err(np.stack([x[0][v] for x in a]), np.stack([x[0][v] for x in b]))
    for c, nm in enumerate(("Bx", "By", "Bz")):
        errs[nm] = H.field_err(np.stack([x[1 + c] for x in a]), np.stack([x[1 + c] for x in b]))
    return errs


def fp32_gate(e32, floor=1e-4, factor=2.0):
    """DESIGN.md R14b: the FP32 gate of a field is the north-star 1e-4, or `factor` x the error that the plain algorithm
    itself has in IEEE single precision (the FP32 instantiation of the oracle against the FP64 oracle, same inputs, same
    dt sequence) where that is larger.  The three momentum components are one vector field: one bound, the largest."""
    g = {k: max(floor, factor * v) for k, v in e32.items()}
    if all(k in g for k in MOM):
        m = max(g[k] for k in MOM)
        for k in MOM:
            g[k] = m
    return g
