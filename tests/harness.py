"""Test harness: periodic uniform-grid stepping on top of a group solver (oracle or CUDA binding).

Stands in for the AMR host layer's preparation/closing steps with periodic copies.
`advance_fn(U_in[G][..], B_in[G][..], dt, dh) -> dict(U=, B=, ...)` is either the oracle or the CUDA path.
"""
from __future__ import annotations

import numpy as np

from paper_1804_03479_b200 import inputs


def step_grid(advance_fn, U, bx, by, bz, dt, dh, N, g, dtype=np.float64):
    """One step of a periodic n^3 grid cut into (n/N)^3 groups.  Returns (U, bx, by, bz, out, shared_face_mismatch)."""
    n = U.shape[-3:]
    U_in, B_in = inputs.pack_groups(U, bx, by, bz, N, g, dtype)
    out = advance_fn(U_in, B_in, dt, dh)
    Un, bxn, byn, bzn, mism = inputs.unpack_groups(np.asarray(out["U"]), np.asarray(out["B"]), n, N)
    return Un, bxn, byn, bzn, out, mism


def totals(U):
    return np.array([np.sum(U[v], dtype=np.float64) for v in range(5)])


def rel_divb(bx, by, bz, dh):
    d = inputs.div_b(bx, by, bz, dh)
    bmax = max(np.max(np.abs(bx)), np.max(np.abs(by)), np.max(np.abs(bz)))
    return float(np.max(np.abs(d)) * dh / bmax)


def field_err(a, b):
    """err_f = max|a-b| / max|b| (reading R14)."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    den = float(np.max(np.abs(b)))
    num = float(np.max(np.abs(a - b)))
    return num / den if den > 0 else num


def pack_boxes(boxes, N, g, dtype=np.float64):
    """Batch of INDEPENDENT periodic N^3 boxes (config 2) -> one ghost-zoned group each (periodic wrap of itself)."""
    sz = inputs.sizes(N, g)
    G = len(boxes)
    U_in = np.empty((G, sz["n_U_in"]), dtype=dtype)
    B_in = np.empty((G, sz["n_B_in"]), dtype=dtype)
    for q, (U, bx, by, bz) in enumerate(boxes):
        u, b = inputs.pack_groups(U, bx, by, bz, N, g, dtype)
        U_in[q], B_in[q] = u[0], b[0]
    return U_in, B_in


def step_boxes(advance_fn, boxes, dt, dh, N, g, dtype=np.float64):
    """One step of a batch of independent periodic boxes through ONE advance call.  boxes: list of (U, bx, by, bz)."""
    U_in, B_in = pack_boxes(boxes, N, g, dtype)
    out = advance_fn(U_in, B_in, dt, dh)
    new = []
    for q in range(len(boxes)):
        Un, bxn, byn, bzn, _ = inputs.unpack_groups(np.asarray(out["U"])[q:q + 1], np.asarray(out["B"])[q:q + 1], N, N)
        new.append((Un, bxn, byn, bzn))
    return new, out
