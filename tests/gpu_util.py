"""Helpers for the -m gpu parity tests: run the CUDA path (through the C ABI binding) on numpy inputs."""
from __future__ import annotations

import numpy as np


def np_dtype(prec):
    return np.float32 if prec == 0 else np.float64


class GpuRunner:
    """advance_fn-compatible wrapper (see tests/harness.py) around paper_1804_03479_b200.mhd.Solver."""

    def __init__(self, N=16, g=3, scheme=0, recon=0, riemann=1, limvar=None, prec=1, max_groups=512, planes=True, limiter=0, hcorr=0, gamma=5.0 / 3.0):
        import torch
        from paper_1804_03479_b200 import mhd
        self.torch = torch
        self.mhd = mhd
        self.cfg = mhd.make_config(N=N, g=g, scheme=scheme, recon=recon, riemann=riemann, limvar=limvar, prec=prec,
                                   max_groups=max_groups, limiter=limiter, hcorr=hcorr, gamma=gamma)
        self.solver = mhd.Solver(self.cfg)
        self.planes = planes
        self.dtype = np_dtype(prec)

    def __call__(self, U_in, B_in, dt, dh):
        torch = self.torch
        G = U_in.shape[0]
        Ui = torch.from_numpy(np.ascontiguousarray(U_in, dtype=self.dtype)).cuda()
        Bi = torch.from_numpy(np.ascontiguousarray(B_in, dtype=self.dtype)).cuda()
        out = self.solver.alloc_outputs(G, planes=self.planes)
        self.solver.advance(Ui, Bi, out["U"], out["B"], out["flux"], out["emf"], G, dt, dh)
        torch.cuda.synchronize()
        res = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}
        return res

    def advance_dt(self, U_in, B_in, dt, dh, cfl):
        """mhd_advance_dt: outputs as __call__, plus (dt_next, maxspeed)"""
        torch = self.torch
        G = U_in.shape[0]
        Ui = torch.from_numpy(np.ascontiguousarray(U_in, dtype=self.dtype)).cuda()
        Bi = torch.from_numpy(np.ascontiguousarray(B_in, dtype=self.dtype)).cuda()
        out = self.solver.alloc_outputs(G, planes=self.planes)
        dtn, smax = self.solver.advance_dt(Ui, Bi, out["U"], out["B"], out["flux"], out["emf"], G, dt, dh, cfl)
        res = {k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}
        return res, dtn, smax

    def dt(self, U, B, ng, dh, cfl):
        torch = self.torch
        G = U.shape[0]
        Ud = torch.from_numpy(np.ascontiguousarray(U, dtype=self.dtype)).cuda()
        Bd = torch.from_numpy(np.ascontiguousarray(B, dtype=self.dtype)).cuda()
        return self.solver.dt_reduce(Ud, Bd, G, ng, dh, cfl)

    def stats(self):
        return self.solver.get_stats()


FIELDS_U = ["rho", "Mx", "My", "Mz", "e"]


def split_fields(out, N):
    """dict of per-field arrays from a solver output dict (U, B, flux, emf), for per-field error norms (R14)."""
    f = {}
    U = np.asarray(out["U"]).reshape(-1, 5, N ** 3)
    for v, name in enumerate(FIELDS_U):
        f[name] = U[:, v]
    nb = N * N * (N + 1)
    B = np.asarray(out["B"])
    f["Bx"], f["By"], f["Bz"] = B[:, :nb], B[:, nb:2 * nb], B[:, 2 * nb:]
    if out.get("flux") is not None:
        F = np.asarray(out["flux"]).reshape(-1, 9, 5, N * N)
        for v, name in enumerate(FIELDS_U):
            f["flux_" + name] = F[:, :, v]
    if out.get("emf") is not None:
        f["emf"] = np.asarray(out["emf"])
    return f


def field_errors(a, b, N):
    """err_f = max|a-b| / max|b| per field (R14); b is the oracle."""
    fa, fb = split_fields(a, N), split_fields(b, N)
    errs = {}
    for k in fb:
        den = float(np.max(np.abs(fb[k])))
        num = float(np.max(np.abs(fa[k].astype(np.float64) - fb[k])))
        errs[k] = num / den if den > 0 else num
    return errs
