"""ctypes binding of the CPU oracle (oracle/mhd_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It never imports the CUDA package's solver; it imports nothing but numpy.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mhd_oracle.cpp")
_LIB = os.path.join(_HERE, "libmhdref.so")

VL, CTU = 0, 1
PLM, PPM = 0, 1
HLLE, HLLD, ROE = 0, 1, 2
LIM_PRIM, LIM_CHAR = 0, 1
MC, MINMOD, VANLEER = 0, 1, 2


class Config(C.Structure):
    _fields_ = [("ps2", C.c_int), ("nghost", C.c_int), ("gamma", C.c_double), ("scheme", C.c_int),
                ("recon", C.c_int), ("riemann", C.c_int), ("limvar", C.c_int),
                ("min_dens", C.c_double), ("min_pres", C.c_double), ("emf_tie", C.c_double), ("limiter", C.c_int)]


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2, no fast-math, no FMA contraction, OpenMP over groups)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        _lib.mhdref_advance.argtypes = [C.POINTER(Config), dp, dp, dp, dp, dp, dp, C.c_int, C.c_double, C.c_double,
                                        C.POINTER(C.c_ulonglong), C.c_int]
        _lib.mhdref_dt.argtypes = [C.POINTER(Config), dp, dp, C.c_int, C.c_int, C.c_double, C.c_double, dp, dp]
        _lib.mhdref_riemann.argtypes = [C.c_int, dp, dp, C.c_double, C.c_double, dp]
        _lib.mhdref_prim2cons.argtypes = [dp, C.c_double, C.c_double, dp]
        _lib.mhdref_physflux.argtypes = [dp, C.c_double, C.c_double, dp]
        _lib.mhdref_fastspeed.argtypes = [dp, C.c_double, C.c_double]
        _lib.mhdref_fastspeed.restype = C.c_double
        _lib.mhdref_eig_prim.argtypes = [dp, C.c_double, C.c_double, dp, dp, dp, dp]
        _lib.mhdref_eig_roe.argtypes = [dp, dp, C.c_double, C.c_double, dp, dp, dp, dp]
        _lib.mhdref_mc.argtypes = [C.c_double, C.c_double]
        _lib.mhdref_mc.restype = C.c_double
        _lib.mhdref_limiter.argtypes = [C.c_int, C.c_double, C.c_double]
        _lib.mhdref_limiter.restype = C.c_double
    return _lib


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def make_config(N=16, g=3, gamma=5.0 / 3.0, scheme=VL, recon=PLM, riemann=HLLD, limvar=None,
                min_dens=1e-10, min_pres=1e-10, emf_tie=1e-12, limiter=MC) -> Config:
    """emf_tie: reading R10a; 1e-12 is the FP64 value, the FP32 path is checked against the oracle run with 1e-5."""
    if limvar is None:
        limvar = LIM_PRIM if scheme == VL else LIM_CHAR
    return Config(N, g, gamma, scheme, recon, riemann, limvar, min_dens, min_pres, emf_tie, limiter)


def advance(cfg: Config, U_in, B_in, dt, dh, want_planes=True, force_ghost_ok=False):
    """Advance G groups.  Returns dict(U, B, flux, emf, stats)."""
    U_in = _c(U_in); B_in = _c(B_in)
    G = U_in.shape[0]
    N = cfg.ps2
    U_out = np.empty((G, 5 * N ** 3)); B_out = np.empty((G, 3 * N * N * (N + 1)))
    flux = np.empty((G, 9 * 5 * N * N)) if want_planes else None
    emf = np.empty((G, 9 * 2 * (N + 1) * N)) if want_planes else None
    stats = (C.c_ulonglong * 3)(0, 0, 0)
    rc = lib().mhdref_advance(C.byref(cfg), _p(U_in), _p(B_in), _p(U_out), _p(B_out), _p(flux), _p(emf), G,
                              float(dt), float(dh), stats, int(force_ghost_ok))
    if rc != 0:
        raise ValueError(f"mhdref_advance failed rc={rc}")
    return dict(U=U_out, B=B_out, flux=flux, emf=emf, stats=tuple(int(s) for s in stats))


def dt_reduce(cfg: Config, U, B, ng, dh, cfl):
    U = _c(U); B = _c(B)
    G = U.shape[0]
    dt = C.c_double(0); sm = C.c_double(0)
    rc = lib().mhdref_dt(C.byref(cfg), _p(U), _p(B), G, ng, float(dh), float(cfl), C.byref(dt), C.byref(sm))
    if rc != 0:
        raise ValueError("mhdref_dt failed")
    return dt.value, sm.value


def riemann(solver, WL, WR, Bn, gamma=5.0 / 3.0):
    WL = _c(WL); WR = _c(WR); F = np.empty(7)
    fb = lib().mhdref_riemann(solver, _p(WL), _p(WR), float(Bn), float(gamma), _p(F))
    return F, fb


def prim2cons(W, Bn, gamma=5.0 / 3.0):
    W = _c(W); U = np.empty(7)
    lib().mhdref_prim2cons(_p(W), float(Bn), float(gamma), _p(U))
    return U


def physflux(W, Bn, gamma=5.0 / 3.0):
    W = _c(W); F = np.empty(7)
    lib().mhdref_physflux(_p(W), float(Bn), float(gamma), _p(F))
    return F


def fastspeed(W, Bn, gamma=5.0 / 3.0):
    return lib().mhdref_fastspeed(_p(_c(W)), float(Bn), float(gamma))


def eig_prim(W, Bn, gamma=5.0 / 3.0):
    """lam[7], R[k] = k-th right eigenvector (rows), L[k] = k-th left eigenvector (rows), A[7][7]."""
    W = _c(W); lam = np.empty(7); R = np.empty((7, 7)); L = np.empty((7, 7)); A = np.empty((7, 7))
    lib().mhdref_eig_prim(_p(W), float(Bn), float(gamma), _p(lam), _p(R), _p(L), _p(A))
    return lam, R, L, A


def eig_roe(WL, WR, Bn, gamma=5.0 / 3.0):
    WL = _c(WL); WR = _c(WR)
    lam = np.empty(7); R = np.empty((7, 7)); L = np.empty((7, 7)); avg = np.empty(9)
    rc = lib().mhdref_eig_roe(_p(WL), _p(WR), float(Bn), float(gamma), _p(lam), _p(R), _p(L), _p(avg))
    return rc, lam, R, L, avg


def mc(a, b):
    return lib().mhdref_mc(float(a), float(b))


def limiter(which, a, b):
    """slope limiter by index: MC, MINMOD, VANLEER"""
    return lib().mhdref_limiter(int(which), float(a), float(b))
