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
_SRC32 = os.path.join(_HERE, "mhd_oracle_f32.cpp")
_LIB32 = os.path.join(_HERE, "libmhdref_f32.so")
_FLAGS = ["-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC"]

VL, CTU = 0, 1
PLM, PPM = 0, 1
HLLE, HLLD, ROE = 0, 1, 2
LIM_PRIM, LIM_CHAR = 0, 1
MC, MINMOD, VANLEER = 0, 1, 2


class Config(C.Structure):
    _fields_ = [("ps2", C.c_int), ("nghost", C.c_int), ("gamma", C.c_double), ("scheme", C.c_int),
                ("recon", C.c_int), ("riemann", C.c_int), ("limvar", C.c_int),
                ("min_dens", C.c_double), ("min_pres", C.c_double), ("emf_tie", C.c_double), ("limiter", C.c_int),
                ("minimal_ranges", C.c_int), ("hcorr", C.c_int)]


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O2, no fast-math, no FMA contraction, OpenMP over groups)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++"] + _FLAGS + ["-o", _LIB, _SRC])
    build32(force)
    return _LIB


def build32(force: bool = False) -> str:
    """The same source instantiated in single precision (mhd_oracle_f32.cpp): the FP32 control of DESIGN.md section 9."""
    newest = max(os.path.getmtime(_SRC), os.path.getmtime(_SRC32))
    if force or not os.path.exists(_LIB32) or os.path.getmtime(_LIB32) < newest:
        subprocess.check_call(["g++"] + _FLAGS + ["-o", _LIB32, _SRC32])
    return _LIB32


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
        _lib.mhdref_roe_eta.argtypes = [dp, dp, C.c_double, C.c_double, C.c_double, dp]
        _lib.mhdref_eta_face.argtypes = [dp, dp, C.c_double, C.c_double]
        _lib.mhdref_eta_face.restype = C.c_double
        _lib.mhdref_emf_up.argtypes = [C.c_double] * 6
        _lib.mhdref_emf_up.restype = C.c_double
        _lib.mhdref_edge_emf.argtypes = [dp, dp, dp, dp, C.c_double]
        _lib.mhdref_edge_emf.restype = C.c_double
    return _lib


_lib32 = None


def lib32():
    global _lib32
    if _lib32 is None:
        _lib32 = C.CDLL(build32())
        fp, dp = C.POINTER(C.c_float), C.POINTER(C.c_double)
        _lib32.mhdref32_advance.argtypes = [C.POINTER(Config), fp, fp, fp, fp, fp, fp, C.c_int, C.c_double, C.c_double,
                                            C.POINTER(C.c_ulonglong), C.c_int]
        _lib32.mhdref32_dt.argtypes = [C.POINTER(Config), fp, fp, C.c_int, C.c_int, C.c_double, C.c_double, dp, dp]
    return _lib32


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def make_config(N=16, g=3, gamma=5.0 / 3.0, scheme=VL, recon=PLM, riemann=HLLD, limvar=None,
                min_dens=1e-10, min_pres=1e-10, emf_tie=1e-12, limiter=MC, minimal_ranges=0, hcorr=0) -> Config:
    """emf_tie: reading R10a; 1e-12 is the FP64 value, the FP32 path is checked against the oracle run with 1e-5."""
    if limvar is None:
        limvar = LIM_PRIM if scheme == VL else LIM_CHAR
    return Config(N, g, gamma, scheme, recon, riemann, limvar, min_dens, min_pres, emf_tie, limiter, minimal_ranges, hcorr)


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


def _p32(a):
    return a.ctypes.data_as(C.POINTER(C.c_float)) if a is not None else None


def advance32(cfg: Config, U_in, B_in, dt, dh, want_planes=True):
    """The oracle in single precision (every operation rounded to float): float32 in, float32 out."""
    U_in = np.ascontiguousarray(U_in, dtype=np.float32); B_in = np.ascontiguousarray(B_in, dtype=np.float32)
    G = U_in.shape[0]
    N = cfg.ps2
    f32 = np.float32
    U_out = np.empty((G, 5 * N ** 3), f32); B_out = np.empty((G, 3 * N * N * (N + 1)), f32)
    flux = np.empty((G, 9 * 5 * N * N), f32) if want_planes else None
    emf = np.empty((G, 9 * 2 * (N + 1) * N), f32) if want_planes else None
    stats = (C.c_ulonglong * 3)(0, 0, 0)
    rc = lib32().mhdref32_advance(C.byref(cfg), _p32(U_in), _p32(B_in), _p32(U_out), _p32(B_out), _p32(flux), _p32(emf), G,
                                  float(dt), float(dh), stats, 0)
    if rc != 0:
        raise ValueError(f"mhdref32_advance failed rc={rc}")
    return dict(U=U_out, B=B_out, flux=flux, emf=emf, stats=tuple(int(s) for s in stats))


def dt_reduce32(cfg: Config, U, B, ng, dh, cfl):
    U = np.ascontiguousarray(U, dtype=np.float32); B = np.ascontiguousarray(B, dtype=np.float32)
    dt = C.c_double(0); sm = C.c_double(0)
    rc = lib32().mhdref32_dt(C.byref(cfg), _p32(U), _p32(B), U.shape[0], ng, float(dh), float(cfl), C.byref(dt), C.byref(sm))
    if rc != 0:
        raise ValueError("mhdref32_dt failed")
    return dt.value, sm.value


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


def roe_eta(WL, WR, Bn, etah, gamma=5.0 / 3.0):
    """Roe flux with every dissipation speed raised to at least etah (reading R19); returns (F, fell back to HLLE)"""
    WL = _c(WL); WR = _c(WR); F = np.empty(7)
    fb = lib().mhdref_roe_eta(_p(WL), _p(WR), float(Bn), float(gamma), float(etah), _p(F))
    return F, fb


def eta_face(WL, WR, Bn, gamma=5.0 / 3.0):
    return lib().mhdref_eta_face(_p(_c(WL)), _p(_c(WR)), float(Bn), float(gamma))


def emf_up(m, rm, rp, qm, qp, tie):
    """R10a: the CT upwind switch; tie = emf_tie * dh / dt"""
    return lib().mhdref_emf_up(float(m), float(rm), float(rp), float(qm), float(qp), float(tie))


def edge_emf(Eface, mface, ec, rho, tie):
    """SURVEY C6 for one edge: Eface/mface = (a-face lo, a-face hi, b-face lo, b-face hi), ec/rho = cells (a-1,b-1), (a,b-1), (a-1,b), (a,b)"""
    return lib().mhdref_edge_emf(_p(_c(Eface)), _p(_c(mface)), _p(_c(ec)), _p(_c(rho)), float(tie))


def mc(a, b):
    return lib().mhdref_mc(float(a), float(b))


def limiter(which, a, b):
    """slope limiter by index: MC, MINMOD, VANLEER"""
    return lib().mhdref_limiter(int(which), float(a), float(b))
