"""Thin Python binding of libmhd.so (include/mhd.h).  Argument marshalling only.

Every step of the update runs in the CUDA kernels behind the C ABI; this module owns no arithmetic and has no
fallback: if the library is missing or no CUDA device is usable it raises.  torch is used for device memory
and streams only (tensor.data_ptr(), torch.cuda.current_stream()).
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# MHD_LIBPATH: another build of the same library (the IEEE-division control build of tests/fp32_controls.py)
_LIBPATH = os.environ.get("MHD_LIBPATH") or os.path.join(_HERE, "libmhd.so")

FP32, FP64 = 0, 1
VL, CTU = 0, 1
PLM, PPM = 0, 1
HLLE, HLLD, ROE = 0, 1, 2
LIM_PRIM, LIM_CHAR = 0, 1
MC, MINMOD, VANLEER = 0, 1, 2
OK, EINVAL, ECUDA, ENOMEM, ESTATE, ELIMIT = 0, -1, -2, -3, -4, -5
NOALLOC_MAX_BLOCKS = 65536      # include/mhd.h MHD_NOALLOC_MAX_BLOCKS

EXPORTS = ["mhd_create", "mhd_destroy", "mhd_sizes", "mhd_advance", "mhd_advance_host", "mhd_advance_host_dt", "mhd_dt_reduce", "mhd_dt_reduce_noalloc", "mhd_advance_dt",
           "mhd_get_stats", "mhd_launch_count", "mhd_grid_pack", "mhd_grid_unpack", "mhd_grid_advance", "mhd_grid_advance_dt", "mhd_grid_dt", "mhd_amr_restrict", "mhd_amr_fixup", "mhd_amr_prolong", "mhd_set_profiling", "mhd_get_profile", "mhd_profile_stage_name",
           "mhd_measure_fma_peak", "mhd_strerror"]


class Config(C.Structure):
    _fields_ = [("ps2", C.c_int), ("nghost", C.c_int), ("gamma", C.c_double), ("scheme", C.c_int),
                ("recon", C.c_int), ("riemann", C.c_int), ("limvar", C.c_int), ("prec", C.c_int),
                ("min_dens", C.c_double), ("min_pres", C.c_double), ("emf_tie", C.c_double), ("max_groups", C.c_int), ("device", C.c_int), ("limiter", C.c_int), ("hcorr", C.c_int)]


class MHDError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libmhd error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libmhd.so (built by paper_1804_03479_b200.build); fail loudly if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIBPATH):
            raise ImportError(f"{_LIBPATH} not found: run `python -m paper_1804_03479_b200.build` (needs nvcc); "
                              "there is no CPU fallback")
        L = C.CDLL(_LIBPATH)
        vp, sp = C.c_void_p, C.POINTER(C.c_size_t)
        L.mhd_create.argtypes = [C.POINTER(Config), C.POINTER(vp)]
        L.mhd_destroy.argtypes = [vp]
        L.mhd_sizes.argtypes = [vp, sp, sp, sp, sp, sp, sp]
        L.mhd_advance.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_double, C.c_double, vp]
        L.mhd_advance_host.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int]
        L.mhd_dt_reduce.argtypes = [vp, vp, vp, C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(C.c_double),
                                    C.POINTER(C.c_double), vp]
        L.mhd_dt_reduce_noalloc.argtypes = [C.c_int, vp, vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_double,
                                            C.c_double, vp, vp]
        L.mhd_advance_host_dt.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                          C.c_double, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.mhd_advance_dt.argtypes = [vp, vp, vp, vp, vp, vp, vp, C.c_int, C.c_double, C.c_double, C.c_double,
                                     C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
        ull = C.POINTER(C.c_ulonglong)
        L.mhd_get_stats.argtypes = [vp, ull, ull, ull]
        L.mhd_launch_count.argtypes = [vp]
        L.mhd_launch_count.restype = C.c_ulonglong
        L.mhd_grid_pack.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, vp, vp, vp]
        L.mhd_grid_unpack.argtypes = [vp, vp, vp, C.c_int, C.c_int, C.c_int, vp, vp, vp, vp, vp]
        L.mhd_grid_advance.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, vp]
        L.mhd_grid_advance_dt.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                          C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
        L.mhd_grid_dt.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                  C.POINTER(C.c_double), C.POINTER(C.c_double), vp]
        ip = C.POINTER(C.c_int)
        L.mhd_amr_restrict.argtypes = [vp, vp, vp, ip, ip, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, vp]
        L.mhd_amr_fixup.argtypes = [vp, vp, vp, vp, vp, ip, ip, C.c_double, C.c_double, C.c_double, C.c_double, vp, vp, vp, vp,
                                    C.c_int, C.c_int, C.c_int, vp]
        L.mhd_amr_prolong.argtypes = [vp, vp, vp, vp, vp, C.c_int, C.c_int, C.c_int, ip, ip, vp, vp, vp, vp, vp]
        L.mhd_set_profiling.argtypes = [vp, C.c_int]
        L.mhd_get_profile.argtypes = [vp, C.POINTER(C.c_double), ull, C.c_int]
        L.mhd_profile_stage_name.argtypes = [C.c_int]
        L.mhd_profile_stage_name.restype = C.c_char_p
        L.mhd_measure_fma_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double)]
        L.mhd_strerror.argtypes = [C.c_int]
        L.mhd_strerror.restype = C.c_char_p
        _lib = L
    return _lib


def strerror(code: int) -> str:
    return lib().mhd_strerror(code).decode()


def _check(rc):
    if rc != OK:
        raise MHDError(rc, strerror(rc))


def _ptr(t):
    """Raw address of a torch tensor (device or pinned host) or numpy array; None -> NULL."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        assert t.is_contiguous()
        return C.c_void_p(t.data_ptr())
    assert t.flags["C_CONTIGUOUS"]
    return C.c_void_p(t.ctypes.data)


def _np_name(prec):
    return "float32" if prec == FP32 else "float64"


def _checked(t, prec, numel, what, device=None):
    """_ptr with the checks a raw pointer cannot carry: element type of the solver's precision, at least `numel` elements,
    and (device calls) a CUDA tensor on the solver's device.  None passes (nullable arguments)."""
    if t is None:
        return None
    want = _np_name(prec)
    if hasattr(t, "data_ptr"):
        if str(t.dtype).split(".")[-1] != want:
            raise TypeError(f"{what}: dtype {t.dtype}, the solver computes in {want}")
        n = t.numel()
        if device is not None and not (t.is_cuda and t.device.index == device):
            raise ValueError(f"{what}: expected a CUDA tensor on device {device}, got {t.device}")
        if device is None and t.is_cuda:
            raise ValueError(f"{what}: expected a host tensor, got {t.device}")
    else:
        if device is not None:
            raise ValueError(f"{what}: expected a CUDA tensor, got a host array")
        if str(t.dtype) != want:
            raise TypeError(f"{what}: dtype {t.dtype}, the solver computes in {want}")
        n = t.size
    if n < numel:
        raise ValueError(f"{what}: {n} elements, the call needs {numel}")
    return _ptr(t)


def _stream_ptr(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def dt_reduce_noalloc(prec, U, B, ngroups, ps2, nghost_of_arrays, gamma, min_dens, min_pres, dh, cfl, dt_speed_out, stream=None):
    """mhd_dt_reduce_noalloc: the CFL reduction with no solver object and no allocation (scratch = a fixed array of the library's
    device image), asynchronous on `stream`; dt_speed_out = CUDA float64 tensor of >= 2 elements that receives (dt, maxspeed).
    Raises MHDError(ELIMIT) beyond ngroups * ceil(ps2^3 / 256) = NOALLOC_MAX_BLOCKS.  Runs on the current device."""
    import torch
    dev = torch.cuda.current_device()
    T = int(ps2) + 2 * int(nghost_of_arrays)
    G = max(int(ngroups), 0)
    if G * ((int(ps2) ** 3 + 255) // 256) > NOALLOC_MAX_BLOCKS or G > 65535:
        G = 0                          # the library rejects the call (MHD_ELIMIT); no size to check against
    _checked(U, prec, G * 5 * T ** 3, "U", dev)
    _checked(B, prec, G * 3 * T * T * (T + 1), "B", dev)
    _checked(dt_speed_out, FP64, 2, "dt_speed_out", dev)
    _check(lib().mhd_dt_reduce_noalloc(int(prec), _ptr(U), _ptr(B), int(ngroups), int(ps2), int(nghost_of_arrays), float(gamma),
                                       float(min_dens), float(min_pres), float(dh), float(cfl), _ptr(dt_speed_out), _stream_ptr(stream)))


def make_config(N=16, g=3, gamma=5.0 / 3.0, scheme=VL, recon=PLM, riemann=HLLD, limvar=None, prec=FP64,
                min_dens=1e-10, min_pres=1e-10, emf_tie=0.0, max_groups=512, device=0, limiter=0, hcorr=0) -> Config:
    if limvar is None:
        limvar = LIM_PRIM if scheme == VL else LIM_CHAR
    return Config(N, g, gamma, scheme, recon, riemann, limvar, prec, min_dens, min_pres, emf_tie, max_groups, device, limiter, hcorr)


class Solver:
    """mhd_create / mhd_destroy wrapped as an object; methods carry the C-ABI names without the prefix."""

    def __init__(self, cfg: Config):
        self.cfg = cfg
        self._h = C.c_void_p()
        _check(lib().mhd_create(C.byref(cfg), C.byref(self._h)))
        n = [C.c_size_t() for _ in range(6)]
        _check(lib().mhd_sizes(self._h, *[C.byref(x) for x in n]))
        self.n_U_in, self.n_B_in, self.n_U_out, self.n_B_out, self.n_flux, self.n_emf = [int(x.value) for x in n]

    def destroy(self):
        if self._h:
            lib().mhd_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @property
    def torch_dtype(self):
        import torch
        return torch.float32 if self.cfg.prec == FP32 else torch.float64

    def sizes(self):
        return dict(n_U_in=self.n_U_in, n_B_in=self.n_B_in, n_U_out=self.n_U_out, n_B_out=self.n_B_out,
                    n_flux=self.n_flux, n_emf=self.n_emf)

    def alloc_outputs(self, G, planes=True, device=None):
        import torch
        dev = device if device is not None else f"cuda:{self.cfg.device}"
        dt = self.torch_dtype
        out = dict(U=torch.empty((G, self.n_U_out), dtype=dt, device=dev),
                   B=torch.empty((G, self.n_B_out), dtype=dt, device=dev))
        out["flux"] = torch.empty((G, self.n_flux), dtype=dt, device=dev) if planes else None
        out["emf"] = torch.empty((G, self.n_emf), dtype=dt, device=dev) if planes else None
        return out

    def _args(self, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, device):
        G, pr = max(int(ngroups), 0), self.cfg.prec
        if G > self.cfg.max_groups:
            G = 0                      # the library rejects the call (MHD_EINVAL); no size to check against
        return (_checked(U_in, pr, G * self.n_U_in, "U_in", device), _checked(B_in, pr, G * self.n_B_in, "B_in", device),
                _checked(U_out, pr, G * self.n_U_out, "U_out", device), _checked(B_out, pr, G * self.n_B_out, "B_out", device),
                _checked(flux_out, pr, G * self.n_flux, "flux_out", device), _checked(emf_out, pr, G * self.n_emf, "emf_out", device))

    def advance(self, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, stream=None):
        """mhd_advance: DEVICE tensors, asynchronous on `stream` (default: torch's current stream)."""
        a = self._args(U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, self.cfg.device)
        _check(lib().mhd_advance(self._h, *a, int(ngroups), float(dt), float(dh), _stream_ptr(stream)))

    def advance_host(self, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, chunk_groups, nstreams=3):
        """mhd_advance_host: HOST arrays (pinned torch tensors or numpy); blocking."""
        a = self._args(U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, None)
        _check(lib().mhd_advance_host(self._h, *a, int(ngroups), float(dt), float(dh), int(chunk_groups), int(nstreams)))

    def advance_host_dt(self, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, chunk_groups, nstreams, cfl):
        """mhd_advance_host_dt: HOST arrays; blocking; returns (dt_next, maxspeed)."""
        dtn, sm = C.c_double(), C.c_double()
        a = self._args(U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, None)
        _check(lib().mhd_advance_host_dt(self._h, *a, int(ngroups), float(dt), float(dh), int(chunk_groups),
                                         int(nstreams), float(cfl), C.byref(dtn), C.byref(sm)))
        return dtn.value, sm.value

    def advance_dt(self, U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, dt, dh, cfl, stream=None):
        dtn, sm = C.c_double(), C.c_double()
        a = self._args(U_in, B_in, U_out, B_out, flux_out, emf_out, ngroups, self.cfg.device)
        _check(lib().mhd_advance_dt(self._h, *a, int(ngroups), float(dt), float(dh), float(cfl), C.byref(dtn), C.byref(sm),
                                    _stream_ptr(stream)))
        return dtn.value, sm.value

    def dt_reduce(self, U, B, ngroups, nghost_of_arrays, dh, cfl, stream=None):
        dt, sm = C.c_double(), C.c_double()
        T = self.cfg.ps2 + 2 * int(nghost_of_arrays)
        G = max(int(ngroups), 0)
        _checked(U, self.cfg.prec, G * 5 * T ** 3, "U", self.cfg.device)
        _checked(B, self.cfg.prec, G * 3 * T * T * (T + 1), "B", self.cfg.device)
        _check(lib().mhd_dt_reduce(self._h, _ptr(U), _ptr(B), int(ngroups), int(nghost_of_arrays), float(dh),
                                   float(cfl), C.byref(dt), C.byref(sm), _stream_ptr(stream)))
        return dt.value, sm.value

    # ---- uniform periodic grid resident on the device (NEXT-1): grid = (U, bx, by, bz) device tensors, shape = (nz, ny, nx)
    def grid_pack(self, U, bx, by, bz, shape, U_in, B_in, stream=None):
        nz, ny, nx = shape
        _check(lib().mhd_grid_pack(self._h, _ptr(U), _ptr(bx), _ptr(by), _ptr(bz), nx, ny, nz, _ptr(U_in), _ptr(B_in),
                                   _stream_ptr(stream)))

    def grid_unpack(self, U_out, B_out, shape, U, bx, by, bz, stream=None):
        nz, ny, nx = shape
        _check(lib().mhd_grid_unpack(self._h, _ptr(U_out), _ptr(B_out), nx, ny, nz, _ptr(U), _ptr(bx), _ptr(by), _ptr(bz),
                                     _stream_ptr(stream)))

    def grid_advance(self, U, bx, by, bz, shape, dt, dh, stream=None):
        nz, ny, nx = shape
        _check(lib().mhd_grid_advance(self._h, _ptr(U), _ptr(bx), _ptr(by), _ptr(bz), nx, ny, nz, float(dt), float(dh),
                                      _stream_ptr(stream)))

    def grid_advance_dt(self, U, bx, by, bz, shape, dt, dh, cfl, stream=None):
        nz, ny, nx = shape
        dtn, sm = C.c_double(), C.c_double()
        _check(lib().mhd_grid_advance_dt(self._h, _ptr(U), _ptr(bx), _ptr(by), _ptr(bz), nx, ny, nz, float(dt), float(dh),
                                         float(cfl), C.byref(dtn), C.byref(sm), _stream_ptr(stream)))
        return dtn.value, sm.value

    def grid_dt(self, U, bx, by, bz, shape, dh, cfl, stream=None):
        nz, ny, nx = shape
        dt, sm = C.c_double(), C.c_double()
        _check(lib().mhd_grid_dt(self._h, _ptr(U), _ptr(bx), _ptr(by), _ptr(bz), nx, ny, nz, float(dh), float(cfl),
                                 C.byref(dt), C.byref(sm), _stream_ptr(stream)))
        return dt.value, sm.value

    # ---- AMR correction operation on a static two-level mesh (NEXT-2); lo, hi: (x, y, z) coarse cell indices of the box
    def amr_restrict(self, U_f, B_f, lo, hi, U, bx, by, bz, shape, stream=None):
        nz, ny, nx = shape
        _check(lib().mhd_amr_restrict(self._h, _ptr(U_f), _ptr(B_f), (C.c_int * 3)(*lo), (C.c_int * 3)(*hi), _ptr(U), _ptr(bx),
                                      _ptr(by), _ptr(bz), nx, ny, nz, _stream_ptr(stream)))

    def amr_fixup(self, flux_c, emf_c, flux_f, emf_f, lo, hi, dt, dh_c, U, bx, by, bz, shape, w_c=1.0, w_f=1.0, stream=None):
        nz, ny, nx = shape
        _check(lib().mhd_amr_fixup(self._h, _ptr(flux_c), _ptr(emf_c), _ptr(flux_f), _ptr(emf_f), (C.c_int * 3)(*lo),
                                   (C.c_int * 3)(*hi), float(dt), float(dh_c), float(w_c), float(w_f), _ptr(U), _ptr(bx), _ptr(by),
                                   _ptr(bz), nx, ny, nz, _stream_ptr(stream)))

    def amr_prolong(self, U, bx, by, bz, shape, lo, hi, U_f, bx_f, by_f, bz_f, stream=None):
        nz, ny, nx = shape
        _check(lib().mhd_amr_prolong(self._h, _ptr(U), _ptr(bx), _ptr(by), _ptr(bz), nx, ny, nz, (C.c_int * 3)(*lo),
                                     (C.c_int * 3)(*hi), _ptr(U_f), _ptr(bx_f), _ptr(by_f), _ptr(bz_f), _stream_ptr(stream)))

    def get_stats(self):
        a, b, c = C.c_ulonglong(), C.c_ulonglong(), C.c_ulonglong()
        _check(lib().mhd_get_stats(self._h, C.byref(a), C.byref(b), C.byref(c)))
        return int(a.value), int(b.value), int(c.value)

    def launch_count(self) -> int:
        return int(lib().mhd_launch_count(self._h))

    def set_profiling(self, on: bool):
        _check(lib().mhd_set_profiling(self._h, int(bool(on))))

    def get_profile(self) -> dict:
        """{stage name: (milliseconds summed over launches, launches)} since set_profiling(True)."""
        n = 16
        ms, cnt = (C.c_double * n)(), (C.c_ulonglong * n)()
        k = lib().mhd_get_profile(self._h, ms, cnt, n)
        if k < 0:
            _check(k)
        return {lib().mhd_profile_stage_name(i).decode(): (float(ms[i]), int(cnt[i])) for i in range(k)}


def measure_fma_peak(device=0, prec=FP64) -> float:
    v = C.c_double()
    _check(lib().mhd_measure_fma_peak(int(device), int(prec), C.byref(v)))
    return v.value
