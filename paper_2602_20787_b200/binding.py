"""Thin ctypes binding of libsteps_cyl.so (include/steps_cyl.h) -- argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch is used for device
memory and the CUDA stream handle, nothing else.  There is no CPU fallback: a missing library
or a missing CUDA device raises.  This module never imports `oracle`.
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsteps_cyl.so")

STEPS_OK, STEPS_EINVAL, STEPS_ESOFT, STEPS_ECUDA, STEPS_ENOMEM, STEPS_EUNSUPPORTED = 0, -1, -2, -3, -4, -5
STEPS_ETOOBIG = -6
NOALLOC_MAX_N = 32768          # STEPS_CYL_NOALLOC_MAX_N
PERIODIC_IMAGES, PERIODIC_EWALD_TABLE = 0, 1
PREC_FP64, PREC_MIXED = 0, 1
BG_FINITE, BG_INFINITE = 0, 1
FLAG_DETERMINISTIC = 1
FLAG_FAR_ORDER2 = 2
FLAG_ORDERED_PAIRS = 4
FLAG_GRAPH = 8
INTERP_CIC, INTERP_TSC = 0, 1

EXPORTS = ["steps_cyl_init", "steps_cyl_destroy", "steps_cyl_accel", "steps_cyl_accel_host",
           "steps_cyl_check", "steps_cyl_background", "steps_cyl_kdk_step",
           "steps_cyl_kdk_step_host",
           "steps_cyl_friedmann_step", "steps_cyl_friedmann_step_cpl", "steps_cyl_ewald_table", "steps_cyl_fp64_peak", "steps_cyl_last_pair_kernel_ms",
           "steps_cyl_strerror", "steps_cyl_last_cuda_error", "steps_cyl_launch_count",
           "steps_cyl_pair_kernel_name", "steps_cyl_pass_stats", "steps_cyl_accel_noalloc"]


class Params(C.Structure):
    """steps_cyl_params (include/steps_cyl.h)."""
    _fields_ = [("n", C.c_int64), ("Lz", C.c_double), ("G", C.c_double),
                ("periodic_mode", C.c_int32), ("n_cut", C.c_int32), ("precision", C.c_int32),
                ("background", C.c_int32), ("R_sim", C.c_double), ("rho0", C.c_double),
                ("device", C.c_int32), ("flags", C.c_int32),
                ("ew_nmax", C.c_int32), ("ew_mmax", C.c_int32), ("ew_alpha", C.c_double),
                ("tab_nrho", C.c_int32), ("tab_nz", C.c_int32), ("tab_rho_max", C.c_double),
                ("interp", C.c_int32), ("tab_fp32", C.c_int32)]


class StepsError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("steps_cyl error %d: %s" % (code, text))
        self.code = code


_lib = None


def lib():
    """Load libsteps_cyl.so; raises if it has not been built (python -m paper_2602_20787_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("libsteps_cyl.so is missing: run `python -m paper_2602_20787_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, dp, d, i64 = C.c_void_p, C.c_void_p, C.c_double, C.c_int64
        L.steps_cyl_init.restype = C.c_int
        L.steps_cyl_init.argtypes = [C.POINTER(Params), C.POINTER(vp)]
        L.steps_cyl_destroy.restype = None
        L.steps_cyl_destroy.argtypes = [vp]
        L.steps_cyl_accel.restype = C.c_int
        L.steps_cyl_accel.argtypes = [vp] + [dp] * 8 + [vp]
        L.steps_cyl_accel_noalloc.restype = C.c_int
        L.steps_cyl_accel_noalloc.argtypes = [i64, d, d, C.c_int32] + [dp] * 8 + [vp]
        L.steps_cyl_accel_host.restype = C.c_int
        L.steps_cyl_accel_host.argtypes = [vp] + [dp] * 8
        L.steps_cyl_check.restype = C.c_int
        L.steps_cyl_check.argtypes = [vp, vp]
        L.steps_cyl_background.restype = C.c_int
        L.steps_cyl_background.argtypes = [vp] + [dp] * 4 + [vp]
        L.steps_cyl_kdk_step.restype = C.c_int
        L.steps_cyl_kdk_step.argtypes = [vp] + [dp] * 11 + [d] * 5 + [vp]
        L.steps_cyl_kdk_step_host.restype = C.c_int
        L.steps_cyl_kdk_step_host.argtypes = [vp] + [dp] * 11 + [d] * 5
        L.steps_cyl_friedmann_step.restype = C.c_int
        L.steps_cyl_friedmann_step.argtypes = [d] * 7 + [C.POINTER(d), C.POINTER(d)]
        L.steps_cyl_friedmann_step_cpl.restype = C.c_int
        L.steps_cyl_friedmann_step_cpl.argtypes = [d] * 9 + [C.POINTER(d), C.POINTER(d)]
        L.steps_cyl_ewald_table.restype = C.c_int
        L.steps_cyl_ewald_table.argtypes = [d, d, C.c_int32, C.c_int32, C.c_int32, C.c_int32, d, dp]
        L.steps_cyl_fp64_peak.restype = C.c_int
        L.steps_cyl_fp64_peak.argtypes = [vp, d, C.POINTER(d)]
        L.steps_cyl_last_pair_kernel_ms.restype = C.c_int
        L.steps_cyl_last_pair_kernel_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.steps_cyl_strerror.restype = C.c_char_p
        L.steps_cyl_strerror.argtypes = [C.c_int]
        L.steps_cyl_last_cuda_error.restype = C.c_char_p
        L.steps_cyl_last_cuda_error.argtypes = [vp]
        L.steps_cyl_pair_kernel_name.restype = C.c_char_p
        L.steps_cyl_pair_kernel_name.argtypes = [vp]
        L.steps_cyl_pass_stats.restype = C.c_int
        L.steps_cyl_pass_stats.argtypes = [vp, vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.steps_cyl_launch_count.restype = i64
        L.steps_cyl_launch_count.argtypes = [vp]
        _lib = L
    return _lib


def friedmann_step(a, dt, H0, Om, Or=0.0, Ok=0.0, OL=0.0):
    """steps_cyl_friedmann_step: one RK4 step of Eq. 18; returns (a_next, H_next).  Host only."""
    an, Hn = C.c_double(), C.c_double()
    rc = lib().steps_cyl_friedmann_step(a, dt, H0, Om, Or, Ok, OL, C.byref(an), C.byref(Hn))
    if rc:
        raise StepsError(rc, lib().steps_cyl_strerror(rc).decode())
    return an.value, Hn.value


def friedmann_step_cpl(a, dt, H0, Om, Or, Ok, ODE, w0, wa):
    """steps_cyl_friedmann_step_cpl: RK4 step of Eq. 18 with CPL dark energy (Eq. 19-20)."""
    an, Hn = C.c_double(), C.c_double()
    rc = lib().steps_cyl_friedmann_step_cpl(a, dt, H0, Om, Or, Ok, ODE, w0, wa, C.byref(an), C.byref(Hn))
    if rc:
        raise StepsError(rc, lib().steps_cyl_strerror(rc).decode())
    return an.value, Hn.value


def ewald_table(Lz, alpha, nmax, mmax, nrho, nz, rho_max):
    """steps_cyl_ewald_table: the Eq. 17 correction table, D[nrho, nz, 2] (host only)."""
    import numpy as np
    D = np.zeros((int(nrho), int(nz), 2))
    rc = lib().steps_cyl_ewald_table(float(Lz), float(alpha), int(nmax), int(mmax), int(nrho), int(nz),
                                     float(rho_max), C.c_void_p(D.ctypes.data))
    if rc:
        raise StepsError(rc, lib().steps_cyl_strerror(rc).decode())
    return D


def _dev_ptr(t, n):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64
            and t.is_contiguous() and t.numel() == n):
        raise ValueError("expected a contiguous float64 CUDA tensor of %d elements" % n)
    return C.c_void_p(t.data_ptr())


def _host_ptr(a, n):
    import numpy as np
    import torch
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != n:
            raise ValueError("expected a contiguous float64 CPU tensor of %d elements" % n)
        return C.c_void_p(a.data_ptr())
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous and a.size == n):
        raise ValueError("expected a contiguous float64 array of %d elements" % n)
    return C.c_void_p(a.ctypes.data)


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def accel_noalloc(n, Lz, G, n_cut, x, y, z, m, h, gx, gy, gz):
    """steps_cyl_accel_noalloc: context-free force evaluation that allocates nothing (n <= NOALLOC_MAX_N),
    on torch's current device and stream (asynchronous); tensors are CUDA float64 of length n."""
    ptrs = [_dev_ptr(t, int(n)) for t in (x, y, z, m, h, gx, gy, gz)]
    rc = lib().steps_cyl_accel_noalloc(int(n), float(Lz), float(G), int(n_cut), *ptrs, _stream())
    if rc:
        raise StepsError(rc, lib().steps_cyl_strerror(rc).decode())


class StepsCyl:
    """One steps_cyl_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, n, Lz, G=1.0, n_cut=5, precision=PREC_FP64, background=BG_FINITE,
                 R_sim=0.0, rho0=0.0, device=0, periodic_mode=PERIODIC_IMAGES, flags=0,
                 ew_nmax=0, ew_mmax=0, ew_alpha=0.0, tab_nrho=0, tab_nz=0, tab_rho_max=0.0,
                 interp=INTERP_CIC, tab_fp32=0):
        self._ctx = C.c_void_p()
        self.params = Params(n=int(n), Lz=float(Lz), G=float(G), periodic_mode=int(periodic_mode),
                             n_cut=int(n_cut), precision=int(precision), background=int(background),
                             R_sim=float(R_sim), rho0=float(rho0), device=int(device), flags=int(flags),
                             ew_nmax=int(ew_nmax), ew_mmax=int(ew_mmax), ew_alpha=float(ew_alpha),
                             tab_nrho=int(tab_nrho), tab_nz=int(tab_nz),
                             tab_rho_max=float(tab_rho_max), interp=int(interp), tab_fp32=int(tab_fp32))
        self.n = int(n)
        rc = lib().steps_cyl_init(C.byref(self.params), C.byref(self._ctx))
        if rc:
            self._ctx = C.c_void_p()
            raise StepsError(rc, lib().steps_cyl_strerror(rc).decode())

    def _raise(self, rc):
        text = lib().steps_cyl_strerror(rc).decode()
        if rc == STEPS_ECUDA:
            text += " [" + lib().steps_cyl_last_cuda_error(self._ctx).decode() + "]"
        raise StepsError(rc, text)

    def close(self):
        if getattr(self, "_ctx", None) is not None and self._ctx:
            lib().steps_cyl_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def accel(self, x, y, z, m, h, gx, gy, gz):
        """steps_cyl_accel on torch's current stream (asynchronous); tensors are CUDA float64."""
        n = self.n
        rc = lib().steps_cyl_accel(self._ctx, *[_dev_ptr(t, n) for t in (x, y, z, m, h, gx, gy, gz)],
                                   _stream())
        if rc:
            self._raise(rc)

    def accel_host(self, x, y, z, m, h, gx, gy, gz):
        """steps_cyl_accel_host: host arrays in, host arrays out, synchronous."""
        n = self.n
        rc = lib().steps_cyl_accel_host(self._ctx, *[_host_ptr(a, n) for a in (x, y, z, m, h, gx, gy, gz)])
        if rc:
            self._raise(rc)

    def check(self):
        rc = lib().steps_cyl_check(self._ctx, _stream())
        if rc:
            self._raise(rc)

    def background(self, x, y, bx, by):
        n = self.n
        rc = lib().steps_cyl_background(self._ctx, *[_dev_ptr(t, n) for t in (x, y, bx, by)], _stream())
        if rc:
            self._raise(rc)

    def kdk_step(self, x, y, z, vx, vy, vz, m, h, gx, gy, gz, a_n, H_n, a_np1, H_np1, dt):
        n = self.n
        ptrs = [_dev_ptr(t, n) for t in (x, y, z, vx, vy, vz, m, h, gx, gy, gz)]
        rc = lib().steps_cyl_kdk_step(self._ctx, *ptrs, a_n, H_n, a_np1, H_np1, dt, _stream())
        if rc:
            self._raise(rc)

    def kdk_step_host(self, x, y, z, vx, vy, vz, m, h, gx, gy, gz, a_n, H_n, a_np1, H_np1, dt):
        """steps_cyl_kdk_step_host: host arrays in and out (updated in place), synchronous."""
        n = self.n
        ptrs = [_host_ptr(a, n) for a in (x, y, z, vx, vy, vz, m, h, gx, gy, gz)]
        rc = lib().steps_cyl_kdk_step_host(self._ctx, *ptrs, a_n, H_n, a_np1, H_np1, dt)
        if rc:
            self._raise(rc)

    def fp64_peak(self, ms=200.0):
        out = C.c_double()
        rc = lib().steps_cyl_fp64_peak(self._ctx, float(ms), C.byref(out))
        if rc:
            self._raise(rc)
        return out.value

    def last_pair_kernel_ms(self):
        out = C.c_float()
        rc = lib().steps_cyl_last_pair_kernel_ms(self._ctx, C.byref(out))
        if rc:
            self._raise(rc)
        return out.value

    def pair_kernel_name(self):
        return lib().steps_cyl_pair_kernel_name(self._ctx).decode()

    def pass_stats(self):
        """(simple, total) two-way ring passes of the mixed image kernel since init."""
        a, t = C.c_uint64(), C.c_uint64()
        rc = lib().steps_cyl_pass_stats(self._ctx, _stream(), C.byref(a), C.byref(t))
        if rc:
            self._raise(rc)
        return int(a.value), int(t.value)

    def launch_count(self):
        return int(lib().steps_cyl_launch_count(self._ctx))
