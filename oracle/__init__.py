"""ctypes front end of the CPU oracle (oracle/steps_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package; the
CUDA path (paper_2602_20787_b200) never does, and this package never imports it.

Every function is a thin argument-marshalling shell around the C function of
the same name; the arithmetic lives in steps_oracle.c, each function there
citing the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "steps_oracle.c")
_LIB = os.path.join(_HERE, "libsteps_oracle.so")
_lib = None

# No -ffast-math, no -march=native: the oracle is plain IEEE double arithmetic.
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off"]


def build(force: bool = False) -> str:
    """Compile steps_oracle.c with gcc into oracle/libsteps_oracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.run(["gcc", *CFLAGS, _SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        d, i, i64, p = C.c_double, C.c_int, C.c_int64, C.POINTER(C.c_double)
        _lib.oracle_spline_F.restype = d
        _lib.oracle_spline_F.argtypes = [d, d]
        _lib.oracle_pair_accel.restype = None
        _lib.oracle_pair_accel.argtypes = [d, d, d, d, d, d, i, p]
        _lib.oracle_accel.restype = i
        _lib.oracle_accel.argtypes = [i64, p, p, p, p, p, d, d, i, i64,
                                      C.POINTER(C.c_int64), p, p, p, i]
        _lib.oracle_max_threads.restype = i
        _lib.oracle_Fh.restype = d
        _lib.oracle_Fh.argtypes = [d, d, d, d, d]
        _lib.oracle_Fh_inf.restype = d
        _lib.oracle_Fh_inf.argtypes = [d, d, d]
        _lib.oracle_Fh_inf_quad.restype = d
        _lib.oracle_Fh_inf_quad.argtypes = [d, d, d, d]
        _lib.oracle_hubble.restype = d
        _lib.oracle_hubble.argtypes = [d] * 6
        _lib.oracle_friedmann_rk4.restype = None
        _lib.oracle_friedmann_rk4.argtypes = [d] * 7 + [p, p]
        _lib.oracle_background.restype = None
        _lib.oracle_background.argtypes = [i64, p, p, d, d, d, d, i, p, p]
        _lib.oracle_omega_de.restype = d
        _lib.oracle_omega_de.argtypes = [d] * 4
        _lib.oracle_hubble_cpl.restype = d
        _lib.oracle_hubble_cpl.argtypes = [d] * 8
        _lib.oracle_friedmann_rk4_cpl.restype = None
        _lib.oracle_friedmann_rk4_cpl.argtypes = [d] * 9 + [p, p]
        _lib.oracle_ewald_force.restype = None
        _lib.oracle_ewald_force.argtypes = [d, d, d, d, i, i, p]
        _lib.oracle_ewald_D.restype = None
        _lib.oracle_ewald_D.argtypes = [d, d, d, d, i, i, p]
        _lib.oracle_ewald_table.restype = None
        _lib.oracle_ewald_table.argtypes = [d, d, i, i, i, i, d, p]
        _lib.oracle_table_interp.restype = None
        _lib.oracle_table_interp.argtypes = [p, i, i, d, d, i, d, d, p]
        _lib.oracle_accel_table.restype = i
        _lib.oracle_accel_table.argtypes = [i64, p, p, p, p, p, d, d, p, i, i, d, i, i64,
                                            C.POINTER(C.c_int64), p, p, p, i]
        _lib.oracle_kdk_step.restype = i
        _lib.oracle_kdk_step.argtypes = [i64] + [p] * 11 + [d, d, i, d, d, i, d, d, d, d, d, i]
    return _lib


def spline_F(r: float, h: float) -> float:
    """Eq. 3, reading G1."""
    return lib().oracle_spline_F(float(r), float(h))


def pair_accel(rx, ry, rz, hh, L, G, ncut):
    """Eq. 8 for one unit-mass source at separation r = x_i - x_j; returns g (3,)."""
    g = np.zeros(3)
    lib().oracle_pair_accel(float(rx), float(ry), float(rz), float(hh), float(L), float(G),
                            int(ncut), _dp(g))
    return g


def accel(x, y, z, m, h, L, G, ncut, targets=None, nthreads=0):
    """g_i = sum_{j!=i} m_j F_{S1xR2}(x_i-x_j, h_i+h_j) (Eq. 1/8/11 pair sum).

    Returns (gx, gy, gz) for `targets` (indices; None = all particles)."""
    x, y, z, m, h = map(_f64, (x, y, z, m, h))
    n = x.shape[0]
    if targets is None:
        nt, tp = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = targets.shape[0], targets.ctypes.data_as(C.POINTER(C.c_int64))
    gx, gy, gz = np.empty(nt), np.empty(nt), np.empty(nt)
    rc = lib().oracle_accel(n, _dp(x), _dp(y), _dp(z), _dp(m), _dp(h), float(L), float(G),
                            int(ncut), nt, tp, _dp(gx), _dp(gy), _dp(gz), int(nthreads))
    if rc:
        raise ValueError("oracle_accel: bad arguments")
    return gx, gy, gz


def max_threads() -> int:
    return lib().oracle_max_threads()


def Fh(rho, R, Lhalf, G, rho0):
    """Eq. 9 (reading G3), L = N_cut*L_z is the half height."""
    return lib().oracle_Fh(float(rho), float(R), float(Lhalf), float(G), float(rho0))


def Fh_inf(rho, G, rho0):
    """Eq. 10."""
    return lib().oracle_Fh_inf(float(rho), float(G), float(rho0))


def Fh_inf_quad(rho, R, G, rho0):
    return lib().oracle_Fh_inf_quad(float(rho), float(R), float(G), float(rho0))


def hubble(a, H0, Om, Or, Ok, OL):
    """Eq. 18 with a cosmological constant."""
    return lib().oracle_hubble(float(a), float(H0), float(Om), float(Or), float(Ok), float(OL))


def friedmann_rk4(a, dt, H0, Om, Or, Ok, OL):
    an, Hn = C.c_double(), C.c_double()
    lib().oracle_friedmann_rk4(float(a), float(dt), float(H0), float(Om), float(Or), float(Ok),
                               float(OL), C.byref(an), C.byref(Hn))
    return an.value, Hn.value


def background(x, y, R, Lhalf, G, rho0, mode):
    """-F_h(rho) e_rho per particle (Eq. 11 background term); returns (bx, by)."""
    x, y = _f64(x), _f64(y)
    bx, by = np.empty_like(x), np.empty_like(y)
    lib().oracle_background(x.shape[0], _dp(x), _dp(y), float(R), float(Lhalf), float(G),
                            float(rho0), int(mode), _dp(bx), _dp(by))
    return bx, by


def kdk_step(x, y, z, vx, vy, vz, m, h, gx, gy, gz, L, G, ncut, R, rho0, mode,
             a_n, H_n, a_np1, H_np1, dt, nthreads=0):
    """One KDK step (reading S4); all twelve arrays are float64, contiguous, updated in place
    except m, h."""
    arrs = (x, y, z, vx, vy, vz, m, h, gx, gy, gz)
    for a in arrs:
        assert a.dtype == np.float64 and a.flags.c_contiguous
    rc = lib().oracle_kdk_step(x.shape[0], *[_dp(a) for a in arrs], float(L), float(G), int(ncut),
                               float(R), float(rho0), int(mode), float(a_n), float(H_n),
                               float(a_np1), float(H_np1), float(dt), int(nthreads))
    if rc:
        raise ValueError("oracle_kdk_step: bad arguments")


def ewald_force(rho, z, L, alpha, nmax, mmax):
    """Eq. 12-16 (reading G4): (F_rho, F_z) per unit G m_i m_j of the one-axis-periodic point mass."""
    F = np.zeros(2)
    lib().oracle_ewald_force(float(rho), float(z), float(L), float(alpha), int(nmax), int(mmax), _dp(F))
    return F


def ewald_D(rho, z, L, alpha, nmax, mmax):
    """Eq. 17 at one point: Ewald force minus the unsoftened nearest-image force."""
    F = np.zeros(2)
    lib().oracle_ewald_D(float(rho), float(z), float(L), float(alpha), int(nmax), int(mmax), _dp(F))
    return F


def ewald_table(L, alpha, nmax, mmax, nrho, nz, rho_max):
    """Eq. 17 on the (nrho x nz) grid; returns D[nrho, nz, 2]."""
    D = np.zeros((int(nrho), int(nz), 2))
    lib().oracle_ewald_table(float(L), float(alpha), int(nmax), int(mmax), int(nrho), int(nz),
                             float(rho_max), _dp(D))
    return D


def table_interp(D, rho_max, L, interp, rho, az):
    D = _f64(D)
    out = np.zeros(2)
    lib().oracle_table_interp(_dp(D), D.shape[0], D.shape[1], float(rho_max), float(L), int(interp),
                              float(rho), float(az), _dp(out))
    return out


def accel_table(x, y, z, m, h, L, G, D, rho_max, interp, targets=None, nthreads=0):
    """Pair sum in EWALD_TABLE mode: softened nearest image + interpolated D (Eq. 17)."""
    x, y, z, m, h, D = map(_f64, (x, y, z, m, h, D))
    n = x.shape[0]
    if targets is None:
        nt, tp = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = targets.shape[0], targets.ctypes.data_as(C.POINTER(C.c_int64))
    gx, gy, gz = np.empty(nt), np.empty(nt), np.empty(nt)
    rc = lib().oracle_accel_table(n, _dp(x), _dp(y), _dp(z), _dp(m), _dp(h), float(L), float(G),
                                  _dp(D), D.shape[0], D.shape[1], float(rho_max), int(interp),
                                  nt, tp, _dp(gx), _dp(gy), _dp(gz), int(nthreads))
    if rc:
        raise ValueError("oracle_accel_table: bad arguments")
    return gx, gy, gz


def omega_de(a, ODE, w0, wa):
    """Eq. 19 with the CPL equation of state Eq. 20 (integral done numerically)."""
    return lib().oracle_omega_de(float(a), float(ODE), float(w0), float(wa))


def hubble_cpl(a, H0, Om, Or, Ok, ODE, w0, wa):
    return lib().oracle_hubble_cpl(*map(float, (a, H0, Om, Or, Ok, ODE, w0, wa)))


def friedmann_rk4_cpl(a, dt, H0, Om, Or, Ok, ODE, w0, wa):
    an, Hn = C.c_double(), C.c_double()
    lib().oracle_friedmann_rk4_cpl(*map(float, (a, dt, H0, Om, Or, Ok, ODE, w0, wa)), C.byref(an), C.byref(Hn))
    return an.value, Hn.value
