"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/steps_cyl.h
declares, validates its arguments, fails loudly without a CUDA device, and its one host-only
entry point (the RK4 Friedmann step, Eq. 18) matches a closed form.  No kernel is launched."""
import ctypes as C
import math
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2602_20787_b200 import build, binding
    build.build()
    return binding.lib()


def test_every_declared_symbol_is_exported(lib):
    hdr = open(os.path.join(ROOT, "include", "steps_cyl.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = sorted(set(re.findall(r"\b(steps_cyl_[a-z0-9_]+)\s*\(", hdr)))
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(lib, name), name
    from paper_2602_20787_b200 import binding
    assert sorted(binding.EXPORTS) == declared


def test_params_struct_layout_matches_header():
    from paper_2602_20787_b200.binding import Params
    # int64, 2 double, 4 int32, 2 double, 2 int32 | 2 int32, double, 2 int32, double, 2 int32
    assert C.sizeof(Params) == 104
    assert Params.R_sim.offset == 40 and Params.device.offset == 56
    assert Params.ew_alpha.offset == 72 and Params.tab_rho_max.offset == 88 and Params.interp.offset == 96
    hdr = open(os.path.join(ROOT, "include", "steps_cyl.h")).read()
    body = hdr[hdr.index("typedef struct {"):hdr.index("} steps_cyl_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"\b(?:int64_t|int32_t|double)\s+(\w+)\s*;", body)
    assert names == [f[0] for f in Params._fields_]


def test_init_rejects_bad_arguments(lib):
    from paper_2602_20787_b200 import binding as b
    ctx = C.c_void_p()
    good = dict(n=16, Lz=100.0, G=1.0, periodic_mode=0, n_cut=5, precision=0, background=0,
                R_sim=0.0, rho0=0.0, device=0, flags=0)
    for bad in (dict(n=0), dict(Lz=0.0), dict(Lz=-1.0), dict(n_cut=0), dict(precision=7),
                dict(background=3), dict(periodic_mode=9), dict(flags=16), dict(device=-1),
                dict(rho0=1.0, R_sim=0.0), dict(n=2 ** 31), dict(n=64 * 65535 * 128 + 1)):
        p = b.Params(**{**good, **bad})
        assert lib.steps_cyl_init(C.byref(p), C.byref(ctx)) == b.STEPS_EINVAL, bad
        assert not ctx.value
    # EWALD_TABLE has no ordered-pair kernel; bad table parameters are EINVAL
    for extra in (dict(flags=b.FLAG_ORDERED_PAIRS), dict(flags=b.FLAG_ORDERED_PAIRS | b.FLAG_DETERMINISTIC)):
        p = b.Params(**{**good, "periodic_mode": b.PERIODIC_EWALD_TABLE, **extra})
        assert lib.steps_cyl_init(C.byref(p), C.byref(ctx)) == b.STEPS_EUNSUPPORTED
    for extra in (dict(tab_nrho=1), dict(ew_alpha=-1.0), dict(interp=5), dict(tab_rho_max=-3.0), dict(tab_fp32=2)):
        p = b.Params(**{**good, "periodic_mode": b.PERIODIC_EWALD_TABLE, **extra})
        assert lib.steps_cyl_init(C.byref(p), C.byref(ctx)) == b.STEPS_EINVAL, extra
    assert lib.steps_cyl_init(None, C.byref(ctx)) == b.STEPS_EINVAL
    assert lib.steps_cyl_accel(None, *([None] * 8), None) == b.STEPS_EINVAL
    assert lib.steps_cyl_kdk_step(None, *([None] * 11), 1.0, 1.0, 1.0, 1.0, 1.0, None) == b.STEPS_EINVAL
    lib.steps_cyl_destroy(None)
    assert lib.steps_cyl_strerror(b.STEPS_ESOFT).decode().startswith("softening")


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2602_20787_b200 import binding as b
    with pytest.raises(b.StepsError) as e:
        b.StepsCyl(n=16, Lz=100.0)
    assert e.value.code == b.STEPS_ECUDA


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2602_20787_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", src, flags=re.M), f
                assert "steps_oracle" not in src, f


def test_friedmann_step_einstein_de_sitter_closed_form(lib):
    """Omega_m = 1: a(t) = (3 H0 t / 2)^(2/3) exactly; RK4 global error is O(dt^4)."""
    from paper_2602_20787_b200 import binding as b
    H0 = 70.0
    errs = []
    for nsteps in (50, 100):
        a0, a1 = 0.1, 0.2
        t0, t1 = (2.0 / (3.0 * H0)) * a0 ** 1.5, (2.0 / (3.0 * H0)) * a1 ** 1.5
        dt = (t1 - t0) / nsteps
        a = a0
        for _ in range(nsteps):
            a, H = b.friedmann_step(a, dt, H0, 1.0)
        errs.append(abs(a - a1))
        assert H == pytest.approx(H0 * a ** -1.5, rel=1e-14)
    assert errs[0] < 1e-9
    assert errs[1] < errs[0] / 12.0          # 4th order: halving dt divides the error by ~16


def test_friedmann_step_lcdm_hubble_value(lib):
    from paper_2602_20787_b200 import binding as b
    a, H = b.friedmann_step(0.5, 0.0, 100.0, 0.3, 1e-4, 0.0, 0.7 - 1e-4)
    assert a == 0.5
    assert H == pytest.approx(100.0 * math.sqrt(1e-4 / 0.5 ** 4 + 0.3 / 0.5 ** 3 + 0.7 - 1e-4), rel=1e-15)
    assert lib.steps_cyl_friedmann_step(-1.0, 0.1, 1.0, 1.0, 0.0, 0.0, 0.0, C.byref(C.c_double()),
                                        C.byref(C.c_double())) == b.STEPS_EINVAL


def test_ewald_table_builder_matches_the_oracle_table(lib, oracle):
    """steps_cyl_ewald_table (host-only entry point; double-exponential quadrature, own series) against
    the oracle's table (Gauss-Legendre panels), written independently from Eq. 12-17."""
    import numpy as np
    from paper_2602_20787_b200 import binding as b
    for (L, aL, nmax, mmax, nrho, nz, rmax) in [(100.0, 2.0, 5, 12, 19, 13, 450.0), (1.0, 3.0, 7, 14, 9, 9, 2.5)]:
        got = b.ewald_table(L, aL / L, nmax, mmax, nrho, nz, rmax)
        want = oracle.ewald_table(L, aL / L, nmax, mmax, nrho, nz, rmax)
        scale = np.abs(want).max()
        assert np.abs(got - want).max() <= 1e-12 * scale
        nz_mask = np.abs(want) > 1e-6 * scale
        assert np.abs(got[nz_mask] / want[nz_mask] - 1).max() <= 1e-9
    assert lib.steps_cyl_ewald_table(1.0, 1.0, 5, 12, 1, 8, 1.0, None) == b.STEPS_EINVAL


def test_friedmann_step_cpl_matches_oracle_and_lcdm(lib, oracle):
    from paper_2602_20787_b200 import binding as b
    for w0, wa in [(-1.0, 0.0), (-0.9, 0.0), (-0.95, 0.3), (-1.1, -0.5)]:
        a, o = 0.02, 0.02
        for _ in range(20):
            a, H = b.friedmann_step_cpl(a, 2e-6, 100.0, 0.3, 8e-5, 0.0, 0.7, w0, wa)
            o, Ho = oracle.friedmann_rk4_cpl(o, 2e-6, 100.0, 0.3, 8e-5, 0.0, 0.7, w0, wa)
        assert a == pytest.approx(o, rel=1e-13) and H == pytest.approx(Ho, rel=1e-13)
    a1, H1 = b.friedmann_step(0.5, 1e-3, 70.0, 0.3, 0.0, 0.0, 0.7)
    a2, H2 = b.friedmann_step_cpl(0.5, 1e-3, 70.0, 0.3, 0.0, 0.0, 0.7, -1.0, 0.0)
    assert a2 == pytest.approx(a1, rel=1e-15) and H2 == pytest.approx(H1, rel=1e-15)
