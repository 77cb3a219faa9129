"""The seeded input generators: shapes, determinism, and the paper-faithful stereographic particle load
(Eq. 21-22) against the numbers the paper prints for its Fig. 4 example."""
import math

import numpy as np
import pytest

from paper_2602_20787_b200 import workloads


def test_configs_are_deterministic_and_shaped():
    for cfg, n in [(0, 2048), (1, 4000), (2, 4000), (3, 4000), (4, 6000)]:
        a, b = workloads.make(cfg, n=n), workloads.make(cfg, n=n)
        assert a.n == n
        for k in ("x", "y", "z", "m", "h"):
            assert np.array_equal(getattr(a, k), getattr(b, k))
        assert np.all((a.z >= 0) & (a.z < a.Lz)) and np.all(a.h > 0) and np.all(a.m > 0)
    w = workloads.make(3, n=4000)
    assert w.vx is not None and w.cosmo["n_steps"] == 10 and w.rho0 > 0


def test_stereographic_load_fig4_parameters():
    """Fig. 4: D_S = 70, R_sim = 500, omega_c = 1.63973, L_z = 500 give a constant-resolution
    core out to rho_c = D_S tan(omega_c/2) = 75.0 Mpc."""
    w = workloads.stereographic_load(n_target=60000)
    assert w.cosmo["rho_c"] == pytest.approx(75.0, abs=5e-4)
    assert abs(w.n - 60000) < 0.15 * 60000
    rho = np.hypot(w.x, w.y)
    assert rho.max() <= 500.0 * (1 + 1e-12) and np.all((w.z >= 0) & (w.z < 500.0))
    # m_i = rho_bar V_i: the cells tile the cylinder, so the masses add up to rho_bar pi R^2 L exactly
    assert w.m.sum() == pytest.approx(math.pi * 500.0 ** 2 * 500.0, rel=1e-12)
    core = rho < 75.0
    assert np.ptp(w.m[core]) < 1e-9 * w.m[core][0]                      # constant mass resolution inside
    # outside, the mass of a cell grows monotonically with its ring (Jacobian of Eq. 22) and joins the
    # core resolution without a jump
    mo, ro = w.m[~core], rho[~core]
    order = np.argsort(ro)
    assert np.all(np.diff(mo[order][:: max(1, mo.size // 200)]) >= -1e-9 * mo.max())
    assert 0.8 < mo.min() / w.m[core][0] < 1.25
    assert mo.max() / mo.min() > 50.0
    # inverse stereographic map, Eq. 21 / 22, are inverses of each other
    om = 2.0 * np.arctan(ro / 70.0)
    assert np.allclose(70.0 * np.tan(0.5 * om), ro, rtol=1e-13)
    assert om.max() <= w.cosmo["omega_max"] * (1 + 1e-12) < math.pi
