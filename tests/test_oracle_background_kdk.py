"""Pins of the oracle's background force (Eq. 9/10), Friedmann RK4 (Eq. 18) and KDK step
(Eq. 11) against independent quadrature, closed forms and invariants.  CPU only."""
import math

import numpy as np
import pytest
from scipy import integrate


# ------------------------------------------------------------------ P8: Eq. 9 / 10
def _cylinder_midplane_field_polar(rho, R, Lh):
    """Independent derivation: integrate the field of the homogeneous cylinder (radius R,
    height 2 Lh, G = rho0 = 1) at a mid-plane point INSIDE it in polar coordinates (s, t)
    centred on the field point.  The z and s integrals are elementary:
      F_x = 2 Lh int_0^{2pi} cos t * asinh(s_max(t)/Lh) dt,
      s_max(t) = -rho cos t + sqrt(R^2 - rho^2 sin^2 t)   (distance to the wall)."""
    f = lambda t: math.cos(t) * math.asinh((-rho * math.cos(t) + math.sqrt(R * R - (rho * math.sin(t)) ** 2)) / Lh)
    val, err = integrate.quad(f, 0.0, 2.0 * math.pi, epsabs=1e-14, epsrel=1e-14, limit=400)
    return 2.0 * Lh * val


@pytest.mark.parametrize("rho,R,Lh", [(0.3, 1.0, 2.0), (0.8, 1.0, 0.5), (20.0, 50.0, 500.0),
                                      (500.0, 1000.0, 500.0), (990.0, 1000.0, 500.0), (1e-3, 1.0, 1.0)])
def test_Fh_matches_independent_quadrature(oracle, rho, R, Lh):
    want = _cylinder_midplane_field_polar(rho, R, Lh)
    got = oracle.Fh(rho, R, Lh, 1.0, 1.0)
    assert got < 0.0                                        # points to the axis
    assert got == pytest.approx(want, rel=2e-11)


@pytest.mark.parametrize("rho", [999.99, 1000.0 * (1 - 1e-12), 1000.0, 1000.0 * (1 + 1e-9), 1001.0])
def test_Fh_at_the_cylinder_edge_against_mpmath(oracle, rho):
    """rho ~ R: a- = (rho - X)^2 + Y^2 nearly vanishes at Y = 0 (logarithmic end-point
    singularity of Eq. 9's second integral).  30-digit tanh-sinh of the same integrand, with
    break points crowding Y = 0, fixes the value; a cancellation-prone a- fails this at 1e-7."""
    import mpmath as mp
    mp.mp.dps = 30
    R, L = mp.mpf(1000), mp.mpf(500)
    r = mp.mpf(rho)

    def f(Y):
        X = mp.sqrt(R * R - Y * Y)
        ap, am = R * R + r * r + 2 * r * X, (r - X) ** 2 + Y * Y      # same a- as Eq. 9, R^2 = X^2 + Y^2
        if am <= 0:
            return mp.mpf(0)
        return 2 * mp.log((mp.sqrt(L * L + ap) + L) / (mp.sqrt(L * L + am) + L)) - mp.log(ap / am)

    want = 2 * mp.quad(f, [0, R * 1e-9, R * 1e-6, R * 1e-3, R / 4, R / 2, R * 0.9, R * 0.99, R * 0.999, R])
    assert oracle.Fh(rho, 1000.0, 500.0, 1.0, 1.0) == pytest.approx(float(want), rel=1e-12)


def test_Fh_brute_force_3d_monte_carlo(oracle):
    """Crude but assumption-free: Monte-Carlo sum of Newtonian pulls of uniformly sampled mass
    elements of the finite cylinder; fixes sign and overall factor of Eq. 9."""
    rng = np.random.default_rng(0)
    R, Lh, rho, n = 1.0, 2.0, 0.5, 4_000_000
    r = R * np.sqrt(rng.random(n))
    t = 2 * np.pi * rng.random(n)
    z = Lh * (2 * rng.random(n) - 1)
    dx, dy = rho - r * np.cos(t), -r * np.sin(t)
    s2 = dx * dx + dy * dy + z * z + 2.5e-3                 # Plummer guard: bounds the MC variance
    V = math.pi * R * R * 2 * Lh
    fx = -np.mean(dx / s2 ** 1.5) * V
    assert oracle.Fh(rho, R, Lh, 1.0, 1.0) == pytest.approx(fx, rel=2e-2)


def test_Fh_limits(oracle):
    # Eq. 10: N_cut -> inf gives -2 pi G rho0 rho inside the cylinder
    assert oracle.Fh(20.0, 50.0, 1e9, 1.0, 1.0) == pytest.approx(-2 * math.pi * 20.0, rel=1e-6)
    assert oracle.Fh_inf_quad(20.0, 50.0, 1.0, 1.0) == pytest.approx(oracle.Fh_inf(20.0, 1.0, 1.0), rel=1e-12)
    assert oracle.Fh_inf(20.0, 2.0, 3.0) == -2 * math.pi * 2.0 * 3.0 * 20.0
    # outside an infinite cylinder: Gauss's law, -2 pi G rho0 R^2 / rho
    assert oracle.Fh_inf_quad(70.0, 50.0, 1.0, 1.0) == pytest.approx(-2 * math.pi * 2500.0 / 70.0, rel=1e-12)
    # finite L is always weaker than the infinite cylinder, and linear in G rho0
    assert 0 > oracle.Fh(20.0, 50.0, 500.0, 1.0, 1.0) > oracle.Fh_inf(20.0, 1.0, 1.0)
    assert oracle.Fh(20.0, 50.0, 500.0, 2.0, 3.0) == pytest.approx(6 * oracle.Fh(20.0, 50.0, 500.0, 1.0, 1.0), rel=1e-14)
    # thin slab limit L << rho, R: the disc pulls sideways only weakly (-> 0 as L -> 0)
    assert abs(oracle.Fh(0.5, 1.0, 1e-6, 1.0, 1.0)) < 1e-4


def test_homogeneous_cylinder_feels_no_net_force(oracle):
    """'The net force in every point should be exactly zero for homogeneous
    matter distribution' -- the Eq. 8 pair sum over a uniform random periodic cylinder is
    cancelled by -F_h(rho, R, N_cut L_z) up to Poisson noise.  Ties Eq. 9's sign, factor and
    height 2 N_cut L_z to the image window of Eq. 8."""
    rng = np.random.default_rng(42)
    n, R, L, ncut = 6000, 10.0, 10.0, 2
    r = R * np.sqrt(rng.random(n))
    t = 2 * np.pi * rng.random(n)
    x, y, z = r * np.cos(t), r * np.sin(t), L * rng.random(n)
    m = np.ones(n)
    h = np.full(n, 1.0)
    rho0 = n / (math.pi * R * R * L)
    sel = np.where((r > 2.0) & (r < 8.0))[0].astype(np.int64)
    gx, gy, _ = oracle.accel(x, y, z, m, h, L, 1.0, ncut, targets=sel)
    g_rad = (gx * x[sel] + gy * y[sel]) / r[sel]
    bx, by = oracle.background(x[sel], y[sel], R, ncut * L, 1.0, rho0, 0)
    b_rad = (bx * x[sel] + by * y[sel]) / r[sel]
    assert np.all(b_rad > 0)                                 # outward
    resid = np.mean(g_rad + b_rad) / np.mean(b_rad)
    assert abs(resid) < 0.02
    # and with the WRONG height (N_cut -> inf form, Eq. 10) the residual is clearly non-zero
    bx2, by2 = oracle.background(x[sel], y[sel], R, ncut * L, 1.0, rho0, 1)
    b2 = (bx2 * x[sel] + by2 * y[sel]) / r[sel]
    assert abs(np.mean(g_rad + b2) / np.mean(b2)) > 0.05


# -------------------------------------------------------------- P12: Friedmann, KDK
def test_friedmann_rk4_einstein_de_sitter(oracle):
    # Omega_m = 1: a(t) = (3 H0 t / 2)^(2/3) exactly
    H0 = 0.07
    a0 = 0.1
    t0 = (2.0 / (3.0 * H0)) * a0 ** 1.5
    a, t, dt = a0, t0, 0.01 * t0
    for _ in range(200):
        a, H = oracle.friedmann_rk4(a, dt, H0, 1.0, 0.0, 0.0, 0.0)
        t += dt
    assert a == pytest.approx((1.5 * H0 * t) ** (2.0 / 3.0), rel=1e-9)
    assert H == pytest.approx(H0 * a ** -1.5, rel=1e-14)
    # de Sitter: a = a0 exp(H0 t)
    a, _ = oracle.friedmann_rk4(1.0, 0.1, 1.0, 0.0, 0.0, 0.0, 1.0)
    assert a == pytest.approx(math.exp(0.1), rel=1e-6)
    # Eq. 18 itself
    assert oracle.hubble(0.5, 70.0, 0.3, 1e-4, 0.01, 0.6899) == pytest.approx(
        70.0 * math.sqrt(1e-4 * 16 + 0.3 * 8 + 0.01 * 4 + 0.6899), rel=1e-15)


def _free_particles(n=8, seed=1):
    rng = np.random.default_rng(seed)
    x, y, z = rng.normal(0, 5, n), rng.normal(0, 5, n), rng.uniform(0, 10, n)
    v = rng.normal(0, 1, (3, n))
    return x, y, z, v[0].copy(), v[1].copy(), v[2].copy()


def test_kdk_free_streaming_conserves_a2v_to_second_order(oracle):
    """m = 0, rho0 = 0: Eq. 11 reduces to xdd = -2 H xd whose solution is a^2 xd = const.
    The KDK of reading S4 must reproduce that with O(dt^2) global error."""
    H0 = 1.0
    errs = []
    for nsteps in (20, 40, 80):
        x, y, z, vx, vy, vz = _free_particles()
        n = len(x)
        m, h = np.zeros(n), np.full(n, 0.1)
        g = [np.zeros(n) for _ in range(3)]
        a0 = 0.5
        t0 = (2.0 / 3.0) * a0 ** 1.5
        a_of = lambda t: (1.5 * H0 * t) ** (2.0 / 3.0)
        T = 0.3 * t0
        dt = T / nsteps
        c0 = a0 ** 2 * vx.copy()
        for k in range(nsteps):
            an, an1 = a_of(t0 + k * dt), a_of(t0 + (k + 1) * dt)
            oracle.kdk_step(x, y, z, vx, vy, vz, m, h, *g, 10.0, 1.0, 2, 50.0, 0.0, 0,
                            an, H0 * an ** -1.5, an1, H0 * an1 ** -1.5, dt)
        errs.append(np.max(np.abs(a_of(t0 + T) ** 2 * vx / c0 - 1.0)))
    assert errs[0] < 2e-3
    assert errs[0] / errs[1] == pytest.approx(4.0, rel=0.1)
    assert errs[1] / errs[2] == pytest.approx(4.0, rel=0.1)


def test_kdk_static_two_body_matches_velocity_verlet(oracle):
    """a = 1, H = 0: the step is plain velocity-Verlet; check one step by hand and that z is
    wrapped into [0, L)."""
    L, G = 10.0, 2.0
    x = np.array([0.0, 3.0]); y = np.array([0.0, 0.0]); z = np.array([9.9, 9.9])
    vx = np.array([0.0, 0.0]); vy = np.array([0.1, -0.1]); vz = np.array([1.0, 1.0])
    m = np.array([1.0, 2.0]); h = np.array([0.01, 0.01])
    gx, gy, gz = oracle.accel(x, y, z, m, h, L, G, 1)
    assert gx[0] == pytest.approx(G * 2.0 / 9.0) and gx[1] == pytest.approx(-G * 1.0 / 9.0)
    dt = 0.05
    vxh = vx + 0.5 * dt * gx
    xn = x + vxh * dt
    g = [gx.copy(), gy.copy(), gz.copy()]
    oracle.kdk_step(x, y, z, vx, vy, vz, m, h, *g, L, G, 1, 50.0, 0.0, 0, 1.0, 0.0, 1.0, 0.0, dt)
    np.testing.assert_allclose(x, xn, rtol=1e-15)
    np.testing.assert_allclose(z, [9.95, 9.95], rtol=1e-13)
    gx2, gy2, gz2 = oracle.accel(x, y, z, m, h, L, G, 1)
    assert np.array_equal(g[0], gx2)
    np.testing.assert_allclose(vx, vxh + 0.5 * dt * gx2, rtol=1e-15)
    # momentum conserved
    assert abs(np.sum(m * vx)) < 1e-16
    z[:] = [9.99, 0.2]; vz[:] = [1.0, -8.0]
    oracle.kdk_step(x, y, z, vx, vy, vz, m, h, *g, L, G, 1, 50.0, 0.0, 0, 1.0, 0.0, 1.0, 0.0, dt)
    assert np.all((z >= 0) & (z < L))


def test_kdk_background_cancels_homogeneous_drag_free_case(oracle):
    """G5: the background term carries the same 1/a^3 as the pair term: with g = 0 (m = 0) one
    kick changes v by (dt/2) b / a^3 exactly."""
    n = 4
    x = np.array([1.0, -2.0, 0.0, 3.0]); y = np.array([0.5, 0.0, -4.0, 3.0]); z = np.zeros(n) + 1.0
    v = [np.zeros(n) for _ in range(3)]
    m, h = np.zeros(n), np.full(n, 0.1)
    g = [np.zeros(n) for _ in range(3)]
    R, L, ncut, rho0, G, a = 10.0, 5.0, 3, 0.7, 1.3, 0.5
    bx, by = oracle.background(x, y, R, ncut * L, G, rho0, 0)
    dt = 1e-3
    x0, y0 = x.copy(), y.copy()
    oracle.kdk_step(x, y, z, *v, m, h, *g, L, G, ncut, R, rho0, 0, a, 0.0, a, 0.0, dt)
    bx1, by1 = oracle.background(x, y, R, ncut * L, G, rho0, 0)
    np.testing.assert_allclose(v[0], 0.5 * dt * (bx + bx1) / a ** 3, rtol=1e-12)
    np.testing.assert_allclose(x, x0 + 0.5 * dt * bx / a ** 3 * dt, rtol=1e-14)
    rho = np.hypot(x0, y0)
    np.testing.assert_allclose(np.hypot(bx, by), [-oracle.Fh(r, R, ncut * L, G, rho0) for r in rho], rtol=1e-13)
    assert np.all(bx * x0 + by * y0 > 0)


# ------------------------------------------------------------- Eq. 19-20: CPL dark energy
def test_cpl_dark_energy_density(oracle):
    """Eq. 19 integrated numerically by the oracle against (i) the textbook constant-w power law
    a^(-3(1+w)), (ii) the closed form of the CPL integral, (iii) 30-digit quadrature of Eq. 19."""
    import mpmath as mp
    assert oracle.omega_de(0.3, 0.7, -1.0, 0.0) == pytest.approx(0.7, rel=1e-14)          # Lambda
    for w in (-0.8, -1.2, 0.0, 1.0 / 3.0):
        assert oracle.omega_de(0.25, 0.7, w, 0.0) == pytest.approx(0.7 * 0.25 ** (-3 * (1 + w)), rel=1e-13)
    for a, w0, wa in [(0.02, -0.9, 0.3), (0.5, -1.1, -0.4), (1.7, -0.7, 0.2)]:
        closed = 0.7 * a ** (-3 * (1 + w0 + wa)) * math.exp(3 * wa * (a - 1))
        quad = 0.7 * mp.exp(-3 * mp.quad(lambda x: (1 + w0 + wa * (1 - x)) / x, [1, a]))
        assert oracle.omega_de(a, 0.7, w0, wa) == pytest.approx(closed, rel=1e-13)
        assert oracle.omega_de(a, 0.7, w0, wa) == pytest.approx(float(quad), rel=1e-13)


def test_cpl_friedmann_reduces_and_has_closed_form(oracle):
    # w0 = -1, wa = 0: identical to the Lambda-CDM step
    a1, H1 = oracle.friedmann_rk4(0.3, 1e-4, 70.0, 0.3, 1e-4, 0.0, 0.7)
    a2, H2 = oracle.friedmann_rk4_cpl(0.3, 1e-4, 70.0, 0.3, 1e-4, 0.0, 0.7, -1.0, 0.0)
    assert a2 == pytest.approx(a1, rel=1e-15) and H2 == pytest.approx(H1, rel=1e-14)
    # dark energy with w = 0 dilutes like matter: Om + ODE = 1 is Einstein-de Sitter, a = (3 H0 t/2)^(2/3)
    H0, n = 70.0, 200
    a0, a_end = 0.1, 0.2
    dt = (2 / (3 * H0)) * (a_end ** 1.5 - a0 ** 1.5) / n
    a = a0
    for _ in range(n):
        a, H = oracle.friedmann_rk4_cpl(a, dt, H0, 0.3, 0.0, 0.0, 0.7, 0.0, 0.0)
    assert a == pytest.approx(a_end, rel=1e-10)
    assert H == pytest.approx(H0 * a ** -1.5, rel=1e-12)
