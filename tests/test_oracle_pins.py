"""Pins of the CPU oracle against things OTHER than itself (CPU only, no GPU).

Each test states what fixes the expected value: a textbook definition, a closed form, an
invariant, an independent quadrature, or brute force.  A dropped term, a wrong sign or
index, or a shifted image window in oracle/steps_oracle.c fails at least one of them.
"""
import math

import mpmath as mp
import numpy as np
import pytest

mp.mp.dps = 40


# ---------------------------------------------------------------- P1: Eq. 3 spline
def _m4_enclosed_mass_over_r2(r, h):
    """Monaghan & Lattanzio (1985) M4 cubic spline with compact support h, unit mass:
    W(u) = 8/(pi h^3) {1 - 6u^2 + 6u^3 (u<=1/2) ; 2(1-u)^3 (1/2<u<=1) ; 0}, u = r/h.
    Newton's shell theorem: force magnitude = M(<r)/r^2 (PAPER.md:61 says Eq. 3
    'corresponds to the cubic spline kernel of Monaghan & Lattanzio')."""
    r, h = mp.mpf(r), mp.mpf(h)

    def W(x):
        u = x / h
        if u <= mp.mpf(1) / 2:
            return 8 / (mp.pi * h ** 3) * (1 - 6 * u ** 2 + 6 * u ** 3)
        if u <= 1:
            return 8 / (mp.pi * h ** 3) * 2 * (1 - u) ** 3
        return mp.mpf(0)

    pts = sorted({mp.mpf(0), min(r, h / 2), min(r, h), r})
    M = mp.quad(lambda x: 4 * mp.pi * x * x * W(x), pts)
    return M / r ** 2


@pytest.mark.parametrize("h", [1.0, 0.7, 2.5, 0.4])
def test_spline_is_m4_enclosed_mass(oracle, h):
    for u in [1e-3, 0.05, 0.1, 0.3, 0.49, 0.5, 0.51, 0.75, 0.9, 0.999, 1.0, 1.2, 3.0]:
        r = u * h
        want = float(_m4_enclosed_mass_over_r2(r, h))
        got = oracle.spline_F(r, h)
        assert got == pytest.approx(want, rel=2e-12), (u, h)


def test_spline_special_values_and_continuity(oracle):
    # closed-form values of M(<r)/r^2: F(h/2,h) = 38/(15 h^2), F(h,h) = 1/h^2
    for h in [1.0, 0.7, 3.0]:
        assert oracle.spline_F(0.5 * h, h) == pytest.approx(38.0 / 15.0 / h ** 2, rel=1e-13)
        assert oracle.spline_F(h, h) == pytest.approx(1.0 / h ** 2, rel=1e-13)
        for rb in (0.5 * h, h):
            lo, hi = oracle.spline_F(rb * (1 - 1e-9), h), oracle.spline_F(rb * (1 + 1e-9), h)
            assert lo == pytest.approx(hi, rel=1e-7)
    # Newton outside the support; linear (homogeneous-sphere-like) at the centre
    assert oracle.spline_F(2.0, 1.0) == 0.25
    assert oracle.spline_F(1e-6, 1.0) == pytest.approx(32.0 / 3.0 * 1e-6, rel=1e-5)


# ---------------------------------------------------- P2: two particles, single image
def test_two_particle_newton_and_softened(oracle):
    # one image (N_cut=1, r_z = 0 -> only n = 0), outside the support: plain Newton -r/|r|^3
    g = oracle.pair_accel(1.0, 0.0, 0.0, 1.0, 100.0, 1.0, 1)
    assert g[0] == -1.0 and g[1] == 0.0 and g[2] == 0.0
    g = oracle.pair_accel(3.0, 4.0, 0.0, 1.0, 1000.0, 2.5, 1)
    np.testing.assert_allclose(g, [-2.5 * 3 / 125, -2.5 * 4 / 125, 0.0], rtol=1e-15)
    # inside the support: enclosed-mass value (independent definition), r = 0.25, h = 1
    want = -float(_m4_enclosed_mass_over_r2(0.25, 1.0))
    g = oracle.pair_accel(0.25, 0.0, 0.0, 1.0, 100.0, 1.0, 1)
    assert g[0] == pytest.approx(want, rel=1e-13)          # = -2.19166...
    assert want == pytest.approx(-2.1916666666666667, rel=1e-13)
    # coincident particles: no force, no NaN
    assert np.all(oracle.pair_accel(0.0, 0.0, 0.0, 1.0, 100.0, 1.0, 4) == 0.0)


# ----------------------------------------- P3: literal transcription of Eq. 8's window
def _literal_eq8(oracle, rx, ry, rz_raw, hh, L, G, ncut):
    """sum_{n=-N_cut}^{N_cut} over images with |r_z - n L| < N_cut L, on the RAW r_z
    (no nearest-image reduction)."""
    g = np.zeros(3)
    cnt = 0
    for n in range(-ncut, ncut + 1):
        d = rz_raw - n * L
        if not abs(d) < ncut * L:
            continue
        cnt += 1
        s = math.sqrt(rx * rx + ry * ry + d * d)
        if s == 0.0:
            continue
        w = oracle.spline_F(s, hh) / s
        g += -G * w * np.array([rx, ry, d])
    return g, cnt


def test_window_matches_literal_eq8(oracle):
    rng = np.random.default_rng(5)
    L = 100.0
    for _ in range(400):
        ncut = int(rng.integers(1, 8))
        rx, ry = rng.normal(0, 30, 2)
        rz = rng.uniform(-L, L)
        hh = rng.uniform(0.1, 5.0)
        lit, cnt = _literal_eq8(oracle, rx, ry, rz, hh, L, 1.0, ncut)
        assert cnt == 2 * ncut
        got = oracle.pair_accel(rx, ry, rz, hh, L, 1.0, ncut)
        np.testing.assert_allclose(got, lit, rtol=1e-13, atol=1e-22)
    # r_z = 0: symmetric set, 2 N_cut - 1 images, no axial force
    lit, cnt = _literal_eq8(oracle, 3.0, 0.0, 0.0, 1.0, L, 1.0, 4)
    assert cnt == 7
    got = oracle.pair_accel(3.0, 0.0, 0.0, 1.0, L, 1.0, 4)
    np.testing.assert_allclose(got, lit, rtol=1e-14, atol=1e-18)
    assert got[2] == 0.0
    # |r_z| = L/2 exactly: the set is symmetric whichever way rint() rounds
    a = oracle.pair_accel(3.0, 1.0, 50.0, 1.0, L, 1.0, 3)
    b = oracle.pair_accel(3.0, 1.0, -50.0, 1.0, L, 1.0, 3)
    assert a[0] == b[0] and a[1] == b[1] and a[2] == -b[2]


# ------------------------------------------------------------------ P4: periodicity
def test_periodicity_bit_exact(oracle):
    base = oracle.pair_accel(3.0, 4.0, 20.0, 1.0, 100.0, 1.0, 5)
    for shift in (100.0, -100.0, 300.0):
        g = oracle.pair_accel(3.0, 4.0, 20.0 + shift, 1.0, 100.0, 1.0, 5)
        assert np.array_equal(g, base)


def test_accel_invariant_under_z_shift_by_L(oracle):
    rng = np.random.default_rng(11)
    n, L = 64, 8.0
    x, y = rng.normal(0, 3, n), rng.normal(0, 3, n)
    z = rng.uniform(0, L, n)
    m, h = rng.uniform(0.5, 2, n), rng.uniform(0.05, 0.3, n)
    g0 = oracle.accel(x, y, z, m, h, L, 1.0, 3)
    z2 = z.copy()
    z2[::3] += L            # exact in fp for these magnitudes? not always -> 1e-13
    z2[1::3] -= 2 * L
    g1 = oracle.accel(x, y, z2, m, h, L, 1.0, 3)
    for a, b in zip(g0, g1):
        np.testing.assert_allclose(a, b, rtol=1e-11, atol=1e-13)


# ------------------------------------------- P5: on-axis closed form with trigamma
@pytest.mark.parametrize("ncut", [1, 3, 10, 37])
def test_on_axis_trigamma(oracle, ncut):
    L = 100.0
    for rz in [17.0, 0.3, 49.0, 50.0]:
        u = mp.mpf(rz) / L
        want = -(mp.psi(1, u) - mp.psi(1, u + ncut) - mp.psi(1, 1 - u) + mp.psi(1, ncut + 1 - u)) / L ** 2
        g = oracle.pair_accel(0.0, 0.0, rz, 1e-3, L, 1.0, ncut)
        assert g[0] == 0.0 and g[1] == 0.0
        if rz == 50.0:
            # |r_z| = L/2: window (-N L, N L) is symmetric about the midpoint between two
            # images, the axial force vanishes by symmetry (either rounding of rint)
            assert abs(g[2]) < 1e-18
        else:
            assert g[2] == pytest.approx(float(want), rel=1e-13)
        gm = oracle.pair_accel(0.0, 0.0, -rz, 1e-3, L, 1.0, ncut)
        assert gm[2] == -g[2]


# ------------------------- P6: exact infinite sum (Bessel series) and exact tails
def _bessel_series(rho, z, L):
    """Field of an infinite periodic line of unit point masses (G = 1), period L, at radial
    distance rho and axial offset z from one of them (Poisson summation of 1/r):
    g_rho = -2/(L rho) - (4/L) sum k K1(k rho) cos(k z), g_z = -(4/L) sum k K0(k rho) sin(k z)."""
    rho, z, L = mp.mpf(rho), mp.mpf(z), mp.mpf(L)
    grho, gz = -2 / (L * rho), mp.mpf(0)
    mmax = int(math.ceil(100.0 * float(L) / (2 * math.pi * float(rho)))) + 2    # K_nu(100) ~ 1e-45
    for m_ in range(1, mmax + 1):
        k = 2 * mp.pi * m_ / L
        grho -= 4 / L * k * mp.besselk(1, k * rho) * mp.cos(k * z)
        gz -= 4 / L * k * mp.besselk(0, k * rho) * mp.sin(k * z)
    return grho, gz


def _tails(rho, rz, L, ncut):
    """Images Eq. 8 EXCLUDES for 0 < r_z <= L/2: d = r_z + kL (k >= N_cut) and
    d = r_z - nL (n >= N_cut + 1); summed to infinity with mpmath.nsum."""
    rho, rz, L = mp.mpf(rho), mp.mpf(rz), mp.mpf(L)
    f_r = lambda d: -rho / (rho ** 2 + d ** 2) ** mp.mpf(1.5)
    f_z = lambda d: -d / (rho ** 2 + d ** 2) ** mp.mpf(1.5)
    tr = mp.nsum(lambda k: f_r(rz + k * L), [ncut, mp.inf]) + mp.nsum(lambda n: f_r(rz - n * L), [ncut + 1, mp.inf])
    tz = mp.nsum(lambda k: f_z(rz + k * L), [ncut, mp.inf]) + mp.nsum(lambda n: f_z(rz - n * L), [ncut + 1, mp.inf])
    return tr, tz


@pytest.mark.parametrize("rho,rz,L,ncut", [(40.0, 30.0, 100.0, 5), (7.0, 11.0, 100.0, 1),
                                           (0.3, 0.2, 1.0, 3), (150.0, 49.0, 100.0, 8)])
def test_truncated_sum_equals_infinite_minus_tails(oracle, rho, rz, L, ncut):
    grho, gz = _bessel_series(rho, rz, L)
    tr, tz = _tails(rho, rz, L, ncut)
    want = np.array([float(grho - tr), float(gz - tz)])
    g = oracle.pair_accel(rho, 0.0, rz, 1e-4 * L, L, 1.0, ncut)
    np.testing.assert_allclose([g[0], g[2]], want, rtol=2e-12)
    # same pair, radial direction along y, negative r_z
    g2 = oracle.pair_accel(0.0, rho, -rz, 1e-4 * L, L, 1.0, ncut)
    np.testing.assert_allclose([g2[1], g2[2]], [want[0], -want[1]], rtol=2e-12)


def test_convergence_to_infinite_sum_is_inverse_square(oracle):
    # PAPER.md:126 "convergence remains exceptionally slow": error ~ N_cut^-2
    grho, gz = _bessel_series(40.0, 30.0, 100.0)
    assert float(grho) == pytest.approx(-4.2917313465578851e-4, rel=1e-12)
    assert float(gz) == pytest.approx(-1.3521024677857938e-4, rel=1e-12)
    errs = []
    for ncut in (5, 20, 100, 1000):
        g = oracle.pair_accel(40.0, 0.0, 30.0, 1e-2, 100.0, 1.0, ncut)
        errs.append(abs(g[0] / float(grho) - 1.0))
    assert errs[0] == pytest.approx(3.7e-3, rel=0.1)
    for (n0, e0), (n1, e1) in zip(zip((5, 20, 100), errs), zip((20, 100, 1000), errs[1:])):
        assert e0 / e1 == pytest.approx((n1 / n0) ** 2, rel=0.15)


# ------------------------------------------------- P7: rod / infinite line-mass limit
def test_line_mass_limit(oracle):
    L, rho = 100.0, 1000.0
    g = oracle.pair_accel(rho, 0.0, 13.0, 1.0, L, 1.0, 50)
    rod = -(2.0 / (L * rho)) * 50 * L / math.sqrt(rho ** 2 + (50 * L) ** 2)
    assert g[0] == pytest.approx(rod, rel=1e-5)
    g = oracle.pair_accel(rho, 0.0, 13.0, 1.0, L, 1.0, 5000)
    assert g[0] == pytest.approx(-2.0 / (L * rho), rel=5e-6)        # 2 G (m/L) / R
    assert abs(g[2]) < 1e-6 * abs(g[0])


# ------------------------------------------------ P10: the paper's qualitative claim
def test_axial_weaker_radial_stronger(oracle):
    # S1xR2 forces are weaker than R^3 only axially, stronger radially
    L, s, ncut = 1.0, 0.17, 2000
    newton = 1.0 / s ** 2
    ax = abs(oracle.pair_accel(0.0, 0.0, s, 1e-4, L, 1.0, ncut)[2])
    ra = abs(oracle.pair_accel(s, 0.0, 0.0, 1e-4, L, 1.0, ncut)[0])
    assert ax < newton < ra
    u = mp.mpf(s)
    assert ax == pytest.approx(float(mp.psi(1, u) - mp.psi(1, 1 - u)), rel=1e-6)   # 33.742136
    assert ra == pytest.approx(-float(_bessel_series(s, 0.0, L)[0]), rel=1e-6)     # 34.996012


# ------------------------------------------------------- brute force + invariants
def _random_set(seed, n=48, L=10.0):
    rng = np.random.default_rng(seed)
    x, y = rng.normal(0, 4, n), rng.normal(0, 4, n)
    z = rng.uniform(-L, 2 * L, n)                 # deliberately outside [0, L)
    m = rng.uniform(0.2, 3.0, n)
    h = rng.uniform(0.05, 1.0, n)                 # many softened pairs
    return x, y, z, m, h, L


def test_accel_is_the_sum_of_pair_terms(oracle):
    x, y, z, m, h, L = _random_set(3)
    n, G, ncut = len(x), 0.7, 3
    gx, gy, gz = oracle.accel(x, y, z, m, h, L, G, ncut)
    ref = np.zeros((n, 3))
    for i in range(n):
        for j in range(n):
            if i != j:
                ref[i] += m[j] * oracle.pair_accel(x[i] - x[j], y[i] - y[j], z[i] - z[j],
                                                   h[i] + h[j], L, G, ncut)
    np.testing.assert_allclose(np.stack([gx, gy, gz], 1), ref, rtol=1e-12, atol=1e-14)
    # target subset = rows of the full result
    t = np.array([5, 17, 40], dtype=np.int64)
    sx, sy, sz = oracle.accel(x, y, z, m, h, L, G, ncut, targets=t)
    assert np.array_equal(sx, gx[t]) and np.array_equal(sy, gy[t]) and np.array_equal(sz, gz[t])
    # G scales linearly, negative G repels
    rx_, _, _ = oracle.accel(x, y, z, m, h, L, -G, ncut)
    np.testing.assert_allclose(rx_, -gx, rtol=1e-14)


def test_momentum_and_axial_angular_momentum_conserved(oracle):
    # translation along z and SO(2) about z => sum m g = 0, sum m (x g_y - y g_x) = 0
    x, y, z, m, h, L = _random_set(8, n=200)
    gx, gy, gz = oracle.accel(x, y, z, m, h, L, 1.0, 4)
    scale = np.sum(m * np.sqrt(gx ** 2 + gy ** 2 + gz ** 2))
    for comp in (gx, gy, gz):
        assert abs(np.sum(m * comp)) < 1e-14 * scale
    tz = np.sum(m * (x * gy - y * gx))
    assert abs(tz) < 1e-13 * np.sum(m * np.hypot(x, y) * np.hypot(gx, gy))


def test_rotation_about_axis(oracle):
    x, y, z, m, h, L = _random_set(9, n=100)
    gx, gy, gz = oracle.accel(x, y, z, m, h, L, 1.0, 3)
    th = 0.7345
    c, s = math.cos(th), math.sin(th)
    gx2, gy2, gz2 = oracle.accel(c * x - s * y, s * x + c * y, z, m, h, L, 1.0, 3)
    np.testing.assert_allclose(gx2, c * gx - s * gy, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(gy2, s * gx + c * gy, rtol=1e-10, atol=1e-13)
    np.testing.assert_allclose(gz2, gz, rtol=1e-10, atol=1e-13)


def test_golden_two_particle_values(oracle):
    """tests/golden/two_particle.txt: values from SURVEY.md 8(c) pin P2 (40-digit evaluation of
    Eq. 3 + Eq. 8 done while surveying).  A regression fixture, not an independent pin."""
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "two_particle.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    assert len(rows) >= 6
    for r in rows:
        rx, ry, rz, hh, L = map(float, r[:5])
        ncut = int(r[5])
        want = np.array(list(map(float, r[6:9])))
        got = oracle.pair_accel(rx, ry, rz, hh, L, 1.0, ncut)
        np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-300)


def test_golden_two_particle_provenance():
    """The stored values are reproduced by the committed 40-digit script (literal Eq. 8 window on the
    raw r_z -- a different route to the image set from the oracle's wrap + sign rule)."""
    import os, subprocess, sys
    script = os.path.join(os.path.dirname(__file__), "golden", "make_two_particle.py")
    r = subprocess.run([sys.executable, script, "--check"], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout + r.stderr
