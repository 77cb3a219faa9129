"""Pins of the oracle's Ewald / lookup-table path (Eq. 12-17; DESIGN.md readings
G4, T1-T3) against things other than itself: the exact Bessel-function series of the
one-axis-periodic point mass, a brute-force image sum, closed-form limits and the symmetries the
boundary rules encode.  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest

mp.mp.dps = 30


def bessel_series(rho, z, L):
    """Exact N_cut -> infinity force of a unit point mass periodic along z (textbook result,
    Poisson summation of 1/r): F_rho = -2/(L rho) - (4/L) sum_m k_m K_1(k_m rho) cos(k_m z),
    F_z = -(4/L) sum_m k_m K_0(k_m rho) sin(k_m z)."""
    rho, z, L = mp.mpf(rho), mp.mpf(z), mp.mpf(L)
    fr, fz = -2 / (L * rho), mp.mpf(0)
    for m in range(1, 2000):
        k = 2 * mp.pi * m / L
        tr = 4 / L * k * mp.besselk(1, k * rho) * mp.cos(k * z)
        tz = 4 / L * k * mp.besselk(0, k * rho) * mp.sin(k * z)
        fr -= tr
        fz -= tz
        if abs(tr) + abs(tz) < mp.mpf(10) ** -35:
            break
    return float(fr), float(fz)


@pytest.mark.parametrize("rho,z,L", [(0.3, 0.2, 1.0), (40.0, 30.0, 100.0), (5.0, 49.0, 100.0),
                                     (150.0, 10.0, 100.0), (12.0, -37.0, 100.0)])
@pytest.mark.parametrize("alphaL", [1.5, 2.0, 4.0])
def test_ewald_equals_exact_bessel_series(oracle, rho, z, L, alphaL):
    """(n_max, m_max) = (5, 12) (the paper's 'medium' setting) with the corrected
    Fourier kernel reproduces the exact sum for any reasonable alpha; the kernel B printed in
    Eq. 15 misses it by 1e-3 or more (reading G4)."""
    want = bessel_series(rho, z, L)
    got = oracle.ewald_force(rho, z, L, alphaL / L, 5, 12)
    assert got[0] == pytest.approx(want[0], rel=2e-11)
    assert got[1] == pytest.approx(want[1], rel=2e-11, abs=1e-18)


def test_ewald_equals_brute_force_image_sum(oracle):
    """Independent of any special function: the truncated image sum of Eq. 8 with many images,
    plus the analytic tail of the two missing half-lines (line-mass integral), converges to the
    Ewald value."""
    L, rho, z = 100.0, 23.0, 31.0
    ncut = 4000
    g = oracle.pair_accel(rho, 0.0, z, 1e-3, L, 1.0, ncut)
    # tail: images beyond +-N L act like a uniform line density 1/L from |d| = N L to infinity:
    # radial pull 2 * (1/L) * [1/rho - (N L)/(rho sqrt(rho^2 + (N L)^2))] ~ rho/(L (N L)^2)
    NL = ncut * L
    tail = 2.0 / (L * rho) * (1.0 - NL / math.sqrt(rho * rho + NL * NL))
    F = oracle.ewald_force(rho, z, L, 2.0 / L, 5, 12)
    assert F[0] == pytest.approx(g[0] - tail, rel=1e-9)
    assert F[1] == pytest.approx(g[2], rel=1e-7)


def test_ewald_alpha_independence_and_terms(oracle):
    """The split parameter only moves weight between Eq. 13 and Eq. 14: the total is the same;
    dropping the m = 0 term (Eq. 16) or the Fourier part is visible at the 10% level."""
    L = 100.0
    a = oracle.ewald_force(30.0, 20.0, L, 1.5 / L, 5, 12)
    b = oracle.ewald_force(30.0, 20.0, L, 3.0 / L, 5, 12)
    assert np.allclose(a, b, rtol=1e-11)
    no_fourier = oracle.ewald_force(30.0, 20.0, L, 3.0 / L, 5, 0)
    assert abs(no_fourier[1] - b[1]) > 0.05 * abs(b[1])
    # large rho: only the line-mass term survives (Eq. 16 with alpha rho >> 1)
    far = oracle.ewald_force(600.0, 17.0, L, 2.0 / L, 5, 12)
    assert far[0] == pytest.approx(-2.0 / (L * 600.0), rel=1e-12)
    assert abs(far[1]) < 1e-18


def test_D_is_ewald_minus_nearest_image_and_regular_at_origin(oracle):
    L, alpha = 100.0, 0.02
    for rho, z in [(10.0, 5.0), (3.0, -40.0), (70.0, 50.0), (0.5, 0.25)]:
        F = oracle.ewald_force(rho, z, L, alpha, 5, 12)
        r3 = (rho * rho + z * z) ** 1.5
        D = oracle.ewald_D(rho, z, L, alpha, 5, 12)
        assert D[0] == pytest.approx(F[0] + rho / r3, rel=1e-9, abs=1e-16)
        assert D[1] == pytest.approx(F[1] + z / r3, rel=1e-9, abs=1e-16)
    # the singular nearest-image term is gone: D -> 0 linearly at the origin, and the series used
    # for alpha r < 0.2 joins the closed form
    d1 = oracle.ewald_D(1e-3, 1e-3, L, alpha, 5, 12)
    d2 = oracle.ewald_D(2e-3, 2e-3, L, alpha, 5, 12)
    assert np.allclose(d2, 2 * d1, rtol=1e-5)
    assert np.all(np.abs(d1) < 1e-8)
    r_lo, r_hi = 0.2 / alpha * (1 - 1e-9), 0.2 / alpha * (1 + 1e-9)
    assert np.allclose(oracle.ewald_D(r_lo, 0.0, L, alpha, 5, 12), oracle.ewald_D(r_hi, 0.0, L, alpha, 5, 12),
                       rtol=1e-7)
    # on the axis (rho = 0) the radial part vanishes; at z = L/2 the FULL axial force vanishes by
    # symmetry, so D_z there is minus the nearest-image force (which jumps at z = L/2)
    assert oracle.ewald_D(0.0, 20.0, L, alpha, 5, 12)[0] == 0.0
    assert abs(oracle.ewald_force(15.0, 50.0, L, alpha, 5, 12)[1]) < 1e-17
    assert oracle.ewald_D(15.0, 50.0, L, alpha, 5, 12)[1] == pytest.approx(50.0 / (15.0 ** 2 + 50.0 ** 2) ** 1.5,
                                                                           rel=1e-12)


@pytest.fixture(scope="module")
def small_table(oracle):
    L, rho_max = 100.0, 300.0
    return L, rho_max, oracle.ewald_table(L, 2.0 / L, 5, 12, 25, 17, rho_max)


def test_table_nodes_and_interpolation_rules(oracle, small_table):
    L, rho_max, D = small_table
    nrho, nz = D.shape[:2]
    dr, dz = rho_max / (nrho - 1), 0.5 * L / (nz - 1)
    for (i, j) in [(0, 0), (3, 5), (24, 16), (7, 0), (0, 9)]:
        want = oracle.ewald_D(i * dr, j * dz, L, 2.0 / L, 5, 12)
        assert np.allclose(D[i, j], want, rtol=1e-12, atol=1e-20)
        # cloud-in-cell reproduces the nodes
        assert np.allclose(oracle.table_interp(D, rho_max, L, 0, i * dr, j * dz), D[i, j], rtol=1e-13, atol=1e-20)
    # CIC is the bilinear form between nodes
    got = oracle.table_interp(D, rho_max, L, 0, 3.25 * dr, 5.5 * dz)
    want = 0.75 * 0.5 * D[3, 5] + 0.25 * 0.5 * D[4, 5] + 0.75 * 0.5 * D[3, 6] + 0.25 * 0.5 * D[4, 6]
    assert np.allclose(got, want, rtol=1e-13)
    # TSC at a node is the (1/8, 3/4, 1/8) x (1/8, 3/4, 1/8) stencil
    w = np.array([0.125, 0.75, 0.125])
    want = np.einsum("a,b,abc->c", w, w, D[2:5, 4:7])
    assert np.allclose(oracle.table_interp(D, rho_max, L, 1, 3 * dr, 5 * dz), want, rtol=1e-13)
    # boundary rules = the symmetries of the true field: TSC on the axis gives no radial force and
    # at z = 0 no axial force (at z = L/2 D_z is odd but jumps, like the nearest-image force)
    assert abs(oracle.table_interp(D, rho_max, L, 1, 0.0, 7.3 * dz)[0]) < 1e-20
    assert abs(oracle.table_interp(D, rho_max, L, 1, 5.2 * dr, 0.0)[1]) < 1e-20
    # and interpolation converges to the function it tabulates (second order)
    e = []
    for n in (13, 25):
        Dn = oracle.ewald_table(L, 2.0 / L, 5, 12, n, 2 * (n - 1) // 3 + 1, rho_max)
        got = oracle.table_interp(Dn, rho_max, L, 0, 61.0, 17.0)
        e.append(np.abs(got - oracle.ewald_D(61.0, 17.0, L, 2.0 / L, 5, 12)).max())
    assert e[1] < e[0] / 2.5


def test_accel_table_two_particles_and_far_branch(oracle, small_table):
    L, rho_max, D = small_table
    x = np.array([0.0, 30.0, 400.0])
    y = np.array([0.0, 40.0, 0.0])
    z = np.array([10.0, 95.0, 50.0])
    m = np.array([2.0, 3.0, 5.0])
    h = np.array([0.5, 0.5, 0.5])
    G = 1.7
    g = np.stack(oracle.accel_table(x, y, z, m, h, L, G, D, rho_max, 0), 1)
    # particle 0 <- particle 1: r = (-30, -40, 15) after wrapping (10 - 95 + 100), rho = 50
    Dv = oracle.table_interp(D, rho_max, L, 0, 50.0, 15.0)
    s3 = (2500.0 + 225.0) ** 1.5
    f01 = np.array([30.0 / s3 - Dv[0] * 30 / 50, 40.0 / s3 - Dv[0] * 40 / 50, -15.0 / s3 + Dv[1]])
    # particle 0 <- particle 2: rho = 400 >= rho_max: line mass, no axial force
    f02 = np.array([2.0 / (L * 400.0), 0.0, 0.0])
    assert np.allclose(g[0], G * (3.0 * f01 + 5.0 * f02), rtol=1e-12)
    # antisymmetry of the pair law: total momentum is conserved
    assert np.all(np.abs((m[:, None] * g).sum(0)) < 1e-15 * np.abs(m[:, None] * g).sum(0))


def test_accel_table_approaches_many_image_sum(oracle):
    """With a fine table the table mode reproduces the image sum of Eq. 8 with very many images
    (the thing it approximates), up to interpolation error and the O(rho/N^2) truncation tail."""
    from paper_2602_20787_b200 import workloads
    w = workloads.make(0, n=160, seed=5)
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, 145, 97, 150.0)
    ref = np.stack(oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, 3000), 1)
    got = np.stack(oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, 150.0, 0), 1)
    err = np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)
    assert err.max() < 2e-3 and np.median(err) < 3e-4
