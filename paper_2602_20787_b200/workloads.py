"""Seeded synthetic particle loads for the five BASELINE.json configs.

This module holds INPUT GENERATION ONLY -- none of the method's arithmetic (no
spline, no image sum, no integrator).  It is the one module that both the CUDA
path's tests/bench and the oracle's tests may import, and it imports neither.

The particle sets stand in for the paper's workloads -- compactified cylindrical
LCDM particle loads made by the glass + stepsic2 pipeline (PAPER.md:205-250,
Sect. 3; Table 1) -- whose IC files and CAMB spectra do not exist
in this environment.  Shapes, sizes and value distributions follow BASELINE.json
`configs`; the recipes are stated in DESIGN.md ("Input recipe").

Every generator draws from numpy.random.default_rng(seed) in the order written
here, so a (config, n, seed) triple always gives bit-identical arrays.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

LZ = 100.0          # periodic length along z, all configs
R_CORE = 20.0       # radius of the constant-resolution core (compactified layout)
N_CUT_DEFAULT = 5   # DESIGN.md reading S3: the paper states no default N_cut

CONFIG_N = {0: 2048, 1: 32768, 2: 262144, 3: 1048576, 4: 4194304}


@dataclass
class Workload:
    name: str
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    m: np.ndarray
    h: np.ndarray
    Lz: float = LZ
    G: float = 1.0
    n_cut: int = N_CUT_DEFAULT
    R_sim: float = 0.0
    rho0: float = 0.0
    vx: np.ndarray | None = None
    vy: np.ndarray | None = None
    vz: np.ndarray | None = None
    cosmo: dict = field(default_factory=dict)

    @property
    def n(self) -> int:
        return int(self.x.shape[0])


def sample_targets(n: int, k: int, seed: int) -> np.ndarray:
    """k distinct, sorted particle indices (the targets the oracle is evaluated on)."""
    k = min(k, n)
    rng = np.random.default_rng(1000003 + seed)
    return np.sort(rng.choice(n, size=k, replace=False)).astype(np.int64)


# --------------------------------------------------------------------- config 0
def uniform_cylinder(n: int = 2048, seed: int = 0, R: float = 50.0, eps: float = 0.5) -> Workload:
    rng = np.random.default_rng(seed)
    r = R * np.sqrt(rng.random(n))
    phi = 2.0 * np.pi * rng.random(n)
    z = LZ * rng.random(n)
    return Workload("cfg0_uniform_cylinder", r * np.cos(phi), r * np.sin(phi), z,
                    np.ones(n), np.full(n, eps), R_sim=R)


# --------------------------------------------------------------------- config 1
def _compactified_radii(rng, n, r_max):
    """Cross-sectional number density flat for r < R_CORE, falling as r^-2 out to r_max."""
    lnr = math.log(r_max / R_CORE)
    f_in = 1.0 / (1.0 + 2.0 * lnr)
    u = rng.random(n)
    inner = u < f_in
    r = np.where(inner, R_CORE * np.sqrt(u / f_in),
                 R_CORE * np.exp((u - f_in) / (1.0 - f_in) * lnr))
    return r, inner


def compactified(n: int = 32768, seed: int = 1, r_max: float = 2000.0, eps_in: float = 0.2,
                 jitter: float = 0.01, name: str = "cfg1_compactified") -> Workload:
    rng = np.random.default_rng(seed)
    r, inner = _compactified_radii(rng, n, r_max)
    phi = 2.0 * np.pi * rng.random(n)
    z = LZ * rng.random(n)
    m = np.maximum(1.0, (r / R_CORE) ** 2)
    h = eps_in * np.cbrt(m)
    n_in = max(int(inner.sum()), 1)
    d0 = (math.pi * R_CORE ** 2 * LZ / n_in) ** (1.0 / 3.0)      # inner mean spacing
    x = r * np.cos(phi)
    y = r * np.sin(phi)
    sig = jitter * d0 * np.cbrt(m)
    x = x + sig * rng.standard_normal(n)
    y = y + sig * rng.standard_normal(n)
    z = np.mod(z + sig * rng.standard_normal(n), LZ)
    w = Workload(name, x, y, z, m, h, R_sim=r_max)
    w.cosmo["d0"] = d0
    w.cosmo["n_in"] = n_in
    return w


# --------------------------------------------------------------------- config 2
def _zeldovich_field(rng, qx, qy, qz, d0, n_modes=256, k_min=2.0 * math.pi / 1000.0):
    """psi(q) = sum_s A_s khat_s sin(k_s.q + theta_s): a Gaussian-like random displacement
    field with P(k) ~ k^-2 (|psi_k| ~ k^-2; modes log-uniform in k, hence A ~ k^-1/2),
    k_z snapped to multiples of 2 pi / LZ so the field is periodic along z.
    Returns the un-normalised (psi_x, psi_y, psi_z)."""
    k_max = math.pi / d0
    k = np.exp(rng.uniform(math.log(k_min), math.log(k_max), n_modes))
    mu = rng.uniform(-1.0, 1.0, n_modes)
    az = rng.uniform(0.0, 2.0 * math.pi, n_modes)
    theta = rng.uniform(-math.pi, math.pi, n_modes)
    st = np.sqrt(1.0 - mu * mu)
    kx, ky, kz = k * st * np.cos(az), k * st * np.sin(az), k * mu
    kz = np.round(kz / (2.0 * math.pi / LZ)) * (2.0 * math.pi / LZ)
    kk = np.sqrt(kx * kx + ky * ky + kz * kz)
    kk = np.where(kk > 0.0, kk, 1.0)
    amp = kk ** -0.5
    K = np.stack([kx, ky, kz])                                  # (3, M)
    W = (amp / kk) * K                                          # (3, M) = A_s khat_s
    n = qx.shape[0]
    psi = np.empty((n, 3))
    step = 16384
    for s in range(0, n, step):
        e = min(s + step, n)
        Q = np.stack([qx[s:e], qy[s:e], qz[s:e]], axis=1)       # (c, 3)
        ph = Q @ K + theta[None, :]
        np.sin(ph, out=ph)
        psi[s:e] = ph @ W.T
    return psi[:, 0], psi[:, 1], psi[:, 2]


def zeldovich(n: int = 262144, seed: int = 2, r_max: float = 2000.0, rms_in_d0: float = 0.5,
              name: str = "cfg2_zeldovich") -> Workload:
    w = compactified(n, seed, r_max, name=name)
    rng = np.random.default_rng(seed + 7919)
    d0 = w.cosmo["d0"]
    px, py, pz = _zeldovich_field(rng, w.x, w.y, w.z, d0)
    inner = np.hypot(w.x, w.y) < R_CORE
    rms = math.sqrt(float(np.mean(px[inner] ** 2 + py[inner] ** 2 + pz[inner] ** 2)))
    s = rms_in_d0 * d0 / rms
    w.cosmo["psi"] = (px * s, py * s, pz * s)
    w.x = w.x + px * s
    w.y = w.y + py * s
    w.z = np.mod(w.z + pz * s, LZ)
    return w


# --------------------------------------------------------------------- config 3
H0_UNITS = 100.0                    # km/s/(Mpc/h)
G_UNITS = 4.30091e-9                # Mpc (km/s)^2 / Msun
RHO_CRIT = 2.77536627e11            # (Msun/h) / (Mpc/h)^3


def lcdm_kdk(n: int = 1048576, seed: int = 3, r_max: float = 1000.0, a_init: float = 0.02,
             a_final: float = 0.025, n_steps: int = 10, Om: float = 0.3, OL: float = 0.7) -> Workload:
    """Comoving LCDM load: Mpc/h, km/s, Msun/h; Zel'dovich positions and velocities at a_init."""
    w = zeldovich(n, seed, r_max, name="cfg3_lcdm_kdk")
    rho_bar = Om * RHO_CRIT
    n_in = w.cosmo["n_in"]
    m_in = rho_bar * math.pi * R_CORE ** 2 * LZ / n_in
    w.m = w.m * m_in                                             # uniform mass density rho_bar
    w.G = G_UNITS
    w.rho0 = rho_bar
    w.R_sim = r_max
    E = lambda a: math.sqrt(Om / a ** 3 + OL)
    H_init = H0_UNITS * E(a_init)
    Om_a = Om / a_init ** 3 / E(a_init) ** 2
    f_growth = Om_a ** 0.55
    px, py, pz = w.cosmo.pop("psi")
    w.vx, w.vy, w.vz = (H_init * f_growth) * px, (H_init * f_growth) * py, (H_init * f_growth) * pz
    # t(a) = int da / (a H): Gauss-Legendre on [a_init, a_final] (smooth integrand)
    xg, wg = np.polynomial.legendre.leggauss(48)
    aa = 0.5 * (a_final - a_init) * xg + 0.5 * (a_final + a_init)
    t_span = 0.5 * (a_final - a_init) * float(np.sum(wg / (aa * H0_UNITS * np.sqrt(Om / aa ** 3 + OL))))
    w.cosmo.update(dict(H0=H0_UNITS, Om=Om, OL=OL, Or=0.0, Ok=0.0, a_init=a_init, a_final=a_final,
                        n_steps=n_steps, dt=t_span / n_steps))
    return w


# --------------------------------------------------------------------- config 4
def clustered(n: int = 4194304, seed: int = 4, n_spheres: int = 512, scale: float = 0.3,
              bg_frac: float = 0.2, r_max: float = 2000.0) -> Workload:
    rng = np.random.default_rng(seed)
    n_bg = int(round(bg_frac * n))
    n_cl = n - n_bg
    bg = compactified(n_bg, seed + 104729, r_max)
    mass = 10.0 ** rng.uniform(0.0, 2.0, n_spheres)
    cnt = np.floor(mass / mass.sum() * n_cl).astype(np.int64)
    cnt[np.argmax(cnt)] += n_cl - int(cnt.sum())
    zc = LZ * rng.random(n_spheres)
    rc = 200.0 * np.sqrt(rng.random(n_spheres))
    pc = 2.0 * np.pi * rng.random(n_spheres)
    cx = np.repeat(rc * np.cos(pc), cnt)
    cy = np.repeat(rc * np.sin(pc), cnt)
    cz = np.repeat(zc, cnt)
    # Plummer radii: r = scale / sqrt(u^(-2/3) - 1), re-drawn beyond 30
    rr = np.empty(n_cl)
    todo = np.arange(n_cl)
    while todo.size:
        u = rng.random(todo.size)
        u = np.where(u > 0.0, u, 0.5)
        val = scale / np.sqrt(u ** (-2.0 / 3.0) - 1.0)
        ok = val <= 30.0
        rr[todo[ok]] = val[ok]
        todo = todo[~ok]
    mu = rng.uniform(-1.0, 1.0, n_cl)
    az = rng.uniform(0.0, 2.0 * np.pi, n_cl)
    st = np.sqrt(1.0 - mu * mu)
    x = np.concatenate([cx + rr * st * np.cos(az), bg.x])
    y = np.concatenate([cy + rr * st * np.sin(az), bg.y])
    z = np.concatenate([np.mod(cz + rr * mu, LZ), bg.z])
    m = np.concatenate([np.ones(n_cl), bg.m])
    h = np.concatenate([np.full(n_cl, 0.2), bg.h])
    w = Workload("cfg4_clustered", x, y, z, m, h, R_sim=r_max)
    w.cosmo["n_clustered"] = n_cl
    return w


# ------------------------------------------- paper-faithful particle load (Sect. 3.1, Eq. 21-22)
def stereographic_load(n_target: int = 200000, D_s: float = 70.0, R_sim: float = 500.0,
                       omega_c: float = 1.63973, Lz: float = 500.0, rho_bar: float = 1.0,
                       eps_core: float | None = None, seed: int = 5) -> Workload:
    """Initial particle load of the cylindrical StePS geometry: the radial
    coordinate is compactified by the inverse stereographic map omega = 2 arctan(rho/D_s) (Eq. 21), the
    compact domain is tessellated uniformly in (omega, phi, z), one particle sits at a random place in
    each cell and carries m_i = rho_bar V_i with V_i the cell's volume in the non-compact
    (rho, phi, z) coordinates; inside the core omega < omega_c the mass resolution is constant
    (equal-volume cells).  Positions come back through rho = D_s tan(omega/2) (Eq. 22).
    Defaults are the parameters of the paper's Fig. 4 (rho_c = D_s tan(omega_c/2) = 75.0 Mpc) at a
    reduced particle number.  Softening: eps_core m^(1/3) scaling as in the BASELINE configs."""
    rng = np.random.default_rng(seed)
    rho_c = D_s * math.tan(0.5 * omega_c)
    omega_max = 2.0 * math.atan(R_sim / D_s)
    # cell sizes: d_omega, d_phi, d_z chosen so that the first ring outside the core is roughly cubic
    # and the total count is close to n_target
    jac_c = 0.5 * D_s / math.cos(0.5 * omega_c) ** 2                 # d rho / d omega at omega_c
    def counts(cell):                                              # cell = physical edge at rho_c
        n_z = max(1, round(Lz / cell))
        n_phi = max(4, round(2.0 * math.pi * rho_c / cell))
        n_om = max(1, round((omega_max - omega_c) / (cell / jac_c)))
        v_first = 0.5 * ((D_s * math.tan(0.5 * (omega_c + (omega_max - omega_c) / n_om))) ** 2 - rho_c ** 2) \
            * (2.0 * math.pi / n_phi) * (Lz / n_z)
        n_r = max(1, round(math.pi * rho_c ** 2 * Lz / v_first / (n_phi * n_z)))
        return n_z, n_phi, n_om, n_r
    lo, hi = 1e-3 * rho_c, 10.0 * rho_c
    for _ in range(60):                                            # bisection on the cell edge
        mid = math.sqrt(lo * hi)
        n_z, n_phi, n_om, n_r = counts(mid)
        if n_z * n_phi * (n_om + n_r) > n_target:
            lo = mid
        else:
            hi = mid
    n_z, n_phi, n_om, n_r = counts(hi)
    d_phi, d_z = 2.0 * math.pi / n_phi, Lz / n_z
    # outer region: uniform rings in omega
    om_edges = np.linspace(omega_c, omega_max, n_om + 1)
    rho_edges_out = D_s * np.tan(0.5 * om_edges)
    # core: rings of equal area (constant mass resolution)
    rho_edges_in = rho_c * np.sqrt(np.linspace(0.0, 1.0, n_r + 1))
    xs, ys, zs, ms = [], [], [], []
    for compact, edges in ((False, rho_edges_in), (True, rho_edges_out)):
        nr = len(edges) - 1
        shape = (nr, n_phi, n_z)
        u = rng.random(shape)
        if compact:      # random place in the COMPACT cell: uniform in omega
            om = om_edges[:-1, None, None] + u * np.diff(om_edges)[:, None, None]
            rho = D_s * np.tan(0.5 * om)
        else:            # equal-volume core cell: uniform in rho^2
            rho = np.sqrt(edges[:-1, None, None] ** 2 + u * np.diff(edges ** 2)[:, None, None])
        phi = (np.arange(n_phi)[None, :, None] + rng.random(shape)) * d_phi
        z = (np.arange(n_z)[None, None, :] + rng.random(shape)) * d_z
        vol = 0.5 * np.diff(edges ** 2)[:, None, None] * d_phi * d_z * np.ones(shape)
        xs.append((rho * np.cos(phi)).ravel()); ys.append((rho * np.sin(phi)).ravel())
        zs.append(z.ravel()); ms.append((rho_bar * vol).ravel())
    x, y, z, m = map(np.concatenate, (xs, ys, zs, ms))
    m_core = float(ms[0].ravel()[0])
    if eps_core is None:
        eps_core = 0.05 * (m_core / rho_bar) ** (1.0 / 3.0)         # 1/20 of the core particle spacing
    h = eps_core * np.cbrt(m / m_core)
    w = Workload("stereographic_load", x, y, z, m, h, Lz=Lz, R_sim=R_sim, rho0=rho_bar)
    w.cosmo.update(dict(rho_c=rho_c, omega_max=omega_max, n_core=int(ms[0].size), n_outer=int(ms[1].size),
                        cells=(n_r, n_om, n_phi, n_z), m_core=m_core))
    return w


def make(config: int, n: int | None = None, seed: int | None = None) -> Workload:
    """The BASELINE.json config `config` (0..4), optionally at a reduced particle count."""
    gens = {0: uniform_cylinder, 1: compactified, 2: zeldovich, 3: lcdm_kdk, 4: clustered}
    kw = {}
    if n is not None:
        kw["n"] = int(n)
    if seed is not None:
        kw["seed"] = int(seed)
    return gens[config](**kw)
