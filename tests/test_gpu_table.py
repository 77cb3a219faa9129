"""GPU-vs-oracle parity of the EWALD_TABLE mode (Eq. 12-17): softened nearest image
+ interpolated correction table D, through the C ABI.  Bar: fp64, per-particle relative error
<= 1e-10 against oracle.accel_table evaluated with the ORACLE's own table."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200; there is no CPU fallback"
    return torch


def gpu_accel_table(torch, arrs, L, G, **kw):
    from paper_2602_20787_b200 import binding as b
    x, y, z, m, h = [np.ascontiguousarray(a, dtype=np.float64) for a in arrs]
    n = x.shape[0]
    ctx = b.StepsCyl(n=n, Lz=L, G=G, periodic_mode=b.PERIODIC_EWALD_TABLE, **kw)
    dev = [torch.from_numpy(a).cuda() for a in (x, y, z, m, h)]
    g = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
    ctx.accel(*dev, *g)
    ctx.check()
    out = [t.cpu().numpy() for t in g]
    ctx.close()
    return out


def rel_err(g, ref):
    g, ref = np.stack(g, 1), np.stack(ref, 1)
    return np.linalg.norm(g - ref, axis=1) / np.linalg.norm(ref, axis=1)


# tab_fp32 (float nodes, fp32 weighted sum) against the oracle interpolating the same float nodes in double
FP32_TABLE_MAX, FP32_TABLE_MEDIAN = 2e-6, 5e-8


@pytest.mark.parametrize("interp", [0, 1])
@pytest.mark.parametrize("cfg,n", [(0, 2048), (1, 6000)])
def test_table_mode_matches_oracle(torch_cuda, oracle, interp, cfg, n):
    from paper_2602_20787_b200 import workloads
    w = workloads.make(cfg, n=n)
    # config 0 lies inside the table (rho < 100 < rho_max); config 1 reaches r = 2000, so most pairs
    # of its outer particles take the line-mass branch
    nrho, nz, rmax = 72, 64, 300.0
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, nrho, nz, rmax)
    ref = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, rmax, interp)
    g = gpu_accel_table(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, tab_nrho=nrho, tab_nz=nz,
                        tab_rho_max=rmax, interp=interp)
    e = rel_err(g, ref)
    assert e.max() <= 1e-10, e.max()


def test_table_mode_defaults_and_clustered(torch_cuda, oracle):
    """Default table (144 x 128 nodes, rho_max = 5 L, (n_max, m_max) = (5, 12), alpha = 2/L) on the
    clustered config-4 recipe: softened pairs, spheres across z = 0 / L."""
    from paper_2602_20787_b200 import workloads
    w = workloads.make(4, n=12000)
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, 144, 128, 5.0 * w.Lz)
    ref = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, 5.0 * w.Lz, 0)
    g = gpu_accel_table(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G)
    assert rel_err(g, ref).max() <= 1e-10


def test_table_mode_degenerate_geometry(torch_cuda, oracle):
    L = 100.0
    x = np.array([0.0, 0.0, 3.0, 3.0, -7.0, 1.0, 1.0, 0.25, 40.0, 40.0, 700.0])
    y = np.array([0.0, 0.0, 4.0, 4.0, 2.0, 1.0, 1.0, 0.0, -9.0, -9.0, 0.0])
    z = np.array([10.0, 10.0, 10.0, 60.0, 110.0, -90.0, 0.0, 100.0, 250.0, -50.0, 33.0])
    m = np.array([1.0, 2.0, 0.5, 1.5, 1.0, 3.0, 1.0, 1.0, 2.0, 2.0, 4.0])
    h = np.array([0.5, 0.5, 0.2, 0.2, 1.0, 0.1, 0.1, 0.3, 0.4, 0.4, 1.0])
    nrho, nz, rmax = 40, 33, 450.0
    D = oracle.ewald_table(L, 2.0 / L, 5, 12, nrho, nz, rmax)
    for interp in (0, 1):
        for G in (1.0, -2.5):
            ref = oracle.accel_table(x, y, z, m, h, L, G, D, rmax, interp)
            g = gpu_accel_table(torch_cuda, (x, y, z, m, h), L, G, tab_nrho=nrho, tab_nz=nz,
                                tab_rho_max=rmax, interp=interp)
            assert rel_err(g, ref).max() <= 1e-10


def test_table_mode_tracks_the_many_image_sum(torch_cuda):
    """What the mode is for: it approximates the N_cut -> infinity sum that the images mode only
    reaches slowly (error ~ N_cut^-2).  Compared on the GPU itself: table mode vs images
    mode with N_cut = 40 and 5."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    torch = torch_cuda
    w = workloads.make(0, n=3000, seed=8)
    dev = [torch.from_numpy(a).cuda() for a in (w.x, w.y, w.z, w.m, w.h)]

    def images(nc):
        ctx = b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, n_cut=nc)
        g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
        ctx.accel(*dev, *g)
        ctx.check()
        ctx.close()
        return [t.cpu().numpy() for t in g]

    tab = gpu_accel_table(torch, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, tab_nrho=289, tab_nz=257,
                          tab_rho_max=120.0)
    e40, e5 = rel_err(tab, images(40)), rel_err(images(5), images(40))
    assert np.median(e40) < 0.2 * np.median(e5)


@pytest.mark.parametrize("interp", [0, 1])
def test_table_mode_fp32_table_in_shared_memory(torch_cuda, oracle, interp):
    """tab_fp32 = 1: the nodes are rounded to float and held in shared memory (512-thread CTAs, eight
    target tiles each); node indices and weights come from the fp64 coordinates, the weighted sum of the
    float nodes is taken in fp32, everything else stays double.  The oracle gets ITS table rounded the
    same way and interpolates in double.  Ragged N (not a multiple of 1024) and pairs beyond rho_max
    included."""
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1, n=7001, seed=31)
    nrho, nz, rmax = 144, 128, 5.0 * w.Lz
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, nrho, nz, rmax)
    D32 = D.astype(np.float32).astype(np.float64)
    ref = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D32, rmax, interp)
    g = gpu_accel_table(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, interp=interp, tab_fp32=1)
    # fp32 interpolation: at most ~4 float roundings (2.4e-7) of each pair's D, uncorrelated between pairs;
    # a particle's relative error is that times sqrt(sum D^2)/|sum|, largest where the sum nearly cancels
    e = rel_err(g, ref)
    assert e.max() <= FP32_TABLE_MAX and np.median(e) <= FP32_TABLE_MEDIAN, (e.max(), np.median(e))
    # and the float table + float interpolation change the answer itself only at this level
    ref64 = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, rmax, interp)
    assert rel_err(g, ref64).max() <= 1e-6


@pytest.mark.parametrize("interp", [0, 1])
def test_table_mode_mixed_precision(torch_cuda, oracle, interp):
    """EWALD_TABLE in mixed precision (float pair terms and float interpolation of the shared-memory
    float table, double accumulation across rings): the mixed-mode bar, RMS <= 1e-5 and max <= 1e-4."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    for cfg, n in [(1, 9000), (4, 12000)]:
        w = workloads.make(cfg, n=n)
        rmax = 5.0 * w.Lz
        D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, 144, 128, rmax).astype(np.float32).astype(np.float64)
        ref = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, rmax, interp)
        g = gpu_accel_table(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, interp=interp,
                            precision=b.PREC_MIXED)
        e = rel_err(g, ref)
        assert np.sqrt(np.mean(e ** 2)) <= 1e-5 and e.max() <= 1e-4, (e.max(), np.sqrt(np.mean(e ** 2)))


@pytest.mark.parametrize("seed", range(4))
def test_table_mode_randomised_parameters(torch_cuda, oracle, seed):
    rng = np.random.default_rng(7000 + seed)
    L = float(rng.choice([1.0, 77.7, 1.0e3]))
    n = int(rng.integers(200, 2500))
    G = float(rng.choice([1.0, -0.37, 6.5]))
    R = L * float(rng.choice([0.5, 3.0, 9.0]))
    r = R * np.sqrt(rng.random(n))
    phi = 2 * np.pi * rng.random(n)
    x, y = r * np.cos(phi), r * np.sin(phi)
    z = L * (rng.random(n) * 5.0 - 2.0)
    m = 10.0 ** rng.uniform(-1.0, 1.0, n)
    h = L * 0.05 * rng.uniform(0.2, 1.0, n)
    nrho, nz = int(rng.integers(20, 60)), int(rng.integers(17, 50))
    rmax = L * float(rng.choice([2.0, 4.0]))
    alpha = float(rng.choice([1.5, 2.0, 3.0])) / L
    interp = int(rng.integers(0, 2))
    D = oracle.ewald_table(L, alpha, 5, 12, nrho, nz, rmax)
    ref = oracle.accel_table(x, y, z, m, h, L, G, D, rmax, interp)
    g = gpu_accel_table(torch_cuda, (x, y, z, m, h), L, G, tab_nrho=nrho, tab_nz=nz, tab_rho_max=rmax,
                        interp=interp, ew_alpha=alpha)
    assert rel_err(g, ref).max() <= 1e-10
    D32 = D.astype(np.float32).astype(np.float64)
    ref32 = oracle.accel_table(x, y, z, m, h, L, G, D32, rmax, interp)
    g = gpu_accel_table(torch_cuda, (x, y, z, m, h), L, G, tab_nrho=nrho, tab_nz=nz, tab_rho_max=rmax,
                        interp=interp, ew_alpha=alpha, tab_fp32=1)
    e = rel_err(g, ref32)
    assert e.max() <= FP32_TABLE_MAX and np.median(e) <= FP32_TABLE_MEDIAN, (e.max(), np.median(e))
    from paper_2602_20787_b200 import binding as b
    g = gpu_accel_table(torch_cuda, (x, y, z, m, h), L, G, tab_nrho=nrho, tab_nz=nz, tab_rho_max=rmax,
                        interp=interp, ew_alpha=alpha, precision=b.PREC_MIXED)
    e = rel_err(g, ref32)
    assert np.sqrt(np.mean(e ** 2)) <= 1e-5 and e.max() <= 1e-4


def test_kdk_step_in_table_mode_is_the_same_leapfrog(torch_cuda, oracle):
    """steps_cyl_kdk_step is mode-agnostic plumbing around the force call: in EWALD_TABLE mode one step must
    equal the leapfrog of reading S4 written out here with the oracle's table-mode accelerations and its
    Eq. 10 background (the kick / drift formulas themselves are pinned in test_oracle_background_kdk.py)."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    torch = torch_cuda
    w = workloads.make(3, n=2500)
    c = w.cosmo
    nrho, nz, rmax = 48, 40, 400.0
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, nrho, nz, rmax)
    a0 = c["a_init"]
    H0 = oracle.hubble(a0, c["H0"], c["Om"], c["Or"], c["Ok"], c["OL"])
    a1, H1 = oracle.friedmann_rk4(a0, c["dt"], c["H0"], c["Om"], c["Or"], c["Ok"], c["OL"])
    dt = c["dt"]
    # oracle side, step by step (reading S4): kick1 + drift, force, kick2
    g0 = np.stack(oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, rmax, 0), 1)
    bx, by = oracle.background(w.x, w.y, w.R_sim, 0.0, w.G, w.rho0, 1)
    v = np.stack([w.vx, w.vy, w.vz], 1)
    acc = g0.copy(); acc[:, 0] += bx; acc[:, 1] += by
    v = v + 0.5 * dt * (acc / a0 ** 3 - 2.0 * H0 * v)
    x, y = w.x + v[:, 0] * dt, w.y + v[:, 1] * dt
    z = np.mod(w.z + v[:, 2] * dt, w.Lz)
    g1 = np.stack(oracle.accel_table(x, y, z, w.m, w.h, w.Lz, w.G, D, rmax, 0), 1)
    bx, by = oracle.background(x, y, w.R_sim, 0.0, w.G, w.rho0, 1)
    acc = g1.copy(); acc[:, 0] += bx; acc[:, 1] += by
    v = (v + 0.5 * dt * acc / a1 ** 3) / (1.0 + H1 * dt)
    # GPU side
    ctx = b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, periodic_mode=b.PERIODIC_EWALD_TABLE, tab_nrho=nrho, tab_nz=nz,
                     tab_rho_max=rmax, background=b.BG_INFINITE, R_sim=w.R_sim, rho0=w.rho0)
    dev = {k: torch.from_numpy(np.ascontiguousarray(getattr(w, k))).cuda()
           for k in ("x", "y", "z", "vx", "vy", "vz", "m", "h")}
    g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
    ctx.accel(dev["x"], dev["y"], dev["z"], dev["m"], dev["h"], *g)
    ctx.kdk_step(*[dev[k] for k in ("x", "y", "z", "vx", "vy", "vz", "m", "h")], *g, a0, H0, a1, H1, dt)
    ctx.check()
    ctx.close()
    gv = np.stack([dev[k].cpu().numpy() for k in ("vx", "vy", "vz")], 1)
    assert np.abs(dev["x"].cpu().numpy() - x).max() <= 1e-12 * np.abs(x).max()
    assert np.abs(gv - v).max() <= 1e-10 * np.abs(v).max()
    gg = np.stack([t.cpu().numpy() for t in g], 1)
    assert (np.linalg.norm(gg - g1, axis=1) / np.linalg.norm(g1, axis=1)).max() <= 1e-10


@pytest.mark.parametrize("interp", [0, 1])
@pytest.mark.parametrize("variant", ["double_global", "float_shared", "mixed"])
def test_table_mode_deterministic_rounds(torch_cuda, oracle, variant, interp):
    """STEPS_FLAG_DETERMINISTIC in EWALD_TABLE mode (pair_table_round.cuh): conflict-free rounds, plain stores.
    Same bars as the atomic kernels, bit-identical between runs, and equal to the atomic kernels up to
    the summation order.  Ragged N; n = 3000 gives 24 tiles (12 groups, 13 rounds), n = 700 one CTA."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    kw = dict(double_global=dict(), float_shared=dict(tab_fp32=1), mixed=dict(precision=b.PREC_MIXED))[variant]
    for cfg, n in [(1, 3000), (4, 700)]:
        w = workloads.make(cfg, n=n, seed=90 + n)
        arrs = (w.x, w.y, w.z, w.m, w.h)
        rmax = 5.0 * w.Lz
        D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, 144, 128, rmax)
        if variant != "double_global":
            D = D.astype(np.float32).astype(np.float64)
        ref = oracle.accel_table(*arrs, w.Lz, w.G, D, rmax, interp)
        g1 = gpu_accel_table(torch_cuda, arrs, w.Lz, w.G, interp=interp, flags=b.FLAG_DETERMINISTIC, **kw)
        g2 = gpu_accel_table(torch_cuda, arrs, w.Lz, w.G, interp=interp, flags=b.FLAG_DETERMINISTIC, **kw)
        for a, c in zip(g1, g2):
            assert np.array_equal(a, c)
        e = rel_err(g1, ref)
        if variant == "double_global":
            assert e.max() <= 1e-10
        elif variant == "float_shared":
            assert e.max() <= FP32_TABLE_MAX and np.median(e) <= FP32_TABLE_MEDIAN, (e.max(), np.median(e))
        else:
            assert np.sqrt(np.mean(e ** 2)) <= 1e-5 and e.max() <= 1e-4, (e.max(), np.sqrt(np.mean(e ** 2)))
        ga = gpu_accel_table(torch_cuda, arrs, w.Lz, w.G, interp=interp, **kw)
        assert rel_err(g1, ga).max() <= (1e-12 if variant != "mixed" else 1e-5)
        # Newton's third law survives the scheduling
        mom = max(abs(np.sum(w.m * g1[c])) / np.sum(w.m * np.abs(g1[c])) for c in range(3))
        assert mom <= (1e-13 if variant != "mixed" else 1e-6)


@pytest.mark.parametrize("variant", ["float_shared", "mixed", "float_shared_deterministic"])
def test_table_mode_bench_size_sampled_targets(torch_cuda, oracle, variant):
    """The table-mode configurations bench.py times (config 3 load, N = 1 048 576, 144 x 128 CIC, rho_max = 5 L,
    same launch configuration) on sampled targets the oracle computes one by one; momentum over ALL particles."""
    import os
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    n = int(os.environ.get("STEPS_TEST_BENCH_N", 1048576))
    w = workloads.make(3, n=n)
    idx = workloads.sample_targets(w.n, 128, seed=33)
    rmax = 5.0 * w.Lz
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, 144, 128, rmax).astype(np.float32).astype(np.float64)
    ref = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D, rmax, 0, targets=idx)
    kw = dict(float_shared=dict(tab_fp32=1), mixed=dict(precision=b.PREC_MIXED),
              float_shared_deterministic=dict(tab_fp32=1, flags=b.FLAG_DETERMINISTIC))[variant]
    g = gpu_accel_table(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, **kw)
    e = rel_err([c[idx] for c in g], ref)
    if variant == "mixed":
        assert np.sqrt(np.mean(e ** 2)) <= 1e-5 and e.max() <= 1e-4, (e.max(), np.sqrt(np.mean(e ** 2)))
    else:
        assert e.max() <= FP32_TABLE_MAX and np.median(e) <= FP32_TABLE_MEDIAN, (e.max(), np.median(e))
    for c in g:
        assert abs(np.sum(w.m * c)) <= (1e-11 if variant != "mixed" else 1e-5) * np.sum(w.m * np.abs(c))


def test_two_live_contexts_with_different_table_sizes(torch_cuda, oracle):
    """The dynamic shared-memory limit of the table kernels is a per-function, process-wide setting: a second
    context with a smaller float table must not lower it under the first one's feet."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    torch = torch_cuda
    w = workloads.make(0, n=1500, seed=4)
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.x, w.y, w.z, w.m, w.h)]
    shapes = [(144, 128, 500.0), (40, 33, 150.0)]
    ctxs = [b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, periodic_mode=b.PERIODIC_EWALD_TABLE, tab_fp32=1, tab_nrho=nr,
                       tab_nz=nz, tab_rho_max=rm) for nr, nz, rm in shapes]        # big first, then small
    for ctx, (nr, nz, rm) in zip(ctxs, shapes):
        D32 = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, nr, nz, rm).astype(np.float32).astype(np.float64)
        ref = oracle.accel_table(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, D32, rm, 0)
        g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
        ctx.accel(*dev, *g)
        ctx.check()
        e = rel_err([t.cpu().numpy() for t in g], ref)
        assert e.max() <= FP32_TABLE_MAX and np.median(e) <= FP32_TABLE_MEDIAN
    for ctx in ctxs:
        ctx.close()


@pytest.mark.parametrize("flags", [0, 8], ids=["plain", "graph"])
def test_table_mode_kdk_across_a_reordering(torch_cuda, oracle, flags):
    """EWALD_TABLE mode keeps its packed arrays in Morton order (order_kernels.cuh) and refreshes the order every 64
    force evaluations; inputs and outputs stay in the CALLER's order.  70 KDK steps cross a re-ordering: the final
    g must be the oracle's table-mode pair sum at the final positions, and m, h must come back untouched."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    torch = torch_cuda
    w = workloads.make(1, n=3001, seed=41)
    nrho, nz, rmax = 72, 64, 300.0
    ctx = b.StepsCyl(n=w.n, Lz=w.Lz, G=w.G, periodic_mode=b.PERIODIC_EWALD_TABLE, tab_nrho=nrho, tab_nz=nz,
                     tab_rho_max=rmax, flags=flags)
    dev = {k: torch.from_numpy(np.ascontiguousarray(getattr(w, k))).cuda() for k in ("x", "y", "z", "m", "h")}
    rng = np.random.default_rng(5)
    v = [torch.from_numpy(rng.normal(0, 0.05, w.n)).cuda() for _ in range(3)]
    g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
    ctx.accel(dev["x"], dev["y"], dev["z"], dev["m"], dev["h"], *g)
    for _ in range(70):
        ctx.kdk_step(dev["x"], dev["y"], dev["z"], *v, dev["m"], dev["h"], *g, 1.0, 0.0, 1.0, 0.0, 0.02)
    ctx.check()
    x, y, z = (dev[k].cpu().numpy() for k in ("x", "y", "z"))
    assert np.array_equal(dev["m"].cpu().numpy(), w.m) and np.array_equal(dev["h"].cpu().numpy(), w.h)
    assert np.abs(x - w.x).max() > 0.01 and z.min() >= 0.0 and z.max() < w.Lz
    D = oracle.ewald_table(w.Lz, 2.0 / w.Lz, 5, 12, nrho, nz, rmax)
    ref = oracle.accel_table(x, y, z, w.m, w.h, w.Lz, w.G, D, rmax, 0)
    assert rel_err([t.cpu().numpy() for t in g], ref).max() <= 1e-10
    ctx.close()
