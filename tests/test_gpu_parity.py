"""GPU-vs-oracle parity of the all-pairs acceleration (steps_cyl_accel), through the C ABI.

Bars (BASELINE.json north_star):
  fp64  : per-particle relative error |g_gpu - g_ref|_2 / |g_ref|_2 <= 1e-10
  mixed : RMS over particles of that error <= 1e-5, max <= 1e-4
The oracle (oracle/steps_oracle.c) is evaluated on the same seeded inputs; nothing it gets
comes from the CUDA path.
"""
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

FP64_TOL = 1e-10
MIXED_RMS, MIXED_MAX = 1e-5, 1e-4


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200; there is no CPU fallback"
    return torch


def gpu_accel(torch, w_arrays, Lz, G, n_cut, precision=0, host=False, flags=0):
    from paper_2602_20787_b200 import binding as b
    x, y, z, m, h = [np.ascontiguousarray(a, dtype=np.float64) for a in w_arrays]
    n = x.shape[0]
    ctx = b.StepsCyl(n=n, Lz=Lz, G=G, n_cut=n_cut, precision=precision, flags=flags)
    try:
        if host:
            out = [np.empty(n) for _ in range(3)]
            ctx.accel_host(x, y, z, m, h, *out)
            return out
        dev = [torch.from_numpy(a).cuda() for a in (x, y, z, m, h)]
        g = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
        ctx.accel(*dev, *g)
        ctx.check()
        assert ctx.launch_count() >= 3        # prestep (pack), all-pairs kernel(s), poststep (reduction)
        return [t.cpu().numpy() for t in g]
    finally:
        ctx.close()


def rel_err(g, ref):
    g = np.stack(g, axis=1)
    ref = np.stack(ref, axis=1)
    return np.linalg.norm(g - ref, axis=1) / np.linalg.norm(ref, axis=1)


def check(g, ref, precision, idx=None):
    if idx is not None:
        g = [a[idx] for a in g]
    e = rel_err(g, ref)
    assert np.all(np.isfinite(e))
    if precision == 0:
        assert e.max() <= FP64_TOL, "fp64 max rel err %.3e" % e.max()
    else:
        rms = float(np.sqrt(np.mean(e ** 2)))
        assert rms <= MIXED_RMS and e.max() <= MIXED_MAX, "mixed rms %.3e max %.3e" % (rms, e.max())
    return e


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("host", [False, True])
def test_config0_full(torch_cuda, oracle, precision, host):
    from paper_2602_20787_b200 import workloads
    w = workloads.make(0)
    ref = oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, w.n_cut)
    g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, w.n_cut, precision, host)
    check(g, ref, precision)


@pytest.mark.parametrize("n", [1, 2, 127, 128, 129, 1000, 2500])
def test_ragged_sizes(torch_cuda, oracle, n):
    from paper_2602_20787_b200 import workloads
    w = workloads.make(0, n=n, seed=11 + n)
    ref = oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, 3)
    for precision in (0, 1):
        g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, 3, precision)
        if n == 1:
            assert all(float(a[0]) == 0.0 for a in g)     # no j != i: empty sum
        else:
            check(g, ref, precision)


@pytest.mark.parametrize("n_cut", [1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 40, 64, 65])
def test_n_cut_unrolled_and_runtime_loops(torch_cuda, oracle, n_cut):
    """N_cut <= 8: unrolled instances; 9 .. 64: run-time loop with tabulated per-image constants;
    above: run-time loop that forms them.  Every kernel family (atomic, rounds, ordered)."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1, n=1500, seed=5)
    ref = oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, n_cut)
    for precision in (0, 1):
        g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, n_cut, precision)
        check(g, ref, precision)
        if n_cut > 8:
            for flag in (b.FLAG_DETERMINISTIC, b.FLAG_ORDERED_PAIRS):
                g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, n_cut, precision, flags=flag)
                check(g, ref, precision)


@pytest.mark.parametrize("precision", [0, 1])
def test_config1_compactified_sampled_targets(torch_cuda, oracle, precision):
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1)
    idx = workloads.sample_targets(w.n, 3072, seed=1)
    ref = oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, w.n_cut, targets=idx)
    g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, w.n_cut, precision)
    check(g, ref, precision, idx)


@pytest.mark.parametrize("precision", [0, 1])
def test_clustered_softening_branches(torch_cuda, oracle, precision):
    """Config-4 recipe at reduced N: dense Plummer cores put many pairs in both spline branches,
    and spheres straddle z = 0 / L."""
    from paper_2602_20787_b200 import workloads
    w = workloads.make(4, n=24000)
    dx = w.x[:2000, None] - w.x[None, :2000]
    dy = w.y[:2000, None] - w.y[None, :2000]
    dz = w.z[:2000, None] - w.z[None, :2000]
    dz -= w.Lz * np.rint(dz / w.Lz)
    s = np.sqrt(dx ** 2 + dy ** 2 + dz ** 2)
    assert ((s > 0) & (s < 0.2)).sum() > 1000 and ((s > 0.2) & (s < 0.4)).sum() > 1000
    ref = oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, w.n_cut)
    g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, w.n_cut, precision)
    check(g, ref, precision)


def test_general_path_when_softening_reaches_other_images(torch_cuda, oracle):
    """2 max(h) > L/2: far images fall inside the spline support; the device picks the general
    kernel on its own (reading S7)."""
    rng = np.random.default_rng(77)
    n, L = 700, 10.0
    x, y = rng.normal(0, 3.0, n), rng.normal(0, 3.0, n)
    z = L * rng.random(n)
    m = rng.uniform(0.5, 2.0, n)
    h = rng.uniform(0.5, 6.0, n)
    assert 2 * h.max() > L / 2
    for n_cut in (1, 2, 5):
        ref = oracle.accel(x, y, z, m, h, L, 1.0, n_cut)
        for precision in (0, 1):          # mixed falls back to the fp64 general kernel
            g = gpu_accel(torch_cuda, (x, y, z, m, h), L, 1.0, n_cut, precision)
            check(g, ref, 0)


def test_degenerate_geometry(torch_cuda, oracle):
    """Coincident particles, equal z (r_z = 0: no end image), |r_z| = L/2 exactly, z outside
    [0, L) and exactly on the boundary, negative G."""
    L = 100.0
    x = np.array([0.0, 0.0, 3.0, 3.0, -7.0, 1.0, 1.0, 0.25, 40.0, 40.0])
    y = np.array([0.0, 0.0, 4.0, 4.0, 2.0, 1.0, 1.0, 0.0, -9.0, -9.0])
    z = np.array([10.0, 10.0, 10.0, 60.0, 110.0, -90.0, 0.0, 100.0, 250.0, -50.0])
    m = np.array([1.0, 2.0, 0.5, 1.5, 1.0, 3.0, 1.0, 1.0, 2.0, 2.0])
    h = np.array([0.5, 0.5, 0.2, 0.2, 1.0, 0.1, 0.1, 0.3, 0.4, 0.4])
    for G in (1.0, -2.5):
        for n_cut in (1, 5):
            ref = oracle.accel(x, y, z, m, h, L, G, n_cut)
            g = gpu_accel(torch_cuda, (x, y, z, m, h), L, G, n_cut, 0)
            check(g, ref, 0)
            gm = gpu_accel(torch_cuda, (x, y, z, m, h), L, G, n_cut, 1)
            assert rel_err(gm, ref).max() < 1e-4


def test_periodicity_and_momentum_on_the_gpu(torch_cuda):
    """Properties that hold at any size: shifting every z by L changes nothing;
    sum_i m_i g_i = 0."""
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1, n=5000, seed=9)
    g0 = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, 5, 0)
    g1 = gpu_accel(torch_cuda, (w.x, w.y, w.z + w.Lz, w.m, w.h), w.Lz, w.G, 5, 0)
    assert rel_err(g1, g0).max() < 1e-12
    for c in g0:
        assert abs(np.sum(w.m * c)) <= 1e-12 * np.sum(w.m * np.abs(c))


def test_nonpositive_softening_is_reported(torch_cuda):
    from paper_2602_20787_b200 import binding as b
    torch = torch_cuda
    n = 300
    rng = np.random.default_rng(1)
    arr = [torch.from_numpy(rng.random(n) * 10).cuda() for _ in range(5)]
    arr[4][17] = 0.0
    g = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
    ctx = b.StepsCyl(n=n, Lz=100.0)
    ctx.accel(*arr, *g)
    with pytest.raises(b.StepsError) as e:
        ctx.check()
    assert e.value.code == b.STEPS_ESOFT
    ctx.close()


@pytest.mark.parametrize("precision", [0, 1])
def test_bench_size_sampled_targets(torch_cuda, oracle, precision):
    """The configuration bench.py times (config 3 particle load, N = 1 048 576, n_cut = 5, same
    launch configuration), checked on sampled targets the oracle computes one by one."""
    from paper_2602_20787_b200 import workloads
    n = int(os.environ.get("STEPS_TEST_BENCH_N", 1048576))
    w = workloads.make(3, n=n)
    idx = workloads.sample_targets(w.n, 192, seed=3)
    ref = oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, w.G, w.n_cut, targets=idx)
    g = gpu_accel(torch_cuda, (w.x, w.y, w.z, w.m, w.h), w.Lz, w.G, w.n_cut, precision)
    check(g, ref, precision, idx)
    # momentum conservation over ALL particles (holds at any size)
    for c in g:
        assert abs(np.sum(w.m * c)) <= (1e-11 if precision == 0 else 1e-5) * np.sum(w.m * np.abs(c))


@pytest.mark.parametrize("n", [2, 129, 257, 700, 5000])
@pytest.mark.parametrize("flag", [1, 4])
def test_deterministic_kernels(torch_cuda, oracle, n, flag):
    """STEPS_FLAG_DETERMINISTIC (round-scheduled symmetric kernel, plain stores) and
    STEPS_FLAG_ORDERED_PAIRS (ordered pairs, fixed-order reduction): same parity bar, and bit-identical
    results from run to run."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1, n=n, seed=21)
    arrs = (w.x, w.y, w.z, w.m, w.h)
    ref = oracle.accel(*arrs, w.Lz, w.G, 5)
    g1 = gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 0, flags=flag)
    g2 = gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 0, flags=flag)
    check(g1, ref, 0)
    for a, c in zip(g1, g2):
        assert np.array_equal(a, c)
    # the default (symmetric, atomics) kernel agrees with it to round-off
    g3 = gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 0)
    assert rel_err(g3, g1).max() < 1e-12


@pytest.mark.parametrize("flag", [1, 4])
def test_deterministic_mixed_kernel(torch_cuda, oracle, flag):
    """Mixed precision with STEPS_FLAG_DETERMINISTIC (round-scheduled symmetric kernel) or
    STEPS_FLAG_ORDERED_PAIRS (ordered pairs, each contribution converted to double before it is
    added): bit-identical from run to run."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1, n=3000, seed=23)
    arrs = (w.x, w.y, w.z, w.m, w.h)
    ref = oracle.accel(*arrs, w.Lz, w.G, 5)
    g1 = gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 1, flags=flag)
    g2 = gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 1, flags=flag)
    check(g1, ref, 1)
    for a, c in zip(g1, g2):
        assert np.array_equal(a, c)


def test_far_order2_flag(torch_cuda, oracle):
    """STEPS_FLAG_FAR_ORDER2: far images refined to first order only -- still far inside the fp64 bar,
    but measurably less accurate than the default (which is at round-off)."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    w = workloads.make(1, n=6000, seed=17)
    arrs = (w.x, w.y, w.z, w.m, w.h)
    ref = oracle.accel(*arrs, w.Lz, w.G, 5)
    e_fast = check(gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 0, flags=b.FLAG_FAR_ORDER2), ref, 0)
    e_def = check(gpu_accel(torch_cuda, arrs, w.Lz, w.G, 5, 0), ref, 0)
    assert e_fast.max() < 2e-11 and e_def.max() < 1e-13


@pytest.mark.parametrize("seed", range(8))
def test_randomised_parameters(torch_cuda, oracle, seed):
    """Seeded random problem set-ups: period not representable in float, length scales from 1e-2 to
    1e4, either sign of G, masses over three decades, softenings up to the point where the general
    path takes over, z far outside [0, L), clustered and diffuse particles mixed."""
    rng = np.random.default_rng(4000 + seed)
    L = float(rng.choice([1.0, 77.7, 0.0123, 1.0e4, 100.0 / 3.0]))
    n = int(rng.integers(100, 2500))
    n_cut = int(rng.integers(1, 10))
    G = float(rng.choice([1.0, -0.37, 4.30091e-9, 6.5]))
    R = L * float(rng.choice([0.3, 2.0, 15.0]))
    r = R * rng.random(n) ** float(rng.choice([0.5, 2.0]))
    phi = 2 * np.pi * rng.random(n)
    x, y = r * np.cos(phi), r * np.sin(phi)
    z = L * (rng.random(n) * 7.0 - 3.0)                       # several periods either side
    k = n // 5                                                # a tight clump: softened pairs
    x[:k] = x[0] + 0.01 * L * rng.normal(size=k)
    y[:k] = y[0] + 0.01 * L * rng.normal(size=k)
    z[:k] = z[0] + 0.01 * L * rng.normal(size=k)
    m = 10.0 ** rng.uniform(-1.5, 1.5, n)
    hmax = L * float(rng.choice([0.002, 0.05, 0.12, 0.4]))    # 0.4 L: 2 hmax > L/2 -> general path
    h = hmax * rng.uniform(0.2, 1.0, n)
    ref = oracle.accel(x, y, z, m, h, L, G, n_cut)
    general = 2 * h.max() > L / 2
    for precision in (0, 1):
        g = gpu_accel(torch_cuda, (x, y, z, m, h), L, G, n_cut, precision)
        check(g, ref, 0 if general else precision)
    for flag in (1, 4):
        g = gpu_accel(torch_cuda, (x, y, z, m, h), L, G, n_cut, 0, flags=flag)
        check(g, ref, 0)
