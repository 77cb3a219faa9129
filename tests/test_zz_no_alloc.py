"""steps_cyl_accel_noalloc: the force evaluation for callers that cannot allocate (include/steps_cyl.h).

Collected LAST on purpose (the suite runs with `pytest -x`: a failure here must not hide another test).
The entry point needs no context and calls no cudaMalloc: its scratch is one static device array of
STEPS_CYL_NOALLOC_MAX_N particle slots that every call shares and that keeps the previous call's contents.
So the GPU test makes calls IN A ROW with different sizes and parameters and checks each against the existing
path (steps_cyl_accel on a context) at the tolerance the other tests use between two fp64 kernels (1e-12), and
against the oracle at the fp64 bar (1e-10)."""
import ctypes as C

import numpy as np
import pytest

KERNEL_VS_KERNEL = 1e-12        # as tests/test_gpu_parity.py: default kernel vs deterministic kernel
FP64_TOL = 1e-10                # north_star bar against the oracle


def _rel(got, ref):
    return np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)


def test_noalloc_rejects_before_touching_the_gpu():
    """Sizes beyond the fixed capacity and bad arguments are refused up front (no device needed)."""
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import build
    build.build()
    lib = b.lib()
    one = C.c_void_p(8)                    # any non-NULL value: it is never dereferenced on these paths
    ptrs = [one] * 8
    assert lib.steps_cyl_accel_noalloc(b.NOALLOC_MAX_N + 1, 100.0, 1.0, 5, *ptrs, None) == b.STEPS_ETOOBIG
    assert lib.steps_cyl_accel_noalloc(10 ** 9, 100.0, 1.0, 5, *ptrs, None) == b.STEPS_ETOOBIG
    assert "STEPS_CYL_NOALLOC_MAX_N" in lib.steps_cyl_strerror(b.STEPS_ETOOBIG).decode()
    assert lib.steps_cyl_accel_noalloc(0, 100.0, 1.0, 5, *ptrs, None) == b.STEPS_EINVAL
    assert lib.steps_cyl_accel_noalloc(16, 0.0, 1.0, 5, *ptrs, None) == b.STEPS_EINVAL
    assert lib.steps_cyl_accel_noalloc(16, 100.0, 1.0, 0, *ptrs, None) == b.STEPS_EINVAL
    assert lib.steps_cyl_accel_noalloc(16, 100.0, 1.0, 5, *([None] + ptrs[1:]), None) == b.STEPS_EINVAL
    hdr = open(__file__.replace("tests/test_zz_no_alloc.py", "include/steps_cyl.h")).read()
    assert "#define STEPS_CYL_NOALLOC_MAX_N ((int64_t)%d)" % b.NOALLOC_MAX_N in hdr


@pytest.mark.gpu
def test_noalloc_matches_the_existing_path_on_calls_in_a_row(oracle):
    import torch
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    assert torch.cuda.is_available(), "this test needs the B200; there is no CPU fallback"

    # (workload, n_cut, G): the capacity itself, then a much smaller set with other parameters (stale contents of
    # the shared array beyond its n must not matter), then a ragged size whose softenings reach the far images
    # (2 max h > L/2: the general pair law, chosen on the device from the flag block the call clears)
    rng = np.random.default_rng(71)
    big = workloads.make(1, n=b.NOALLOC_MAX_N, seed=61)
    small = workloads.make(1, n=1301, seed=62)
    soft = workloads.make(0, n=700, seed=63)
    soft.h = rng.uniform(5.0, 30.0, soft.n)
    cases = [(big, 5, 1.0), (small, 3, -2.5), (soft, 2, 1.0), (small, 5, 1.0)]

    def existing(w, n_cut, G):
        dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.x, w.y, w.z, w.m, w.h)]
        g = [torch.empty(w.n, dtype=torch.float64, device="cuda") for _ in range(3)]
        ctx = b.StepsCyl(n=w.n, Lz=w.Lz, G=G, n_cut=n_cut)
        ctx.accel(*dev, *g)
        ctx.check()
        ctx.close()
        return np.stack([t.cpu().numpy() for t in g], 1)

    refs = [existing(w, nc, G) for w, nc, G in cases]
    ins = [[torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.x, w.y, w.z, w.m, w.h)] for w, _, _ in cases]
    outs = [[torch.full((w.n,), float("nan"), dtype=torch.float64, device="cuda") for _ in range(3)] for w, _, _ in cases]

    def run_all():
        for (w, nc, G), i, o in zip(cases, ins, outs):
            b.accel_noalloc(w.n, w.Lz, G, nc, *i, *o)          # back to back on one stream, no sync in between
        torch.cuda.synchronize()

    run_all()                                                   # first pass: set-up + lazy kernel loading
    free_before = torch.cuda.mem_get_info()[0]
    for o in outs:
        for t in o:
            t.fill_(float("nan"))
    run_all()                                                   # second pass: the array holds the first pass's data
    free_after = torch.cuda.mem_get_info()[0]
    assert free_after >= free_before, "the no-allocation entry point took device memory"

    for (w, nc, G), o, ref in zip(cases, outs, refs):
        got = np.stack([t.cpu().numpy() for t in o], 1)
        assert np.all(np.isfinite(got))
        e = _rel(got, ref)
        assert e.max() <= KERNEL_VS_KERNEL, "N=%d n_cut=%d: %.3e vs the existing path" % (w.n, nc, e.max())
    # and against the oracle itself where it finishes in seconds
    for k in (1, 2):
        w, nc, G = cases[k]
        ref = np.stack(oracle.accel(w.x, w.y, w.z, w.m, w.h, w.Lz, G, nc), 1)
        got = np.stack([t.cpu().numpy() for t in outs[k]], 1)
        assert _rel(got, ref).max() <= FP64_TOL

    # one more particle than the capacity: refused, nothing launched, the outputs untouched
    n_big = b.NOALLOC_MAX_N + 1
    t = [torch.zeros(n_big, dtype=torch.float64, device="cuda") for _ in range(8)]
    with pytest.raises(b.StepsError) as err:
        b.accel_noalloc(n_big, 100.0, 1.0, 5, *t)
    assert err.value.code == b.STEPS_ETOOBIG
    torch.cuda.synchronize()
    assert all(float(a.abs().max()) == 0.0 for a in t[5:])


@pytest.mark.gpu
def test_noalloc_can_be_captured_in_a_cuda_graph():
    """What the entry point is for: after one ordinary call (the one-time set-up), a call under stream capture
    records one memset and three kernels and nothing else; replaying the graph on new inputs written into the same
    buffers gives what steps_cyl_accel gives for them."""
    import torch
    from paper_2602_20787_b200 import binding as b
    from paper_2602_20787_b200 import workloads
    assert torch.cuda.is_available(), "this test needs the B200; there is no CPU fallback"
    wa = workloads.make(1, n=4000, seed=81)
    wb = workloads.make(1, n=4000, seed=82)
    n, L, G, nc = wa.n, wa.Lz, 1.0, 5
    ins = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (wa.x, wa.y, wa.z, wa.m, wa.h)]
    out = [torch.zeros(n, dtype=torch.float64, device="cuda") for _ in range(3)]
    b.accel_noalloc(n, L, G, nc, *ins, *out)                 # set-up happens here, outside capture
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        b.accel_noalloc(n, L, G, nc, *ins, *out)             # torch's current stream is the capturing stream
    ctx = b.StepsCyl(n=n, Lz=L, G=G, n_cut=nc)
    ref = [torch.empty(n, dtype=torch.float64, device="cuda") for _ in range(3)]
    for w in (wa, wb, wa):
        for t, a in zip(ins, (w.x, w.y, w.z, w.m, w.h)):
            t.copy_(torch.from_numpy(np.ascontiguousarray(a)))
        for t in out:
            t.fill_(float("nan"))
        graph.replay()
        ctx.accel(*ins, *ref)
        ctx.check()
        got = np.stack([t.cpu().numpy() for t in out], 1)
        want = np.stack([t.cpu().numpy() for t in ref], 1)
        assert np.all(np.isfinite(got)) and _rel(got, want).max() <= KERNEL_VS_KERNEL
    ctx.close()
