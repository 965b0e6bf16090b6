"""poisson_solve_batch / poisson_solve_batch_host (several densities, one K^F, solves dealt to lanes with
their own intermediates and streams -- PAPER.md:53,89) against the oracle and against one-by-one solves."""
import numpy as np
import pytest

import oracle
from workloads import generators as gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pk():
    import torch
    import paper_1211_5244_b200 as pk
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the solve has no fallback")
    pk.load_library()
    torch.cuda.set_device(0)
    return pk


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def _even_kernel(rng, s):
    sx, sy, sz = s
    K = rng.standard_normal((sz, sy, sx))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    return K


@pytest.mark.parametrize("n,bc,prec", [((32, 32, 32), (0, 0, 0), "fp64"), ((24, 16, 32), (1, 0, 0), "fp64"),
                                       ((16, 8, 4), (0, 1, 0), "fp32")])
@pytest.mark.parametrize("wide", ["auto", "0", "3"])
def test_batch_matches_oracle_and_single_solves(pk, n, bc, prec, wide, monkeypatch):
    """wide = auto: small grids go several densities per launch; 0: the lane path; 3: chunks of 3 (7 = 3 + 3 + 1)."""
    import torch
    if wide != "auto":
        monkeypatch.setenv("POISSON_WIDE", wide)
    rng = np.random.default_rng(4242 + n[0])
    dt = np.float64 if prec == "fp64" else np.float32
    tol = 1e-12 if prec == "fp64" else 1e-5
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s)).astype(dt)
    count = 7                                                      # more solves than lanes, not a multiple of them
    rhos_np = [rng.standard_normal((n[2], n[1], n[0])).astype(dt) for _ in range(count)]
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64 if prec == "fp64" else pk.FP32)
    try:
        plan.set_kernel(torch.from_numpy(Kf).cuda())
        rhos = [torch.from_numpy(r).cuda() for r in rhos_np]
        Vs = plan.solve_batch(rhos)
        torch.cuda.synchronize()
        single = [plan.solve(r) for r in rhos]
        torch.cuda.synchronize()
        for i in range(count):
            ref = oracle.solve(rhos_np[i].astype(np.float64), Kf.astype(np.float64), bc)
            assert rel_l2(Vs[i].cpu().numpy().astype(np.float64), ref) <= tol, (i, n, bc, prec)
            assert rel_l2(Vs[i].cpu().numpy().astype(np.float64), single[i].cpu().numpy().astype(np.float64)) <= tol * 1e-2
        # in place (rho[i] == V[i]) and a second batch on the same lanes
        work = [r.clone() for r in rhos]
        plan.solve_batch(work, work)
        torch.cuda.synchronize()
        for i in range(count):
            assert torch.equal(work[i], Vs[i])                     # same kernels, same order: bitwise
        # host variant: H2D + passes + D2H per lane, returns with every V on the host
        hr = [torch.from_numpy(r).pin_memory() for r in rhos_np]
        hv = [torch.empty_like(h).pin_memory() for h in hr]
        plan.solve_batch_host(hr, hv)
        for i in range(count):
            assert torch.equal(hv[i], Vs[i].cpu())
        plan.solve_batch([], [])                                   # empty batch is a no-op
    finally:
        plan.close()


def test_batch_error_codes(pk):
    import ctypes
    import torch
    plan = pk.PoissonPlan((8, 8, 8), (0, 0, 0), 0.1, pk.FP64)
    rho = torch.zeros(8, 8, 8, dtype=torch.float64, device="cuda")
    lib = pk.load_library()
    arr = (ctypes.c_void_p * 1)(rho.data_ptr())
    assert lib.poisson_solve_batch(plan.handle, arr, arr, 1, None) == 4          # ENOKERNEL
    plan.set_kernel(torch.ones(16, 16, 9, dtype=torch.float64, device="cuda"))
    assert lib.poisson_solve_batch(plan.handle, arr, arr, -1, None) == 1         # EINVAL
    bad = (ctypes.c_void_p * 1)(rho.data_ptr() + 8)
    assert lib.poisson_solve_batch(plan.handle, bad, arr, 1, None) == 1          # misaligned
    assert lib.poisson_solve_batch(plan.handle, None, arr, 1, None) == 1         # null
    assert lib.poisson_solve_batch(plan.handle, arr, arr, 1, None) == 0          # K^F == 1: V = rho
    torch.cuda.synchronize()
    plan.close()


def test_wide_batch_more_densities_than_one_launch_takes(pk):
    """40 densities on a 16x8x12 grid: two launches' worth (32 + 8) through the several-densities-per-launch route,
    compared with one-by-one solves of the same plan."""
    import torch
    rng = np.random.default_rng(99)
    n, bc = (16, 8, 12), (0, 1, 0)
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
    try:
        plan.set_kernel(torch.from_numpy(Kf).cuda())
        rhos = [torch.from_numpy(rng.standard_normal((n[2], n[1], n[0]))).cuda() for _ in range(40)]
        Vs = plan.solve_batch(rhos)
        torch.cuda.synchronize()
        for i in (0, 1, 31, 32, 39):
            ref = oracle.solve(rhos[i].cpu().numpy(), Kf, bc)
            assert rel_l2(Vs[i].cpu().numpy(), ref) <= 1e-12
        for i in range(40):
            assert torch.equal(plan.solve(rhos[i]), Vs[i])     # same kernels, same arithmetic per tile: bitwise
    finally:
        plan.close()


def test_config1_batch_in_the_bench_configuration(pk):
    """configs[1] (128^3 -> 256^3 fp64) through poisson_solve_batch the way bench.py times it (device batch, 2 lanes,
    marshalled once): every V equals the single-stream solve of the same density bitwise (that solve is checked against the
    oracle in test_named_config_vs_oracle), and the shift property V = rho displaced holds for a delta kernel."""
    import torch
    cfg = gen.get_config("c1")
    rng = np.random.default_rng(7)
    n = cfg.n
    s = gen.padded_shape(n, cfg.bc)
    # K = delta at displacement d (and at -d, the kernel is inversion symmetric): K_f = 2 cos(2 pi k.d / S), analytic
    d = (3, 5, 7)
    kz = np.arange(s[2])[:, None, None] * d[2] / s[2]
    ky = np.arange(s[1])[None, :, None] * d[1] / s[1]
    kx = np.arange(s[0] // 2 + 1)[None, None, :] * d[0] / s[0]
    Kf = 2.0 * np.cos(2 * np.pi * (kx + ky + kz))
    plan = pk.PoissonPlan(n, cfg.bc, cfg.h, pk.FP64)
    try:
        plan.set_kernel(torch.from_numpy(Kf).cuda())
        assert plan.batch_width(8) == 0 and plan.batch_lanes(8) == 2 and plan.batch_lanes(8, host=True) == 3
        rhos = [torch.from_numpy(rng.standard_normal((n[2], n[1], n[0]))).cuda() for _ in range(8)]
        Vs = [torch.empty_like(r) for r in rhos]
        pb = plan.pointer_batch(rhos, Vs)
        plan.solve_pointer_batch(pb)
        plan.solve_pointer_batch(pb)
        torch.cuda.synchronize()
        for i in range(8):
            assert torch.equal(plan.solve(rhos[i]), Vs[i])
        r = rhos[3].cpu().numpy()
        exp = np.zeros_like(r)
        exp[d[2]:, d[1]:, d[0]:] += r[:-d[2], :-d[1], :-d[0]]          # zero fill on free axes: nothing wraps around
        exp[:-d[2], :-d[1], :-d[0]] += r[d[2]:, d[1]:, d[0]:]
        assert rel_l2(Vs[3].cpu().numpy(), exp) <= 1e-12
    finally:
        plan.close()


def test_lane_graphs_survive_a_kernel_switch(pk, monkeypatch):
    """Lane path in graph mode: solve_batch -> set_kernel_even -> solve_batch -> set_kernel_complex -> solve_batch ->
    set_kernel -> solve_batch.  Every kernel switch drops the lanes' instantiated graphs; the next batch must rebuild them
    (it used to launch a NULL graph exec and return ECUDA) and solve with the NEW kernel."""
    import torch
    monkeypatch.setenv("POISSON_WIDE", "0")      # small grid, but the lane route (as grids above 16 MB per lane take)
    monkeypatch.setenv("POISSON_GRAPH", "1")
    n, bc = (48, 32, 32), (0, 0, 0)
    rng = np.random.default_rng(99)
    s = gen.padded_shape(n, bc)
    Kf1 = oracle.kernel_spectrum(_even_kernel(rng, s))
    Kf2 = oracle.kernel_spectrum(_even_kernel(rng, s))
    rhos_np = [rng.standard_normal((n[2], n[1], n[0])) for _ in range(5)]
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
    try:
        assert plan.batch_width(5) == 0 and plan.batch_lanes(5) >= 2
        rhos = [torch.from_numpy(r).cuda() for r in rhos_np]

        def check(Kf):
            Vs = plan.solve_batch(rhos)
            torch.cuda.synchronize()
            for i in (0, 4):
                assert rel_l2(Vs[i].cpu().numpy(), oracle.solve(rhos_np[i], Kf, bc)) <= 1e-12

        plan.set_kernel(torch.from_numpy(Kf1).cuda());        check(Kf1)
        plan.set_kernel_even(torch.from_numpy(Kf2).cuda());   check(Kf2)
        plan.set_kernel_complex(torch.from_numpy(Kf1.astype(np.complex128)).cuda()); check(Kf1)
        plan.set_kernel(torch.from_numpy(Kf2).cuda());        check(Kf2)
    finally:
        plan.close()


@pytest.mark.parametrize("max_lanes,host", [(1, False), (2, True)], ids=["device_1_of_2", "host_2_of_3"])
def test_batch_falls_back_to_the_lanes_that_fit(pk, monkeypatch, max_lanes, host):
    """ensure_lanes running out of device memory (injected: POISSON_TEST_MAX_LANES) must not fail the batch: it runs on the
    lanes that could be allocated, the caller's stream stays ordered after them, and the results are those of single solves."""
    import torch
    monkeypatch.setenv("POISSON_WIDE", "0")
    monkeypatch.setenv("POISSON_TEST_MAX_LANES", str(max_lanes))
    n, bc = (32, 24, 40), (0, 0, 0)
    rng = np.random.default_rng(17)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, gen.padded_shape(n, bc)))
    rhos_np = [rng.standard_normal((n[2], n[1], n[0])) for _ in range(7)]
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
    try:
        plan.set_kernel(torch.from_numpy(Kf).cuda())
        assert plan.batch_lanes(7, host=host) > max_lanes          # more lanes wanted than the injected limit allows
        rhos = [torch.from_numpy(r).cuda() for r in rhos_np]
        singles = [plan.solve(r).clone() for r in rhos]
        torch.cuda.synchronize()
        if host:
            hin = [torch.from_numpy(r).pin_memory() for r in rhos_np]
            hout = [torch.empty_like(r).pin_memory() for r in hin]
            for rep in range(2):
                plan.solve_batch_host(hin, hout)
                for i in range(7):
                    assert torch.equal(hout[i], singles[i].cpu())
        else:
            for rep in range(2):
                Vs = plan.solve_batch(rhos)
                after = Vs[6] + 0            # queued on the caller's stream: must see the finished batch
                torch.cuda.synchronize()
                assert torch.equal(after, singles[6])
                for i in range(7):
                    assert torch.equal(Vs[i], singles[i])
        assert rel_l2(singles[3].cpu().numpy(), oracle.solve(rhos_np[3], Kf, bc)) <= 1e-12
    finally:
        plan.close()
