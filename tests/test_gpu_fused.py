"""The one-launch fused solve kernel (csrc/solve_kernel.cuh: F1 | F2 -> F3 -> I2 per plane | I1 in one
cooperative launch) against the CPU oracle, and against the 5-launch path on the same inputs."""
import os

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


def _solve(pk, rho, Kf, n, bc, prec, fused, repeats=1):
    import torch
    dt = np.float64 if prec == "fp64" else np.float32
    old = os.environ.get("POISSON_FUSED")
    os.environ["POISSON_FUSED"] = "1" if fused else "0"
    try:
        plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64 if prec == "fp64" else pk.FP32)
    finally:
        if old is None:
            del os.environ["POISSON_FUSED"]
        else:
            os.environ["POISSON_FUSED"] = old
    try:
        J, R = plan.graph_shape()      # the tuner may keep a shaped graph (parallel chains) when not fused
        assert plan.launches_per_solve() == (1 if fused else (5 if (J, R) == (1, 1) else 2 * R + 2 * R * J + J))
        plan.set_kernel(torch.from_numpy(np.ascontiguousarray(Kf.astype(dt))).cuda())
        r = torch.from_numpy(np.ascontiguousarray(rho.astype(dt))).cuda()
        outs = []
        for _ in range(repeats):   # back-to-back solves: the kernel must re-arm its own counters
            outs.append(plan.solve(r))
        torch.cuda.synchronize()
        return [o.cpu().numpy().astype(np.float64) for o in outs]
    finally:
        plan.close()


# (n, bc, precisions): combinations with a compiled fused kernel (csrc/fused_*.cu)
FUSED_CASES = [
    ((4, 4, 4), (0, 0, 0), ("fp64", "fp32")),
    ((8, 8, 8), (0, 0, 0), ("fp64",)),
    ((16, 16, 16), (1, 1, 1), ("fp64",)),
    ((16, 16, 16), (0, 0, 0), ("fp64", "fp32")),
    ((6, 24, 12), (0, 0, 0), ("fp64",)),          # three different lengths 12 / 48 / 24, ragged tiles
    ((32, 32, 32), (0, 0, 0), ("fp64", "fp32")),
]


@pytest.mark.parametrize("n,bc,precs", FUSED_CASES, ids=lambda v: "x".join(map(str, v)) if isinstance(v, tuple) and isinstance(v[0], int) else None)
def test_fused_kernel_vs_oracle_and_vs_five_launches(pk, n, bc, precs):
    rng = np.random.default_rng(77 + sum(n))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
    for prec in precs:
        tol = 1e-12 if prec == "fp64" else 1e-5
        if prec == "fp32":
            r_in, k_in = rho.astype(np.float32).astype(np.float64), Kf.astype(np.float32).astype(np.float64)
        else:
            r_in, k_in = rho, Kf
        ref = oracle.solve(r_in, k_in, bc)
        outs = _solve(pk, rho, Kf, n, bc, prec, fused=True, repeats=3)
        for V in outs:
            assert rel_l2(V, ref) <= tol, (n, bc, prec)
        assert np.array_equal(outs[0], outs[1]) and np.array_equal(outs[0], outs[2])   # bitwise repeatable
        five = _solve(pk, rho, Kf, n, bc, prec, fused=False)[0]
        # same butterflies, but two separately compiled kernels may contract multiply-adds differently
        assert rel_l2(outs[0], five) <= (1e-14 if prec == "fp64" else 1e-6)


@pytest.mark.parametrize("key", ["c0", "c1", "c2", "c3"])
def test_named_configs_run_fused(pk, key):
    """configs[0..3] take the one-launch path, and it matches the oracle."""
    cfg = gen.get_config(key)
    rho = gen.gaussian_density(cfg)
    K = gen.green_kernel_realspace(cfg.n, cfg.bc, cfg.h, cfg.images)
    Kf = oracle.kernel_spectrum(K)
    V = _solve(pk, rho, Kf, cfg.n, cfg.bc, "fp64", fused=True, repeats=2)
    ref = oracle.solve(rho, Kf, cfg.bc)
    assert rel_l2(V[0], ref) <= 1e-12 and np.array_equal(V[0], V[1])


@pytest.mark.parametrize("pdl", [False, True])
def test_graph_launch_mode_matches_five_launches_bitwise(pk, monkeypatch, pdl):
    """POISSON_GRAPH=1: the five launches as one CUDA graph launch (rho / V patched into the F1 / I1 nodes per call).
    Same kernels, same arithmetic: bitwise equal to the five stream launches, also when the buffers change between
    calls and when rho == V."""
    import torch
    rng = np.random.default_rng(31)
    n, bc = (24, 16, 32), (0, 1, 0)
    s = gen.padded_shape(n, bc)
    Kf = torch.from_numpy(rng.standard_normal((s[2], s[1], s[0] // 2 + 1))).cuda()
    rhos = [torch.from_numpy(rng.standard_normal((n[2], n[1], n[0]))).cuda() for _ in range(3)]
    monkeypatch.setenv("POISSON_TUNE", "0")
    ref_plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64)
    ref_plan.set_kernel(Kf)
    assert ref_plan.launch_mode()[0] == "five"
    refs = [ref_plan.solve(r).clone() for r in rhos]
    ref_plan.close()
    monkeypatch.setenv("POISSON_GRAPH", "1")
    if pdl:
        monkeypatch.setenv("POISSON_PDL", "1")     # graph captured from the PDL launches: programmatic edges
    plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64)
    try:
        plan.set_kernel(Kf)
        assert plan.launch_mode()[0] == ("graph_pdl" if pdl else "graph")
        outs = [torch.empty_like(r) for r in rhos]
        for rep in range(2):
            for r, o, ref in zip(rhos, outs, refs):
                plan.solve(r, o)
                assert torch.equal(o, ref)
        w = rhos[1].clone()
        plan.solve(w, w)                                   # in place
        assert torch.equal(w, refs[1])
        s2 = torch.cuda.Stream()
        with torch.cuda.stream(s2):
            plan.solve(rhos[2], outs[0], stream=s2)        # another stream, another (rho, V) pair
        s2.synchronize()
        assert torch.equal(outs[0], refs[2])
    finally:
        plan.close()


@pytest.mark.parametrize("n,bc,prec", [((24, 16, 32), (0, 0, 0), "fp64"), ((32, 24, 16), (1, 1, 0), "fp64"), ((16, 40, 12), (0, 0, 1), "fp32"),
                                       ((15, 9, 14), (0, 1, 0), "fp64")])
@pytest.mark.parametrize("mode", ["five", "graph", "graph_pdl"])
def test_plane_chunked_middle_passes(pk, monkeypatch, n, bc, prec, mode):
    """Large grids run F2 -> F3 -> I2 chunk by chunk of k_a planes through an A2 buffer that holds one chunk (csrc/api.cu:
    for_each_launch).  Forced here on small grids (POISSON_CHUNK = planes per chunk, ragged last chunk): the result equals the
    unchunked plan's bitwise (same kernels, same arithmetic per tile) and matches the oracle, in every launch mode and through
    the batch lanes."""
    import torch
    dt = np.float64 if prec == "fp64" else np.float32
    rng = np.random.default_rng(606 + sum(n))
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s)).astype(dt)
    rhos_np = [rng.standard_normal((n[2], n[1], n[0])).astype(dt) for _ in range(3)]
    monkeypatch.setenv("POISSON_TUNE", "0")
    if mode != "five":
        monkeypatch.setenv("POISSON_GRAPH", "1")
    if mode == "graph_pdl":
        monkeypatch.setenv("POISSON_PDL", "1")
    prec_id = pk.FP64 if prec == "fp64" else pk.FP32
    ref_plan = pk.PoissonPlan(n, bc, 0.3, prec_id)
    ref_plan.set_kernel(torch.from_numpy(Kf).cuda())
    rhos = [torch.from_numpy(r).cuda() for r in rhos_np]
    refs = [ref_plan.solve(r).clone() for r in rhos]
    assert ref_plan.launches_per_solve() == 5
    ref_plan.close()
    monkeypatch.setenv("POISSON_CHUNK", "3")
    plan = pk.PoissonPlan(n, bc, 0.3, prec_id)
    try:
        planes = plan.info.half_len
        assert plan.launches_per_solve() == 2 + 3 * ((planes + 2) // 3)
        assert plan.launch_mode()[0] == mode
        plan.set_kernel(torch.from_numpy(Kf).cuda())
        for rep in range(2):
            for r, ref in zip(rhos, refs):
                assert torch.equal(plan.solve(r), ref)
        err = rel_l2(refs[0].cpu().numpy().astype(np.float64), oracle.solve(rhos_np[0].astype(np.float64), Kf.astype(np.float64), bc))
        assert err <= (1e-12 if prec == "fp64" else 1e-5)
        monkeypatch.setenv("POISSON_WIDE", "0")
        for v, ref in zip(plan.solve_batch(rhos), refs):          # batch lanes carry their own chunk-sized A2
            torch.cuda.synchronize()
            assert torch.equal(v, ref)
        for i in range(4):
            plan.solve_profiled(rhos[0], refs[0].clone())
        ms, cnt = plan.profile_read()
        assert cnt == 4 and all(m > 0 for m in ms)
        with pytest.raises(pk.PoissonError) as ei:
            plan.debug_workspace(1)
        assert ei.value.status == 2                                # A2 is never whole in memory on a chunked plan
    finally:
        plan.close()


MODE_ENV = {"five": {"POISSON_TUNE": "0"}, "five_pdl": {"POISSON_PDL": "1"}, "graph": {"POISSON_GRAPH": "1"},
            "graph_pdl": {"POISSON_GRAPH": "1", "POISSON_PDL": "1"}, "fused": {"POISSON_FUSED": "1"}}


@pytest.mark.parametrize("mode", list(MODE_ENV))
@pytest.mark.parametrize("n", [(16, 8, 4), (24, 16, 32), (32, 32, 32), (20, 40, 36), (7, 12, 10)], ids=lambda n: "x".join(map(str, n)))
def test_every_launch_mode_all_bc_vs_oracle(pk, monkeypatch, n, mode):
    """poisson_plan_create normally keeps whichever launch mode its timing run found fastest, so a sweep only exercises the
    winner.  Here every mode is FORCED in turn (all 8 BC combinations per size, compiled and any-length kernels) and compared
    with the oracle; the mode actually used is asserted (the fused kernel exists only for the combinations of csrc/fused.def
    and falls back to five launches elsewhere)."""
    import itertools
    import torch
    for k, v in MODE_ENV[mode].items():
        monkeypatch.setenv(k, v)
    rng = np.random.default_rng(2024 + sum(n))
    used = set()
    for bc in itertools.product((0, 1), repeat=3):
        s = gen.padded_shape(n, bc)
        rho = rng.standard_normal((n[2], n[1], n[0]))
        Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
        plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
        try:
            got_mode = plan.launch_mode()[0]
            used.add(got_mode)
            assert got_mode == mode or (mode == "fused" and got_mode == "five")
            plan.set_kernel(torch.from_numpy(Kf).cuda())
            r = torch.from_numpy(rho).cuda()
            V1 = plan.solve(r).cpu().numpy()
            V2 = plan.solve(r).cpu().numpy()              # a second solve on the same plan (counters / graph nodes re-armed)
        finally:
            plan.close()
        assert np.array_equal(V1, V2)
        assert rel_l2(V1, oracle.solve(rho, Kf, bc)) <= 1e-12, (n, bc, mode)
    print(n, mode, "modes used:", sorted(used))


SHAPES = [(2, 1), (3, 1), (4, 1), (1, 2), (2, 2), (2, 4), (3, 2)]


@pytest.mark.parametrize("pdl", [False, True], ids=["graph", "graph_pdl"])
@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: f"J{s[0]}R{s[1]}")
def test_shaped_graph_bitwise_and_vs_oracle(pk, monkeypatch, shape, pdl):
    """The solve graph as parallel chains (poisson_plan_graph_shape: J ranges of k_a planes, R ranges of x), FORCED with
    POISSON_BRANCHES / POISSON_XCHAINS: same kernels on the same tiles, so the result is bitwise the five stream launches';
    it is also compared with the oracle.  Grids: x last-processed with whole tiles per x range (R applies), surface
    boundary conditions and an odd N_x (R must fall back to 1), rho / V changing between calls, rho == V, another stream."""
    import torch
    J, R = shape
    # x ranges need whole tiles: 128 x values = 4 ranges of 2 P = 32 reals in F1 / I1 (S = 64: 8 threads per pencil, P = 16)
    # the surface grid processes x second: its chains run over ranges of z (F1 / I1's group index, F2 / I2's pencil index), 64 = 4 x 16 pencils
    cases = [((128, 32, 32), (0, 0, 0), True), ((128, 32, 64), (0, 0, 1), True), ((64, 16, 64), (1, 1, 0), True), ((64, 64, 12), (1, 0, 0), True),
             ((32, 24, 16), (1, 1, 0), False), ((15, 12, 10), (0, 1, 0), False)]
    for n, bc, x_ok in cases:
        rng = np.random.default_rng(77 + sum(n) + J + 10 * R)
        s = gen.padded_shape(n, bc)
        Kf_np = oracle.kernel_spectrum(_even_kernel(rng, s))
        rhos_np = [rng.standard_normal((n[2], n[1], n[0])) for _ in range(3)]
        Kf = torch.from_numpy(Kf_np).cuda()
        rhos = [torch.from_numpy(r).cuda() for r in rhos_np]
        for k in ("POISSON_GRAPH", "POISSON_PDL", "POISSON_BRANCHES", "POISSON_XCHAINS"):
            monkeypatch.delenv(k, raising=False)
        monkeypatch.setenv("POISSON_TUNE", "0")
        ref_plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64)
        ref_plan.set_kernel(Kf)
        assert ref_plan.launch_mode()[0] == "five" and ref_plan.graph_shape() == (1, 1)
        refs = [ref_plan.solve(r).clone() for r in rhos]
        ref_plan.close()
        monkeypatch.setenv("POISSON_GRAPH", "1")
        monkeypatch.setenv("POISSON_BRANCHES", str(J))
        monkeypatch.setenv("POISSON_XCHAINS", str(R))
        if pdl:
            monkeypatch.setenv("POISSON_PDL", "1")
        plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64)
        try:
            plan.set_kernel(Kf)
            assert plan.launch_mode()[0] == ("graph_pdl" if pdl else "graph")
            want_r = R if x_ok else 1
            assert plan.graph_shape() == (J, want_r), (n, bc, plan.graph_shape())
            if J > 1 or want_r > 1:
                assert plan.launches_per_solve() == 2 * want_r + 2 * want_r * J + J
            outs = [torch.empty_like(r) for r in rhos]
            for rep in range(2):
                for r, o, ref in zip(rhos, outs, refs):
                    plan.solve(r, o)
                    assert torch.equal(o, ref), (n, bc, shape)
            w = rhos[1].clone()
            plan.solve(w, w)                                   # in place
            assert torch.equal(w, refs[1])
            s2 = torch.cuda.Stream()
            with torch.cuda.stream(s2):
                plan.solve(rhos[2], outs[0], stream=s2)
            s2.synchronize()
            assert torch.equal(outs[0], refs[2])
            for v, ref in zip(plan.solve_batch(rhos), refs):   # the batch lanes keep plain chains
                torch.cuda.synchronize()
                assert torch.equal(v, ref)
        finally:
            plan.close()
        assert rel_l2(refs[0].cpu().numpy(), oracle.solve(rhos_np[0], Kf_np, bc)) <= 1e-12


def test_tuner_reports_graph_shape(pk):
    """poisson_plan_create times a few graph shapes with the launch modes; whatever it keeps is reported consistently."""
    import torch
    plan = pk.PoissonPlan((64, 64, 64), (0, 0, 0), 0.2, pk.FP64)
    try:
        mode, ms = plan.launch_mode()
        J, R = plan.graph_shape()
        print("launch mode", mode, "graph shape", (J, R), ms)
        assert J >= 1 and R >= 1
        if mode not in ("graph", "graph_pdl"):
            assert (J, R) == (1, 1)
        if (J, R) != (1, 1):
            assert plan.launches_per_solve() == 2 * R + 2 * R * J + J
        rng = np.random.default_rng(5)
        Kf = oracle.kernel_spectrum(_even_kernel(rng, (128, 128, 128)))
        rho = rng.standard_normal((64, 64, 64))
        plan.set_kernel(torch.from_numpy(Kf).cuda())
        V = plan.solve(torch.from_numpy(rho).cuda()).cpu().numpy()
    finally:
        plan.close()
    assert rel_l2(V, oracle.solve(rho, Kf, (0, 0, 0))) <= 1e-12


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_even_kernel_folded_storage(pk, monkeypatch, prec):
    """poisson_set_kernel_even (less K^F traffic): K^F of a kernel that is even along every axis is kept for
    the pencils k_b <= S_b / 2 only; pass F3 reads the mirror pencil's values for the rest.  Same values, same arithmetic:
    bitwise the result of poisson_set_kernel, for all 8 BCs (contiguous and strided F3, ragged tiles), in a forced graph of
    parallel chains, through the batch route and plane chunks; the K^F buffer shrinks; switching back and forth works; a kernel
    that is NOT even per axis differs (the evenness is the caller's statement)."""
    import itertools
    import torch
    dt = np.float64 if prec == "fp64" else np.float32
    prec_id = pk.FP64 if prec == "fp64" else pk.FP32
    for n, env in (((24, 16, 32), {}), ((20, 40, 36), {"POISSON_GRAPH": "1", "POISSON_BRANCHES": "3"}), ((32, 12, 20), {"POISSON_CHUNK": "4"})):
        for k in ("POISSON_GRAPH", "POISSON_BRANCHES", "POISSON_CHUNK"):
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        for bc in itertools.product((0, 1), repeat=3):
            rng = np.random.default_rng(4242 + sum(n) + sum(b << i for i, b in enumerate(bc)))
            s = gen.padded_shape(n, bc)
            Kf = oracle.kernel_spectrum(_even_kernel(rng, s)).astype(dt)
            # the computed spectrum is even along y and z up to rounding only: make it so exactly (a + b == b + a), so that
            # the mirror pencil holds the SAME values and the comparison below can be bitwise
            Kf = 0.5 * (Kf + np.roll(np.flip(Kf, axis=1), 1, axis=1))
            Kf = np.ascontiguousarray(0.5 * (Kf + np.roll(np.flip(Kf, axis=0), 1, axis=0))).astype(dt)
            rhos = [torch.from_numpy(rng.standard_normal((n[2], n[1], n[0])).astype(dt)).cuda() for _ in range(3)]
            Kf_t = torch.from_numpy(Kf).cuda()
            plan = pk.PoissonPlan(n, bc, 0.25, prec_id)
            try:
                plan.set_kernel(Kf_t)
                refs = [plan.solve(r).clone() for r in rhos]
                plan.solve_batch(rhos)                         # the batch route allocates its own intermediates: before the sizes are compared
                torch.cuda.synchronize()
                full_ws = plan.workspace_bytes()
                plan.set_kernel_even(Kf_t)
                assert plan.workspace_bytes() <= full_ws      # whole tiles of pencils are kept: tiny planes may not shrink
                for rep in range(2):
                    for r, ref in zip(rhos, refs):
                        assert torch.equal(plan.solve(r), ref), (n, bc, prec)
                for v, ref in zip(plan.solve_batch(rhos), refs):
                    torch.cuda.synchronize()
                    assert torch.equal(v, ref)
                plan.set_kernel(Kf_t)                       # back to the full layout
                assert plan.workspace_bytes() == full_ws
                assert torch.equal(plan.solve(rhos[0]), refs[0])
            finally:
                plan.close()
            if bc == (0, 1, 0) and not env:
                ref = oracle.solve(rhos[0].cpu().numpy().astype(np.float64), Kf.astype(np.float64), bc)
                assert rel_l2(refs[0].cpu().numpy().astype(np.float64), ref) <= (1e-12 if prec == "fp64" else 1e-5)
    # a grid with many tiles per plane: the K^F copy shrinks to (S_b / 2 + 1) / S_b of its size, rounded up to whole tiles
    plan = pk.PoissonPlan((64, 64, 64), (0, 0, 0), 0.2, prec_id)
    try:
        rng = np.random.default_rng(8)
        Kf_t = torch.from_numpy(rng.standard_normal((128, 128, 65)).astype(dt)).cuda()
        Kf_t = 0.5 * (Kf_t + torch.roll(torch.flip(Kf_t, dims=(1,)), 1, dims=(1,))).contiguous()     # even along y (= axis b)
        rho = torch.from_numpy(rng.standard_normal((64, 64, 64)).astype(dt)).cuda()
        plan.set_kernel(Kf_t)
        full_ws = plan.workspace_bytes()
        ref = plan.solve(rho).clone()
        plan.set_kernel_even(Kf_t)
        k_bytes = 65 * 128 * 128 * (8 if prec == "fp64" else 4)
        assert full_ws - plan.workspace_bytes() >= 0.3 * k_bytes
        assert torch.equal(plan.solve(rho), ref)
    finally:
        plan.close()
    # inversion symmetric but not even per axis: the folded copy is a different kernel
    n, bc = (8, 12, 4), (0, 1, 0)
    rng = np.random.default_rng(5)
    s = gen.padded_shape(n, bc)
    K = rng.standard_normal((s[2], s[1], s[0]))
    K = 0.5 * (K + np.roll(np.flip(K, axis=(0, 1, 2)), 1, axis=(0, 1, 2)))
    Kf_t = torch.from_numpy(oracle.kernel_spectrum(K).astype(dt)).cuda()
    rho = torch.from_numpy(rng.standard_normal((n[2], n[1], n[0])).astype(dt)).cuda()
    plan = pk.PoissonPlan(n, bc, 0.3, prec_id)
    try:
        plan.set_kernel(Kf_t)
        a = plan.solve(rho).clone()
        plan.set_kernel_even(Kf_t)
        assert not torch.equal(plan.solve(rho), a)
    finally:
        plan.close()


def test_fused_mode_comes_back_after_an_even_kernel(pk, monkeypatch):
    """poisson_set_kernel_even drops the one-launch FUSED mode (that kernel reads the full K^F layout); poisson_set_kernel
    afterwards must put the plan back into the mode it was created in, as include/poisson.h says ("switches back")."""
    import torch
    monkeypatch.setenv("POISSON_FUSED", "1")
    n, bc = (32, 32, 32), (0, 0, 0)
    rng = np.random.default_rng(31)
    Kf = torch.from_numpy(oracle.kernel_spectrum(_even_kernel(rng, gen.padded_shape(n, bc)))).cuda()
    rho = torch.from_numpy(rng.standard_normal((n[2], n[1], n[0]))).cuda()
    plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64)
    try:
        assert plan.launch_mode()[0] == "fused"
        plan.set_kernel(Kf)
        ref = plan.solve(rho).clone()
        plan.set_kernel_even(Kf)
        assert plan.launch_mode()[0] != "fused"
        V_even = plan.solve(rho).clone()
        plan.set_kernel(Kf)
        assert plan.launch_mode()[0] == "fused"
        assert torch.equal(plan.solve(rho), ref)
        torch.cuda.synchronize()
        assert rel_l2(V_even.cpu().numpy(), ref.cpu().numpy()) <= 1e-12   # Kf is even to rounding only: not bitwise here
    finally:
        plan.close()
