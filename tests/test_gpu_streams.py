"""How poisson_solve behaves around streams (include/poisson.h: "asynchronous on `stream`", "one plan = one solve in flight"):
captured into a caller's CUDA graph, two plans on two streams at once, and a soak of repeated solves whose results must
stay bitwise the same (the substitute for a race detector on this pool: DESIGN.md section 10)."""
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


def _setup(pk, n, bc, seed):
    import torch
    rng = np.random.default_rng(seed)
    s = gen.padded_shape(n, bc)
    K = rng.standard_normal((s[2], s[1], s[0]))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    Kf = oracle.kernel_spectrum(K)
    rhos = [rng.standard_normal((n[2], n[1], n[0])) for _ in range(4)]
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
    plan.set_kernel(torch.from_numpy(Kf).cuda())
    return plan, Kf, rhos


@pytest.mark.parametrize("mode_env", [{"POISSON_GRAPH": "1"}, {"POISSON_GRAPH": "1", "POISSON_PDL": "1"}, {"POISSON_TUNE": "0"}, {}],
                         ids=["plan_graph", "plan_graph_pdl", "five", "tuned"])
def test_solve_captured_into_a_callers_graph(pk, monkeypatch, mode_env):
    """A caller that is capturing its stream gets the five passes as plain launches (nodes of ITS graph) even when the plan's
    own launch mode is an instantiated graph; replaying the caller's graph gives the bits of the direct call, also after the
    density buffer's contents changed."""
    import torch
    for k, v in mode_env.items():
        monkeypatch.setenv(k, v)
    n, bc = (32, 24, 16), (0, 0, 1)
    plan, Kf, rhos = _setup(pk, n, bc, 11)
    try:
        rho = torch.from_numpy(rhos[0]).cuda()
        ref0 = plan.solve(rho).clone()
        ref1 = plan.solve(torch.from_numpy(rhos[1]).cuda()).clone()
        torch.cuda.synchronize()
        assert rel_l2(ref0.cpu().numpy(), oracle.solve(rhos[0], Kf, bc)) <= 1e-12
        V = torch.empty_like(rho)
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):                  # the current stream is capturing inside this block
            plan.solve(rho, V)
        V.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(V, ref0)
        rho.copy_(torch.from_numpy(rhos[1]).cuda())
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(V, ref1)
        assert torch.equal(plan.solve(torch.from_numpy(rhos[0]).cuda()), ref0)   # the plan's own mode still works afterwards
    finally:
        plan.close()


def test_two_plans_on_two_streams(pk):
    """Plans share nothing but read-only kernels: two of them solving at the same time on their own streams give the bits
    each gives alone."""
    import torch
    pa, Kfa, ra = _setup(pk, (32, 32, 32), (0, 0, 0), 21)
    pb, Kfb, rb = _setup(pk, (24, 40, 16), (1, 0, 0), 22)
    try:
        da = [torch.from_numpy(r).cuda() for r in ra]
        db = [torch.from_numpy(r).cuda() for r in rb]
        refa = [pa.solve(r).clone() for r in da]
        refb = [pb.solve(r).clone() for r in db]
        torch.cuda.synchronize()
        sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
        outa = [torch.empty_like(r) for r in da]
        outb = [torch.empty_like(r) for r in db]
        for rep in range(25):
            for i in range(4):
                pa.solve(da[i], outa[i], stream=sa)
                pb.solve(db[i], outb[i], stream=sb)
        torch.cuda.synchronize()
        for i in range(4):
            assert torch.equal(outa[i], refa[i]) and torch.equal(outb[i], refb[i])
    finally:
        pa.close()
        pb.close()


@pytest.mark.slow
@pytest.mark.parametrize("n,bc", [((32, 32, 32), (0, 0, 0)), ((64, 64, 64), (0, 0, 0)), ((48, 48, 128), (0, 0, 1))],
                         ids=["c0_shape", "free_64", "wire_48"])
def test_soak_repeated_solves_stay_bitwise_equal(pk, n, bc):
    """2 000 solves per grid in the plan's tuned launch mode (graphs of parallel chains included), cycling over four densities
    and two output buffers: every result equals the first solve of its density bit for bit.  A missing dependency between
    passes, a tile written twice or a stale intermediate would show up as a differing bit sooner or later."""
    import torch
    plan, Kf, rhos = _setup(pk, n, bc, 4242)
    try:
        d = [torch.from_numpy(r).cuda() for r in rhos]
        ref = [plan.solve(r).clone() for r in d]
        torch.cuda.synchronize()
        assert rel_l2(ref[0].cpu().numpy(), oracle.solve(rhos[0], Kf, bc)) <= 1e-12
        out = [torch.empty_like(d[0]) for _ in range(2)]
        bad = torch.zeros((), dtype=torch.int64, device="cuda")
        for it in range(2000):
            i = (it * 7 + it // 5) % 4
            V = plan.solve(d[i], out[it % 2])
            bad += (V != ref[i]).sum()            # stream-ordered with the solves: no host sync inside the loop
        torch.cuda.synchronize()
        assert int(bad.item()) == 0
    finally:
        plan.close()
