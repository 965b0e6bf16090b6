"""GPU tests of the sharded single solve (include/poisson.h: poisson_shard_*).

Only one GPU is available, so the R ranks of a sharded solve are R shard plans in ONE process on ONE device, run stage by
stage (every rank's forward, then every rank's middle, then every rank's inverse): the "peer" slabs are ordinary device
buffers, which is exactly what a peer-mapped pointer is to the kernels.  That exercises everything the library does for a
multi-GPU solve -- the partition, the local strides, passes F1 / I2 scattering their stores over the ranks' slabs, the
rank-local share of K^F -- and leaves out only what torch.distributed provides (peer mapping and the two barriers)."""
import itertools

import numpy as np
import pytest

import oracle
from workloads import generators as gen

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pk():
    import torch
    import paper_1211_5244_b200 as pk_
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the solve has no fallback")
    pk_.load_library()
    torch.cuda.set_device(0)
    return pk_


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def _even_kernel(rng, s):
    sx, sy, sz = s
    K = rng.standard_normal((sz, sy, sx))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    return K


def _sharded_solve(pk, n, bc, prec, R, rho_t, Kf_t, repeats=2):
    """V of the whole box from R virtual ranks (list over repeats)."""
    import torch
    dt = rho_t.dtype
    plans = [pk.ShardPlan(n, bc, 0.25, prec, r, R) for r in range(R)]
    try:
        infos = [p.info for p in plans]
        axis = 2 - infos[0].split_axis                      # numpy axis of [z][y][x]
        # partition properties the kernels rely on
        assert infos[0].o0 == 0 and infos[-1].o1 == n[infos[0].split_axis]
        assert infos[0].k0 == 0 and infos[-1].k1 == gen.padded_shape(n, bc)[infos[0].plane_axis] // 2 + 1
        for a, b in zip(infos[:-1], infos[1:]):
            assert a.o1 == b.o0 and a.k1 == b.k0 and a.o1 > a.o0 and a.k1 > a.k0
        csize = 16 if prec == pk.FP64 else 8
        mids = [torch.full((i.mid_bytes // csize * 2,), float("nan"), dtype=dt, device="cuda") for i in infos]
        backs = [torch.full((i.back_bytes // csize * 2,), float("nan"), dtype=dt, device="cuda") for i in infos]
        for p in plans:
            p.set_slabs([m.data_ptr() for m in mids], [b.data_ptr() for b in backs], keep=(mids, backs))
            p.set_kernel(Kf_t)
        outs = []
        for rep in range(repeats):
            for m in mids: m.fill_(float("nan"))            # an element no rank writes would poison the result
            for b in backs: b.fill_(float("nan"))
            locs = []
            for p, i in zip(plans, infos):
                sl = [slice(None)] * 3
                sl[axis] = slice(i.o0, i.o1)
                locs.append(rho_t[tuple(sl)].contiguous())
                assert tuple(locs[-1].shape) == p.local_shape
            for p, r in zip(plans, locs): p.forward(r)
            torch.cuda.synchronize()                         # barrier A
            assert all(bool(torch.isfinite(m).all()) for m in mids)
            for p in plans: p.middle()
            torch.cuda.synchronize()                         # barrier B
            assert all(bool(torch.isfinite(b).all()) for b in backs)
            Vs = [torch.empty_like(r) for r in locs]
            for p, v in zip(plans, Vs): p.inverse(v)
            torch.cuda.synchronize()
            outs.append(torch.cat(Vs, dim=axis))
        return outs, infos
    finally:
        for p in plans: p.close()


@pytest.mark.parametrize("R", [1, 2, 3, 4])
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_sharded_solve_all_bc_bitwise_and_vs_oracle(pk, R, prec):
    """All 8 boundary-condition combinations (axis orders (z,y,x), (y,x,z), (z,x,y): split axis y or z, I2 along y or along x),
    ragged partitions (R = 3), both precisions: bitwise equal to poisson_solve on one GPU, and within tolerance of the oracle."""
    import torch
    dt_np = np.float64 if prec == "fp64" else np.float32
    prec_id = pk.FP64 if prec == "fp64" else pk.FP32
    n = (32, 20, 24)
    for bc in itertools.product((0, 1), repeat=3):
        rng = np.random.default_rng(900 + R + 8 * sum(b << i for i, b in enumerate(bc)))
        s = gen.padded_shape(n, bc)
        Kf = oracle.kernel_spectrum(_even_kernel(rng, s)).astype(dt_np)
        rho = rng.standard_normal((n[2], n[1], n[0])).astype(dt_np)
        rho_t, Kf_t = torch.from_numpy(rho).cuda(), torch.from_numpy(Kf).cuda()
        ref_plan = pk.PoissonPlan(n, bc, 0.25, prec_id)
        try:
            ref_plan.set_kernel(Kf_t)
            V_ref = ref_plan.solve(rho_t).clone()
        finally:
            ref_plan.close()
        outs, infos = _sharded_solve(pk, n, bc, prec_id, R, rho_t, Kf_t)
        for V in outs:
            assert torch.equal(V, V_ref), (bc, R, prec)
        ref = oracle.solve(rho.astype(np.float64), Kf.astype(np.float64), bc)
        assert rel_l2(V_ref.cpu().numpy().astype(np.float64), ref) <= (1e-12 if prec == "fp64" else 1e-5)
        if R > 1:
            assert all(i.sent_bytes[0] > 0 and i.sent_bytes[1] > 0 for i in infos)


def test_sharded_config1_four_ranks(pk):
    """configs[1] (128^3 -> 256^3 fp64) over 4 virtual ranks: bitwise the single-GPU result; exchange volume = A1 minus the
    part that stays on its rank, twice (SURVEY.md 8e quotes the A2 volume; the exchange here is on the smaller A1)."""
    import torch
    cfg = gen.get_config("c1")
    rho = gen.gaussian_density(cfg)
    rng = np.random.default_rng(3)
    s = gen.padded_shape(cfg.n, cfg.bc)
    Kf = rng.standard_normal((s[2], s[1], s[0] // 2 + 1))          # any real spectrum: the comparison is bitwise
    rho_t, Kf_t = torch.from_numpy(rho).cuda(), torch.from_numpy(Kf).cuda()
    ref_plan = pk.PoissonPlan(cfg.n, cfg.bc, cfg.h, pk.FP64)
    try:
        ref_plan.set_kernel(Kf_t)
        V_ref = ref_plan.solve(rho_t).clone()
    finally:
        ref_plan.close()
    outs, infos = _sharded_solve(pk, cfg.n, cfg.bc, pk.FP64, 4, rho_t, Kf_t, repeats=1)
    assert torch.equal(outs[0], V_ref)
    a1_bytes = 129 * 128 * 128 * 16
    assert sum(i.sent_bytes[0] for i in infos) == a1_bytes - sum((i.k1 - i.k0) * (i.o1 - i.o0) * 128 * 16 for i in infos)
    assert sum(i.mid_bytes for i in infos) == a1_bytes and sum(i.back_bytes for i in infos) == a1_bytes


def test_sharded_solver_world_size_one(pk):
    """ShardedSolver (the torch.distributed wrapper) without a process group = one rank: same result as poisson_solve."""
    import torch
    n, bc = (32, 24, 16), (0, 0, 1)
    rng = np.random.default_rng(17)
    s = gen.padded_shape(n, bc)
    Kf = torch.from_numpy(oracle.kernel_spectrum(_even_kernel(rng, s))).cuda()
    rho = torch.from_numpy(rng.standard_normal((n[2], n[1], n[0]))).cuda()
    ref_plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64)
    try:
        ref_plan.set_kernel(Kf)
        V_ref = ref_plan.solve(rho).clone()
    finally:
        ref_plan.close()
    solver = pk.ShardedSolver(n, bc, 0.3, pk.FP64)
    solver.set_kernel(Kf)
    assert torch.equal(solver.solve(rho), V_ref)
    assert torch.equal(solver.solve(rho), V_ref)
    solver.plan.close()


def test_shard_plan_refuses_plain_calls_and_bad_arguments(pk):
    import ctypes
    import torch
    lib = pk.load_library()
    with pytest.raises(pk.PoissonError) as ei:
        pk.ShardPlan((32, 32, 32), (0, 0, 0), 0.2, pk.FP64, 2, 2)          # rank out of range
    assert ei.value.status == 1
    with pytest.raises(pk.PoissonError) as ei:
        pk.ShardPlan((30, 22, 12), (0, 0, 0), 0.2, pk.FP64, 0, 2)          # S = 44: no register-engine kernel
    assert ei.value.status == 2
    p = pk.ShardPlan((32, 32, 32), (0, 0, 0), 0.2, pk.FP64, 0, 2)
    try:
        x = torch.zeros(p.local_shape, dtype=torch.float64, device="cuda")
        with pytest.raises(pk.PoissonError):                                # slabs not set
            p.forward(x)
        full = torch.zeros((32, 32, 32), dtype=torch.float64, device="cuda")
        assert lib.poisson_solve(p._h, full.data_ptr(), full.data_ptr(), 0) == 1   # EINVAL: not a plain plan
    finally:
        p.close()
