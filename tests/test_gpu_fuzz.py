"""Seeded random sweep of the CUDA path against the oracle: random sizes (compiled register-engine lengths, factor-7 lengths, odd and prime
ones through the any-length kernel, mixed per axis), random boundary conditions, precision, launch mode / graph shape forced at random,
plain or folded K^F, single solves and the batch route -- the combinations no hand-written case list covers."""
import os
import random

import numpy as np
import pytest

import oracle
from workloads import generators as gen

pytestmark = pytest.mark.gpu

SIZES = [2, 3, 4, 5, 6, 7, 8, 9, 10, 12, 14, 15, 16, 18, 20, 21, 24, 28, 30, 32, 35, 36, 40, 48, 56, 60, 64, 72]
KNOBS = ("POISSON_GRAPH", "POISSON_PDL", "POISSON_BRANCHES", "POISSON_XCHAINS", "POISSON_TUNE")


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
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def _even_kernel(rng, s):
    K = rng.standard_normal((s[2], s[1], s[0]))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    return K


@pytest.mark.parametrize("seed", range(8))
def test_random_cases_vs_oracle(pk, monkeypatch, seed):
    import torch
    rnd = random.Random(5244 + seed)
    for it in range(10):
        while True:
            n = (rnd.choice(SIZES), rnd.choice(SIZES), rnd.choice(SIZES))
            if n[0] * n[1] * n[2] <= 40_000:
                break
        bc = tuple(rnd.randint(0, 1) for _ in range(3))
        prec = rnd.choice(["fp64", "fp64", "fp32"])
        mode = rnd.choice(["tuned", "graph", "graph_pdl", "five_pdl", "five"])
        env = {"tuned": {}, "five": {"POISSON_TUNE": "0"}, "five_pdl": {"POISSON_PDL": "1"},
               "graph": {"POISSON_GRAPH": "1", "POISSON_BRANCHES": str(rnd.choice([1, 2, 3, 4])), "POISSON_XCHAINS": str(rnd.choice([1, 2, 4]))},
               "graph_pdl": {"POISSON_GRAPH": "1", "POISSON_PDL": "1", "POISSON_BRANCHES": str(rnd.choice([1, 2, 3])),
                             "POISSON_XCHAINS": str(rnd.choice([1, 2]))}}[mode]
        for k in KNOBS:
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        rng = np.random.default_rng(100 * seed + it)
        s = gen.padded_shape(n, bc)
        dt = np.float64 if prec == "fp64" else np.float32
        Kf = oracle.kernel_spectrum(_even_kernel(rng, s)).astype(dt)
        rho = rng.standard_normal((n[2], n[1], n[0])).astype(dt)
        ref = oracle.solve(rho.astype(np.float64), Kf.astype(np.float64), bc)
        plan = pk.PoissonPlan(n, bc, 0.3, pk.FP64 if prec == "fp64" else pk.FP32)
        try:
            even = rnd.random() < 0.3
            Kf_t = torch.from_numpy(Kf).cuda()
            try:
                (plan.set_kernel_even if even else plan.set_kernel)(Kf_t)
            except pk.PoissonError as e:                       # folded storage: register-engine F3 only
                assert even and e.status == 2
                plan.set_kernel(Kf_t)
                even = False
            r = torch.from_numpy(rho).cuda()
            V = plan.solve(r).cpu().numpy().astype(np.float64)
            Vb = [v for v in plan.solve_batch([r, r, r])]
            torch.cuda.synchronize()
            what = (n, bc, prec, env, even, plan.launch_mode()[0], plan.graph_shape())
        finally:
            plan.close()
        # a folded copy reads the mirror pencil's K^F, equal to the pencil's own only up to the rounding of the computed spectrum
        tol = (1e-12 if prec == "fp64" else 1e-5) * (2.0 if even else 1.0)
        assert rel_l2(V, ref) <= tol, what
        for v in Vb:
            assert rel_l2(v.cpu().numpy().astype(np.float64), ref) <= tol, what
