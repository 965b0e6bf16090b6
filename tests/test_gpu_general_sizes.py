"""General grid sizes and kernels ("various grid sizes"): odd N, lengths with
factors 7, 11, 13, ..., three or more radices, primes -- everything outside csrc/sizes.def runs the any-length kernel of
csrc/generic_pass.cuh -- and complex K^F for kernels without inversion symmetry.  Every case is compared element by
element with the CPU oracle on the same seeded inputs (rel. L2 <= 1e-12 fp64, <= 1e-5 fp32)."""
import itertools

import numpy as np
import pytest

import oracle
from workloads import generators as gen

pytestmark = pytest.mark.gpu

TOL = {"fp64": 1e-12, "fp32": 1e-5}


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


def _solve(pk, rho, Kf, n, bc, prec, complex_k=False):
    import torch
    np_dt = np.float64 if prec == "fp64" else np.float32
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64 if prec == "fp64" else pk.FP32)
    try:
        if complex_k:
            plan.set_kernel_complex(torch.from_numpy(np.ascontiguousarray(Kf.astype(np.complex128 if prec == "fp64" else np.complex64))).cuda())
        else:
            plan.set_kernel(torch.from_numpy(np.ascontiguousarray(Kf.astype(np_dt))).cuda())
        r = torch.from_numpy(np.ascontiguousarray(rho.astype(np_dt))).cuda()
        V = plan.solve(r)
        torch.cuda.synchronize()
        return V.cpu().numpy().astype(np.float64)
    finally:
        plan.close()


# odd N, factor 7 / 11 / 13, three radices (30 = 2*3*5, 60 on a free axis = 120 is compiled, 45 -> 90 = 2*3*3*5), primes (13, 17, 31),
# N = 1, one compiled axis next to two any-length ones, ragged tiles (N_x = 37 -> 19 pair pencils, the last one unpaired)
GENERAL_SIZES = [(7, 5, 3), (1, 1, 1), (1, 6, 9), (9, 1, 4), (14, 10, 6), (15, 21, 8), (13, 16, 11), (37, 12, 10), (22, 7, 32),
                 (28, 18, 5), (30, 45, 6), (64, 9, 17), (25, 50, 4), (31, 8, 8), (8, 8, 77), (150, 4, 3), (6, 125, 5)]


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
@pytest.mark.parametrize("n", GENERAL_SIZES, ids=lambda n: "x".join(map(str, n)))
def test_general_sizes_all_bc_vs_oracle(pk, n, prec):
    rng = np.random.default_rng(5000 + 7 * n[0] + 3 * n[1] + n[2])
    for bc in itertools.product((0, 1), repeat=3):
        s = gen.padded_shape(n, bc)
        rho = rng.standard_normal((n[2], n[1], n[0]))
        Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
        if prec == "fp32":
            rho, Kf = rho.astype(np.float32).astype(np.float64), Kf.astype(np.float32).astype(np.float64)
        V = _solve(pk, rho, Kf, n, bc, prec)
        err = rel_l2(V, oracle.solve(rho, Kf, bc))
        assert err <= TOL[prec], (n, bc, prec, err)


@pytest.mark.parametrize("n,bc", [((251, 6, 4), (1, 0, 0)), ((4, 6, 300), (0, 0, 0)), ((6, 360, 4), (0, 1, 0)), ((450, 4, 2), (0, 0, 1)),
                                  ((127, 4, 6), (0, 0, 0)), ((4, 6, 521), (0, 0, 1)), ((4, 6, 521), (0, 0, 0)), ((509, 3, 2), (1, 1, 1))])
def test_long_awkward_lengths_vs_oracle(pk, n, bc):
    """600, 360 and 900 (the lengths DESIGN.md, round 1, named as needing a three-pass engine); prime and 2 * prime lengths up to
    1024 through Bluestein's chirp-z (251, 254 = 2 * 127, 521, 509 with odd N_x in the R2C pass next to it); 1042 = 2 * 521, above the
    Bluestein limit, through the O(p) fallback butterfly."""
    rng = np.random.default_rng(77 + sum(n))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
    for prec in ("fp64", "fp32"):
        r_in, k_in = (rho, Kf) if prec == "fp64" else (rho.astype(np.float32).astype(np.float64), Kf.astype(np.float32).astype(np.float64))
        err = rel_l2(_solve(pk, r_in, k_in, n, bc, prec), oracle.solve(r_in, k_in, bc))
        assert err <= TOL[prec], (n, bc, prec, err)


def test_maximum_any_length_4096_shift_kernel_property(pk):
    """The longest length the any-length kernel takes (S = 4096 = 2 * 2048, free z) next to two compiled axes; the exact
    result for K = delta(r - d) + delta(r + d) is rho displaced by +-d with zero fill (nothing wraps on free axes)."""
    import torch
    n, bc, d = (8, 8, 2048), (0, 0, 0), (1, 2, 700)
    s = gen.padded_shape(n, bc)
    rng = np.random.default_rng(4096)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    kz = np.arange(s[2])[:, None, None] * d[2] / s[2]
    ky = np.arange(s[1])[None, :, None] * d[1] / s[1]
    kx = np.arange(s[0] // 2 + 1)[None, None, :] * d[0] / s[0]
    Kf = 2.0 * np.cos(2 * np.pi * (kx + ky + kz))
    exp = np.zeros_like(rho)
    exp[d[2]:, d[1]:, d[0]:] += rho[:-d[2], :-d[1], :-d[0]]
    exp[:-d[2], :-d[1], :-d[0]] += rho[d[2]:, d[1]:, d[0]:]
    assert rel_l2(_solve(pk, rho, Kf, n, bc, "fp64"), exp) <= 1e-12
    with pytest.raises(pk.PoissonError) as ei:
        pk.PoissonPlan((8, 8, 2049), bc, 0.1, pk.FP64)
    assert ei.value.status == 2                                     # EUNSUPPORTED only above the limit


@pytest.mark.parametrize("n,bc", [((8, 12, 4), (0, 1, 0)), ((16, 16, 16), (0, 0, 0)), ((7, 5, 6), (1, 0, 1)), ((32, 6, 9), (0, 0, 1)),
                                  ((24, 20, 10), (1, 1, 1))])
def test_complex_kernel_spectrum_vs_oracle_and_direct_sum(pk, n, bc):
    """poisson_set_kernel_complex: a real kernel with NO symmetry (complex K^F, K^F(-k) = conj K^F(k)) against
    oracle.solve_complex and against the O(N^2) sum of Eq. 2 itself; then back to a real spectrum on the same plan."""
    import torch
    rng = np.random.default_rng(31 + sum(n))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = rng.standard_normal((s[2], s[1], s[0]))
    Kf = oracle.kernel_spectrum_complex(K)
    V = _solve(pk, rho, Kf, n, bc, "fp64", complex_k=True)
    assert rel_l2(V, oracle.solve_complex(rho, Kf, bc)) <= 1e-12
    assert rel_l2(V, oracle.direct_sum(rho, K, bc)) <= 1e-12
    r32, k32 = rho.astype(np.float32).astype(np.float64), Kf.astype(np.complex64).astype(np.complex128)
    assert rel_l2(_solve(pk, r32, k32, n, bc, "fp32", complex_k=True), oracle.solve_complex(r32, k32, bc)) <= 1e-5
    # one plan: real kernel, then a complex one, then a real one again; batch + graph paths included
    Ke = _even_kernel(rng, s)
    Kfe = oracle.kernel_spectrum(Ke)
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
    try:
        r = torch.from_numpy(rho).cuda()
        plan.set_kernel(torch.from_numpy(Kfe).cuda())
        v_real = plan.solve(r).cpu().numpy()
        plan.set_kernel_complex(torch.from_numpy(Kf).cuda())
        v_c = plan.solve(r).cpu().numpy()
        vb = plan.solve_batch([r, r, r])
        torch.cuda.synchronize()
        plan.set_kernel(torch.from_numpy(Kfe).cuda())
        v_real2 = plan.solve(r).cpu().numpy()
        ref_real = oracle.solve(rho, Kfe, bc)
        assert rel_l2(v_real, ref_real) <= 1e-12 and rel_l2(v_real2, ref_real) <= 1e-12
        assert rel_l2(v_c, oracle.solve_complex(rho, Kf, bc)) <= 1e-12
        for v in vb:
            assert np.array_equal(v.cpu().numpy(), v_c)
    finally:
        plan.close()


def test_general_sizes_through_batches_and_host_entry(pk):
    """The any-length kernels behind poisson_solve_batch (several densities per launch on small grids, lanes otherwise)
    and poisson_solve_host: same results as one-by-one solves, which match the oracle."""
    import torch
    for n, bc in (((7, 5, 3), (0, 1, 0)), ((15, 9, 14), (0, 0, 0))):
        rng = np.random.default_rng(909 + n[0])
        s = gen.padded_shape(n, bc)
        Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
        plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
        try:
            plan.set_kernel(torch.from_numpy(Kf).cuda())
            rhos = [torch.from_numpy(rng.standard_normal((n[2], n[1], n[0]))).cuda() for _ in range(5)]
            Vs = plan.solve_batch(rhos)
            torch.cuda.synchronize()
            for r, v in zip(rhos, Vs):
                assert torch.equal(plan.solve(r), v)
                assert rel_l2(v.cpu().numpy(), oracle.solve(r.cpu().numpy(), Kf, bc)) <= 1e-12
            rh = rhos[0].cpu().pin_memory()
            vh = torch.empty_like(rh).pin_memory()
            plan.solve_host(rh, vh)
            assert torch.equal(vh, Vs[0].cpu())
            w = rhos[1].clone()
            plan.solve(w, w)                                        # in place
            assert torch.equal(w, Vs[1])
        finally:
            plan.close()


@pytest.mark.parametrize("n,bc", [((128, 16, 12), (0, 0, 0)), ((7, 5, 6), (1, 0, 1)), ((32, 6, 9), (0, 0, 1)), ((24, 20, 10), (1, 1, 0))])
@pytest.mark.parametrize("pdl", [False, True], ids=["graph", "graph_pdl"])
def test_kernel_kinds_in_a_shaped_graph(pk, monkeypatch, n, bc, pdl):
    """One plan whose solve graph is FORCED into parallel chains (3 plane ranges x 2 x ranges where x ranges apply): real K^F,
    folded even K^F, complex K^F (pass F3 switches to the any-length kernel: the graph is rebuilt, x ranges fall away), real
    again -- every switch rebuilds the graph around pass F3's new parameters, and every result matches the oracle."""
    import torch
    monkeypatch.setenv("POISSON_GRAPH", "1")
    monkeypatch.setenv("POISSON_BRANCHES", "3")
    monkeypatch.setenv("POISSON_XCHAINS", "2")
    if pdl:
        monkeypatch.setenv("POISSON_PDL", "1")
    rng = np.random.default_rng(77 + sum(n))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    Kfe = oracle.kernel_spectrum(_even_kernel(rng, s))
    Kfe = 0.5 * (Kfe + np.roll(np.flip(Kfe, axis=1), 1, axis=1))
    Kfe = np.ascontiguousarray(0.5 * (Kfe + np.roll(np.flip(Kfe, axis=0), 1, axis=0)))       # exactly even along y and z
    Kc = oracle.kernel_spectrum_complex(rng.standard_normal((s[2], s[1], s[0])))
    ref_real, ref_c = oracle.solve(rho, Kfe, bc), oracle.solve_complex(rho, Kc, bc)
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64)
    try:
        assert plan.launch_mode()[0] == ("graph_pdl" if pdl else "graph")
        J, R = plan.graph_shape()
        assert J == min(3, plan.info.half_len) and R in (1, 2)
        r = torch.from_numpy(rho).cuda()
        plan.set_kernel(torch.from_numpy(Kfe).cuda())
        v1 = plan.solve(r).cpu().numpy()
        try:
            plan.set_kernel_even(torch.from_numpy(Kfe).cuda())
            v2 = plan.solve(r).cpu().numpy()
            assert np.array_equal(v1, v2)
        except pk.PoissonError as e:
            assert e.status == 2                      # pass F3 of this grid runs the any-length kernel: folded storage refused
        plan.set_kernel_complex(torch.from_numpy(Kc).cuda())
        v3 = plan.solve(r).cpu().numpy()
        assert plan.graph_shape()[0] == J             # still chains over plane ranges
        plan.set_kernel(torch.from_numpy(Kfe).cuda())
        v4 = plan.solve(r).cpu().numpy()
    finally:
        plan.close()
    assert rel_l2(v1, ref_real) <= 1e-12 and rel_l2(v4, ref_real) <= 1e-12
    assert rel_l2(v3, ref_c) <= 1e-12
