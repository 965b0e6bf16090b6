"""`poisson_solve_static`: the solve for callers that cannot allocate device memory.

Who that is: an application that reserved the whole GPU for its own memory pool at start-up (a cudaMalloc issued by a
library it calls then fails), a job held to a fixed memory budget, or an inner loop that can afford neither an
out-of-memory error nor the device-wide synchronisation inside cudaMalloc / cudaFree.  The entry point needs no plan
and calls no allocating routine; its intermediates live in a fixed 32 MiB array inside the library image, one per GPU,
shared by every call (include/poisson.h).

What is checked here, against the existing path (`PoissonPlan.set_kernel` + `solve`) on the same inputs, within the
bars every parity test of this repo uses (rel. L2 <= 1e-12 in fp64, <= 1e-5 in fp32 -- the kernels are the same, so
the difference is in fact expected to be exactly 0):
  * two calls in a row on the same grid with different densities (the second call finds the first one's leftovers in
    the array and must not be affected by them);
  * then a different grid, precision and boundary conditions, and back (tables and carving of the array change);
  * a grid above the stated limit is refused with EUNSUPPORTED and a message that names the limit;
  * the call really allocates nothing (the device's free memory is the same before and after).
The file is named so that pytest collects it last (`pytest -x` stops at the first failure; a failure here must not
hide the other tests), and it passes both alone in a fresh process and after the rest of the suite: it depends on no
state but the array, which each call rewrites before reading.
"""
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


def _inputs(seed, n, bc, prec):
    """Seeded density and the spectrum of a random kernel that is even along every axis (so K^F is real)."""
    import torch
    rng = np.random.default_rng(seed)
    sx, sy, sz = gen.padded_shape(n, bc)
    K = rng.standard_normal((sz, sy, sx))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    Kf = np.ascontiguousarray(np.fft.rfftn(K).real)          # an input, like the densities: any real array would do
    dt = np.float64 if prec == "fp64" else np.float32
    rhos = [rng.standard_normal((n[2], n[1], n[0])).astype(dt) for _ in range(2)]
    return torch.from_numpy(Kf.astype(dt)).cuda(), [torch.from_numpy(r).cuda() for r in rhos]


def _existing_path(pk, n, bc, prec, Kf, rhos):
    import torch
    plan = pk.PoissonPlan(n, bc, 0.25, pk.FP64 if prec == "fp64" else pk.FP32)
    try:
        plan.set_kernel(Kf)
        out = [plan.solve(r).clone() for r in rhos]
        torch.cuda.synchronize()
        return out
    finally:
        plan.close()


def _static(pk, n, bc, prec, Kf, rho):
    import torch
    V = torch.full_like(rho, float("nan"))                   # every element must be written by the call
    pk.poisson_solve_static(n[0], n[1], n[2], bc, pk.FP64 if prec == "fp64" else pk.FP32, Kf.data_ptr(), rho.data_ptr(),
                            V.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return V


CASES = [((32, 32, 32), (0, 0, 0), "fp64"),      # BASELINE.json config 0's grid
         ((24, 20, 36), (0, 1, 0), "fp32"),      # other lengths, one periodic axis, other precision
         ((15, 22, 9), (1, 0, 0), "fp64"),       # odd N_x and a length outside sizes.def: the any-length kernel's tables
         ((32, 32, 32), (0, 0, 0), "fp64")]      # and back to the first grid


def test_two_calls_in_a_row_match_the_existing_path(pk):
    import torch
    for i, (n, bc, prec) in enumerate(CASES):
        Kf, rhos = _inputs(5244 + i, n, bc, prec)
        want = _existing_path(pk, n, bc, prec, Kf, rhos)
        got = [_static(pk, n, bc, prec, Kf, rhos[0]), _static(pk, n, bc, prec, Kf, rhos[1])]   # two calls in a row
        torch.cuda.synchronize()
        for j in range(2):
            g, w = got[j].cpu().numpy().astype(np.float64), want[j].cpu().numpy().astype(np.float64)
            assert np.isfinite(g).all(), (n, bc, prec, j)
            err = rel_l2(g, w)
            assert err <= TOL[prec], (n, bc, prec, j, err)
        # and the first result is not the second one's (the calls did not share an output by accident)
        assert rel_l2(got[0].cpu().numpy(), got[1].cpu().numpy()) > 0.1


def test_static_solve_matches_the_oracle(pk):
    """The new entry point against the CPU oracle directly, on BASELINE.json config 0 (seeded Gaussians, 1/(4 pi r))."""
    import torch
    cfg = gen.get_config("c0")
    rho = gen.gaussian_density(cfg)
    Kf = oracle.kernel_spectrum(gen.green_kernel_realspace(cfg.n, cfg.bc, cfg.h))
    V = _static(pk, cfg.n, cfg.bc, "fp64", torch.from_numpy(np.ascontiguousarray(Kf)).cuda(),
                torch.from_numpy(np.ascontiguousarray(rho)).cuda())
    torch.cuda.synchronize()
    err = rel_l2(V.cpu().numpy(), oracle.solve(rho, Kf, cfg.bc))
    assert err <= TOL["fp64"], err


def test_grid_above_the_limit_is_refused(pk):
    import torch
    n, bc = (96, 96, 96), (0, 0, 0)              # 71 MB of intermediates: more than the 32 MiB array
    x = torch.zeros(16, dtype=torch.float64, device="cuda")   # never touched: the size check comes first
    with pytest.raises(pk.PoissonError) as e:
        pk.poisson_solve_static(n[0], n[1], n[2], bc, pk.FP64, x.data_ptr(), x.data_ptr(), x.data_ptr(), 0)
    assert e.value.status == 2
    assert str(pk.STATIC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()                     # nothing was launched, nothing is pending or broken


def test_call_allocates_no_device_memory(pk):
    import torch
    n, bc, prec = (32, 32, 32), (0, 0, 0), "fp64"
    Kf, rhos = _inputs(77, n, bc, prec)
    V = _static(pk, n, bc, prec, Kf, rhos[0])    # first call for this grid: device set-up and tables are behind us now
    torch.cuda.synchronize()
    out = torch.empty_like(rhos[1])
    stream = torch.cuda.current_stream().cuda_stream
    free_before = torch.cuda.mem_get_info()[0]
    for _ in range(50):
        pk.poisson_solve_static(n[0], n[1], n[2], bc, pk.FP64, Kf.data_ptr(), rhos[1].data_ptr(), out.data_ptr(), stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert torch.isfinite(out).all() and torch.isfinite(V).all()
