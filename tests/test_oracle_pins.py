"""Pins for the CPU oracle (oracle/poisson_oracle.c) against things that are NOT the oracle:
the O(N^2) real-space sum of Eq. 2, closed forms, invariants, explicit index
shifting, and numpy's pocketfft as a library second opinion.  All CPU-only.

The paper prints no worked numerical example, hence no value fixtures here;
the closed-form 1D-FFT-count ratios of PAPER.md:51 are pinned in test_plan_host.py from
tests/golden/fft_count_ratios.txt.
"""
import itertools
import math

import numpy as np
import pytest

import oracle
from workloads import generators as gen

FREE, PER = gen.FREE, gen.PERIODIC
ALL_BC = list(itertools.product((FREE, PER), repeat=3))


def _rng(seed):
    return np.random.default_rng(seed)


def _even_kernel(rng, s):
    """Random real kernel on the padded grid, even along every axis (so K_f is real)."""
    sx, sy, sz = s
    K = rng.standard_normal((sz, sy, sx))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    return K


def _inversion_kernel(rng, s):
    """Random real kernel with K(-r) = K(r) only (NOT even per axis): K_f real but K_f(kx,ky,kz) != K_f(-kx,ky,kz)."""
    sx, sy, sz = s
    K = rng.standard_normal((sz, sy, sx))
    Kinv = np.roll(np.flip(K, axis=(0, 1, 2)), 1, axis=(0, 1, 2))
    return 0.5 * (K + Kinv)


def _pad(rho, s):
    sx, sy, sz = s
    nz, ny, nx = rho.shape
    p = np.zeros((sz, sy, sx))
    p[:nz, :ny, :nx] = rho
    return p


def rel_l2(a, b):
    return np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300)


# ----------------------------------------------------------------------------- the DFT itself
@pytest.mark.parametrize("shape", [(4, 6, 8), (5, 3, 7), (1, 16, 2)])
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_dft_axis_matches_library_fft_and_sign_convention(shape, axis):
    rng = _rng(1)
    a = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    fwd = oracle.dft_axis(a, axis, -1)
    inv = oracle.dft_axis(a, axis, +1)
    assert rel_l2(fwd, np.fft.fft(a, axis=axis)) < 1e-14          # forward = exp(-2 pi i jk/S)
    assert rel_l2(inv, np.fft.ifft(a, axis=axis) * shape[axis]) < 1e-14   # inverse is unnormalised


def test_dft_of_delta_is_a_pure_phase_closed_form():
    S, j0 = 12, 5
    a = np.zeros((1, 1, S), dtype=complex)
    a[0, 0, j0] = 1.0
    X = oracle.dft_axis(a, 2, -1)[0, 0]
    k = np.arange(S)
    # closed form, with exact values at the quarter turns
    assert np.allclose(X, np.cos(2 * np.pi * j0 * k / S) - 1j * np.sin(2 * np.pi * j0 * k / S), atol=1e-15)
    assert np.allclose(np.abs(X), 1.0, atol=1e-15)
    assert X[0] == 1.0 and abs(X[6] - (-1.0)) < 1e-15  # k=6: exp(-i pi 5) = -1


def test_parseval_and_roundtrip():
    rng = _rng(2)
    a = rng.standard_normal((6, 10, 8)) + 1j * rng.standard_normal((6, 10, 8))
    X = a
    for ax in range(3):
        X = oracle.dft_axis(X, ax, -1)
    assert abs(np.sum(np.abs(a) ** 2) - np.sum(np.abs(X) ** 2) / a.size) < 1e-12 * np.sum(np.abs(a) ** 2)
    back = X
    for ax in range(3):
        back = oracle.dft_axis(back, ax, +1)
    assert rel_l2(back / a.size, a) < 1e-14


def test_long_double_accumulation_agrees_with_double():
    rng = _rng(3)
    a = rng.standard_normal((3, 4, 96)) + 1j * rng.standard_normal((3, 4, 96))
    assert rel_l2(oracle.dft_axis(a, 2, -1, accum_ld=False), oracle.dft_axis(a, 2, -1, accum_ld=True)) < 5e-15


# ----------------------------------------------------------------------------- Eq. 3 == Eq. 2 (brute force)
@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("n", [(6, 4, 8), (3, 5, 2)])
def test_solve_equals_direct_sum_all_bc(bc, n):
    """Padding, indexing, free-vs-periodic semantics and normalisation against the O(N^2) sum of Eq. 2."""
    rng = _rng(10 + sum(b << i for i, b in enumerate(bc)))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = _even_kernel(rng, s)
    Kf, max_imag = oracle.kernel_spectrum(K, return_max_imag=True)
    assert max_imag < 1e-12 * np.abs(Kf).max()
    V, vimag = oracle.solve(rho, Kf, bc, return_max_imag=True)
    assert vimag < 1e-13 * np.abs(V).max()            # PAPER.md:55 "yielding a real potential"
    assert rel_l2(V, oracle.direct_sum(rho, K, bc)) < 1e-13


@pytest.mark.parametrize("bc", [(FREE, FREE, FREE), (PER, FREE, PER), (PER, PER, PER)])
def test_half_spectrum_reflection_with_inversion_symmetric_kernel(bc):
    """K(-r)=K(r) but not even per axis: pins the (-kz,-ky,Sx-kx) reflection of the half spectrum."""
    n = (4, 6, 4)
    rng = _rng(77)
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = _inversion_kernel(rng, s)
    Kf, max_imag = oracle.kernel_spectrum(K, return_max_imag=True)
    assert max_imag < 1e-12 * np.abs(Kf).max()
    assert rel_l2(oracle.solve(rho, Kf, bc), oracle.direct_sum(rho, K, bc)) < 1e-13


def test_direct_sum_at_matches_full_direct_sum():
    rng = _rng(5)
    n, bc = (5, 4, 3), (FREE, PER, FREE)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = _even_kernel(rng, gen.padded_shape(n, bc))
    full = oracle.direct_sum(rho, K, bc).ravel()
    pts = np.array([0, 7, 13, 59])
    assert np.allclose(oracle.direct_sum_at(rho, K, bc, pts), full[pts], rtol=0, atol=1e-14)


def test_direct_sum_is_the_textbook_convolution_python_loops():
    """Eq. 2 once more, in pure-Python loops, on a tiny grid (pins the C brute force itself)."""
    n, bc = (3, 2, 2), (FREE, PER, FREE)
    s = gen.padded_shape(n, bc)
    rng = _rng(6)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = rng.standard_normal((s[2], s[1], s[0]))  # need not be even for Eq. 2
    V = np.zeros_like(rho)
    for iz, iy, ix in itertools.product(range(n[2]), range(n[1]), range(n[0])):
        acc = 0.0
        for jz, jy, jx in itertools.product(range(n[2]), range(n[1]), range(n[0])):
            acc += K[(iz - jz) % s[2], (iy - jy) % s[1], (ix - jx) % s[0]] * rho[jz, jy, jx]
        V[iz, iy, ix] = acc
    assert np.allclose(oracle.direct_sum(rho, K, bc), V, rtol=0, atol=1e-13)


# ----------------------------------------------------------------------------- invariants of the whole solve
@pytest.mark.parametrize("bc", ALL_BC)
def test_delta_density_returns_the_kernel(bc):
    n = (4, 6, 4)
    s = gen.padded_shape(n, bc)
    rng = _rng(20)
    K = _even_kernel(rng, s)
    Kf = oracle.kernel_spectrum(K)
    i0 = (1, 2, 3)  # (z, y, x)
    rho = np.zeros((n[2], n[1], n[0]))
    rho[i0] = 1.0
    V = oracle.solve(rho, Kf, bc)
    z, y, x = np.meshgrid(range(n[2]), range(n[1]), range(n[0]), indexing="ij")
    expect = K[(z - i0[0]) % s[2], (y - i0[1]) % s[1], (x - i0[2]) % s[0]]
    assert np.allclose(V, expect, rtol=0, atol=1e-13)


@pytest.mark.parametrize("bc", ALL_BC)
def test_identity_kernel_returns_rho(bc):
    n = (6, 4, 2)
    s = gen.padded_shape(n, bc)
    rho = _rng(21).standard_normal((n[2], n[1], n[0]))
    Kf = np.ones((s[2], s[1], s[0] // 2 + 1))
    assert rel_l2(oracle.solve(rho, Kf, bc), rho) < 1e-14


@pytest.mark.parametrize("bc", ALL_BC)
def test_symmetric_shift_kernel_zero_fill_vs_wrap(bc):
    """K = prod_a (delta_{d_a} + delta_{-d_a})/2 has the analytic spectrum prod_a cos(2 pi k_a d_a / S_a).
    V must be the average of the 8 shifted copies of rho: zero-filled on free axes (no wrap-around
    leaks), wrapped on periodic axes.  Expected value built by index shifting only."""
    n = (6, 4, 8)
    d = (2, 1, 3)  # shift in x, y, z (smaller than n)
    s = gen.padded_shape(n, bc)
    rho = _rng(22).standard_normal((n[2], n[1], n[0]))
    kx = np.arange(s[0] // 2 + 1); ky = np.arange(s[1]); kz = np.arange(s[2])
    Kf = (np.cos(2 * np.pi * kz * d[2] / s[2])[:, None, None]
          * np.cos(2 * np.pi * ky * d[1] / s[1])[None, :, None]
          * np.cos(2 * np.pi * kx * d[0] / s[0])[None, None, :])
    expect = np.zeros_like(rho)
    for sg in itertools.product((-1, 1), repeat=3):
        shifted = rho
        for a, arr_axis in ((0, 2), (1, 1), (2, 0)):  # a = x,y,z ; numpy axis of that coordinate
            sh = sg[a] * d[a]
            if bc[a] == PER:
                shifted = np.roll(shifted, sh, axis=arr_axis)
            else:
                out = np.zeros_like(shifted)
                sl_src = [slice(None)] * 3; sl_dst = [slice(None)] * 3
                if sh > 0:
                    sl_src[arr_axis] = slice(0, n[a] - sh); sl_dst[arr_axis] = slice(sh, n[a])
                else:
                    sl_src[arr_axis] = slice(-sh, n[a]); sl_dst[arr_axis] = slice(0, n[a] + sh)
                out[tuple(sl_dst)] = shifted[tuple(sl_src)]
                shifted = out
        expect += shifted / 8.0
    assert np.allclose(oracle.solve(rho, Kf, bc), expect, rtol=0, atol=1e-13)


def test_linearity():
    n, bc = (6, 6, 4), (FREE, PER, FREE)
    rng = _rng(23)
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
    r1 = rng.standard_normal((n[2], n[1], n[0])); r2 = rng.standard_normal((n[2], n[1], n[0]))
    a, b = 0.7, -1.9
    lhs = oracle.solve(a * r1 + b * r2, Kf, bc)
    rhs = a * oracle.solve(r1, Kf, bc) + b * oracle.solve(r2, Kf, bc)
    assert rel_l2(lhs, rhs) < 1e-14


def test_fully_periodic_plane_wave_closed_form():
    """rho = cos(k.r), K_f = -1/|k|^2  =>  V = -rho/|k|^2 exactly on the grid."""
    n, h = (8, 12, 6), 0.3
    m = (1, 2, 1)
    bc = (PER, PER, PER)
    kvec = [2 * math.pi * m[a] / (n[a] * h) for a in range(3)]
    z, y, x = np.meshgrid(np.arange(n[2]) * h, np.arange(n[1]) * h, np.arange(n[0]) * h, indexing="ij")
    rho = np.cos(kvec[0] * x + kvec[1] * y + kvec[2] * z)
    Kf = gen.periodic_kernel_spectrum(n, h)
    V = oracle.solve(rho, Kf, bc)
    k2 = sum(kk * kk for kk in kvec)
    assert np.allclose(V, -rho / k2, rtol=0, atol=1e-14)


def test_mirror_symmetric_density_gives_mirror_symmetric_potential():
    n, bc = (6, 4, 4), (FREE, FREE, PER)
    rng = _rng(24)
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
    rho = rng.standard_normal((n[2], n[1], n[0]))
    rho = 0.5 * (rho + rho[:, :, ::-1])  # mirror in x about the box centre
    V = oracle.solve(rho, Kf, bc)
    assert rel_l2(V, V[:, :, ::-1]) < 1e-13


@pytest.mark.parametrize("bc", [(FREE, FREE, FREE), (PER, PER, FREE), (FREE, FREE, PER)])
def test_library_second_opinion_pocketfft(bc):
    """irfftn(rfftn(pad) * K_f) from numpy's pocketfft -- a different algorithm, test-only."""
    n = (8, 6, 10)
    rng = _rng(25)
    s = gen.padded_shape(n, bc)
    K = _even_kernel(rng, s)
    Kf = oracle.kernel_spectrum(K)
    assert rel_l2(Kf, np.fft.rfftn(K).real) < 1e-13
    rho = rng.standard_normal((n[2], n[1], n[0]))
    ref = np.fft.irfftn(np.fft.rfftn(_pad(rho, s)) * Kf, s=(s[2], s[1], s[0]), axes=(0, 1, 2))[: n[2], : n[1], : n[0]]
    assert rel_l2(oracle.solve(rho, Kf, bc), ref) < 1e-13


def test_stages_and_axis_order_independence():
    n, bc = (4, 6, 4), (FREE, PER, FREE)
    rng = _rng(26)
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
    rho = rng.standard_normal((n[2], n[1], n[0]))
    V0, st0 = oracle.solve(rho, Kf, bc, axis_order=(0, 1, 2), return_stages=True)
    V1, st1 = oracle.solve(rho, Kf, bc, axis_order=(2, 1, 0), return_stages=True)
    assert rel_l2(V1, V0) < 1e-14
    pad = _pad(rho, s)
    assert rel_l2(st0[0], np.fft.fft(pad, axis=2)) < 1e-14      # after the x sweep
    assert rel_l2(st1[0], np.fft.fft(pad, axis=0)) < 1e-14      # after the z sweep
    assert rel_l2(st0[2], np.fft.fftn(pad)) < 1e-13
    assert rel_l2(st1[2], st0[2]) < 1e-13


def _full_spectrum(Kf_half, s):
    """Full [Sz][Sy][Sx] spectrum from the half the data contract holds: K_f(-k) = K_f(k) (index reflection only)."""
    sx, sy, sz = s
    full = np.empty((sz, sy, sx))
    full[:, :, : sx // 2 + 1] = Kf_half
    kx = np.arange(sx // 2 + 1, sx)
    full[:, :, sx // 2 + 1:] = Kf_half[(-np.arange(sz)) % sz][:, (-np.arange(sy)) % sy][:, :, sx - kx]
    return full


@pytest.mark.parametrize("bc,order", [((FREE, PER, FREE), (1, 2, 0)), ((FREE, FREE, FREE), (2, 1, 0)), ((PER, PER, FREE), (1, 0, 2)),
                                      ((FREE, FREE, PER), (2, 1, 0))])
def test_every_stage_of_oracle_solve_against_library_fft_per_axis(bc, order):
    """All six intermediates oracle.solve exposes (the per-pass parity references of the GPU tests), each against
    numpy's FFT applied one axis at a time in the same order: after each forward sweep (0, 1, 2), after the K_f
    multiply (3), after the first and second inverse sweep (4, 5).  Array axis of grid axis q is 2 - q.
    A kernel that is inversion symmetric but not even per axis makes stage 3 sensitive to the half-spectrum reflection."""
    n = (6, 4, 10)
    rng = _rng(260 + sum(order) + 7 * sum(bc))
    s = gen.padded_shape(n, bc)
    Kf = oracle.kernel_spectrum(_inversion_kernel(rng, s))
    rho = rng.standard_normal((n[2], n[1], n[0]))
    V, st = oracle.solve(rho, Kf, bc, axis_order=order, return_stages=True)
    a = _pad(rho, s).astype(complex)
    for i in range(3):
        a = np.fft.fft(a, axis=2 - order[i])
        assert rel_l2(st[i], a) < 1e-13, ("forward", i)
    a = a * _full_spectrum(Kf, s)
    assert rel_l2(st[3], a) < 1e-13
    for j, i in enumerate((2, 1)):                                   # inverse sweeps run in reverse order: c, then b
        a = np.fft.ifft(a, axis=2 - order[i]) * s[order[i]]          # unnormalised inverse
        assert rel_l2(st[4 + j], a) < 1e-13, ("inverse", j)
    a = np.fft.ifft(a, axis=2 - order[0]) * s[order[0]]
    assert rel_l2(V, a.real[: n[2], : n[1], : n[0]] / (s[0] * s[1] * s[2])) < 1e-13


@pytest.mark.parametrize("bc", ALL_BC)
def test_solve_equals_direct_sum_16_cubed(bc):
    """north_star: the oracle against the O(N^2) sum of Eq. 2 by brute force "on grids up to 16^3" -- the 16^3 case,
    all 8 BC combinations (padded up to 32^3; 16.8 M kernel-density products per BC)."""
    n = (16, 16, 16)
    rng = _rng(1600 + sum(b << i for i, b in enumerate(bc)))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = _even_kernel(rng, s)
    Kf = oracle.kernel_spectrum(K)
    assert rel_l2(oracle.solve(rho, Kf, bc), oracle.direct_sum(rho, K, bc)) < 1e-13


@pytest.mark.parametrize("bc", ALL_BC)
@pytest.mark.parametrize("n", [(6, 4, 8), (5, 3, 7)])
def test_complex_spectrum_solve_equals_direct_sum_all_bc(bc, n):
    """Eq. 2 holds for ANY real kernel: a random K with no symmetry has a complex spectrum with
    K_f(-k) = conj K_f(k); oracle.solve_complex against the O(N^2) sum, even and odd sizes, all 8 BC combinations."""
    rng = _rng(300 + sum(b << i for i, b in enumerate(bc)) + n[0])
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = rng.standard_normal((s[2], s[1], s[0]))
    Kf = oracle.kernel_spectrum_complex(K)
    assert rel_l2(Kf, np.fft.rfftn(K)) < 1e-13                        # library second opinion on the spectrum itself
    V, vimag = oracle.solve_complex(rho, Kf, bc, return_max_imag=True)
    assert vimag < 1e-13 * np.abs(V).max()
    assert rel_l2(V, oracle.direct_sum(rho, K, bc)) < 1e-13
    # a symmetric kernel through the complex route reproduces the real route
    Ke = _even_kernel(rng, s)
    assert rel_l2(oracle.solve_complex(rho, oracle.kernel_spectrum_complex(Ke), bc), oracle.solve(rho, oracle.kernel_spectrum(Ke), bc)) < 1e-13


@pytest.mark.parametrize("bc", ALL_BC)
def test_solve_equals_direct_sum_odd_and_prime_sizes(bc):
    """Odd N on every axis (S = N on periodic axes is then odd: the half spectrum has S/2+1 = (S+1)/2 entries)."""
    n = (7, 5, 3)
    rng = _rng(700 + sum(b << i for i, b in enumerate(bc)))
    s = gen.padded_shape(n, bc)
    rho = rng.standard_normal((n[2], n[1], n[0]))
    K = _even_kernel(rng, s)
    assert rel_l2(oracle.solve(rho, oracle.kernel_spectrum(K), bc), oracle.direct_sum(rho, K, bc)) < 1e-13


# ----------------------------------------------------------------------------- the workloads themselves
def test_workload_generators_are_seeded_and_shaped():
    cfg = gen.get_config("c0")
    r1 = gen.gaussian_density(cfg); r2 = gen.gaussian_density(cfg)
    assert r1.shape == (32, 32, 32) and np.array_equal(r1, r2)
    assert abs(r1.sum() * cfg.h ** 3) < 2e-2                    # "net charge 0" up to tail truncation (reading 10)
    K = gen.green_kernel_realspace(cfg.n, cfg.bc, cfg.h)
    assert K.shape == (64, 64, 64)
    assert K[0, 0, 0] == pytest.approx(1.0 / (4 * math.pi * 0.5 * cfg.h))
    assert K[0, 0, 1] == pytest.approx(1.0 / (4 * math.pi * cfg.h))
    for ax in range(3):                                         # even along every axis
        assert np.array_equal(K, np.roll(np.flip(K, axis=ax), 1, axis=ax))
    rng = gen.SplitMix64(1234567)
    assert rng.next_u64() == 6457827717110365317                # splitmix64 reference value for seed 1234567


def test_config0_oracle_vs_direct_sum_samples():
    """Config 0 end to end: K_f from the naive DFT of the Green's function, solve, and Eq. 2 at samples."""
    cfg = gen.get_config("c0")
    rho = gen.gaussian_density(cfg)
    K = gen.green_kernel_realspace(cfg.n, cfg.bc, cfg.h)
    Kf, max_imag = oracle.kernel_spectrum(K, return_max_imag=True)
    assert max_imag < 1e-12 * np.abs(Kf).max()
    V = oracle.solve(rho, Kf, cfg.bc)
    pts = _rng(30).integers(0, rho.size, size=64)
    ref = oracle.direct_sum_at(rho, K, cfg.bc, pts)
    assert np.allclose(V.ravel()[pts], ref, rtol=0, atol=1e-13 * np.abs(ref).max())
