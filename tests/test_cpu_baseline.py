"""The timed CPU baseline (baseline/cpu_fft.cpp: the paper's customised FFT on the host) against the oracle.
CPU only.  The baseline is reported by bench.py, it is not the product and not the oracle."""
import itertools

import numpy as np
import pytest

import baseline
import oracle
from workloads import generators as gen


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / max(np.linalg.norm(b.ravel()), 1e-300))


def _even_kernel(rng, s):
    sx, sy, sz = s
    K = rng.standard_normal((sz, sy, sx))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    return K


@pytest.mark.parametrize("n", [(8, 6, 4), (16, 12, 10), (7, 5, 3), (9, 20, 15), (32, 3, 14)])
def test_cpu_baseline_matches_oracle_all_bc(n):
    rng = np.random.default_rng(11 + sum(n))
    for bc in itertools.product((0, 1), repeat=3):
        s = gen.padded_shape(n, bc)
        rho = rng.standard_normal((n[2], n[1], n[0]))
        Kf = oracle.kernel_spectrum(_even_kernel(rng, s))
        ref = oracle.solve(rho, Kf, bc)
        assert rel_l2(baseline.solve(rho, Kf, bc), ref) < 1e-12, (n, bc)
        assert rel_l2(baseline.solve(rho, Kf, bc, threads=1), ref) < 1e-12, (n, bc)


def test_cpu_baseline_on_config0():
    cfg = gen.get_config("c0")
    rho = gen.gaussian_density(cfg)
    Kf = oracle.kernel_spectrum(gen.green_kernel_realspace(cfg.n, cfg.bc, cfg.h))
    assert rel_l2(baseline.solve(rho, Kf, cfg.bc), oracle.solve(rho, Kf, cfg.bc)) < 1e-12
    assert baseline.max_threads() >= 1
