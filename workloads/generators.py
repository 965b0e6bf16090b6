"""Seeded synthetic workloads for the free/wire/surface/periodic Poisson solve.

The paper (§4) benchmarks on "various grid sizes" with BigDFT-style smooth
localised charge densities; the sizes and data live in figures that are not available.  The
inputs below are the stand-ins BASELINE.json's `configs` spell out (recipe restated in
DESIGN.md §"Input recipe").  Everything is a pure function of (config, seed).

No DFT / convolution / solver arithmetic lives here -- only
  * rho: sums of normalised isotropic Gaussians (separable evaluation),
  * K  : samples of the real-space Green's function 1/(4 pi r) (+ periodic images),
  * K_f: the one kernel that is *defined* in Fourier space, -1/|k|^2 (fully periodic case).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Tuple

import numpy as np

FREE = 0      # matches POISSON_BC_FREE in include/poisson.h
PERIODIC = 1  # matches POISSON_BC_PERIODIC

BASE_SEED = 12115244  # arxiv id 1211.5244


class SplitMix64:
    """Counter-based splitmix64; doubles are the top 53 bits / 2^53."""

    MASK = (1 << 64) - 1

    def __init__(self, seed: int):
        self.state = seed & self.MASK

    def next_u64(self) -> int:
        self.state = (self.state + 0x9E3779B97F4A7C15) & self.MASK
        z = self.state
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & self.MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & self.MASK
        return z ^ (z >> 31)

    def uniform(self, lo: float = 0.0, hi: float = 1.0) -> float:
        u = (self.next_u64() >> 11) * (1.0 / (1 << 53))
        return lo + (hi - lo) * u


@dataclass(frozen=True)
class WorkloadConfig:
    name: str
    n: Tuple[int, int, int]            # physical grid (nx, ny, nz)
    bc: Tuple[int, int, int]           # per axis x,y,z: FREE / PERIODIC
    h: float
    n_gauss: int
    sigma_h: Tuple[float, float]       # sigma range in units of h
    centre: Tuple[Tuple[float, float], Tuple[float, float], Tuple[float, float]]  # per axis, fraction of L
    seed: int
    precision: str = "fp64"
    chain_z: bool = False              # config 3: centres equally spaced along z
    kernel: str = "green"              # "green" (1/(4 pi r) + images) or "periodic_k2" (-1/k^2)
    images: int = 4                    # |m| <= images on periodic axes (reading 9)
    extra: dict = field(default_factory=dict, compare=False)

    @property
    def s(self) -> Tuple[int, int, int]:
        return tuple(ni * (2 if b == FREE else 1) for ni, b in zip(self.n, self.bc))


def _cfg(idx, name, n, bc, h, ng, sig, centre, **kw):
    return WorkloadConfig(name=name, n=n, bc=bc, h=h, n_gauss=ng, sigma_h=sig, centre=centre,
                          seed=BASE_SEED + idx, **kw)


_INNER = ((0.2, 0.8),) * 3
CONFIGS = {
    # BASELINE.json configs[0..4]; 4a/4b/4p are the three legs of configs[4].
    "c0": _cfg(0, "c0_free_32", (32, 32, 32), (FREE, FREE, FREE), 0.3, 4, (1.0, 2.5), _INNER),
    "c1": _cfg(1, "c1_free_128", (128, 128, 128), (FREE, FREE, FREE), 0.2, 32, (1.0, 4.0), _INNER),
    "c2": _cfg(2, "c2_surface_128", (128, 128, 128), (PERIODIC, PERIODIC, FREE), 0.2, 32, (1.0, 4.0),
               ((0.0, 1.0), (0.0, 1.0), (0.2, 0.8))),
    "c3": _cfg(3, "c3_wire_96x96x256", (96, 96, 256), (FREE, FREE, PERIODIC), 0.2, 64, (1.0, 3.0),
               ((0.4, 0.6), (0.4, 0.6), (0.0, 1.0)), chain_z=True),
    "c4a": _cfg(4, "c4a_free_256_fp64", (256, 256, 256), (FREE, FREE, FREE), 0.2, 256, (1.0, 4.0), _INNER),
    "c4b": _cfg(4, "c4b_free_256_fp32", (256, 256, 256), (FREE, FREE, FREE), 0.2, 256, (1.0, 4.0), _INNER,
                precision="fp32"),
    "c4p": _cfg(4, "c4p_periodic_256", (256, 256, 256), (PERIODIC, PERIODIC, PERIODIC), 0.2, 256, (1.0, 4.0),
                _INNER, kernel="periodic_k2"),
}


def get_config(key: str) -> WorkloadConfig:
    return CONFIGS[key]


def padded_shape(n, bc):
    """S_i = N_i * B_i with B = 1 periodic, 2 free."""
    return tuple(int(ni) * (2 if b == FREE else 1) for ni, b in zip(n, bc))


def signed_displacement(s: int) -> np.ndarray:
    """d(j) = j for j <= S/2, j - S otherwise (kernel origin at index 0, wrap-around order)."""
    j = np.arange(s)
    return np.where(j <= s // 2, j, j - s).astype(np.float64)


def draw_gaussians(cfg: WorkloadConfig):
    """Per Gaussian four draws in the order c_x, c_y, c_z, sigma; q = +1 (even index), -1 (odd)."""
    rng = SplitMix64(cfg.seed)
    nx, ny, nz = cfg.n
    L = (nx * cfg.h, ny * cfg.h, nz * cfg.h)
    out = []
    for g in range(cfg.n_gauss):
        c = [rng.uniform(cfg.centre[a][0] * L[a], cfg.centre[a][1] * L[a]) for a in range(3)]
        sigma = rng.uniform(cfg.sigma_h[0], cfg.sigma_h[1]) * cfg.h
        if cfg.chain_z:
            c[2] = (g + 0.5) * L[2] / cfg.n_gauss
        out.append((c[0], c[1], c[2], sigma, 1.0 if g % 2 == 0 else -1.0))
    return out


def gaussian_density(cfg: WorkloadConfig, dtype=np.float64) -> np.ndarray:
    """rho[z][y][x] = sum_g q_g (2 pi)^{-3/2} sigma_g^{-3} exp(-|r - c_g|^2 / (2 sigma_g^2)).

    Grid point i sits at r = i*h; on periodic axes the minimum-image distance is used.
    Evaluated separably (a Gaussian is a product of three 1D Gaussians)."""
    nx, ny, nz = cfg.n
    gs = draw_gaussians(cfg)
    G = len(gs)
    fx = np.empty((G, nx)); fy = np.empty((G, ny)); fz = np.empty((G, nz))
    for gi, (cx, cy, cz, sig, q) in enumerate(gs):
        for arr, c, n_a, b in ((fx, cx, nx, cfg.bc[0]), (fy, cy, ny, cfg.bc[1]), (fz, cz, nz, cfg.bc[2])):
            d = np.arange(n_a) * cfg.h - c
            if b == PERIODIC:
                La = n_a * cfg.h
                d = d - La * np.round(d / La)
            arr[gi] = np.exp(-0.5 * (d / sig) ** 2)
        fz[gi] *= q / ((2.0 * math.pi) ** 1.5 * sig ** 3)
    yx = (fy[:, :, None] * fx[:, None, :]).reshape(G, ny * nx)
    rho = (fz.T @ yx).reshape(nz, ny, nx)
    return np.ascontiguousarray(rho.astype(dtype))


def green_kernel_realspace(n, bc, h, images: int = 4) -> np.ndarray:
    """K[jz][jy][jx] on the padded S grid: 1/(4 pi |d|), d the signed displacement times h.

    * K(0) = 1/(4 pi 0.5 h)                                   (BASELINE.json configs[0])
    * periodic axes add images d_i + m N_i h, |m| <= images   (configs[2], [3]; reading 9)
    The result is even along every axis, so its DFT is real."""
    s = padded_shape(n, bc)
    d = [signed_displacement(s[a]) * h for a in range(3)]
    ms = [range(-images, images + 1) if bc[a] == PERIODIC else (0,) for a in range(3)]
    K = np.zeros((s[2], s[1], s[0]))
    inv4pi = 1.0 / (4.0 * math.pi)
    for mz in ms[2]:
        dz2 = (d[2] + mz * n[2] * h) ** 2
        for my in ms[1]:
            dy2 = (d[1] + my * n[1] * h) ** 2
            for mx in ms[0]:
                dx2 = (d[0] + mx * n[0] * h) ** 2
                r2 = dz2[:, None, None] + dy2[None, :, None] + dx2[None, None, :]
                if mx == 0 and my == 0 and mz == 0:
                    r2[0, 0, 0] = (0.5 * h) ** 2
                K += inv4pi / np.sqrt(r2)
    return K


def periodic_kernel_spectrum(n, h) -> np.ndarray:
    """K_f[kz][ky][kx<=nx/2] = -1/|k|^2, k_i = 2 pi f_i / (N_i h), f_i the signed frequency; K_f(0)=0."""
    nx, ny, nz = n
    kx = 2.0 * math.pi * np.fft.rfftfreq(nx, d=h)
    ky = 2.0 * math.pi * np.fft.fftfreq(ny, d=h)
    kz = 2.0 * math.pi * np.fft.fftfreq(nz, d=h)
    k2 = kz[:, None, None] ** 2 + ky[None, :, None] ** 2 + kx[None, None, :] ** 2
    k2[0, 0, 0] = 1.0
    out = -1.0 / k2
    out[0, 0, 0] = 0.0
    return out
