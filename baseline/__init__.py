"""ctypes binding of the timed CPU baseline (baseline/cpu_fft.cpp): the paper's customised-FFT Poisson solve on the host with
an FFTW-free Stockham FFT -- the analogue of the paper's "CPU implementation of the same method".

Reported by bench.py beside the GPU numbers.  Not the product (no CUDA here), not the oracle (tests/test_cpu_baseline.py
checks it AGAINST the oracle); it shares no code with either."""
from __future__ import annotations

import ctypes
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "cpu_fft.cpp"
_LIB = _HERE / "libcpu_fft.so"
_lib = None


def build(force: bool = False) -> Path:
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        subprocess.run(["g++", "-std=c++17", "-O3", "-march=native", "-fcx-limited-range", "-fopenmp", "-fPIC", "-shared", str(_SRC), "-o", str(_LIB)],
                       check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        lib.cpu_poisson_solve.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int * 3, ctypes.c_int * 3, ctypes.c_int]
        lib.cpu_poisson_solve.restype = ctypes.c_int
        lib.cpu_fft_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().cpu_fft_max_threads())


def solve(rho: np.ndarray, Kf_half: np.ndarray, bc, threads: int = 0) -> np.ndarray:
    """rho [nz][ny][nx] float64, Kf_half [Sz][Sy][Sx/2+1] float64, bc = (x, y, z) with 0 free / 1 periodic."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    Kf_half = np.ascontiguousarray(Kf_half, dtype=np.float64)
    nz, ny, nx = rho.shape
    s = [nx * (2 if bc[0] == 0 else 1), ny * (2 if bc[1] == 0 else 1), nz * (2 if bc[2] == 0 else 1)]
    assert Kf_half.shape == (s[2], s[1], s[0] // 2 + 1), (Kf_half.shape, s)
    V = np.empty_like(rho)
    st = _load().cpu_poisson_solve(rho.ctypes.data, Kf_half.ctypes.data, V.ctypes.data, (ctypes.c_int * 3)(nx, ny, nz),
                                   (ctypes.c_int * 3)(*[int(b) for b in bc]), int(threads))
    if st != 0:
        raise RuntimeError(f"cpu_poisson_solve failed with status {st}")
    return V
