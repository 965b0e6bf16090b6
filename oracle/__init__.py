"""ctypes binding of the CPU oracle (oracle/poisson_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It never imports paper_1211_5244_b200 (the CUDA path) and shares no code
with it.  See the header of poisson_oracle.c for what each function computes and which passage
of the paper it follows.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "poisson_oracle.c"
_LIB = _HERE / "liboracle.so"
_lib = None

_LL3 = ctypes.c_longlong * 3
_I3 = ctypes.c_int * 3


def build(force: bool = False) -> Path:
    """gcc -O2 -fopenmp; -ffp-contract=off keeps every multiply and add separately rounded."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        cmd = ["gcc", "-std=c11", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               str(_SRC), "-o", str(_LIB), "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(str(_LIB))
        p = ctypes.c_void_p
        lib.oracle_dft_axis.argtypes = [p, _LL3, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.oracle_kernel_spectrum.argtypes = [p, _LL3, p, ctypes.POINTER(ctypes.c_double), ctypes.c_int]
        lib.oracle_solve.argtypes = [p, p, p, _LL3, _I3, p, p, ctypes.POINTER(ctypes.c_double), ctypes.c_int]
        lib.oracle_kernel_spectrum_c.argtypes = [p, _LL3, p, ctypes.c_int]
        lib.oracle_solve_c.argtypes = [p, p, p, _LL3, _I3, p, p, ctypes.POINTER(ctypes.c_double), ctypes.c_int]
        lib.oracle_direct_sum_at.argtypes = [p, p, _LL3, _I3, p, ctypes.c_longlong, p]
        lib.oracle_direct_sum.argtypes = [p, p, _LL3, _I3, p]
        for f in (lib.oracle_dft_axis, lib.oracle_kernel_spectrum, lib.oracle_solve, lib.oracle_kernel_spectrum_c, lib.oracle_solve_c,
                  lib.oracle_direct_sum_at, lib.oracle_direct_sum):
            f.restype = ctypes.c_int
        _lib = lib
    return _lib


def _check(st, what):
    if st != 0:
        raise RuntimeError(f"oracle: {what} failed with status {st}")


def _ptr(a: np.ndarray):
    return ctypes.c_void_p(a.ctypes.data)


def n_threads() -> int:
    """Threads the OpenMP loops will use (OMP_NUM_THREADS or all cores)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def dft_axis(a: np.ndarray, axis: int, sign: int = -1, accum_ld: bool = False) -> np.ndarray:
    """DFT by definition along `axis` of a 3D complex array (sign -1 forward, +1 inverse, unnormalised)."""
    out = np.ascontiguousarray(a, dtype=np.complex128).copy()
    assert out.ndim == 3
    _check(_load().oracle_dft_axis(_ptr(out), _LL3(*out.shape), axis, sign, int(accum_ld)), "dft_axis")
    return out


def kernel_spectrum(K: np.ndarray, accum_ld: bool = False, return_max_imag: bool = False):
    """K real [Sz][Sy][Sx] -> K_f real [Sz][Sy][Sx/2+1] (library data contract) by the naive DFT."""
    K = np.ascontiguousarray(K, dtype=np.float64)
    sz, sy, sx = K.shape
    full = np.empty_like(K)
    mi = ctypes.c_double(0.0)
    _check(_load().oracle_kernel_spectrum(_ptr(K), _LL3(sx, sy, sz), _ptr(full), ctypes.byref(mi),
                                          int(accum_ld)), "kernel_spectrum")
    half = np.ascontiguousarray(full[:, :, : sx // 2 + 1])
    return (half, mi.value) if return_max_imag else half


def solve(rho: np.ndarray, Kf_half: np.ndarray, bc, axis_order=(0, 1, 2), return_stages: bool = False,
          accum_ld: bool = False, return_max_imag: bool = False):
    """Eq. 3 on the explicitly zero-padded grid.  rho [nz][ny][nx]; Kf_half [Sz][Sy][Sx/2+1]; bc = (x,y,z)."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    Kf_half = np.ascontiguousarray(Kf_half, dtype=np.float64)
    nz, ny, nx = rho.shape
    s = [nx * (2 if bc[0] == 0 else 1), ny * (2 if bc[1] == 0 else 1), nz * (2 if bc[2] == 0 else 1)]
    assert Kf_half.shape == (s[2], s[1], s[0] // 2 + 1), (Kf_half.shape, s)
    V = np.empty_like(rho)
    stages = np.empty((6, s[2], s[1], s[0]), dtype=np.complex128) if return_stages else None
    mi = ctypes.c_double(0.0)
    _check(_load().oracle_solve(_ptr(rho), _ptr(Kf_half), _ptr(V), _LL3(nx, ny, nz), _I3(*[int(b) for b in bc]),
                                _ptr(np.asarray(axis_order, dtype=np.int32)),
                                _ptr(stages) if stages is not None else None, ctypes.byref(mi), int(accum_ld)),
           "solve")
    res = [V]
    if return_stages:
        res.append(stages)
    if return_max_imag:
        res.append(mi.value)
    return res[0] if len(res) == 1 else tuple(res)


def kernel_spectrum_complex(K: np.ndarray, accum_ld: bool = False) -> np.ndarray:
    """K real [Sz][Sy][Sx] with NO symmetry -> complex K_f [Sz][Sy][Sx/2+1] (numpy rfftn shape) by the naive DFT."""
    K = np.ascontiguousarray(K, dtype=np.float64)
    sz, sy, sx = K.shape
    full = np.empty(K.shape, dtype=np.complex128)
    _check(_load().oracle_kernel_spectrum_c(_ptr(K), _LL3(sx, sy, sz), _ptr(full), int(accum_ld)), "kernel_spectrum_c")
    return np.ascontiguousarray(full[:, :, : sx // 2 + 1])


def solve_complex(rho: np.ndarray, Kf_half: np.ndarray, bc, axis_order=(0, 1, 2), accum_ld: bool = False,
                  return_max_imag: bool = False):
    """Eq. 3 with a complex half spectrum (real kernel without inversion symmetry; K_f(-k) = conj K_f(k))."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    Kf_half = np.ascontiguousarray(Kf_half, dtype=np.complex128)
    nz, ny, nx = rho.shape
    s = [nx * (2 if bc[0] == 0 else 1), ny * (2 if bc[1] == 0 else 1), nz * (2 if bc[2] == 0 else 1)]
    assert Kf_half.shape == (s[2], s[1], s[0] // 2 + 1), (Kf_half.shape, s)
    V = np.empty_like(rho)
    mi = ctypes.c_double(0.0)
    _check(_load().oracle_solve_c(_ptr(rho), _ptr(Kf_half), _ptr(V), _LL3(nx, ny, nz), _I3(*[int(b) for b in bc]),
                                  _ptr(np.asarray(axis_order, dtype=np.int32)), None, ctypes.byref(mi), int(accum_ld)),
           "solve_c")
    return (V, mi.value) if return_max_imag else V


def direct_sum(rho: np.ndarray, K: np.ndarray, bc) -> np.ndarray:
    """Eq. 2 by brute force over the whole box (tiny grids only)."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    K = np.ascontiguousarray(K, dtype=np.float64)
    nz, ny, nx = rho.shape
    V = np.empty_like(rho)
    _check(_load().oracle_direct_sum(_ptr(rho), _ptr(K), _LL3(nx, ny, nz), _I3(*[int(b) for b in bc]), _ptr(V)),
           "direct_sum")
    return V


def direct_sum_at(rho: np.ndarray, K: np.ndarray, bc, flat_points) -> np.ndarray:
    """Eq. 2 by brute force at sampled output points (flat indices into [nz][ny][nx])."""
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    K = np.ascontiguousarray(K, dtype=np.float64)
    nz, ny, nx = rho.shape
    pts = np.ascontiguousarray(flat_points, dtype=np.int64)
    out = np.empty(pts.shape[0], dtype=np.float64)
    _check(_load().oracle_direct_sum_at(_ptr(rho), _ptr(K), _LL3(nx, ny, nz), _I3(*[int(b) for b in bc]),
                                        _ptr(pts), pts.shape[0], _ptr(out)), "direct_sum_at")
    return out
