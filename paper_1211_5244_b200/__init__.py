"""paper_1211_5244_b200 -- thin Python binding of the C-ABI library in include/poisson.h.

Argument marshalling only: every step of the solve runs in the hand-written sm_100a kernels of
libpoisson_b200.so.  PyTorch is used by callers for device memory and streams; this module only
needs `.data_ptr()` integers and a raw cudaStream_t.  There is no CPU fallback: if the library
is missing or no B200 is present the calls raise.
"""
from __future__ import annotations

import ctypes
from pathlib import Path

__all__ = [
    "FREE", "PERIODIC", "FP64", "FP32", "PoissonError", "PlanInfo", "lib_path", "load_library",
    "poisson_plan_describe", "poisson_plan_create", "poisson_set_kernel", "poisson_solve",
    "poisson_solve_host", "poisson_plan_destroy", "poisson_measure_fma_peak", "PoissonPlan", "EXPORTED_SYMBOLS",
    "poisson_set_kernel_even", "poisson_set_kernel_complex", "poisson_shard_describe", "ShardInfo", "ShardPlan", "ShardedSolver",
    "poisson_solve_static", "STATIC_SCRATCH_BYTES",
]

FREE, PERIODIC = 0, 1
FP64, FP32 = 0, 1
PASS_NAMES = ("F1", "F2", "F3", "I2", "I1")

EXPORTED_SYMBOLS = (
    "poisson_plan_describe", "poisson_plan_create", "poisson_plan_kernel_dims", "poisson_plan_get_info",
    "poisson_set_kernel", "poisson_set_kernel_complex", "poisson_solve", "poisson_solve_host", "poisson_debug_workspace",
    "poisson_debug_run_passes", "poisson_solve_profiled", "poisson_profile_read", "poisson_plan_launches_per_solve", "poisson_measure_fma_peak", "poisson_plan_workspace_bytes",
    "poisson_plan_destroy", "poisson_status_string", "poisson_last_error", "poisson_build_arch", "poisson_plan_launch_mode", "poisson_plan_graph_shape", "poisson_set_kernel_even", "poisson_shard_describe", "poisson_shard_plan_create", "poisson_shard_get_info", "poisson_shard_set_slabs", "poisson_shard_set_kernel", "poisson_shard_forward", "poisson_shard_middle", "poisson_shard_inverse", "poisson_solve_batch", "poisson_solve_batch_host", "poisson_plan_batch_lanes", "poisson_plan_batch_width",
    "poisson_solve_static",
)

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libpoisson_b200.so"
_lib = None


class PoissonError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        super().__init__(f"{where}: status {status} ({detail})")


class PlanInfo(ctypes.Structure):
    """Mirror of `poisson_plan_info` (include/poisson.h)."""
    _fields_ = [
        ("n", ctypes.c_int * 3), ("bc", ctypes.c_int * 3), ("s", ctypes.c_int * 3),
        ("precision", ctypes.c_int), ("order", ctypes.c_int * 3), ("half_len", ctypes.c_int),
        ("rows", ctypes.c_longlong * 5), ("length", ctypes.c_longlong * 5), ("bytes", ctypes.c_longlong * 5),
        ("bytes_total", ctypes.c_longlong), ("workspace_bytes", ctypes.c_longlong),
        ("fft_fraction", ctypes.c_double),
    ]

    def as_dict(self):
        return {
            "n": list(self.n), "bc": list(self.bc), "s": list(self.s), "precision": self.precision,
            "order": list(self.order), "half_len": self.half_len, "rows": list(self.rows),
            "length": list(self.length), "bytes": list(self.bytes), "bytes_total": self.bytes_total,
            "workspace_bytes": self.workspace_bytes, "fft_fraction": self.fft_fraction,
        }


class ShardInfo(ctypes.Structure):
    """Mirror of `poisson_shard_info` (include/poisson.h)."""
    _fields_ = [
        ("rank", ctypes.c_int), ("nranks", ctypes.c_int), ("split_axis", ctypes.c_int), ("plane_axis", ctypes.c_int),
        ("o0", ctypes.c_int), ("o1", ctypes.c_int), ("k0", ctypes.c_int), ("k1", ctypes.c_int),
        ("local_dims", ctypes.c_longlong * 3), ("mid_dims", ctypes.c_longlong * 3), ("back_dims", ctypes.c_longlong * 3),
        ("mid_bytes", ctypes.c_longlong), ("back_bytes", ctypes.c_longlong), ("sent_bytes", ctypes.c_longlong * 2),
        ("workspace_bytes", ctypes.c_longlong),
    ]

    def as_dict(self):
        return {k: (list(getattr(self, k)) if hasattr(getattr(self, k), "__len__") else getattr(self, k)) for k, _ in self._fields_}


def lib_path() -> Path:
    return _LIB_PATH


def load_library():
    """dlopen the in-tree library.  Fails loudly when it has not been built (no fallback exists)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise ImportError(
            f"{_LIB_PATH} is missing: run `python -m paper_1211_5244_b200.build` (or __graft_entry__.build()). "
            "The solve has no CPU or library fallback.")
    lib = ctypes.CDLL(str(_LIB_PATH))
    vp, i, ll = ctypes.c_void_p, ctypes.c_int, ctypes.c_longlong
    i3 = ctypes.c_int * 3
    lib.poisson_plan_describe.argtypes = [i, i, i, i3, i, ctypes.POINTER(PlanInfo)]
    lib.poisson_plan_create.argtypes = [ctypes.POINTER(vp), i, i, i, i3, ctypes.c_double, i]
    lib.poisson_plan_kernel_dims.argtypes = [vp, ll * 3]
    lib.poisson_plan_get_info.argtypes = [vp, ctypes.POINTER(PlanInfo)]
    lib.poisson_set_kernel.argtypes = [vp, vp, vp]
    lib.poisson_set_kernel_complex.argtypes = [vp, vp, vp]
    lib.poisson_set_kernel_even.argtypes = [vp, vp, vp]
    lib.poisson_solve.argtypes = [vp, vp, vp, vp]
    lib.poisson_solve_host.argtypes = [vp, vp, vp, vp]
    lib.poisson_debug_workspace.argtypes = [vp, i, ctypes.POINTER(vp), ll * 3]
    lib.poisson_debug_run_passes.argtypes = [vp, vp, vp, vp, i, i]
    lib.poisson_solve_profiled.argtypes = [vp, vp, vp, vp]
    lib.poisson_profile_read.argtypes = [vp, ctypes.c_double * 5, ctypes.POINTER(i)]
    lib.poisson_measure_fma_peak.argtypes = [i, ctypes.POINTER(ctypes.c_double)]
    lib.poisson_plan_launches_per_solve.argtypes = [vp]
    lib.poisson_plan_batch_lanes.argtypes = [vp, i, i]
    lib.poisson_plan_batch_width.argtypes = [vp, i]
    lib.poisson_plan_batch_width.restype = i
    lib.poisson_solve_batch.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), i, vp]
    lib.poisson_solve_batch_host.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp), i, vp]
    lib.poisson_plan_launch_mode.argtypes = [vp, ctypes.POINTER(i), ctypes.c_double * 5]
    lib.poisson_plan_graph_shape.argtypes = [vp, ctypes.POINTER(i), ctypes.POINTER(i)]
    lib.poisson_shard_describe.argtypes = [i, i, i, i3, i, i, i, ctypes.POINTER(ShardInfo)]
    lib.poisson_shard_plan_create.argtypes = [ctypes.POINTER(vp), i, i, i, i3, ctypes.c_double, i, i, i]
    lib.poisson_shard_get_info.argtypes = [vp, ctypes.POINTER(ShardInfo)]
    lib.poisson_shard_set_slabs.argtypes = [vp, ctypes.POINTER(vp), ctypes.POINTER(vp)]
    lib.poisson_shard_set_kernel.argtypes = [vp, vp, vp]
    lib.poisson_shard_forward.argtypes = [vp, vp, vp]
    lib.poisson_shard_middle.argtypes = [vp, vp]
    lib.poisson_shard_inverse.argtypes = [vp, vp, vp]
    lib.poisson_solve_static.argtypes = [i, i, i, i3, i, vp, vp, vp, vp]
    lib.poisson_plan_workspace_bytes.argtypes = [vp]
    lib.poisson_plan_workspace_bytes.restype = ctypes.c_size_t
    lib.poisson_plan_destroy.argtypes = [vp]
    lib.poisson_status_string.argtypes = [i]
    lib.poisson_status_string.restype = ctypes.c_char_p
    lib.poisson_last_error.restype = ctypes.c_char_p
    lib.poisson_build_arch.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _check(status: int, where: str):
    if status != 0:
        lib = load_library()
        msg = lib.poisson_status_string(status).decode()
        extra = lib.poisson_last_error().decode()
        raise PoissonError(status, where, msg + (f"; {extra}" if extra else ""))


# ------------------------------------------------------------------ function-level API (same names as the C ABI)
def poisson_plan_describe(nx: int, ny: int, nz: int, bc, precision: int = FP64) -> PlanInfo:
    info = PlanInfo()
    _check(load_library().poisson_plan_describe(nx, ny, nz, (ctypes.c_int * 3)(*bc), precision, ctypes.byref(info)),
           "poisson_plan_describe")
    return info


def poisson_plan_create(nx: int, ny: int, nz: int, bc, h: float, precision: int = FP64) -> int:
    """Returns the opaque plan handle (an integer address)."""
    handle = ctypes.c_void_p()
    _check(load_library().poisson_plan_create(ctypes.byref(handle), nx, ny, nz, (ctypes.c_int * 3)(*bc), float(h),
                                              precision), "poisson_plan_create")
    return handle.value


def poisson_set_kernel(plan: int, K_f_dev_ptr: int, stream: int = 0) -> None:
    _check(load_library().poisson_set_kernel(plan, K_f_dev_ptr, stream), "poisson_set_kernel")


def poisson_set_kernel_even(plan: int, K_f_dev_ptr: int, stream: int = 0) -> None:
    _check(load_library().poisson_set_kernel_even(plan, K_f_dev_ptr, stream), "poisson_set_kernel_even")


def poisson_set_kernel_complex(plan: int, K_f_dev_ptr: int, stream: int = 0) -> None:
    _check(load_library().poisson_set_kernel_complex(plan, K_f_dev_ptr, stream), "poisson_set_kernel_complex")


def poisson_solve(plan: int, rho_dev_ptr: int, V_dev_ptr: int, stream: int = 0) -> None:
    _check(load_library().poisson_solve(plan, rho_dev_ptr, V_dev_ptr, stream), "poisson_solve")


def poisson_solve_host(plan: int, rho_host_ptr: int, V_host_ptr: int, stream: int = 0) -> None:
    _check(load_library().poisson_solve_host(plan, rho_host_ptr, V_host_ptr, stream), "poisson_solve_host")


STATIC_SCRATCH_BYTES = 32 << 20   # POISSON_STATIC_SCRATCH_BYTES of include/poisson.h


def poisson_solve_static(nx: int, ny: int, nz: int, bc, precision: int, K_f_dev_ptr: int, rho_dev_ptr: int, V_dev_ptr: int,
                         stream: int = 0) -> None:
    """A whole solve without a plan and without any device allocation, for callers that cannot cudaMalloc (all device
    memory already in the application's own pool, a fixed memory budget, an inner loop that must not hit an allocation
    failure or cudaMalloc's device-wide synchronisation).  Scratch is the library's fixed STATIC_SCRATCH_BYTES array, one
    per GPU, shared by every call: grids that do not fit raise PoissonError (status 2), and calls whose GPU work could
    overlap must be ordered by the caller.  Same kernels and bits as PoissonPlan.solve.  See include/poisson.h."""
    _check(load_library().poisson_solve_static(nx, ny, nz, (ctypes.c_int * 3)(*bc), precision, K_f_dev_ptr, rho_dev_ptr,
                                               V_dev_ptr, stream), "poisson_solve_static")


def poisson_measure_fma_peak(precision: int = FP64) -> float:
    """Plain-ALU FMA peak of the current device in TFLOP/s (FMA = 2 flops)."""
    out = ctypes.c_double()
    _check(load_library().poisson_measure_fma_peak(precision, ctypes.byref(out)), "poisson_measure_fma_peak")
    return out.value


def poisson_plan_destroy(plan: int) -> None:
    _check(load_library().poisson_plan_destroy(plan), "poisson_plan_destroy")


def poisson_shard_describe(nx: int, ny: int, nz: int, bc, precision: int, rank: int, nranks: int) -> ShardInfo:
    info = ShardInfo()
    _check(load_library().poisson_shard_describe(nx, ny, nz, (ctypes.c_int * 3)(*bc), precision, rank, nranks, ctypes.byref(info)),
           "poisson_shard_describe")
    return info


# ------------------------------------------------------------------ small convenience wrapper over torch tensors
class PoissonPlan:
    """Owns a plan handle; takes torch CUDA tensors and forwards their pointers (no arithmetic here)."""

    def __init__(self, n, bc, h: float, precision: int = FP64):
        self.n = tuple(int(v) for v in n)          # (nx, ny, nz)
        self.bc = tuple(int(v) for v in bc)
        self.precision = precision
        self._h = poisson_plan_create(self.n[0], self.n[1], self.n[2], self.bc, h, precision)
        info = PlanInfo()
        _check(load_library().poisson_plan_get_info(self._h, ctypes.byref(info)), "poisson_plan_get_info")
        self.info = info
        dims = (ctypes.c_longlong * 3)()
        _check(load_library().poisson_plan_kernel_dims(self._h, dims), "poisson_plan_kernel_dims")
        self.kernel_dims = tuple(dims)

    @property
    def handle(self) -> int:
        return self._h

    @staticmethod
    def _stream(stream):
        if stream is None:
            import torch
            return torch.cuda.current_stream().cuda_stream
        return int(getattr(stream, "cuda_stream", stream))

    def _dtype(self):
        import torch
        return torch.float64 if self.precision == FP64 else torch.float32

    def set_kernel(self, K_f, stream=None):
        assert K_f.is_cuda and K_f.is_contiguous() and K_f.dtype == self._dtype()
        assert tuple(K_f.shape) == self.kernel_dims, (tuple(K_f.shape), self.kernel_dims)
        poisson_set_kernel(self._h, K_f.data_ptr(), self._stream(stream))

    def set_kernel_even(self, K_f, stream=None):
        """K_f of a kernel that is even along every axis: stored folded, half the size (poisson_set_kernel_even)."""
        assert K_f.is_cuda and K_f.is_contiguous() and K_f.dtype == self._dtype()
        assert tuple(K_f.shape) == self.kernel_dims, (tuple(K_f.shape), self.kernel_dims)
        poisson_set_kernel_even(self._h, K_f.data_ptr(), self._stream(stream))

    def set_kernel_complex(self, K_f, stream=None):
        """K_f: complex CUDA tensor [S_z][S_y][S_x/2+1] (rfftn of a real kernel without inversion symmetry)."""
        import torch
        want = torch.complex128 if self.precision == FP64 else torch.complex64
        assert K_f.is_cuda and K_f.is_contiguous() and K_f.dtype == want
        assert tuple(K_f.shape) == self.kernel_dims, (tuple(K_f.shape), self.kernel_dims)
        poisson_set_kernel_complex(self._h, K_f.data_ptr(), self._stream(stream))

    def solve(self, rho, V=None, stream=None):
        import torch
        assert rho.is_cuda and rho.is_contiguous() and rho.dtype == self._dtype()
        assert tuple(rho.shape) == (self.n[2], self.n[1], self.n[0])
        if V is None:
            V = torch.empty_like(rho)
        assert V.is_cuda and V.is_contiguous() and V.dtype == rho.dtype and V.shape == rho.shape
        poisson_solve(self._h, rho.data_ptr(), V.data_ptr(), self._stream(stream))
        return V

    def solve_host(self, rho_host, V_host, stream=None):
        """rho_host / V_host: CPU tensors (pinned for full speed); H2D + solve + D2H + sync inside the C call."""
        assert not rho_host.is_cuda and not V_host.is_cuda and rho_host.is_contiguous() and V_host.is_contiguous()
        assert rho_host.dtype == self._dtype() and V_host.dtype == self._dtype()
        poisson_solve_host(self._h, rho_host.data_ptr(), V_host.data_ptr(), self._stream(stream))
        return V_host

    def solve_profiled(self, rho, V, stream=None):
        _check(load_library().poisson_solve_profiled(self._h, rho.data_ptr(), V.data_ptr(), self._stream(stream)),
               "poisson_solve_profiled")
        return V

    def profile_read(self):
        """(per-pass milliseconds summed over the profiled solves, number of solves); resets the pool."""
        ms = (ctypes.c_double * 5)()
        n = ctypes.c_int()
        _check(load_library().poisson_profile_read(self._h, ms, ctypes.byref(n)), "poisson_profile_read")
        return list(ms), n.value

    def launches_per_solve(self) -> int:
        return load_library().poisson_plan_launches_per_solve(self._h)

    def solve_batch(self, rhos, Vs=None, stream=None):
        """poisson_solve_batch on lists of device tensors (asynchronous; returns the list of V tensors)."""
        import torch
        if Vs is None:
            Vs = [torch.empty_like(r) for r in rhos]
        for r, v in zip(rhos, Vs):
            assert r.is_cuda and r.is_contiguous() and r.dtype == self._dtype() and tuple(r.shape) == (self.n[2], self.n[1], self.n[0])
            assert v.is_cuda and v.is_contiguous() and v.dtype == r.dtype and v.shape == r.shape
        n = len(rhos)
        rp = (ctypes.c_void_p * n)(*[r.data_ptr() for r in rhos])
        vp_ = (ctypes.c_void_p * n)(*[v.data_ptr() for v in Vs])
        _check(load_library().poisson_solve_batch(self._h, rp, vp_, n, self._stream(stream)), "poisson_solve_batch")
        return Vs

    def pointer_batch(self, rhos, Vs):
        """Marshal a batch ONCE: validates the device tensors and returns the two pointer arrays poisson_solve_batch
        takes (what a C caller holds anyway), for repeated solve_pointer_batch calls on the same buffers."""
        for r, v in zip(rhos, Vs):
            assert r.is_cuda and r.is_contiguous() and r.dtype == self._dtype() and tuple(r.shape) == (self.n[2], self.n[1], self.n[0])
            assert v.is_cuda and v.is_contiguous() and v.dtype == r.dtype and v.shape == r.shape
        n = len(rhos)
        rp = (ctypes.c_void_p * n)(*[r.data_ptr() for r in rhos])
        vp_ = (ctypes.c_void_p * n)(*[v.data_ptr() for v in Vs])
        return (rp, vp_, n, list(rhos), list(Vs))     # the tensor lists keep the buffers alive

    def solve_pointer_batch(self, batch, stream=None):
        rp, vp_, n = batch[0], batch[1], batch[2]
        _check(load_library().poisson_solve_batch(self._h, rp, vp_, n, self._stream(stream)), "poisson_solve_batch")

    def solve_batch_host(self, rhos, Vs, stream=None):
        """poisson_solve_batch_host on lists of (pinned) host tensors; returns when every V is on the host."""
        for r, v in zip(rhos, Vs):
            assert (not r.is_cuda) and r.is_contiguous() and r.dtype == self._dtype()
            assert (not v.is_cuda) and v.is_contiguous() and v.dtype == r.dtype and v.shape == r.shape
        n = len(rhos)
        rp = (ctypes.c_void_p * n)(*[r.data_ptr() for r in rhos])
        vp_ = (ctypes.c_void_p * n)(*[v.data_ptr() for v in Vs])
        _check(load_library().poisson_solve_batch_host(self._h, rp, vp_, n, self._stream(stream)), "poisson_solve_batch_host")
        return Vs

    def batch_lanes(self, count: int, host: bool = False) -> int:
        return load_library().poisson_plan_batch_lanes(self._h, count, 1 if host else 0)

    def batch_width(self, count: int) -> int:
        """Densities per launch of a device batch of `count` solves (small grids), 0 = the lane route."""
        return load_library().poisson_plan_batch_width(self._h, count)

    def launch_mode(self):
        """(mode name, {mode name: measured ms per solve at plan creation}) -- see poisson_plan_launch_mode."""
        mode = ctypes.c_int()
        ms = (ctypes.c_double * 5)()
        _check(load_library().poisson_plan_launch_mode(self._h, ctypes.byref(mode), ms), "poisson_plan_launch_mode")
        names = ("five", "five_pdl", "fused", "graph", "graph_pdl")
        return names[mode.value], {names[k]: ms[k] for k in range(5) if ms[k] > 0}

    def graph_shape(self):
        """(chains over k_a plane ranges, chains over x ranges) of the solve graph -- see poisson_plan_graph_shape."""
        j, r = ctypes.c_int(), ctypes.c_int()
        _check(load_library().poisson_plan_graph_shape(self._h, ctypes.byref(j), ctypes.byref(r)), "poisson_plan_graph_shape")
        return j.value, r.value

    def workspace_bytes(self) -> int:
        return load_library().poisson_plan_workspace_bytes(self._h)

    def debug_workspace(self, which: int):
        """(device pointer, (ez, ey, ex)) of intermediate A1 (which=0) or A2 (which=1)."""
        ptr = ctypes.c_void_p()
        dims = (ctypes.c_longlong * 3)()
        _check(load_library().poisson_debug_workspace(self._h, which, ctypes.byref(ptr), dims), "poisson_debug_workspace")
        return ptr.value, tuple(dims)

    def debug_run_passes(self, rho, V, first: int, last: int, stream=None):
        _check(load_library().poisson_debug_run_passes(
            self._h, rho.data_ptr() if rho is not None else None, V.data_ptr() if V is not None else None,
            self._stream(stream), first, last), "poisson_debug_run_passes")

    def close(self):
        if self._h:
            poisson_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class ShardPlan:
    """One rank of a solve sharded over several GPUs (include/poisson.h: poisson_shard_*).  Marshalling only: the caller
    owns the exchange slabs and enqueues the two cross-rank barriers (see ShardedSolver for the torch.distributed plumbing)."""

    def __init__(self, n, bc, h: float, precision: int, rank: int, nranks: int):
        self.n = tuple(int(v) for v in n)
        self.bc = tuple(int(v) for v in bc)
        self.precision = precision
        handle = ctypes.c_void_p()
        _check(load_library().poisson_shard_plan_create(ctypes.byref(handle), self.n[0], self.n[1], self.n[2], (ctypes.c_int * 3)(*self.bc),
                                                        float(h), precision, rank, nranks), "poisson_shard_plan_create")
        self._h = handle.value
        self.info = ShardInfo()
        _check(load_library().poisson_shard_get_info(self._h, ctypes.byref(self.info)), "poisson_shard_get_info")
        dims = (ctypes.c_longlong * 3)()
        _check(load_library().poisson_plan_kernel_dims(self._h, dims), "poisson_plan_kernel_dims")
        self.kernel_dims = tuple(dims)
        self._keep = None

    @property
    def local_shape(self):
        return tuple(self.info.local_dims)

    def set_slabs(self, mid_ptrs, back_ptrs, keep=None):
        """mid_ptrs / back_ptrs: one device pointer per rank (as THIS device addresses that rank's slab)."""
        n = self.info.nranks
        assert len(mid_ptrs) == n and len(back_ptrs) == n
        m = (ctypes.c_void_p * n)(*[int(p) for p in mid_ptrs])
        b = (ctypes.c_void_p * n)(*[int(p) for p in back_ptrs])
        _check(load_library().poisson_shard_set_slabs(self._h, m, b), "poisson_shard_set_slabs")
        self._keep = keep     # whatever owns the memory

    def set_kernel(self, K_f, stream=None):
        assert K_f.is_cuda and K_f.is_contiguous() and tuple(K_f.shape) == self.kernel_dims
        _check(load_library().poisson_shard_set_kernel(self._h, K_f.data_ptr(), PoissonPlan._stream(stream)), "poisson_shard_set_kernel")

    def forward(self, rho_local, stream=None):
        assert rho_local.is_cuda and rho_local.is_contiguous() and tuple(rho_local.shape) == self.local_shape
        _check(load_library().poisson_shard_forward(self._h, rho_local.data_ptr(), PoissonPlan._stream(stream)), "poisson_shard_forward")

    def middle(self, stream=None):
        _check(load_library().poisson_shard_middle(self._h, PoissonPlan._stream(stream)), "poisson_shard_middle")

    def inverse(self, V_local, stream=None):
        assert V_local.is_cuda and V_local.is_contiguous() and tuple(V_local.shape) == self.local_shape
        _check(load_library().poisson_shard_inverse(self._h, V_local.data_ptr(), PoissonPlan._stream(stream)), "poisson_shard_inverse")

    def close(self):
        if self._h:
            poisson_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class ShardedSolver:
    """One solve over the GPUs of a torch.distributed process group (one process per GPU, NCCL): this rank's ShardPlan, its two
    exchange slabs in symmetric memory (every peer's slab mapped into this process over NVLink), and the two barriers as
    one-element all-reduces on the compute stream.  torch supplies memory, peer mapping and the barrier; every step of the
    path runs in the library's kernels, which store straight into the peers' slabs.

    EXPERIMENTAL for world > 1: that branch (symmetric-memory allocation, rendezvous, all-reduce as the barrier) has never
    run on hardware -- no box with two GPUs was available to this build; only world == 1 and the library's own sharded
    passes (virtual ranks on one GPU, tests/test_gpu_shard.py) are verified.  Every process must have made ITS GPU current
    (torch.cuda.set_device(local_rank)) before constructing this object: the plan binds to the current device."""

    def __init__(self, n, bc, h: float, precision: int = FP64, group=None):
        import torch
        import torch.distributed as dist
        self.group = group
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        if self.world > 1:
            import os
            local = os.environ.get("LOCAL_RANK")
            if local is not None and torch.cuda.device_count() > 1 and torch.cuda.current_device() != int(local):
                raise RuntimeError(f"ShardedSolver: current CUDA device {torch.cuda.current_device()} is not LOCAL_RANK {local}: "
                                   "call torch.cuda.set_device(local_rank) first (the plan and its slabs bind to the current device)")
        self.plan = ShardPlan(n, bc, h, precision, self.rank, self.world)
        info = self.plan.info
        if self.world == 1:
            self._mid = torch.empty(info.mid_bytes, dtype=torch.uint8, device="cuda")
            self._back = torch.empty(info.back_bytes, dtype=torch.uint8, device="cuda")
            mids, backs = [self._mid.data_ptr()], [self._back.data_ptr()]
        else:
            import torch.distributed._symmetric_memory as symm
            # symmetric allocations have one size on every rank: the largest slab of any rank
            sizes = torch.tensor([info.mid_bytes, info.back_bytes], dtype=torch.int64, device="cuda")
            dist.all_reduce(sizes, op=dist.ReduceOp.MAX, group=group)
            mid_b, back_b = (int(v) for v in sizes.tolist())
            pg = group or dist.group.WORLD
            self._mid = symm.empty(mid_b, dtype=torch.uint8, device="cuda")
            self._back = symm.empty(back_b, dtype=torch.uint8, device="cuda")
            hm, hb = symm.rendezvous(self._mid, pg), symm.rendezvous(self._back, pg)
            mids, backs = list(hm.buffer_ptrs), list(hb.buffer_ptrs)
        self.plan.set_slabs(mids, backs, keep=(self._mid, self._back))
        self._flag = torch.zeros(1, dtype=torch.int32, device="cuda")

    def _barrier(self):
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(self._flag, group=self.group)     # stream-ordered: enqueued on the current stream

    def set_kernel(self, K_f):
        self.plan.set_kernel(K_f)

    def solve(self, rho_local, V_local=None):
        import torch
        if V_local is None:
            V_local = torch.empty_like(rho_local)
        self.plan.forward(rho_local)
        self._barrier()
        self.plan.middle()
        self._barrier()
        self.plan.inverse(V_local)
        return V_local
