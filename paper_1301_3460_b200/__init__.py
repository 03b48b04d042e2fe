"""paper_1301_3460_b200 -- B200 (sm_100a) Fourier-accelerated Landau gauge fixing (arXiv 1301.3460).

Thin ctypes binding over the C ABI of ``include/lgf.h`` (``paper_1301_3460_b200/liblgf.so``, built from
``csrc/`` by ``python -m paper_1301_3460_b200._build``).  The functions here carry the C names and do argument
marshalling only: every step of the iteration (Delta/theta/F, 4-D FFT, p2max/p2 filter, g build, link update,
stop test) runs in the library's CUDA kernels.  PyTorch is used for device memory and streams only.

There is no CPU fallback.  If the shared library is missing or no CUDA device is present the calls raise.
This package never imports ``oracle`` (the CPU oracle is test infrastructure).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

__all__ = [
    "LgfError", "lib", "library_path", "GaugeFixer", "ShardedGaugeFixer", "measure_static", "LGF_STATIC_MAX_SITES", "copy_peak_gbs", "stream_peak_gbs", "fp64_peak_tflops",
    "LGF_OK", "LGF_NOT_CONVERGED", "LGF_FP64", "LGF_FP32", "LGF_MIXED", "LGF_STORE_12", "LGF_STORE_18",
    "LGF_FIELD_DELTA", "LGF_FIELD_X", "LGF_FIELD_G",
    "LGF_OPT_STORE_G", "LGF_OPT_GRAPH", "LGF_OPT_BATCH", "LGF_OPT_PDL", "LGF_OPT_FAST_FFT", "LGF_OPT_FOURIER_ACCEL",
    "LGF_OPT_GAUGE_DIRECTIONS", "LGF_OPT_MIXED_FP32_ITERS", "LGF_OPT_MIXED_SWITCH", "LGF_OPT_TMA",
    "EXPORTS",
]

LGF_OK = 0
LGF_ERR_INVALID_ARG = 1
LGF_ERR_UNSUPPORTED = 2
LGF_ERR_OOM = 3
LGF_ERR_CUDA = 4
LGF_ERR_NOT_LOADED = 5
LGF_ERR_NUMERIC = 6
LGF_NOT_CONVERGED = 100
LGF_FP64, LGF_FP32, LGF_MIXED = 0, 1, 2
LGF_STORE_18, LGF_STORE_12 = 18, 12
LGF_FIELD_DELTA, LGF_FIELD_X, LGF_FIELD_G = 0, 1, 2
LGF_OPT_STORE_G, LGF_OPT_GRAPH, LGF_OPT_BATCH, LGF_OPT_PDL, LGF_OPT_FAST_FFT = 0, 1, 2, 3, 4
LGF_OPT_FOURIER_ACCEL, LGF_OPT_GAUGE_DIRECTIONS, LGF_OPT_MIXED_FP32_ITERS, LGF_OPT_MIXED_SWITCH, LGF_OPT_TMA = 5, 6, 7, 8, 9
LGF_MAX_KERNELS = 32
LGF_STATIC_MAX_SITES = 1 << 24

# every symbol include/lgf.h declares (checked by tests/test_abi.py against the header text)
EXPORTS = [
    "lgf_workspace_bytes", "lgf_create", "lgf_create_ex", "lgf_destroy", "lgf_load_links", "lgf_load_links_device",
    "lgf_get_links", "lgf_get_links_device", "lgf_load_links_12", "lgf_get_links_12", "lgf_iterate", "lgf_fix", "lgf_scan_alpha", "lgf_measure", "lgf_get_history",
    "lgf_get_field", "lgf_set_option", "lgf_get_option", "lgf_set_profiling", "lgf_get_profile", "lgf_kernel_name",
    "lgf_launch_count", "lgf_copy_peak", "lgf_stream_peak", "lgf_fp64_peak", "lgf_status_string", "lgf_last_error",
    "lgf_create_sharded", "lgf_destroy_sharded", "lgf_sharded_ranks", "lgf_load_links_sharded", "lgf_get_links_sharded",
    "lgf_iterate_sharded", "lgf_fix_sharded", "lgf_get_history_sharded", "lgf_sharded_traffic", "lgf_last_error_sharded",
    "lgf_measure_static", "lgf_measure_static_error",
]

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


class LgfError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = status
        msg = f"{where}: lgf_status {status}"
        try:
            msg += " (" + lib().lgf_status_string(status).decode() + ")"
        except Exception:
            pass
        if detail:
            msg += ": " + detail
        super().__init__(msg)


def library_path() -> str:
    """The in-tree library; LGF_LIBRARY points at another build of the same sources (kernel A/B timing)."""
    return os.environ.get("LGF_LIBRARY") or os.path.join(_HERE, "liblgf.so")


def lib():
    """Load liblgf.so (building it first if the sources are newer and nvcc is present).  Raises if it cannot
    be had: the product path has no fallback."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.environ.get("LGF_LIBRARY"):
        from . import _build
        if _build.have_nvcc():
            _build.build()                    # no-op when the .so is newer than every source
        elif os.path.exists(path) and not _build.up_to_date():
            import warnings
            warnings.warn("paper_1301_3460_b200/liblgf.so is older than its sources and nvcc is not available")
    if not os.path.exists(path):
        raise ImportError("paper_1301_3460_b200/liblgf.so is missing; run python -m paper_1301_3460_b200._build")
    L = C.CDLL(path)
    P, D, I = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
    I4 = C.POINTER(C.c_int)
    L.lgf_workspace_bytes.restype = C.c_size_t
    L.lgf_workspace_bytes.argtypes = [I4, C.c_int, C.c_int]
    L.lgf_create.argtypes = [I4, C.c_int, C.c_int, C.POINTER(P)]
    L.lgf_create_ex.argtypes = [I4, C.c_int, C.c_int, P, C.c_size_t, P, C.POINTER(P)]
    L.lgf_destroy.restype = None
    L.lgf_destroy.argtypes = [P]
    L.lgf_load_links.argtypes = [P, P]
    L.lgf_load_links_device.argtypes = [P, P]
    L.lgf_get_links.argtypes = [P, P]
    L.lgf_get_links_device.argtypes = [P, P]
    L.lgf_load_links_12.argtypes = [P, P]
    L.lgf_get_links_12.argtypes = [P, P]
    L.lgf_iterate.argtypes = [P, C.c_int, C.c_double, D, D]
    L.lgf_fix.argtypes = [P, C.c_double, C.c_double, C.c_int, I, D, D]
    L.lgf_measure.argtypes = [P, D, D, D]
    L.lgf_scan_alpha.argtypes = [P, D, C.c_int, C.c_double, C.c_int, I, D, I]
    L.lgf_get_history.argtypes = [P, P, C.c_int, I]
    L.lgf_get_field.argtypes = [P, C.c_int, C.c_double, P]
    L.lgf_set_option.argtypes = [P, C.c_int, C.c_int]
    L.lgf_get_option.argtypes = [P, C.c_int, I]
    L.lgf_set_profiling.argtypes = [P, C.c_int]
    L.lgf_get_profile.argtypes = [P, D, C.POINTER(C.c_longlong)]
    L.lgf_kernel_name.restype = C.c_char_p
    L.lgf_kernel_name.argtypes = [C.c_int]
    L.lgf_launch_count.restype = C.c_longlong
    L.lgf_launch_count.argtypes = [P]
    L.lgf_copy_peak.argtypes = [P, P, C.c_size_t, C.c_int, P, D]
    L.lgf_stream_peak.argtypes = [P, C.c_size_t, C.c_int, C.c_int, P, D]
    L.lgf_fp64_peak.argtypes = [C.c_int, P, D]
    L.lgf_status_string.restype = C.c_char_p
    L.lgf_status_string.argtypes = [C.c_int]
    L.lgf_last_error.restype = C.c_char_p
    L.lgf_last_error.argtypes = [P]
    L.lgf_create_sharded.argtypes = [I4, C.c_int, C.c_int, C.POINTER(P)]
    L.lgf_destroy_sharded.restype = None
    L.lgf_destroy_sharded.argtypes = [P]
    L.lgf_sharded_ranks.argtypes = [P]
    L.lgf_load_links_sharded.argtypes = [P, P]
    L.lgf_get_links_sharded.argtypes = [P, P]
    L.lgf_iterate_sharded.argtypes = [P, C.c_int, C.c_double, D, D]
    L.lgf_fix_sharded.argtypes = [P, C.c_double, C.c_double, C.c_int, I, D, D]
    L.lgf_get_history_sharded.argtypes = [P, P, C.c_int, I]
    L.lgf_sharded_traffic.argtypes = [P, C.POINTER(C.c_longlong)]
    L.lgf_last_error_sharded.restype = C.c_char_p
    L.lgf_last_error_sharded.argtypes = [P]
    L.lgf_measure_static.argtypes = [P, I4, P, P]
    L.lgf_measure_static_error.restype = C.c_char_p
    L.lgf_measure_static_error.argtypes = []
    _lib = L
    return L


def _dims(dims):
    d = [int(v) for v in dims]
    if len(d) != 4:
        raise ValueError("dims must have 4 entries")
    return (C.c_int * 4)(*d)


def _host_f64(a, n_doubles: int) -> np.ndarray:
    """View a host array (complex128 or float64, C-contiguous) as float64 without changing its bytes."""
    a = np.asarray(a)
    if a.dtype == np.complex128:
        a = np.ascontiguousarray(a).view(np.float64)
    elif a.dtype != np.float64:
        raise TypeError("links must be float64 [V,4,3,3,2] or complex128 [V,4,3,3]")
    a = np.ascontiguousarray(a)
    if a.size != n_doubles:
        raise ValueError(f"expected {n_doubles} doubles, got {a.size}")
    return a


class GaugeFixer:
    """One lattice on one GPU.  Methods are the lgf_* calls of include/lgf.h with the ``lgf_`` prefix dropped.

    ``use_torch_workspace=True`` (default) allocates the device workspace with ``torch.empty`` on the current
    CUDA device and orders all work on a ``torch.cuda.Stream`` owned by this object (``self.stream``;
    lgf_create_ex); ``False`` lets the library cudaMalloc and create its own stream (lgf_create).  Every call
    is synchronous for the host on return.
    """

    def __init__(self, dims, storage: int = LGF_STORE_12, precision: int = LGF_FP64, use_torch_workspace: bool = True):
        L = lib()
        self.dims = tuple(int(v) for v in dims)
        self.V = int(np.prod(self.dims))
        self.storage = int(storage)
        self._h = C.c_void_p()
        self._ws = None
        if use_torch_workspace:
            import torch
            if not torch.cuda.is_available():
                raise LgfError(LGF_ERR_CUDA, "lgf_create_ex", "no CUDA device (there is no CPU fallback)")
            nbytes = L.lgf_workspace_bytes(_dims(self.dims), precision, self.storage)
            if nbytes == 0:
                raise LgfError(LGF_ERR_UNSUPPORTED, "lgf_workspace_bytes", f"dims={self.dims}")
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            base = (self._ws.data_ptr() + 255) // 256 * 256
            # a stream of the context's own: the legacy default stream cannot be captured into a CUDA graph
            self._stream = torch.cuda.Stream()
            self._stream.wait_stream(torch.cuda.current_stream())
            st = L.lgf_create_ex(_dims(self.dims), precision, self.storage, C.c_void_p(base), nbytes,
                                 C.c_void_p(self._stream.cuda_stream), C.byref(self._h))
            where = "lgf_create_ex"
        else:
            st = L.lgf_create(_dims(self.dims), precision, self.storage, C.byref(self._h))
            where = "lgf_create"
        if st != LGF_OK:
            self._h = C.c_void_p()
            raise LgfError(st, where, f"dims={self.dims} " + L.lgf_last_error(None).decode())

    # ---- lifetime
    def destroy(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().lgf_destroy(self._h)
            self._h = C.c_void_p()
        self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _ck(self, st: int, where: str, ok=(LGF_OK,)):
        if st not in ok:
            raise LgfError(st, where, lib().lgf_last_error(self._h).decode())
        return st

    # ---- links
    def load_links(self, host_links):
        a = _host_f64(host_links, self.V * 72)
        self._ck(lib().lgf_load_links(self._h, a.ctypes.data), "lgf_load_links")

    @property
    def stream(self):
        """The torch.cuda.Stream the context runs on (None when the library owns its stream)."""
        return getattr(self, "_stream", None)

    def _after_current_stream(self):
        if self.stream is not None:
            import torch
            self._stream.wait_stream(torch.cuda.current_stream())

    def load_links_device(self, dev_ptr: int):
        self._after_current_stream()      # the producer of dev_ptr may still be running on torch's current stream
        self._ck(lib().lgf_load_links_device(self._h, C.c_void_p(int(dev_ptr))), "lgf_load_links_device")

    def get_links(self, out=None) -> np.ndarray:
        """Returns complex128 [V,4,3,3] (canonical order)."""
        if out is None:
            out = np.empty((self.V, 4, 3, 3), dtype=np.complex128)
        elif not (isinstance(out, np.ndarray) and out.flags.c_contiguous and out.flags.writeable
                  and out.dtype in (np.complex128, np.float64)):
            raise TypeError("out must be a writeable C-contiguous complex128 [V,4,3,3] or float64 [V,4,3,3,2] array")
        a = _host_f64(out, self.V * 72)
        self._ck(lib().lgf_get_links(self._h, a.ctypes.data), "lgf_get_links")
        return out

    def load_links_12(self, host_rows):
        """Two-row host format: complex128 [V,4,2,3] (rows 0,1 of every link); LGF_STORE_12 contexts only."""
        a = _host_f64(host_rows, self.V * 48)
        self._ck(lib().lgf_load_links_12(self._h, a.ctypes.data), "lgf_load_links_12")

    def get_links_12(self, out=None) -> np.ndarray:
        """Returns complex128 [V,4,2,3]: rows 0,1 of every link (two-row host format)."""
        if out is None:
            out = np.empty((self.V, 4, 2, 3), dtype=np.complex128)
        elif not (isinstance(out, np.ndarray) and out.flags.c_contiguous and out.flags.writeable
                  and out.dtype in (np.complex128, np.float64)):
            raise TypeError("out must be a writeable C-contiguous complex128 [V,4,2,3] or float64 [V,4,2,3,2] array")
        a = _host_f64(out, self.V * 48)
        self._ck(lib().lgf_get_links_12(self._h, a.ctypes.data), "lgf_get_links_12")
        return out

    def get_links_device(self, dev_ptr: int):
        self._after_current_stream()
        self._ck(lib().lgf_get_links_device(self._h, C.c_void_p(int(dev_ptr))), "lgf_get_links_device")

    # ---- the iteration
    def iterate(self, n: int, alpha: float):
        F, th = C.c_double(), C.c_double()
        self._ck(lib().lgf_iterate(self._h, int(n), float(alpha), C.byref(F), C.byref(th)), "lgf_iterate")
        return F.value, th.value

    def fix(self, alpha: float, theta_tol: float, max_iter: int) -> dict:
        F, th, n = C.c_double(), C.c_double(), C.c_int()
        st = self._ck(lib().lgf_fix(self._h, float(alpha), float(theta_tol), int(max_iter), C.byref(n), C.byref(F), C.byref(th)),
                      "lgf_fix", ok=(LGF_OK, LGF_NOT_CONVERGED))
        return dict(status=st, n_iter=n.value, F=F.value, theta=th.value)

    def scan_alpha(self, alphas, theta_tol: float, max_iter: int) -> dict:
        """One lgf_fix per alpha from the links now loaded (which the call leaves unchanged): iteration counts
        (-1: not converged within max_iter, -2: diverged), F at the stop, index of the best alpha (-1: none)."""
        a = np.ascontiguousarray(alphas, dtype=np.float64)
        n = len(a)
        counts = (C.c_int * n)()
        F = (C.c_double * n)()
        best = C.c_int(-1)
        self._ck(lib().lgf_scan_alpha(self._h, a.ctypes.data_as(C.POINTER(C.c_double)), n, float(theta_tol), int(max_iter), counts, F, C.byref(best)),
                 "lgf_scan_alpha")
        return dict(alphas=[float(v) for v in a], counts=[int(v) for v in counts], F=[float(v) for v in F], best=int(best.value))

    def measure(self):
        F, th, p = C.c_double(), C.c_double(), C.c_double()
        self._ck(lib().lgf_measure(self._h, C.byref(F), C.byref(th), C.byref(p)), "lgf_measure")
        return F.value, th.value, p.value

    def get_history(self, capacity: int = 65536) -> np.ndarray:
        h = np.zeros((capacity, 2), dtype=np.float64)
        n = C.c_int()
        self._ck(lib().lgf_get_history(self._h, h.ctypes.data, capacity, C.byref(n)), "lgf_get_history")
        return h[: n.value].copy()

    def get_field(self, which: int, alpha: float = 0.0) -> np.ndarray:
        """Delta, X or g of the current links as complex128 [V,3,3] (kernel-level parity read-out)."""
        out = np.empty((self.V, 3, 3), dtype=np.complex128)
        self._ck(lib().lgf_get_field(self._h, int(which), float(alpha), out.ctypes.data), "lgf_get_field")
        return out

    # ---- options / instrumentation
    def set_option(self, opt: int, value: int):
        self._ck(lib().lgf_set_option(self._h, int(opt), int(value)), "lgf_set_option")

    def get_option(self, opt: int) -> int:
        v = C.c_int()
        self._ck(lib().lgf_get_option(self._h, int(opt), C.byref(v)), "lgf_get_option")
        return v.value

    def set_profiling(self, on: bool):
        self._ck(lib().lgf_set_profiling(self._h, 1 if on else 0), "lgf_set_profiling")

    def get_profile(self) -> dict:
        ms = (C.c_double * LGF_MAX_KERNELS)()
        n = (C.c_longlong * LGF_MAX_KERNELS)()
        self._ck(lib().lgf_get_profile(self._h, ms, n), "lgf_get_profile")
        out = {}
        for i in range(LGF_MAX_KERNELS):
            if n[i]:
                out[lib().lgf_kernel_name(i).decode()] = dict(ms=ms[i], launches=int(n[i]))
        return out

    def launch_count(self) -> int:
        return int(lib().lgf_launch_count(self._h))


class ShardedGaugeFixer:
    """Slab-decomposed context (include/lgf.h lgf_*_sharded): n_ranks virtual ranks on the current device, each with its
    own workspace; argument marshalling only."""

    def __init__(self, dims, n_ranks: int, storage: int = LGF_STORE_12):
        self.dims = _dims(dims)
        self.V = int(np.prod(self.dims))
        self.n_ranks = int(n_ranks)
        h = C.c_void_p()
        st = lib().lgf_create_sharded((C.c_int * 4)(*self.dims), self.n_ranks, int(storage), C.byref(h))
        if st != LGF_OK:
            raise LgfError(st, "lgf_create_sharded", f"dims={tuple(self.dims)} n_ranks={self.n_ranks} " + lib().lgf_last_error_sharded(None).decode())
        self._h = h

    def destroy(self):
        if getattr(self, "_h", None):
            lib().lgf_destroy_sharded(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _ck(self, st: int, where: str, ok=(LGF_OK,)):
        if st not in ok:
            raise LgfError(st, where, lib().lgf_last_error_sharded(self._h).decode())
        return st

    def load_links(self, host_links):
        a = _host_f64(host_links, self.V * 72)
        self._ck(lib().lgf_load_links_sharded(self._h, a.ctypes.data), "lgf_load_links_sharded")

    def get_links(self) -> np.ndarray:
        out = np.empty((self.V, 4, 3, 3), dtype=np.complex128)
        self._ck(lib().lgf_get_links_sharded(self._h, out.ctypes.data), "lgf_get_links_sharded")
        return out

    def iterate(self, n: int, alpha: float):
        F, th = C.c_double(), C.c_double()
        self._ck(lib().lgf_iterate_sharded(self._h, int(n), float(alpha), C.byref(F), C.byref(th)), "lgf_iterate_sharded")
        return F.value, th.value

    def fix(self, alpha: float, theta_tol: float, max_iter: int) -> dict:
        F, th, n = C.c_double(), C.c_double(), C.c_int()
        st = self._ck(lib().lgf_fix_sharded(self._h, float(alpha), float(theta_tol), int(max_iter), C.byref(n), C.byref(F), C.byref(th)),
                      "lgf_fix_sharded", ok=(LGF_OK, LGF_NOT_CONVERGED))
        return dict(status=st, n_iter=n.value, F=F.value, theta=th.value)

    def get_history(self, capacity: int = 65536) -> np.ndarray:
        h = np.zeros((capacity, 2))
        n = C.c_int()
        self._ck(lib().lgf_get_history_sharded(self._h, h.ctypes.data, capacity, C.byref(n)), "lgf_get_history_sharded")
        return h[: n.value].copy()

    def traffic(self) -> dict:
        o = (C.c_longlong * 5)()
        self._ck(lib().lgf_sharded_traffic(self._h, o), "lgf_sharded_traffic")
        return dict(halo_u_bytes=int(o[0]), halo_x_bytes=int(o[1]), transpose_bytes=int(o[2]), launches=int(o[3]), copies=int(o[4]))


def measure_static(dev_links_ptr: int, dims, dev_out_ptr: int, cuda_stream: int = 0) -> None:
    """lgf_measure_static: F and theta of the links at ``dev_links_ptr`` (DEVICE, canonical [V,4,3,3] complex128) into the
    two doubles at ``dev_out_ptr`` (DEVICE: F, theta), for callers that cannot let the library allocate -- their own pool
    or a framework's caching allocator holds the HBM, or they run inside a loop that a device-wide cudaMalloc/cudaFree
    synchronisation would stall.  No context and no allocation: the scratch memory is a fixed 2 MiB array inside the library, so at most
    ``LGF_STATIC_MAX_SITES`` sites.  The call only enqueues work on ``cuda_stream`` (a raw cudaStream_t as int, 0 = default
    stream) and does not wait; calls that overlap on the GPU share the scratch array and race, so keep them on one
    stream.  Make the first call on a device before any stream capture.  Marshalling only."""
    L = lib()
    st = L.lgf_measure_static(C.c_void_p(int(dev_links_ptr)), _dims(dims), C.c_void_p(int(cuda_stream)), C.c_void_p(int(dev_out_ptr)))
    if st != LGF_OK:
        raise LgfError(st, "lgf_measure_static", L.lgf_measure_static_error().decode())


def copy_peak_gbs(nbytes: int = 1 << 30, reps: int = 10) -> float:
    """GB/s (read + write bytes) of the library's own double2 streaming copy kernel: the measured copy peak."""
    import torch
    a = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    b = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    a.zero_()
    ms = C.c_double()
    s = torch.cuda.current_stream()
    st = lib().lgf_copy_peak(C.c_void_p(b.data_ptr()), C.c_void_p(a.data_ptr()), nbytes, reps, C.c_void_p(s.cuda_stream), C.byref(ms))
    if st != LGF_OK:
        raise LgfError(st, "lgf_copy_peak")
    return 2.0 * nbytes / ms.value / 1e6


def fp64_peak_tflops(reps: int = 5) -> float:
    """FP64 FMA rate of the device in TFLOP/s (lgf_fp64_peak)."""
    import torch
    v = C.c_double()
    st = lib().lgf_fp64_peak(int(reps), C.c_void_p(torch.cuda.current_stream().cuda_stream), C.byref(v))
    if st != LGF_OK:
        raise LgfError(st, "lgf_fp64_peak")
    return v.value


def stream_peak_gbs(n_sites: int = 1 << 20, write: bool = False, reps: int = 10) -> float:
    """GB/s of the 24-stream yardstick (lgf_stream_peak): the link kernels' access pattern without their arithmetic."""
    import torch
    a = torch.zeros(n_sites * 24 * 2, dtype=torch.float64, device="cuda")
    ms = C.c_double()
    s = torch.cuda.current_stream()
    st = lib().lgf_stream_peak(C.c_void_p(a.data_ptr()), n_sites, 1 if write else 0, reps, C.c_void_p(s.cuda_stream), C.byref(ms))
    if st != LGF_OK:
        raise LgfError(st, "lgf_stream_peak")
    return 384.0 * n_sites * (2 if write else 1) / ms.value / 1e6
