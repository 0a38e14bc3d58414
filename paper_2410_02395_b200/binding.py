"""Thin ctypes binding over libmbs_b200.so (include/mbs.h): argument marshalling only.

The functions carry the C names (mbs_create, mbs_set_potential, mbs_apply_operator, mbs_solve,
mbs_solve_host, mbs_get_info, mbs_destroy, mbs_last_error).  `Solver` is a convenience wrapper
that lets PyTorch own the device memory (workspace, fields) and the stream.  Every step of the
path runs in the library's CUDA kernels; if the library is missing this module raises at import:
there is no fallback.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmbs_b200.so")      # the in-tree build; no environment override

if not os.path.exists(LIB_PATH):
    raise ImportError(
        "libmbs_b200.so is not built (%s). Run `python -m paper_2410_02395_b200.build` "
        "(or __graft_entry__.build()); there is no CPU fallback." % LIB_PATH)

_lib = ctypes.CDLL(LIB_PATH)

MBS_OK, MBS_ERR_INVALID_ARG, MBS_ERR_UNSUPPORTED_SIZE, MBS_ERR_OOM = 0, 1, 2, 3
MBS_ERR_CUDA, MBS_ERR_NOT_CONVERGED, MBS_ERR_NUMERIC, MBS_ERR_STATE = 4, 5, 6, 7
MBS_OP_B, MBS_OP_PROPAGATOR, MBS_OP_A, MBS_OP_PRECOND_A = 0, 1, 2, 3
MBS_OPT_FUSED, MBS_OPT_CHECK_INTERVAL, MBS_OPT_USE_GRAPH, MBS_OPT_PROFILE, MBS_OPT_TMA, MBS_OPT_LINE = 0, 1, 2, 3, 4, 5
MBS_OPT_REFINE = 7

STATUS_NAMES = {0: "MBS_OK", 1: "MBS_ERR_INVALID_ARG", 2: "MBS_ERR_UNSUPPORTED_SIZE", 3: "MBS_ERR_OOM",
                4: "MBS_ERR_CUDA", 5: "MBS_ERR_NOT_CONVERGED", 6: "MBS_ERR_NUMERIC", 7: "MBS_ERR_STATE"}

# every symbol include/mbs.h declares (tests/test_abi.py checks the library exports them all)
DECLARED_SYMBOLS = ("mbs_create", "mbs_fft_supported", "mbs_workspace_bytes", "mbs_set_workspace", "mbs_set_option",
                    "mbs_set_potential", "mbs_apply_operator", "mbs_solve", "mbs_solve_host", "mbs_iterate",
                    "mbs_get_info", "mbs_get_kernel_stats", "mbs_reset_kernel_stats", "mbs_destroy", "mbs_last_error",
                    "mbs_set_activation", "mbs_get_activation", "mbs_apply_B_static", "mbs_solve_batch")
MBS_STATIC_SCRATCH_BYTES = 16 << 20


class mbs_info(ctypes.Structure):
    _fields_ = [("c_re", ctypes.c_double), ("c_im", ctypes.c_double),
                ("k02_re", ctypes.c_double), ("k02_im", ctypes.c_double),
                ("v_max", ctypes.c_double), ("norm_A12", ctypes.c_double),
                ("sum_a", ctypes.c_int32), ("ndim", ctypes.c_int32),
                ("voxels", ctypes.c_int64), ("subdomain_shape", ctypes.c_int64 * 3),
                ("alpha", ctypes.c_double), ("norm_rhs", ctypes.c_double),
                ("algorithmic_bytes_per_iteration", ctypes.c_double),
                ("workspace_bytes", ctypes.c_uint64), ("kernel_launches", ctypes.c_int64),
                ("last_solve_ms", ctypes.c_double), ("sparse_source_bytes_per_iteration", ctypes.c_double)]


class mbs_kernel_stat(ctypes.Structure):
    _fields_ = [("name", ctypes.c_char * 48), ("launches", ctypes.c_int64), ("total_ms", ctypes.c_double),
                ("algorithmic_bytes", ctypes.c_double)]


_vp = ctypes.c_void_p
_lib.mbs_create.argtypes = [ctypes.POINTER(_vp), ctypes.c_int, ctypes.POINTER(ctypes.c_int64), ctypes.c_double,
                            ctypes.c_double, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                            ctypes.POINTER(ctypes.c_uint8), ctypes.c_int32, _vp]
_lib.mbs_create.restype = ctypes.c_int
_lib.mbs_fft_supported.argtypes = [ctypes.c_int64]
_lib.mbs_fft_supported.restype = ctypes.c_int
_lib.mbs_workspace_bytes.argtypes = [_vp]
_lib.mbs_workspace_bytes.restype = ctypes.c_size_t
_lib.mbs_set_workspace.argtypes = [_vp, _vp, ctypes.c_size_t]
_lib.mbs_set_workspace.restype = ctypes.c_int
_lib.mbs_set_option.argtypes = [_vp, ctypes.c_int, ctypes.c_int64]
_lib.mbs_set_option.restype = ctypes.c_int
_lib.mbs_set_potential.argtypes = [_vp, _vp]
_lib.mbs_set_potential.restype = ctypes.c_int
_lib.mbs_apply_operator.argtypes = [_vp, ctypes.c_int, _vp, _vp]
_lib.mbs_apply_operator.restype = ctypes.c_int
_lib.mbs_apply_B_static.argtypes = [_vp, _vp, _vp]
_lib.mbs_apply_B_static.restype = ctypes.c_int
_lib.mbs_solve.argtypes = [_vp, _vp, _vp, ctypes.c_double, ctypes.c_int32, ctypes.POINTER(ctypes.c_double),
                           ctypes.POINTER(ctypes.c_int32)]
_lib.mbs_solve.restype = ctypes.c_int
_lib.mbs_solve_batch.argtypes = [_vp, ctypes.c_int32] + list(_lib.mbs_solve.argtypes[1:])
_lib.mbs_solve_batch.restype = ctypes.c_int
_lib.mbs_solve_host.argtypes = _lib.mbs_solve.argtypes
_lib.mbs_solve_host.restype = ctypes.c_int
_lib.mbs_iterate.argtypes = [_vp, _vp, _vp, ctypes.c_int32, ctypes.c_double, ctypes.POINTER(ctypes.c_double)]
_lib.mbs_iterate.restype = ctypes.c_int
_lib.mbs_get_kernel_stats.argtypes = [_vp, ctypes.POINTER(mbs_kernel_stat), ctypes.c_int32, ctypes.POINTER(ctypes.c_int32)]
_lib.mbs_get_kernel_stats.restype = ctypes.c_int
_lib.mbs_reset_kernel_stats.argtypes = [_vp]
_lib.mbs_reset_kernel_stats.restype = ctypes.c_int
_lib.mbs_set_activation.argtypes = [_vp, ctypes.c_int, ctypes.c_double]
_lib.mbs_set_activation.restype = ctypes.c_int
_lib.mbs_get_activation.argtypes = [_vp, ctypes.POINTER(ctypes.c_int32), ctypes.c_int32, ctypes.POINTER(ctypes.c_int32)]
_lib.mbs_get_activation.restype = ctypes.c_int
_lib.mbs_get_info.argtypes = [_vp, ctypes.POINTER(mbs_info)]
_lib.mbs_get_info.restype = ctypes.c_int
_lib.mbs_destroy.argtypes = [_vp]
_lib.mbs_destroy.restype = None
_lib.mbs_last_error.argtypes = [_vp]
_lib.mbs_last_error.restype = ctypes.c_char_p


class MBSError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__("%s: %s" % (STATUS_NAMES.get(status, str(status)), message))
        self.status = status


# --------------------------------------------------------------------------------------------
# C-named functions (pointers are plain integers / ctypes values)
# --------------------------------------------------------------------------------------------
def mbs_last_error(ctx) -> str:
    s = _lib.mbs_last_error(ctx)
    return s.decode() if s else ""


def mbs_create(shape: Sequence[int], pixel_size: float, wavelength: float, boundary_width: Sequence[int],
               n_subdomains: Sequence[int], periodic: Optional[Sequence[int]], n_correction: int, cuda_stream: int = 0):
    nd = len(shape)
    ctx = _vp()
    sh = (ctypes.c_int64 * max(nd, 1))(*[int(s) for s in shape])
    bw = (ctypes.c_int32 * max(nd, 1))(*[int(s) for s in boundary_width])
    ns = (ctypes.c_int32 * max(nd, 1))(*[int(s) for s in n_subdomains])
    per = None
    if periodic is not None:
        per = (ctypes.c_uint8 * max(nd, 1))(*[int(bool(p)) for p in periodic])
    rc = _lib.mbs_create(ctypes.byref(ctx), nd, sh, float(pixel_size), float(wavelength), bw, ns, per,
                         int(n_correction), _vp(cuda_stream))
    if rc != MBS_OK:
        raise MBSError(rc, mbs_last_error(None))
    return ctx


def mbs_fft_supported(M: int) -> bool:
    return bool(_lib.mbs_fft_supported(int(M)))


def mbs_workspace_bytes(ctx) -> int:
    return int(_lib.mbs_workspace_bytes(ctx))


def _check(ctx, rc, allow=()):
    if rc != MBS_OK and rc not in allow:
        raise MBSError(rc, mbs_last_error(ctx))
    return rc


def mbs_set_workspace(ctx, device_ptr: int, nbytes: int):
    _check(ctx, _lib.mbs_set_workspace(ctx, _vp(device_ptr), nbytes))


def mbs_set_option(ctx, option: int, value: int):
    _check(ctx, _lib.mbs_set_option(ctx, option, int(value)))


def mbs_set_potential(ctx, n_map_device_ptr: int):
    _check(ctx, _lib.mbs_set_potential(ctx, _vp(n_map_device_ptr)))


def mbs_apply_operator(ctx, which: int, in_ptr: int, out_ptr: int):
    _check(ctx, _lib.mbs_apply_operator(ctx, which, _vp(in_ptr), _vp(out_ptr)))


def mbs_apply_B_static(ctx, in_ptr: int, out_ptr: int):
    """out = B in with the slab scratch in the library's static device array: no allocation (include/mbs.h)."""
    _check(ctx, _lib.mbs_apply_B_static(ctx, _vp(in_ptr), _vp(out_ptr)))


def _solve(fn, ctx, y_ptr, x_ptr, tol, max_iter, want_history):
    hist = np.empty(max_iter if want_history else 0, dtype=np.float64)
    n_iter = ctypes.c_int32(0)
    hp = hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if want_history else None
    rc = fn(ctx, _vp(y_ptr), _vp(x_ptr), float(tol), int(max_iter), hp, ctypes.byref(n_iter))
    _check(ctx, rc, allow=(MBS_ERR_NOT_CONVERGED,))
    return rc, hist[:n_iter.value], n_iter.value


def mbs_solve(ctx, y_ptr: int, x_ptr: int, tol: float, max_iter: int, want_history: bool = True):
    """Device pointers.  Returns (status, residual_history, n_iter); status is MBS_OK or MBS_ERR_NOT_CONVERGED."""
    return _solve(_lib.mbs_solve, ctx, y_ptr, x_ptr, tol, max_iter, want_history)


def mbs_solve_batch(ctx, n_batch: int, y_ptr: int, x_ptr: int, tol: float, max_iter: int, want_history: bool = True):
    """n_batch sources, one medium (device pointers to [n_batch][shape] arrays).  Returns (status, history, n_iter)."""
    hist = np.empty(max_iter if want_history else 0, dtype=np.float64)
    n_iter = ctypes.c_int32(0)
    hp = hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if want_history else None
    rc = _lib.mbs_solve_batch(ctx, int(n_batch), _vp(y_ptr), _vp(x_ptr), float(tol), int(max_iter), hp, ctypes.byref(n_iter))
    _check(ctx, rc, allow=(MBS_ERR_NOT_CONVERGED,))
    return rc, hist[:n_iter.value], n_iter.value


def mbs_solve_host(ctx, y_ptr: int, x_ptr: int, tol: float, max_iter: int, want_history: bool = True):
    """Host pointers (e.g. pinned torch tensors or numpy arrays)."""
    return _solve(_lib.mbs_solve_host, ctx, y_ptr, x_ptr, tol, max_iter, want_history)


def mbs_iterate(ctx, y_ptr: int, x_ptr: int, n_iter: int, nu: float = 0.0, want_history: bool = True):
    """Exactly n_iter updates, no stop test (device pointers).  Returns the residual history."""
    hist = np.empty(n_iter if want_history else 0, dtype=np.float64)
    hp = hist.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if want_history else None
    _check(ctx, _lib.mbs_iterate(ctx, _vp(y_ptr), _vp(x_ptr), int(n_iter), float(nu), hp))
    return hist


def mbs_get_kernel_stats(ctx) -> list:
    cap = 64
    arr = (mbs_kernel_stat * cap)()
    n = ctypes.c_int32(0)
    _check(ctx, _lib.mbs_get_kernel_stats(ctx, arr, cap, ctypes.byref(n)))
    return [dict(name=arr[i].name.decode(), launches=int(arr[i].launches), total_ms=float(arr[i].total_ms),
                 algorithmic_bytes=float(arr[i].algorithmic_bytes)) for i in range(min(n.value, cap))]


def mbs_reset_kernel_stats(ctx):
    _check(ctx, _lib.mbs_reset_kernel_stats(ctx))


def mbs_set_activation(ctx, enable: bool, threshold: float = -1.0):
    _check(ctx, _lib.mbs_set_activation(ctx, int(bool(enable)), float(threshold)))


def mbs_get_activation(ctx) -> list:
    """Iteration at which each subdomain was activated in the last solve (subdomains in np.ndindex(S) order)."""
    n = ctypes.c_int32(0)
    _check(ctx, _lib.mbs_get_activation(ctx, None, 0, ctypes.byref(n)))
    arr = (ctypes.c_int32 * max(n.value, 1))()
    _check(ctx, _lib.mbs_get_activation(ctx, arr, n.value, ctypes.byref(n)))
    return [int(arr[i]) for i in range(n.value)]


def mbs_get_info(ctx) -> dict:
    info = mbs_info()
    _check(ctx, _lib.mbs_get_info(ctx, ctypes.byref(info)))
    out = {name: getattr(info, name) for name, _ in mbs_info._fields_ if name != "subdomain_shape"}
    out["subdomain_shape"] = tuple(info.subdomain_shape[d] for d in range(info.ndim))
    out["c"] = complex(info.c_re, info.c_im)
    out["k02"] = complex(info.k02_re, info.k02_im)
    return out


def mbs_destroy(ctx):
    _lib.mbs_destroy(ctx)


# --------------------------------------------------------------------------------------------
# convenience wrapper: PyTorch owns device memory and the stream
# --------------------------------------------------------------------------------------------
class Solver:
    def __init__(self, shape, pixel_size, wavelength, boundary_width, n_subdomains, periodic=None,
                 n_correction: int = 8, device="cuda:0", stream=None):
        import torch
        self._torch = torch
        self.device = torch.device(device)
        self.shape = tuple(int(s) for s in shape)
        if self.device.type != "cuda" or not torch.cuda.is_available():
            raise RuntimeError("paper_2410_02395_b200 needs a CUDA device; there is no CPU fallback")
        torch.cuda.set_device(self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.ctx = mbs_create(self.shape, pixel_size, wavelength, boundary_width, n_subdomains, periodic,
                              n_correction, self.stream.cuda_stream)
        nbytes = mbs_workspace_bytes(self.ctx)
        with torch.cuda.stream(self.stream):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ptr = (self.workspace.data_ptr() + 255) // 256 * 256
        mbs_set_workspace(self.ctx, ptr, nbytes)

    @classmethod
    def from_workload(cls, w, device="cuda:0", stream=None):
        return cls(w.shape, w.pixel_size, w.wavelength, w.boundary_width, w.n_subdomains,
                   periodic=w.periodic_flags(), n_correction=w.n_correction, device=device, stream=stream)

    def _dev(self, a):
        """complex64 device tensor of the grid shape.  Copies and conversions are enqueued on the solver's stream, so
        the library's kernels (same stream) are ordered after them; a tensor that is already right is passed through
        (the caller orders its producer with the solver's stream, as with any CUDA library)."""
        torch = self._torch
        if not isinstance(a, torch.Tensor):
            a = torch.from_numpy(np.ascontiguousarray(a))
        with torch.cuda.stream(self.stream):
            a = a.to(device=self.device, dtype=torch.complex64).contiguous()
        assert tuple(a.shape) == self.shape, (tuple(a.shape), self.shape)
        return a

    def _sync(self):
        """Temporaries created by this wrapper are released to torch's caching allocator on return; the library's
        asynchronous kernels may still read them, so the wrapper waits for the stream first."""
        self.stream.synchronize()

    def set_option(self, option: int, value: int):
        mbs_set_option(self.ctx, option, value)

    def set_potential(self, n_map):
        n = self._dev(n_map)
        mbs_set_potential(self.ctx, n.data_ptr())       # synchronises the stream itself (include/mbs.h)

    def apply_operator(self, which: int, inp, out=None):
        torch = self._torch
        a = self._dev(inp)
        if out is None:
            with torch.cuda.stream(self.stream):
                out = torch.empty_like(a)
        mbs_apply_operator(self.ctx, which, a.data_ptr(), out.data_ptr())
        if a is not inp:
            self._sync()                                # `a` is a temporary of this call
        return out

    def solve(self, y, x0=None, tol: float = 1e-6, max_iter: int = 1000):
        """Returns (x [device tensor], history [numpy], status)."""
        torch = self._torch
        yd = self._dev(y)
        if x0 is None:
            with torch.cuda.stream(self.stream):
                xd = torch.zeros(self.shape, dtype=torch.complex64, device=self.device)
        else:
            xd = self._dev(x0)
            if xd is x0:
                with torch.cuda.stream(self.stream):
                    xd = xd.clone()
        rc, hist, _ = mbs_solve(self.ctx, yd.data_ptr(), xd.data_ptr(), tol, max_iter)   # returns after a stream sync
        return xd, hist, rc

    def solve_batch(self, ys, x0s=None, tol: float = 1e-6, max_iter: int = 1000):
        """ys: [n_batch, *shape] (numpy or tensor).  Returns (x [n_batch, *shape] device tensor, history, status)."""
        torch = self._torch
        if not isinstance(ys, torch.Tensor):
            ys = torch.from_numpy(np.ascontiguousarray(ys))
        with torch.cuda.stream(self.stream):
            yd = ys.to(device=self.device, dtype=torch.complex64).contiguous()
            if x0s is None:
                xd = torch.zeros_like(yd)
            else:
                if not isinstance(x0s, torch.Tensor):
                    x0s = torch.from_numpy(np.ascontiguousarray(x0s))
                xd = x0s.to(device=self.device, dtype=torch.complex64).contiguous().clone()
        assert tuple(yd.shape[1:]) == self.shape and xd.shape == yd.shape
        rc, hist, _ = mbs_solve_batch(self.ctx, yd.shape[0], yd.data_ptr(), xd.data_ptr(), tol, max_iter)
        return xd, hist, rc

    def solve_host(self, y_host, x_host, tol: float, max_iter: int):
        """y_host, x_host: complex64 host arrays (numpy or CPU torch tensors, ideally pinned); x_host is in/out."""
        def ptr(a):
            return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
        rc, hist, n = mbs_solve_host(self.ctx, ptr(y_host), ptr(x_host), tol, max_iter)
        return hist, rc

    def iterate(self, y_dev, x_dev, n_iter: int, nu: float = 0.0, want_history: bool = True):
        """y_dev, x_dev: complex64 device tensors of the grid shape; x_dev is updated in place."""
        return mbs_iterate(self.ctx, y_dev.data_ptr(), x_dev.data_ptr(), n_iter, nu, want_history)

    def set_activation(self, enable: bool, threshold: float = -1.0):
        mbs_set_activation(self.ctx, enable, threshold)

    def activation(self) -> list:
        return mbs_get_activation(self.ctx)

    def kernel_stats(self) -> list:
        return mbs_get_kernel_stats(self.ctx)

    def reset_kernel_stats(self):
        mbs_reset_kernel_stats(self.ctx)

    def info(self) -> dict:
        return mbs_get_info(self.ctx)

    def close(self):
        if getattr(self, "ctx", None):
            mbs_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
