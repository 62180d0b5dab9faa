"""paper_1503_05768_b200 -- thin Python binding of libtnrd (include/tnrd.h).

The hot path of the trained nonlinear reaction-diffusion model (Chen, Yu, Pock, arXiv 1503.05768, Main
Eq. 7) runs entirely inside the hand-written sm_100a kernels of ``libtnrd.so``.  This module
only marshals arguments: it loads the shared library with ``ctypes`` and passes ``tensor.data_ptr()`` and the
current CUDA stream.  PyTorch supplies device memory and streams, nothing else.  There is NO CPU fallback:
if the library is missing, loading fails loudly.

Function names and argument order are those of the C ABI.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtnrd.so")
NUM_RBF = 63

OK, ERR_NULL, ERR_SHAPE, ERR_UNSUPPORTED, ERR_ALIAS, ERR_CUDA, ERR_PARAM, ERR_TOO_LARGE = 0, -1, -2, -3, -4, -5, -6, -7
STATIC_SCRATCH_BYTES = 64 << 20                                     # TNRD_STATIC_SCRATCH_BYTES (include/tnrd.h)
PHI_DENSE, PHI_WINDOW, PHI_LUT, PHI_FACTORED = 0, 1, 2, 3          # tnrd_set_phi_mode (include/tnrd.h)
KERNEL_AUTO, KERNEL_REF, KERNEL_TILE, KERNEL_TC, KERNEL_SMALL = 0, 1, 2, 3, 4     # tnrd_set_kernel (include/tnrd.h)

_lib = None


class TnrdError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libtnrd status {status}: {msg}")
        self.status = status


def build(verbose: bool = False, force: bool = False) -> str:
    """Compile libtnrd.so in-tree for sm_100a (nvcc cross-compiles without a GPU)."""
    from . import _build
    return _build.build(verbose=verbose, force=force)


def lib() -> ctypes.CDLL:
    """Load libtnrd.so (raises if it has not been built -- never falls back to anything else)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                f"{LIB_PATH} is missing: build it with `python -m paper_1503_05768_b200._build` "
                "(there is no CPU fallback for the TNRD hot path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cf = ctypes.c_void_p, ctypes.c_int, ctypes.c_float
        L.tnrd_stage.argtypes = [vp, vp, ci, ci, ci, ci, ci, vp, vp, vp, cf, cf, vp, vp]
        L.tnrd_stage.restype = ci
        L.tnrd_stage_static.argtypes = L.tnrd_stage.argtypes
        L.tnrd_stage_static.restype = ci
        dargs = [vp, vp, ci, ci, ci, ci, ci, ci, vp, vp, vp, cf, vp, vp, vp]
        L.tnrd_diffuse.argtypes = dargs
        L.tnrd_diffuse.restype = ci
        L.tnrd_diffuse_host.argtypes = dargs
        L.tnrd_diffuse_host.restype = ci
        L.tnrd_deblock_diffuse.argtypes = [vp, ci, ci, ci, ci, ci, ci, vp, vp, vp, cf, vp, vp, vp, vp]
        L.tnrd_deblock_diffuse.restype = ci
        L.tnrd_qcs_project.argtypes = [vp, ci, ci, ci, vp, vp, vp, vp]
        L.tnrd_qcs_project.restype = ci
        L.tnrd_stage_backward.argtypes = [vp, vp, vp, ci, ci, ci, ci, ci, vp, vp, vp, cf, cf, vp, vp, vp, vp, vp]
        L.tnrd_stage_backward.restype = ci
        L.tnrd_diffuse_backward.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, ci, ci, vp, vp, vp, cf, vp, vp, vp, vp, vp,
                                            vp, vp]
        L.tnrd_diffuse_backward.restype = ci
        L.tnrd_set_kernel.argtypes = [ci]
        L.tnrd_set_kernel.restype = ci
        L.tnrd_set_phi_mode.argtypes = [ci]
        L.tnrd_set_phi_mode.restype = ci
        L.tnrd_set_rbf_basis.argtypes = [ci]
        L.tnrd_set_rbf_basis.restype = ci
        L.tnrd_plan_query.argtypes = [ci, ci, ci, ci, ci, ci, ctypes.POINTER(ctypes.c_longlong)]
        L.tnrd_plan_query.restype = ci
        L.tnrd_tc_plan_query.argtypes = [ci, ci, ci, ci, ci, ci, ctypes.POINTER(ctypes.c_longlong)]
        L.tnrd_tc_plan_query.restype = ci
        L.tnrd_phi_stats.argtypes = [ci, ctypes.POINTER(ctypes.c_ulonglong), ctypes.POINTER(ctypes.c_ulonglong), vp]
        L.tnrd_phi_stats.restype = ci
        L.tnrd_launch_count.restype = ctypes.c_ulonglong
        L.tnrd_reset_launch_count.restype = None
        L.tnrd_microbench.argtypes = [ci, ctypes.POINTER(ctypes.c_double), vp]
        L.tnrd_microbench.restype = ci
        L.tnrd_strerror.argtypes = [ci]
        L.tnrd_strerror.restype = ctypes.c_char_p
        L.tnrd_last_cuda_error.restype = ctypes.c_char_p
        L.tnrd_version.restype = ci
        L.tnrd_shutdown.restype = None
        _lib = L
    return _lib


def _ptr(x):
    """Raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(f"cannot take the address of {type(x)}")


def _stream(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _check(rc: int):
    if rc != 0:
        L = lib()
        msg = L.tnrd_strerror(rc).decode()
        if rc == ERR_CUDA:
            msg += " -- " + L.tnrd_last_cuda_error().decode()
        raise TnrdError(rc, msg)


def tnrd_stage(f, u_in, B, H, W, N_k, ksize, filters_t, rbf_w_t, rbf_mu, rbf_gamma, lambda_t, u_out,
               stream=None):
    """One stage on device buffers (include/tnrd.h: tnrd_stage)."""
    _check(lib().tnrd_stage(_ptr(f), _ptr(u_in), B, H, W, N_k, ksize, _ptr(filters_t), _ptr(rbf_w_t),
                            _ptr(rbf_mu), float(rbf_gamma), float(lambda_t), _ptr(u_out), _stream(stream)))
    return u_out


def tnrd_stage_static(f, u_in, B, H, W, N_k, ksize, filters_t, rbf_w_t, rbf_mu, rbf_gamma, lambda_t, u_out,
                      stream=None):
    """One stage on device buffers without any allocation (include/tnrd.h: tnrd_stage_static)."""
    _check(lib().tnrd_stage_static(_ptr(f), _ptr(u_in), B, H, W, N_k, ksize, _ptr(filters_t), _ptr(rbf_w_t),
                                   _ptr(rbf_mu), float(rbf_gamma), float(lambda_t), _ptr(u_out), _stream(stream)))
    return u_out


def tnrd_diffuse(f, u0, B, H, W, T, N_k, ksize, filters, rbf_w, rbf_mu, rbf_gamma, lam, out, stream=None):
    """T stages on device buffers (include/tnrd.h: tnrd_diffuse)."""
    _check(lib().tnrd_diffuse(_ptr(f), _ptr(u0), B, H, W, T, N_k, ksize, _ptr(filters), _ptr(rbf_w),
                              _ptr(rbf_mu), float(rbf_gamma), _ptr(lam), _ptr(out), _stream(stream)))
    return out


def tnrd_diffuse_host(f, u0, B, H, W, T, N_k, ksize, filters, rbf_w, rbf_mu, rbf_gamma, lam, out,
                      stream=None):
    """T stages on HOST buffers, copies included (include/tnrd.h: tnrd_diffuse_host)."""
    _check(lib().tnrd_diffuse_host(_ptr(f), _ptr(u0), B, H, W, T, N_k, ksize, _ptr(filters), _ptr(rbf_w),
                                   _ptr(rbf_mu), float(rbf_gamma), _ptr(lam), _ptr(out), _stream(stream)))
    return out


def tnrd_deblock_diffuse(u0, B, H, W, T, N_k, ksize, filters, rbf_w, rbf_mu, rbf_gamma, qcs_lo, qcs_hi, out,
                         stream=None):
    """T JPEG-deblocking stages on device buffers (include/tnrd.h: tnrd_deblock_diffuse)."""
    _check(lib().tnrd_deblock_diffuse(_ptr(u0), B, H, W, T, N_k, ksize, _ptr(filters), _ptr(rbf_w), _ptr(rbf_mu),
                                      float(rbf_gamma), _ptr(qcs_lo), _ptr(qcs_hi), _ptr(out), _stream(stream)))
    return out


def tnrd_qcs_project(y, B, H, W, qcs_lo, qcs_hi, u_out, stream=None):
    """u_out = D^T eta(D y) on device buffers (include/tnrd.h: tnrd_qcs_project)."""
    _check(lib().tnrd_qcs_project(_ptr(y), B, H, W, _ptr(qcs_lo), _ptr(qcs_hi), _ptr(u_out), _stream(stream)))
    return u_out


def tnrd_stage_backward(f, u_in, e, B, H, W, N_k, ksize, filters_t, rbf_w_t, rbf_mu, rbf_gamma, lambda_t, grad_u=None,
                        grad_filters=None, grad_w=None, grad_lambda=None, stream=None):
    """Backward pass of one stage on device buffers (include/tnrd.h: tnrd_stage_backward)."""
    _check(lib().tnrd_stage_backward(_ptr(f), _ptr(u_in), _ptr(e), B, H, W, N_k, ksize, _ptr(filters_t), _ptr(rbf_w_t),
                                     _ptr(rbf_mu), float(rbf_gamma), float(lambda_t), _ptr(grad_u), _ptr(grad_filters),
                                     _ptr(grad_w), _ptr(grad_lambda), _stream(stream)))


def tnrd_diffuse_backward(f, u0, u_gt, e_T, B, H, W, T, N_k, ksize, filters, rbf_w, rbf_mu, rbf_gamma, lam, u_T=None,
                          grad_u0=None, grad_filters=None, grad_w=None, grad_lambda=None, stream=None):
    """Forward T stages + back-propagation on device buffers (include/tnrd.h: tnrd_diffuse_backward)."""
    _check(lib().tnrd_diffuse_backward(_ptr(f), _ptr(u0), _ptr(u_gt), _ptr(e_T), B, H, W, T, N_k, ksize, _ptr(filters),
                                       _ptr(rbf_w), _ptr(rbf_mu), float(rbf_gamma), _ptr(lam), _ptr(u_T), _ptr(grad_u0),
                                       _ptr(grad_filters), _ptr(grad_w), _ptr(grad_lambda), _stream(stream)))


def tnrd_set_kernel(which: int):
    _check(lib().tnrd_set_kernel(int(which)))


def tnrd_set_phi_mode(mode: int):
    """3 = factorised 63-term phi (default), 0 = direct 63-term phi, 1 = windowed evaluator, 2 = lookup table + linear
    interpolation (include/tnrd.h: tnrd_set_phi_mode)."""
    _check(lib().tnrd_set_phi_mode(int(mode)))


def tnrd_set_rbf_basis(basis: int):
    """0 = Gaussian radial basis (default), 1 = triangular-shaped (include/tnrd.h: tnrd_set_rbf_basis)."""
    _check(lib().tnrd_set_rbf_basis(int(basis)))


def tnrd_plan_query(B, H, W, N_k, ksize, num_sms=148) -> dict:
    """Launch plan of one stage (include/tnrd.h: tnrd_plan_query); host logic only, works without a GPU."""
    buf = (ctypes.c_longlong * 10)()
    _check(lib().tnrd_plan_query(B, H, W, N_k, ksize, num_sms, buf))
    keys = ("cfg", "ntx", "nty", "tw", "th", "n_full", "nsplit", "ctas", "cta_floats", "part_floats")
    return dict(zip(keys, (int(v) for v in buf)))


def tnrd_tc_plan_query(B, H, W, N_k, ksize, num_sms=148) -> dict:
    """Work decomposition of the tensor-core stage kernel (include/tnrd.h: tnrd_tc_plan_query); host logic only."""
    buf = (ctypes.c_longlong * 7)()
    _check(lib().tnrd_tc_plan_query(B, H, W, N_k, ksize, num_sms, buf))
    keys = ("applies", "nxs", "nys", "seg_rows", "units", "out_cols", "nchunk")
    return dict(zip(keys, (int(v) for v in buf)))


def tnrd_phi_stats(enable: bool, stream=None):
    """(executed, defined) phi group evaluations of the tensor-core kernel since the last call; switches counting on or
    off for later calls (include/tnrd.h: tnrd_phi_stats)."""
    ex, de = ctypes.c_ulonglong(0), ctypes.c_ulonglong(0)
    _check(lib().tnrd_phi_stats(int(bool(enable)), ctypes.byref(ex), ctypes.byref(de), _stream(stream)))
    return int(ex.value), int(de.value)


def tnrd_launch_count() -> int:
    return int(lib().tnrd_launch_count())


def tnrd_reset_launch_count():
    lib().tnrd_reset_launch_count()


def tnrd_microbench(which: int, stream=None) -> float:
    r = ctypes.c_double(0.0)
    _check(lib().tnrd_microbench(int(which), ctypes.byref(r), _stream(stream)))
    return r.value


def tnrd_strerror(status: int) -> str:
    return lib().tnrd_strerror(int(status)).decode()


def tnrd_last_cuda_error() -> str:
    return lib().tnrd_last_cuda_error().decode()


def tnrd_version() -> int:
    return int(lib().tnrd_version())


def tnrd_shutdown():
    lib().tnrd_shutdown()
