"""CPU oracle for the TNRD hot path -- TEST INFRASTRUCTURE, not product code.

Thin ctypes binding of ``oracle/tnrd_oracle.c`` (plain C, IEEE double, libm exp; the header
of that file states what it follows in PAPER.md and what pins it).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs
may import this package.  It imports nothing from ``paper_1503_05768_b200`` and that package
imports nothing from here.

All arrays are promoted to float64 (exact for float32 inputs) before the call; results are
float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tnrd_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "tnrd_oracle_bwd.c")]
_LIB = os.path.join(_HERE, "liboracle_tnrd.so")

SYMMETRIC_2R = 0   # reading A, the default boundary handling
ZERO_SAME = 1      # Main Eq. 2 with K^T under zero padding -- pins only

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 (no fast-math).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < max(os.path.getmtime(s) for s in _SRCS):
        cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-o", _LIB] + _SRCS + ["-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        ci, cd = ctypes.c_int, ctypes.c_double
        lib.oracle_num_threads.restype = ci
        lib.oracle_set_num_threads.argtypes = [ci]
        lib.oracle_mirror.argtypes = [ci, ci]
        lib.oracle_mirror.restype = ci
        lib.oracle_pad.argtypes = [dp, ci, ci, ci, ci, dp]
        lib.oracle_pad.restype = None
        lib.oracle_conv_valid.argtypes = [dp, ci, ci, dp, ci, dp]
        lib.oracle_conv_valid.restype = None
        lib.oracle_corr_valid.argtypes = [dp, ci, ci, dp, ci, dp]
        lib.oracle_corr_valid.restype = None
        lib.oracle_phi.argtypes = [dp, ctypes.c_size_t, dp, dp, ci, cd, dp]
        lib.oracle_phi.restype = None
        lib.oracle_set_basis.argtypes = [ci]
        lib.oracle_set_basis.restype = None
        lib.oracle_get_basis.restype = ci
        lib.oracle_stage.argtypes = [dp, dp, ci, ci, ci, ci, ci, dp, dp, dp, ci, cd, cd, dp, ci]
        lib.oracle_stage.restype = ci
        lib.oracle_diffuse.argtypes = [dp, dp, ci, ci, ci, ci, ci, ci, dp, dp, dp, ci, cd, dp, dp, ci]
        lib.oracle_diffuse.restype = ci
        _lib = lib
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


GAUSSIAN, TRIANGLE = 0, 1   # radial basis of phi


class basis:
    """Context manager: evaluate phi with the given radial basis inside the block (the oracle's switch is restored)."""

    def __init__(self, which: int):
        self.which = int(which)

    def __enter__(self):
        self.old = int(_load().oracle_get_basis())
        _load().oracle_set_basis(self.which)
        return self

    def __exit__(self, *exc):
        _load().oracle_set_basis(self.old)


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().oracle_set_num_threads(int(n))


def mirror(q: int, n: int) -> int:
    """O1 mirror map (edge pixel repeated)."""
    return int(_load().oracle_mirror(int(q), int(n)))


def pad(u, p: int, symmetric: bool = True):
    u = _d(u)
    H, W = u.shape
    out = np.empty((H + 2 * p, W + 2 * p), dtype=np.float64)
    _load().oracle_pad(_p(u), H, W, int(p), int(bool(symmetric)), _p(out))
    return out


def conv_valid(img, k):
    """O2: true convolution, valid extent."""
    img, k = _d(img), _d(k)
    K = k.shape[0]
    out = np.empty((img.shape[0] - K + 1, img.shape[1] - K + 1), dtype=np.float64)
    _load().oracle_conv_valid(_p(img), img.shape[0], img.shape[1], _p(k), K, _p(out))
    return out


def corr_valid(img, k):
    """O4: convolution with rot180(k) == correlation with k, valid extent."""
    img, k = _d(img), _d(k)
    K = k.shape[0]
    out = np.empty((img.shape[0] - K + 1, img.shape[1] - K + 1), dtype=np.float64)
    _load().oracle_corr_valid(_p(img), img.shape[0], img.shape[1], _p(k), K, _p(out))
    return out


def phi(z, w, mu, gamma: float):
    """O3: Gaussian-RBF influence function, point-wise."""
    z, w, mu = _d(z), _d(w), _d(mu)
    out = np.empty_like(z)
    _load().oracle_phi(_p(z), z.size, _p(w), _p(mu), mu.size, float(gamma), _p(out))
    return out


def _img3(a):
    a = _d(a)
    if a.ndim == 2:
        a = a[None]
    assert a.ndim == 3, "images are [B][H][W] or [H][W]"
    return a


def stage(f, u_in, filters_t, rbf_w_t, rbf_mu, rbf_gamma: float, lambda_t: float,
          mode: int = SYMMETRIC_2R):
    """One stage (O1-O5) on a batch; returns float64 [B][H][W]."""
    f3, u3 = _img3(f), _img3(u_in)
    k, w, mu = _d(filters_t), _d(rbf_w_t), _d(rbf_mu)
    B, H, W = u3.shape
    n_k, K = k.shape[0], k.shape[1]
    assert f3.shape == u3.shape and k.shape == (n_k, K, K) and w.shape == (n_k, mu.size)
    out = np.empty_like(u3)
    rc = _load().oracle_stage(_p(f3), _p(u3), B, H, W, n_k, K, _p(k), _p(w), _p(mu), mu.size,
                              float(rbf_gamma), float(lambda_t), _p(out), int(mode))
    if rc != 0:
        raise ValueError(f"oracle_stage failed with {rc}")
    return out if np.ndim(u_in) == 3 else out[0]


def diffuse(f, u0, filters, rbf_w, rbf_mu, rbf_gamma: float, lambdas, mode: int = SYMMETRIC_2R):
    """T stages (O6); returns float64 [B][H][W]."""
    f3, u3 = _img3(f), _img3(u0)
    k, w, mu, lam = _d(filters), _d(rbf_w), _d(rbf_mu), _d(lambdas)
    B, H, W = u3.shape
    T = lam.size
    if T > 0:
        n_k, K = k.shape[1], k.shape[2]
        assert k.shape == (T, n_k, K, K) and w.shape == (T, n_k, mu.size)
    else:
        n_k, K = 1, 1
    assert f3.shape == u3.shape
    out = np.empty_like(u3)
    rc = _load().oracle_diffuse(_p(f3), _p(u3), B, H, W, T, n_k, K, _p(k), _p(w), _p(mu), mu.size,
                                float(rbf_gamma), _p(lam), _p(out), int(mode))
    if rc != 0:
        raise ValueError(f"oracle_diffuse failed with {rc}")
    return out if np.ndim(u0) == 3 else out[0]


def diffuse_window(f, u0, filters, rbf_w, rbf_mu, rbf_gamma, lambdas, y0, x0, h, w):
    """u_T restricted to the window [y0,y0+h) x [x0,x0+w) of ONE image, from a crop.

    The update is local: u_T inside a window depends only on u0, f within 2r*T pixels of it
    (mirror-extended at true image borders).  The crop keeps a 2r*T margin and cuts it off
    only where it reaches a real image border (where the crop border IS the image border, so
    the mirror extension is the true one).  Everything is still computed by diffuse().
    """
    f2, u2 = _d(f), _d(u0)
    assert f2.ndim == 2
    H, W = f2.shape
    T = int(np.size(lambdas))
    K = int(np.shape(filters)[-1])
    m = (K - 1) * T            # 2 r T
    ya, yb = max(0, y0 - m), min(H, y0 + h + m)
    xa, xb = max(0, x0 - m), min(W, x0 + w + m)
    res = diffuse(f2[ya:yb, xa:xb], u2[ya:yb, xa:xb], filters, rbf_w, rbf_mu, rbf_gamma, lambdas)
    return res[y0 - ya:y0 - ya + h, x0 - xa:x0 - xa + w]


# ---- JPEG-deblocking stage (Main Eq. 9; Supp. Eq. 26-29) -----------------------------------------------------
def _load_deblock():
    lib = _load()
    if not getattr(lib, "_deblock_ready", False):
        dp, ci, cd = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double
        lib.oracle_block_dct8.argtypes = [dp, ci, ci, ci, dp]
        lib.oracle_block_dct8.restype = ci
        lib.oracle_qcs_project.argtypes = [dp, ci, ci, dp, dp, dp]
        lib.oracle_qcs_project.restype = ci
        lib.oracle_deblock_stage.argtypes = [dp, ci, ci, ci, ci, ci, dp, dp, dp, ci, cd, dp, dp, dp]
        lib.oracle_deblock_stage.restype = ci
        lib.oracle_deblock_diffuse.argtypes = [dp, ci, ci, ci, ci, ci, ci, dp, dp, dp, ci, cd, dp, dp, dp]
        lib.oracle_deblock_diffuse.restype = ci
        lib._deblock_ready = True
    return lib


def block_dct8(img, inverse: bool = False):
    """Orthonormal 2-D DCT-II (inverse: DCT-III) of every 8x8 block of one image; coefficient layout in place."""
    a = _d(img)
    out = np.empty_like(a)
    rc = _load_deblock().oracle_block_dct8(_p(a), a.shape[0], a.shape[1], int(bool(inverse)), _p(out))
    if rc != 0:
        raise ValueError(f"oracle_block_dct8 failed with {rc}")
    return out


def qcs_project(y, lo, hi):
    """u = D^T eta(D y) for one image (Supp. Eq. 26-27)."""
    y, lo, hi = _d(y), _d(lo), _d(hi)
    out = np.empty_like(y)
    rc = _load_deblock().oracle_qcs_project(_p(y), y.shape[0], y.shape[1], _p(lo), _p(hi), _p(out))
    if rc != 0:
        raise ValueError(f"oracle_qcs_project failed with {rc}")
    return out


def deblock_diffuse(u0, filters, rbf_w, rbf_mu, rbf_gamma: float, qcs_lo, qcs_hi):
    """T deblocking stages (Supp. Eq. 28-29); T = filters.shape[0]; returns float64 [B][H][W]."""
    u3, lo, hi = _img3(u0), _img3(qcs_lo), _img3(qcs_hi)
    k, w, mu = _d(filters), _d(rbf_w), _d(rbf_mu)
    B, H, W = u3.shape
    T = k.shape[0]
    n_k, K = (k.shape[1], k.shape[2]) if T > 0 else (1, 1)
    assert lo.shape == u3.shape and hi.shape == u3.shape
    out = np.empty_like(u3)
    rc = _load_deblock().oracle_deblock_diffuse(_p(u3), B, H, W, T, n_k, K, _p(k), _p(w), _p(mu), mu.size,
                                                float(rbf_gamma), _p(lo), _p(hi), _p(out))
    if rc != 0:
        raise ValueError(f"oracle_deblock_diffuse failed with {rc}")
    return out if np.ndim(u0) == 3 else out[0]


# ---- backward pass of a stage (Supp. Sec. 2: Eq. 7, 10, 19, 21) -- oracle/tnrd_oracle_bwd.c ---------------------
def _load_bwd():
    lib = _load()
    if not getattr(lib, "_bwd_ready", False):
        dp, ci, cd = ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_double
        lib.oracle_pad_T.argtypes = [dp, ci, ci, ci, dp]
        lib.oracle_pad_T.restype = None
        lib.oracle_conv_valid_T.argtypes = [dp, ci, ci, dp, ci, dp]
        lib.oracle_conv_valid_T.restype = None
        lib.oracle_corr_valid_T.argtypes = [dp, ci, ci, dp, ci, dp]
        lib.oracle_corr_valid_T.restype = None
        lib.oracle_dphi.argtypes = [dp, ctypes.c_size_t, dp, dp, ci, cd, dp]
        lib.oracle_dphi.restype = None
        lib.oracle_stage_backward.argtypes = [dp, dp, dp, ci, ci, ci, ci, ci, dp, dp, dp, ci, cd, cd, dp, dp, dp, dp]
        lib.oracle_stage_backward.restype = ci
        lib.oracle_diffuse_backward.argtypes = [dp, dp, dp, dp, ci, ci, ci, ci, ci, ci, dp, dp, dp, ci, cd, dp,
                                                dp, dp, dp, dp, dp]
        lib.oracle_diffuse_backward.restype = ci
        lib._bwd_ready = True
    return lib


def pad_T(up, H: int, W: int, p: int):
    """Adjoint of pad(symmetric): folds a (H+2p) x (W+2p) image back onto H x W."""
    up = _d(up)
    assert up.shape == (H + 2 * p, W + 2 * p)
    out = np.empty((H, W), dtype=np.float64)
    _load_bwd().oracle_pad_T(_p(up), H, W, int(p), _p(out))
    return out


def conv_valid_T(out_img, k):
    """Adjoint of conv_valid: (Ho, Wo) -> (Ho + K - 1, Wo + K - 1)."""
    o, k = _d(out_img), _d(k)
    K = k.shape[0]
    res = np.empty((o.shape[0] + K - 1, o.shape[1] + K - 1), dtype=np.float64)
    _load_bwd().oracle_conv_valid_T(_p(o), res.shape[0], res.shape[1], _p(k), K, _p(res))
    return res


def corr_valid_T(out_img, k):
    """Adjoint of corr_valid: (Ho, Wo) -> (Ho + K - 1, Wo + K - 1)."""
    o, k = _d(out_img), _d(k)
    K = k.shape[0]
    res = np.empty((o.shape[0] + K - 1, o.shape[1] + K - 1), dtype=np.float64)
    _load_bwd().oracle_corr_valid_T(_p(o), res.shape[0], res.shape[1], _p(k), K, _p(res))
    return res


def dphi(z, w, mu, gamma: float):
    """phi'(z), point-wise (derivative of PAPER.md:553)."""
    z, w, mu = _d(z), _d(w), _d(mu)
    out = np.empty_like(z)
    _load_bwd().oracle_dphi(_p(z), z.size, _p(w), _p(mu), mu.size, float(gamma), _p(out))
    return out


def stage_backward(f, u_in, e, filters_t, rbf_w_t, rbf_mu, rbf_gamma: float, lambda_t: float):
    """Backward pass of one stage; returns dict(g_u [B][H][W], g_k [N_k][K][K], g_w [N_k][M], g_lambda float)."""
    f3, u3, e3 = _img3(f), _img3(u_in), _img3(e)
    k, w, mu = _d(filters_t), _d(rbf_w_t), _d(rbf_mu)
    B, H, W = u3.shape
    n_k, K = k.shape[0], k.shape[1]
    assert f3.shape == u3.shape == e3.shape and k.shape == (n_k, K, K) and w.shape == (n_k, mu.size)
    g_u, g_k, g_w, g_l = np.empty_like(u3), np.empty_like(k), np.empty_like(w), np.zeros(1)
    rc = _load_bwd().oracle_stage_backward(_p(f3), _p(u3), _p(e3), B, H, W, n_k, K, _p(k), _p(w), _p(mu), mu.size,
                                           float(rbf_gamma), float(lambda_t), _p(g_u), _p(g_k), _p(g_w), _p(g_l))
    if rc != 0:
        raise ValueError(f"oracle_stage_backward failed with {rc}")
    return {"g_u": g_u if np.ndim(u_in) == 3 else g_u[0], "g_k": g_k, "g_w": g_w, "g_lambda": float(g_l[0])}


def diffuse_backward(f, u0, filters, rbf_w, rbf_mu, rbf_gamma: float, lambdas, u_gt=None, e_T=None):
    """Forward T stages + back-propagation (Supp. Eq. 20-21).  Loss 1/2 ||u_T - u_gt||^2 when u_gt is given, else
    e_T = dl/du_T is used.  Returns dict(u_T, g_u0, g_k [T][N_k][K][K], g_w [T][N_k][M], g_lambda [T])."""
    f3, u3 = _img3(f), _img3(u0)
    k, w, mu, lam = _d(filters), _d(rbf_w), _d(rbf_mu), _d(lambdas)
    B, H, W = u3.shape
    T, n_k, K = k.shape[0], k.shape[1], k.shape[2]
    gt = _img3(u_gt) if u_gt is not None else None
    eT = _img3(e_T) if e_T is not None else None
    u_T, g_u0, g_k, g_w, g_l = np.empty_like(u3), np.empty_like(u3), np.empty_like(k), np.empty_like(w), np.zeros(T)
    rc = _load_bwd().oracle_diffuse_backward(_p(f3), _p(u3), _p(gt) if gt is not None else None,
                                             _p(eT) if eT is not None else None, B, H, W, T, n_k, K, _p(k), _p(w),
                                             _p(mu), mu.size, float(rbf_gamma), _p(lam), _p(u_T), _p(g_u0), _p(g_k),
                                             _p(g_w), _p(g_l))
    if rc != 0:
        raise ValueError(f"oracle_diffuse_backward failed with {rc}")
    return {"u_T": u_T, "g_u0": g_u0, "g_k": g_k, "g_w": g_w, "g_lambda": g_l}
