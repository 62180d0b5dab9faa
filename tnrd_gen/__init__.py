"""Seeded synthetic inputs and parameters for the TNRD hot path (NumPy; SciPy only for the JPEG-like codec simulator).

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_1503_05768_b200``).  It holds none of the method's arithmetic: no
convolution of an image with a model filter, no influence function, no stage
update.  It only draws images, noise, filter coefficients and RBF weights with
the shapes and statistics of the paper's workloads (PAPER.md:162, :198-200,
:168-176, :484-488; recipe in DESIGN.md "Input recipe").

The paper measures on natural images (68 test images of 481x321, sigma 15/25)
that are not available here; the generators below stand in for them.

Every array is generated in float64, rounded ONCE to float32 and returned as
float32, so that the oracle (which promotes to double) and the GPU (fp32) read
bit-identical inputs.
"""
from __future__ import annotations

import numpy as np

MASTER_SEED = 150305768
NUM_RBF = 63                      # M
RBF_MU0, RBF_STEP = -310.0, 10.0  # BASELINE.json configs: mu_j = -310 + 10 (j-1)
RBF_GAMMA = 10.0                  # "width 10"
W_STD = 0.05                      # DESIGN.md reading S13: N(0, 0.05) is a std


def rng_for(cfg: int, item: int = 0, what: int = 0) -> np.random.Generator:
    """Independent stream for (config, item, purpose)."""
    return np.random.default_rng([MASTER_SEED, int(cfg), int(item), int(what)])


# --------------------------------------------------------------------------
# parameters
# --------------------------------------------------------------------------
def dct_basis(ksize: int) -> np.ndarray:
    """Orthonormal 2-D DCT-II atoms of a ksize x ksize patch WITHOUT the DC atom.

    Returns B with shape [ksize*ksize - 1][ksize][ksize]; atom (p, q), row-major
    in (p, q) with (0, 0) removed:  alpha_p alpha_q cos(pi (2a+1) p / 2m)
    cos(pi (2b+1) q / 2m).  ("DCT basis without the
    DC-component" -> zero-mean filters.)
    """
    m = ksize
    a = np.arange(m, dtype=np.float64)
    one_d = np.empty((m, m), dtype=np.float64)          # [p][a]
    for p in range(m):
        alpha = np.sqrt(1.0 / m) if p == 0 else np.sqrt(2.0 / m)
        one_d[p] = alpha * np.cos(np.pi * (2.0 * a + 1.0) * p / (2.0 * m))
    atoms = []
    for p in range(m):
        for q in range(m):
            if p == 0 and q == 0:
                continue
            atoms.append(np.outer(one_d[p], one_d[q]))
    return np.stack(atoms, axis=0)


def dct_filters(ksize: int, n_k: int, rng: np.random.Generator) -> np.ndarray:
    """n_k unit-norm zero-mean filters k = B c / ||c||_2, c ~ N(0,1)."""
    basis = dct_basis(ksize)                             # [R-1][m][m]
    c = rng.standard_normal((n_k, basis.shape[0]))
    c /= np.linalg.norm(c, axis=1, keepdims=True)
    return np.tensordot(c, basis, axes=(1, 0))           # [n_k][m][m], float64


def rbf_centres() -> np.ndarray:
    return RBF_MU0 + RBF_STEP * np.arange(NUM_RBF, dtype=np.float64)


def make_params(cfg: int, T: int, n_k: int, ksize: int, lam: str = "uniform") -> dict:
    """Per-stage parameter set Theta_t = {lambda^t, w^t_ij, k^t_i}."""
    rng = rng_for(cfg, 0, 1)
    filters = np.stack([dct_filters(ksize, n_k, rng) for _ in range(T)], axis=0)
    rbf_w = W_STD * rng.standard_normal((T, n_k, NUM_RBF))
    if lam == "const":
        lambdas = np.full((T,), 0.1)
    else:
        lambdas = rng.uniform(0.05, 0.2, size=(T,))
    return {
        "T": T, "N_k": n_k, "ksize": ksize,
        "filters": np.ascontiguousarray(filters, dtype=np.float32),
        "rbf_w": np.ascontiguousarray(rbf_w, dtype=np.float32),
        "rbf_mu": rbf_centres().astype(np.float32),
        "rbf_gamma": float(np.float32(RBF_GAMMA)),
        "lambda": lambdas.astype(np.float32),
    }


# --------------------------------------------------------------------------
# images
# --------------------------------------------------------------------------
def image_rectangles(H: int, W: int, rng: np.random.Generator, n_rect: int = 6) -> np.ndarray:
    """Piecewise-constant image: background U(0,255) + n_rect rectangles painted in order."""
    img = np.full((H, W), rng.uniform(0.0, 255.0))
    for _ in range(n_rect):
        y0 = int(rng.integers(0, H))
        x0 = int(rng.integers(0, W))
        hh = int(rng.integers(8, 49))
        ww = int(rng.integers(8, 49))
        img[y0:min(H, y0 + hh), x0:min(W, x0 + ww)] = rng.uniform(0.0, 255.0)
    return img


def image_field_texture(H: int, W: int, rng: np.random.Generator,
                        n_patches: int | None = None, blur_sigma: float = 12.0) -> np.ndarray:
    """Smooth Gaussian-random-field background in [0,255] + oriented sinusoidal texture patches."""
    if n_patches is None:
        n_patches = max(1, int(round(12.0 * (H * W) / (321.0 * 481.0))))
    white = rng.standard_normal((H, W))
    fy = np.fft.fftfreq(H)[:, None]
    fx = np.fft.rfftfreq(W)[None, :]
    gauss = np.exp(-2.0 * (np.pi ** 2) * (blur_sigma ** 2) * (fy * fy + fx * fx))
    field = np.fft.irfft2(np.fft.rfft2(white) * gauss, s=(H, W))
    lo, hi = field.min(), field.max()
    img = (field - lo) * (255.0 / (hi - lo))
    yy = np.arange(H, dtype=np.float64)[:, None]
    xx = np.arange(W, dtype=np.float64)[None, :]
    # patches are applied on a bounded window (4 sigma) so 4096^2 stays cheap
    for _ in range(n_patches):
        cy, cx = rng.uniform(0, H), rng.uniform(0, W)
        sp = rng.uniform(15.0, 40.0)
        amp = rng.uniform(15.0, 45.0)
        wav = rng.uniform(4.0, 14.0)
        th = rng.uniform(0.0, np.pi)
        ph = rng.uniform(0.0, 2.0 * np.pi)
        y0, y1 = max(0, int(cy - 4 * sp)), min(H, int(cy + 4 * sp) + 1)
        x0, x1 = max(0, int(cx - 4 * sp)), min(W, int(cx + 4 * sp) + 1)
        if y0 >= y1 or x0 >= x1:
            continue
        ys, xs = yy[y0:y1], xx[:, x0:x1]
        win = np.exp(-((ys - cy) ** 2 + (xs - cx) ** 2) / (2.0 * sp * sp))
        img[y0:y1, x0:x1] += amp * win * np.sin(
            2.0 * np.pi * (xs * np.cos(th) + ys * np.sin(th)) / wav + ph)
    return np.clip(img, 0.0, 255.0)


def add_noise(clean: np.ndarray, sigma: float, rng: np.random.Generator) -> np.ndarray:
    """f = clean + sigma N(0,1), NOT clipped (sigma on the 0..255 scale)."""
    return clean + sigma * rng.standard_normal(clean.shape)


# --------------------------------------------------------------------------
# the five BASELINE.json configs
# --------------------------------------------------------------------------
CONFIG_SHAPES = {
    1: dict(B=1, H=64, W=64, T=2, N_k=8, ksize=3),
    2: dict(B=1, H=321, W=481, T=5, N_k=24, ksize=5),
    3: dict(B=1, H=321, W=481, T=5, N_k=48, ksize=7),
    4: dict(B=1, H=4096, W=4096, T=5, N_k=48, ksize=7),
    5: dict(B=128, H=321, W=481, T=5, N_k=48, ksize=7),
}


def make_config(cfg: int, *, size: int | None = None, T: int | None = None,
                B: int | None = None) -> dict:
    """Inputs + parameters of BASELINE.json configs[cfg-1].

    cfg 4 takes ``size`` in {1024, 2048, 4096, ...} and ``T`` in {5, 8}; its T=5
    model is the first five stages of its T=8 parameter set.  cfg 5 takes ``B``
    (<=128) to draw only the first B items of the batch.
    Returns dict with float32 arrays f, u0 [B][H][W], clean, and the params.
    """
    shp = dict(CONFIG_SHAPES[cfg])
    if cfg == 4:
        if size is not None:
            shp["H"] = shp["W"] = int(size)
        if T is not None:
            shp["T"] = int(T)
    if cfg == 5 and B is not None:
        shp["B"] = int(B)
    H, W, nb = shp["H"], shp["W"], shp["B"]

    if cfg == 1:
        params = make_params(1, shp["T"], shp["N_k"], shp["ksize"], lam="const")
    elif cfg == 4:
        full = make_params(4, 8, shp["N_k"], shp["ksize"])
        t = shp["T"]
        params = dict(full, T=t, filters=full["filters"][:t].copy(),
                      rbf_w=full["rbf_w"][:t].copy(), **{"lambda": full["lambda"][:t].copy()})
    elif cfg == 5:
        params = make_params(3, shp["T"], shp["N_k"], shp["ksize"])   # C3's set, shared
    else:
        params = make_params(cfg, shp["T"], shp["N_k"], shp["ksize"])

    clean = np.empty((nb, H, W), dtype=np.float64)
    noisy = np.empty((nb, H, W), dtype=np.float64)
    sigmas = []
    for n in range(nb):
        if cfg == 1:
            r = rng_for(1, n, 0)
            clean[n] = image_rectangles(H, W, r)
            sigma = 15.0
        elif cfg in (2, 3):
            r = rng_for(2, n, 0)                 # C3 = same image and noise as C2
            clean[n] = image_field_texture(H, W, r)
            sigma = 25.0
        elif cfg == 4:
            r = rng_for(4, H * 100000 + W, 0)
            clean[n] = image_field_texture(H, W, r)
            sigma = 25.0
        else:
            r = rng_for(5, n, 0)
            clean[n] = image_field_texture(H, W, r)
            sigma = float(r.choice([15.0, 25.0, 50.0]))
        noisy[n] = add_noise(clean[n], sigma, r)
        sigmas.append(sigma)

    f = np.ascontiguousarray(noisy, dtype=np.float32)
    out = dict(shp)
    out.update(params)
    out.update(cfg=cfg, f=f, u0=f.copy(), clean=clean.astype(np.float32), sigma=sigmas)
    return out


def make_small(seed: int, B: int, H: int, W: int, T: int, n_k: int, ksize: int,
               sigma: float = 25.0) -> dict:
    """Ad-hoc small/odd-shaped case for parity tests (same generators, own seed stream)."""
    rng = rng_for(1000 + seed, 0, 0)
    prm = make_params(1000 + seed, T, n_k, ksize)
    clean = np.stack([image_field_texture(H, W, rng, n_patches=3, blur_sigma=4.0)
                      for _ in range(B)], axis=0)
    f = np.ascontiguousarray(add_noise(clean, sigma, rng), dtype=np.float32)
    out = dict(B=B, H=H, W=W, cfg=0, f=f, u0=f.copy(), clean=clean.astype(np.float32))
    out.update(prm)
    return out


# --------------------------------------------------------------------------
# JPEG-deblocking inputs: a synthetic compress / decompress round trip
# --------------------------------------------------------------------------
def synthetic_quant_table(strength: float) -> np.ndarray:
    """8x8 quantisation steps growing with frequency, Q[i][j] = strength * (1 + 0.6 (i + j) + 0.15 i j).

    A stand-in for a JPEG luminance table at some quality (the real tables and JPEG files are not available
    here); `strength` plays the role of the quality factor (larger = coarser)."""
    i = np.arange(8, dtype=np.float64)[:, None]
    j = np.arange(8, dtype=np.float64)[None, :]
    return strength * (1.0 + 0.6 * (i + j) + 0.15 * i * j)


def jpeg_like_roundtrip(clean: np.ndarray, qtable: np.ndarray):
    """Block-DCT, quantise, dequantise, inverse DCT of one image (H, W multiples of 8).

    Returns (decoded image, qcs_lo, qcs_hi): the decoder output u0 and the quantisation constraint set
    S = [Q (d - 1/2), Q (d + 1/2)] in block-coefficient layout.  Uses scipy's DCT: this is data
    synthesis (a codec simulator), not the method under test."""
    import scipy.fft as sfft
    H, W = clean.shape
    assert H % 8 == 0 and W % 8 == 0
    blocks = clean.reshape(H // 8, 8, W // 8, 8).transpose(0, 2, 1, 3)
    coef = sfft.dctn(blocks, type=2, norm="ortho", axes=(2, 3))
    d = np.rint(coef / qtable)
    lo, hi = qtable * (d - 0.5), qtable * (d + 0.5)
    dec = sfft.idctn(qtable * d, type=2, norm="ortho", axes=(2, 3))
    back = lambda a: a.transpose(0, 2, 1, 3).reshape(H, W)  # noqa: E731
    return back(dec), back(lo), back(hi)


def make_deblock(seed: int, B: int, H: int, W: int, T: int, n_k: int, ksize: int,
                 strength: float = 6.0) -> dict:
    """Deblocking case: decoded images u0, QCS bounds and per-stage parameters (no lambda: PAPER.md:716)."""
    rng = rng_for(2000 + seed, 0, 0)
    prm = make_params(2000 + seed, T, n_k, ksize)
    q = synthetic_quant_table(strength)
    u0, lo, hi, clean = [], [], [], []
    for _ in range(B):
        c = image_field_texture(H, W, rng, blur_sigma=max(2.0, min(12.0, H / 16.0)))
        d, a, b = jpeg_like_roundtrip(c, q)
        clean.append(c); u0.append(d); lo.append(a); hi.append(b)
    f32 = lambda xs: np.ascontiguousarray(np.stack(xs), dtype=np.float32)  # noqa: E731
    out = dict(B=B, H=H, W=W, u0=f32(u0), qcs_lo=f32(lo), qcs_hi=f32(hi), clean=f32(clean))
    out.update(prm)
    return out


def hash_image(H: int, W: int, y0: int = 0, y1: int | None = None) -> np.ndarray:
    """Rows [y0, y1) of an H x W image given by an integer formula of (y, x) -- blocks of two grey levels plus hash noise,
    values 0 .. 191, exactly representable -- so that a billion-pixel image (the `B*H*W < 2^31` edge case) can be made in row
    chunks and any window of it again later, without keeping or copying the whole image.  float32 [y1 - y0][W]."""
    y1 = H if y1 is None else y1
    y = np.arange(y0, y1, dtype=np.uint64)[:, None]
    x = np.arange(W, dtype=np.uint64)[None, :]
    h = (y * np.uint64(2654435761) + x * np.uint64(40503)) ^ ((y * x) >> np.uint64(3))
    h ^= h >> np.uint64(15)
    v = (h & np.uint64(127)) + np.uint64(64) * (((y // np.uint64(97)) + (x // np.uint64(89))) & np.uint64(1))
    return v.astype(np.float32)
