"""Pins of the CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the pin and the PAPER.md passage it rests on.  None of
them compares the oracle with itself: they use textbook definitions, closed forms (libm
erf / exp constants), library routines (scipy.signal, numpy.pad), dense-matrix brute force
and invariants.
"""
import math
import os

import numpy as np
import pytest
import scipy.signal as sig
from scipy.special import erf

import oracle
import tnrd_gen

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
MU = tnrd_gen.rbf_centres()
GAMMA = tnrd_gen.RBF_GAMMA
M = tnrd_gen.NUM_RBF


def _rng(n):
    return np.random.default_rng([20150305, n])


def _params(n_k, K, seed, T=1, w_std=0.05):
    r = _rng(seed)
    k = np.stack([tnrd_gen.dct_filters(K, n_k, r) for _ in range(T)])
    w = w_std * r.standard_normal((T, n_k, M))
    lam = r.uniform(0.05, 0.2, size=T)
    return k, w, lam


def _phi_np(z, w):
    """phi_g written with numpy broadcasting; used only inside brute-force pins
    whose point is the LINEAR structure; phi itself is pinned by P3 and P5."""
    return np.sum(w * np.exp(-((z[..., None] - MU) ** 2) / (2.0 * GAMMA ** 2)), axis=-1)


# ----------------------------------------------------------------------------------------
# O1: the mirror map is numpy's / Matlab's 'symmetric' (edge pixel repeated), NOT 'reflect'
# (PAPER.md:383 "mirror reflections", :387 "symmetric boundary condition"; reading S2)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("H,W,p", [(5, 7, 4), (8, 8, 6), (6, 9, 6), (3, 4, 2)])
def test_mirror_pad_is_numpy_symmetric(H, W, p):
    u = _rng(1).standard_normal((H, W))
    got = oracle.pad(u, p, symmetric=True)
    assert np.array_equal(got, np.pad(u, p, mode="symmetric"))
    assert not np.array_equal(got, np.pad(u, p, mode="reflect"))
    assert np.array_equal(oracle.pad(u, p, symmetric=False), np.pad(u, p, mode="constant"))


def test_mirror_index_values():
    # ... b a | a b ... : q = -1 -> 0, -2 -> 1 ; q = n -> n-1, n+1 -> n-2
    assert [oracle.mirror(q, 5) for q in (-3, -2, -1, 0, 4, 5, 6, 7)] == [2, 1, 0, 0, 4, 4, 3, 2]


# ----------------------------------------------------------------------------------------
# P1: orientation, tap indexing and centring (PAPER.md:70 "2D convolution", :125 rot180)
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [3, 5, 7, 9])
def test_P1_delta_response(K):
    r = (K - 1) // 2
    H, W, y0, x0 = 2 * K + 3, 2 * K + 5, K + 1, K + 2
    k = _rng(K).standard_normal((K, K))
    d = np.zeros((H, W)); d[y0, x0] = 1.0
    z = oracle.conv_valid(oracle.pad(d, r, symmetric=False), k)          # K u, zero-same
    s = oracle.corr_valid(oracle.pad(d, r, symmetric=False), k)          # Kbar v
    assert z.shape == (H, W) and s.shape == (H, W)
    for a in range(K):
        for b in range(K):
            assert z[y0 + a - r, x0 + b - r] == k[a, b]      # convolution: the kernel itself
            assert s[y0 - a + r, x0 - b + r] == k[a, b]      # rot180 kernel
    assert np.count_nonzero(z) == np.count_nonzero(k) and np.count_nonzero(s) == np.count_nonzero(k)


@pytest.mark.parametrize("K", [3, 5, 7])
def test_P1b_conv_corr_equal_scipy(K):
    img = _rng(10 + K).standard_normal((13, 17))
    k = _rng(20 + K).standard_normal((K, K))
    np.testing.assert_allclose(oracle.conv_valid(img, k), sig.convolve2d(img, k, mode="valid"),
                               rtol=0, atol=1e-13)
    np.testing.assert_allclose(oracle.corr_valid(img, k), sig.correlate2d(img, k, mode="valid"),
                               rtol=0, atol=1e-13)
    np.testing.assert_allclose(oracle.corr_valid(img, k),
                               sig.convolve2d(img, k[::-1, ::-1], mode="valid"), rtol=0, atol=1e-13)


# ----------------------------------------------------------------------------------------
# P2: constant image, zero-mean filters => u_t = u - lambda (u - f)   (north_star (d);
# PAPER.md:484-488 zero-mean filters; :123)
# ----------------------------------------------------------------------------------------
def test_P2_constant_image_dct_filters():
    k, w, lam = _params(24, 5, 2)
    f = _rng(3).uniform(0, 255, size=(12, 15))
    u = np.full_like(f, 93.25)
    got = oracle.stage(f, u, k[0], w[0], MU, GAMMA, lam[0])
    np.testing.assert_allclose(got, u - lam[0] * (u - f), rtol=0, atol=1e-9)


def test_P2_constant_image_integer_filters_bit_exact():
    k = np.zeros((3, 3, 3))
    k[0, 1] = [-1, 2, -1]; k[1, :, 1] = [-1, 2, -1]; k[2, 0, 0], k[2, 2, 2] = 1, -1
    w = 0.05 * _rng(4).standard_normal((3, M))
    f = _rng(5).uniform(0, 255, size=(9, 10))
    u = np.full_like(f, 128.0)
    got = oracle.stage(f, u, k, w, MU, GAMMA, 0.125)
    assert np.array_equal(got, u - (0.0 + 0.125 * (u - f)))


# ----------------------------------------------------------------------------------------
# P3: closed form of phi for a single non-zero weight (reading S5: gamma is a
# width, factor 2 in the denominator).  Constants from tests/golden/phi_closed_form.txt.
# ----------------------------------------------------------------------------------------
def test_P3_phi_single_weight_closed_form():
    table = np.loadtxt(os.path.join(GOLDEN, "phi_closed_form.txt"))
    for j in (0, 17, 31, 62):
        w = np.zeros(M); w[j] = -0.73
        for d, val in table:
            for sgn in (+1.0, -1.0):
                z = np.array([MU[j] + sgn * d * GAMMA])
                got = oracle.phi(z, w, MU, GAMMA)[0]
                assert got == pytest.approx(-0.73 * val, rel=1e-13, abs=0)
    # a different gamma / mu grid: phi(mu_j + gamma) = w e^{-1/2}
    mu2 = np.linspace(-3, 3, 7); w2 = np.zeros(7); w2[2] = 2.0
    assert oracle.phi(np.array([mu2[2] + 0.25]), w2, mu2, 0.25)[0] == pytest.approx(
        2.0 * 0.6065306597126334, rel=1e-14)


def test_P3b_phi_partition_of_unity():
    # sum_j exp(-(z-mu_j)^2/2g^2) with delta = gamma equals sqrt(2 pi) to ~1e-8 (Poisson summation):
    # a property of the equidistant Gaussian grid, checks that all 63 terms are summed.
    z = np.linspace(-200, 200, 401)
    got = oracle.phi(z, np.ones(M), MU, GAMMA)
    np.testing.assert_allclose(got, math.sqrt(2 * math.pi), rtol=1e-7)


# ----------------------------------------------------------------------------------------
# P4: O4 is the exact adjoint of O2 under zero padding  <K u, v> = <u, K^T v>
# (north_star (d); "K^T can be computed by convolution with kbar")
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [3, 5, 7])
def test_P4_adjoint_identity(K):
    r = (K - 1) // 2
    g = _rng(30 + K)
    u, v, k = g.standard_normal((11, 14)), g.standard_normal((11, 14)), g.standard_normal((K, K))
    Ku = oracle.conv_valid(oracle.pad(u, r, symmetric=False), k)
    Ktv = oracle.corr_valid(oracle.pad(v, r, symmetric=False), k)
    lhs, rhs = np.sum(Ku * v), np.sum(u * Ktv)
    assert abs(lhs - rhs) <= 1e-12 * max(1.0, abs(lhs))


# ----------------------------------------------------------------------------------------
# P5: the stage is one gradient step on the FoE energy (Main Eq. 3, rho' = phi).
# rho_i(z) = sum_j w_ij gamma sqrt(pi/2) erf((z-mu_j)/(gamma sqrt 2)); E by scipy 'same' zero
# boundary convolution; central differences against <u - u_t, d>.
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K,n_k", [(3, 8), (5, 6), (7, 5)])
def test_P5_energy_finite_difference(K, n_k):
    k, w, lam = _params(n_k, K, 40 + K)
    k, w, lam = k[0], w[0], lam[0]
    g = _rng(50 + K)
    f = g.uniform(0, 255, size=(12, 13))
    u = f + 10.0 * g.standard_normal(f.shape)

    def energy(img):
        e = 0.5 * lam * np.sum((img - f) ** 2)
        for i in range(n_k):
            zi = sig.convolve2d(img, k[i], mode="same", boundary="fill", fillvalue=0.0)
            rho = np.sum(w[i] * GAMMA * math.sqrt(math.pi / 2.0)
                         * erf((zi[..., None] - MU) / (GAMMA * math.sqrt(2.0))), axis=-1)
            e += np.sum(rho)
        return e

    ut = oracle.stage(f, u, k, w, MU, GAMMA, lam, mode=oracle.ZERO_SAME)
    grad = u - ut                                    # = sum K^T phi(K u) + lam (u - f)
    for trial in range(3):
        d = g.standard_normal(f.shape)
        eps = 1e-3
        fd = (energy(u + eps * d) - energy(u - eps * d)) / (2 * eps)
        an = np.sum(grad * d)
        assert abs(fd - an) <= 2e-6 * max(1.0, abs(an)), (fd, an)


# ----------------------------------------------------------------------------------------
# P6: special case -> library routine.  w_ij = a mu_j delta / (gamma sqrt(2 pi)) makes phi(z) = a z
# (to ~1e-6 a |z| on |z| <= 250), so the stage is linear and equals scipy convolutions on the
# numpy-'symmetric'-padded image.  With +-1 taps this is the linearised Perona-Malik step
# (PAPER.md:50-66).
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [3, 5])
def test_P6_linear_phi_equals_scipy(K):
    r = (K - 1) // 2
    n_k = 4
    k, _, lam = _params(n_k, K, 60 + K)
    k, lam = k[0], lam[0]
    if K == 3:                                   # embed k_x = [-1, 1], k_y = [-1, 1]^T
        k[0] = 0; k[0, 1, 1], k[0, 1, 2] = -1, 1
        k[1] = 0; k[1, 1, 1], k[1, 2, 1] = -1, 1
    a = np.array([0.05, -0.02, 0.03, 0.01])
    w = a[:, None] * MU[None, :] * tnrd_gen.RBF_STEP / (GAMMA * math.sqrt(2 * math.pi))
    g = _rng(70 + K)
    f = g.uniform(60, 200, size=(14, 11))
    u = f + 5.0 * g.standard_normal(f.shape)
    got = oracle.stage(f, u, k, w, MU, GAMMA, lam)
    up = np.pad(u, 2 * r, mode="symmetric")
    s = np.zeros_like(u)
    for i in range(n_k):
        zi = sig.convolve2d(up, k[i], mode="valid")
        assert np.max(np.abs(zi)) < 250
        s += a[i] * sig.correlate2d(zi, k[i], mode="valid")
    want = u - (s + lam * (u - f))
    np.testing.assert_allclose(got, want, rtol=0, atol=2e-4)      # 1.4e-6 * a * |z| * taps
    # and the deviation is NOT zero-tolerance luck: a wrong orientation fails by far more
    bad = np.zeros_like(u)
    for i in range(n_k):
        zi = sig.correlate2d(up, k[i], mode="valid")
        bad += a[i] * sig.correlate2d(zi, k[i], mode="valid")
    assert np.max(np.abs((u - (bad + lam * (u - f))) - got)) > 1e-2


# ----------------------------------------------------------------------------------------
# P7: brute force with dense matrices (PAPER.md:70 "K_i in R^{NxN}", :383 P and T matrices)
# ----------------------------------------------------------------------------------------
def _dense_ops(H, W, K):
    """Mirror-pad matrix P2r, valid-convolution matrix builder, valid-correlation matrix builder."""
    r = (K - 1) // 2
    idx = np.arange(H * W).reshape(H, W)
    pidx = np.pad(idx, 2 * r, mode="symmetric")              # numpy's index map, not oracle_mirror
    Hu, Wu = pidx.shape
    P = np.zeros((Hu * Wu, H * W)); P[np.arange(Hu * Wu), pidx.ravel()] = 1.0
    Hz, Wz = H + 2 * r, W + 2 * r

    def conv_mat(k):                                          # (Hz*Wz) x (Hu*Wu)
        A = np.zeros((Hz * Wz, Hu * Wu))
        for y in range(Hz):
            for x in range(Wz):
                for a in range(K):
                    for b in range(K):
                        # (k * u)[n] = sum_m k[m] u[n - m], output index offset by K-1 ('valid')
                        A[y * Wz + x, (y + K - 1 - a) * Wu + (x + K - 1 - b)] += k[a, b]
        return A

    def corr_mat(k):                                          # (H*W) x (Hz*Wz): conv with rot180(k)
        kb = k[::-1, ::-1]
        A = np.zeros((H * W, Hz * Wz))
        for y in range(H):
            for x in range(W):
                for a in range(K):
                    for b in range(K):
                        A[y * W + x, (y + K - 1 - a) * Wz + (x + K - 1 - b)] += kb[a, b]
        return A
    return P, conv_mat, corr_mat


@pytest.mark.parametrize("H,W,K,n_k", [(8, 8, 3, 8), (8, 11, 5, 4), (7, 7, 3, 3), (8, 8, 5, 5), (6, 7, 7, 2)])
def test_P7_dense_matrix_brute_force(H, W, K, n_k):
    k, w, lam = _params(n_k, K, 80 + H + W + K)
    k, w, lam = k[0], w[0], lam[0]
    g = _rng(90 + H)
    f = g.uniform(0, 255, size=(H, W)); u = f + 20.0 * g.standard_normal((H, W))
    P, conv_mat, corr_mat = _dense_ops(H, W, K)
    uv = u.ravel()
    s = np.zeros(H * W)
    for i in range(n_k):
        z = conv_mat(k[i]) @ (P @ uv)
        s += corr_mat(k[i]) @ _phi_np(z, w[i])
    want = (uv - (s + lam * (uv - f.ravel()))).reshape(H, W)
    got = oracle.stage(f, u, k, w, MU, GAMMA, lam)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-11)


# ----------------------------------------------------------------------------------------
# P8: reading S1.  Literal Supp. procedure: pad u and f by omega with mirror
# reflections, both convolutions 'same' with symmetric boundary ON THE PADDED IMAGE, crop.
# Equal to O1-O5 for every omega >= 2r; reading B (Main fn. 2 literally) differs at the border only.
# ----------------------------------------------------------------------------------------
def _literal_pad_crop_stage(f, u, k, w, lam, omega):
    up = np.pad(u, omega, mode="symmetric"); fp = np.pad(f, omega, mode="symmetric")
    s = np.zeros_like(up)
    for i in range(k.shape[0]):
        z = sig.convolve2d(up, k[i], mode="same", boundary="symm")
        s += sig.convolve2d(_phi_np(z, w[i]), k[i][::-1, ::-1], mode="same", boundary="symm")
    utp = up - (s + lam * (up - fp))
    return utp[omega:utp.shape[0] - omega, omega:utp.shape[1] - omega] if omega else utp


@pytest.mark.parametrize("K", [3, 5])
def test_P8_pad_crop_procedure_any_omega(K):
    r = (K - 1) // 2
    k, w, lam = _params(6, K, 100 + K)
    k, w, lam = k[0], w[0], lam[0]
    g = _rng(110 + K)
    f = g.uniform(0, 255, size=(16, 19)); u = f + 15.0 * g.standard_normal(f.shape)
    got = oracle.stage(f, u, k, w, MU, GAMMA, lam)
    for omega in (2 * r, 2 * r + 3, 8):
        np.testing.assert_allclose(got, _literal_pad_crop_stage(f, u, k, w, lam, omega), rtol=0, atol=1e-11)
    # omega too small (< 2r) is NOT the same thing
    short = _literal_pad_crop_stage(f, u, k, w, lam, 2 * r - 1)
    assert np.max(np.abs(short - got)) > 1e-3
    # reading B = omega 0: differs within r pixels of the border, agrees in the interior
    rb = _literal_pad_crop_stage(f, u, k, w, lam, 0)
    assert np.max(np.abs(rb - got)) > 1e-3
    np.testing.assert_allclose(rb[r:-r, r:-r], got[r:-r, r:-r], rtol=0, atol=1e-11)


# ----------------------------------------------------------------------------------------
# P9: no hidden asymmetry: flips and transposition commute with the stage
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [3, 5, 7])
def test_P9_flip_transpose_equivariance(K):
    k, w, lam = _params(5, K, 120 + K, T=2)
    g = _rng(130 + K)
    f = g.uniform(0, 255, size=(13, 18)); u = f + 15.0 * g.standard_normal(f.shape)
    base = oracle.diffuse(f, u, k, w, MU, GAMMA, lam)
    lr = oracle.diffuse(f[:, ::-1], u[:, ::-1], k[..., ::-1], w, MU, GAMMA, lam)
    ud = oracle.diffuse(f[::-1], u[::-1], k[:, :, ::-1, :], w, MU, GAMMA, lam)
    tr = oracle.diffuse(f.T, u.T, np.swapaxes(k, -1, -2), w, MU, GAMMA, lam)
    np.testing.assert_allclose(lr[:, ::-1], base, rtol=0, atol=1e-11)
    np.testing.assert_allclose(ud[::-1], base, rtol=0, atol=1e-11)
    np.testing.assert_allclose(tr.T, base, rtol=0, atol=1e-11)


# ----------------------------------------------------------------------------------------
# P10 / P11 / P12: batch independence, composition, degenerate parameters
# ----------------------------------------------------------------------------------------
def test_P10_P11_batch_and_composition():
    k, w, lam = _params(6, 5, 140, T=3)
    g = _rng(141)
    f = g.uniform(0, 255, size=(3, 10, 12)); u0 = f + 10 * g.standard_normal(f.shape)
    full = oracle.diffuse(f, u0, k, w, MU, GAMMA, lam)
    for b in range(3):
        assert np.array_equal(full[b], oracle.diffuse(f[b], u0[b], k, w, MU, GAMMA, lam))
    u = u0
    for t in range(3):
        u = oracle.stage(f, u, k[t], w[t], MU, GAMMA, lam[t])
    assert np.array_equal(u, full)


def test_P12_degenerate_parameters():
    k, w, lam = _params(4, 3, 150, T=2)
    g = _rng(151)
    f = g.uniform(0, 255, size=(9, 9)); u0 = f + 10 * g.standard_normal(f.shape)
    assert np.array_equal(oracle.diffuse(f, u0, k[:0], w[:0], MU, GAMMA, lam[:0]), u0)       # T = 0
    got = oracle.stage(f, u0, k[0], np.zeros_like(w[0]), MU, GAMMA, 0.25)                      # w = 0
    assert np.array_equal(got, u0 - (0.0 + 0.25 * (u0 - f)))
    got = oracle.stage(f, u0, k[0], np.zeros_like(w[0]), MU, GAMMA, 1.0)                       # lambda = 1
    np.testing.assert_allclose(got, f, rtol=0, atol=1e-13)
    with pytest.raises(ValueError):                                                            # min(H,W) < 2r
        oracle.stage(f[:1], u0[:1], k[0], w[0], MU, GAMMA, 0.1)
    with pytest.raises(ValueError):                                                            # gamma <= 0
        oracle.stage(f, u0, k[0], w[0], MU, 0.0, 0.1)


# ----------------------------------------------------------------------------------------
# P13 + locality: interior shift-equivariance and the crop-with-margin window oracle
# ----------------------------------------------------------------------------------------
def test_P13_interior_shift_equivariance_and_window():
    K, T = 5, 2
    k, w, lam = _params(5, K, 160, T=T)
    g = _rng(161)
    f = g.uniform(0, 255, size=(40, 44)); u0 = f + 10 * g.standard_normal(f.shape)
    full = oracle.diffuse(f, u0, k, w, MU, GAMMA, lam)
    m = (K - 1) * T
    dy, dx = 3, 5
    sh = oracle.diffuse(f[dy:, dx:], u0[dy:, dx:], k, w, MU, GAMMA, lam)
    assert np.array_equal(sh[m:-m, m:-m], full[dy + m:-m, dx + m:-m])
    for (y0, x0, h, ww) in [(0, 0, 9, 9), (14, 17, 8, 6), (31, 35, 9, 9), (0, 20, 5, 7)]:
        win = oracle.diffuse_window(f, u0, k, w, MU, GAMMA, lam, y0, x0, h, ww)
        assert np.array_equal(win, full[y0:y0 + h, x0:x0 + ww])
    # a margin one pixel short is visible
    ya, xa = 14 - (m - 1), 17 - (m - 1)
    short = oracle.diffuse(f[ya:14 + 8 + m - 1, xa:17 + 6 + m - 1], u0[ya:14 + 8 + m - 1, xa:17 + 6 + m - 1],
                           k, w, MU, GAMMA, lam)[m - 1:m - 1 + 8, m - 1:m - 1 + 6]
    assert not np.array_equal(short, full[14:22, 17:23])


# ----------------------------------------------------------------------------------------
# generator properties the configs rely on: zero-mean, unit-norm filters
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("K", [3, 5, 7, 9])
def test_generator_filters_zero_mean_unit_norm(K):
    k = tnrd_gen.dct_filters(K, K * K - 1, _rng(170 + K))
    np.testing.assert_allclose(k.sum(axis=(1, 2)), 0.0, atol=1e-13)
    np.testing.assert_allclose(np.sqrt((k ** 2).sum(axis=(1, 2))), 1.0, rtol=1e-13)
    B = tnrd_gen.dct_basis(K).reshape(K * K - 1, -1)
    np.testing.assert_allclose(B @ B.T, np.eye(K * K - 1), atol=1e-13)


def test_config1_runs_and_is_stable():
    c = tnrd_gen.make_config(1)
    out = oracle.diffuse(c["f"], c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"])
    assert out.shape == (1, 64, 64) and np.all(np.isfinite(out))
    assert np.max(np.abs(out - c["f"].astype(np.float64))) < 100.0
    c2 = tnrd_gen.make_config(1)
    assert np.array_equal(c["f"], c2["f"]) and np.array_equal(c["filters"], c2["filters"])
