"""Pins of the deblocking part of the oracle (Main Eq. 9; Supp. Eq. 26-29) -- no GPU."""
import math

import numpy as np
import pytest
import scipy.fft as sfft

import oracle
import tnrd_gen

MU, GAMMA = tnrd_gen.rbf_centres(), tnrd_gen.RBF_GAMMA


def _rng(n):
    return np.random.default_rng([20150306, n])


def _blocks(a):
    H, W = a.shape
    return a.reshape(H // 8, 8, W // 8, 8).transpose(0, 2, 1, 3)


def test_D1_block_dct_equals_scipy_ortho():
    x = _rng(1).standard_normal((24, 40))
    c = oracle.block_dct8(x)
    np.testing.assert_allclose(_blocks(c), sfft.dctn(_blocks(x), type=2, norm="ortho", axes=(2, 3)), atol=1e-13)
    np.testing.assert_allclose(_blocks(oracle.block_dct8(x, inverse=True)),
                               sfft.idctn(_blocks(x), type=2, norm="ortho", axes=(2, 3)), atol=1e-13)


def test_D2_orthogonality_and_parseval():
    # "DCT is an orthogonal transform, D^T D = D D^T = I"
    x = _rng(2).standard_normal((16, 16))
    np.testing.assert_allclose(oracle.block_dct8(oracle.block_dct8(x), inverse=True), x, atol=1e-13)
    np.testing.assert_allclose(oracle.block_dct8(oracle.block_dct8(x, inverse=True)), x, atol=1e-13)
    assert np.sum(oracle.block_dct8(x) ** 2) == pytest.approx(np.sum(x ** 2), rel=1e-13)
    y = _rng(3).standard_normal((16, 16))                      # <D x, y> = <x, D^T y>
    assert np.sum(oracle.block_dct8(x) * y) == pytest.approx(np.sum(x * oracle.block_dct8(y, inverse=True)), rel=1e-12)


def test_D3_closed_forms():
    c = oracle.block_dct8(np.full((8, 16), 3.5))               # constant block: only DC, value 8 c
    want = np.zeros((8, 16)); want[0, 0] = want[0, 8] = 8 * 3.5
    np.testing.assert_allclose(c, want, atol=1e-13)
    yy, xx = np.mgrid[0:8, 0:8]
    p, q = 2, 5                                                # one cosine atom -> one coefficient (p, q)
    atom = 0.5 * 0.5 * np.cos(math.pi * (2 * yy + 1) * p / 16) * np.cos(math.pi * (2 * xx + 1) * q / 16)
    c = oracle.block_dct8(atom)
    want = np.zeros((8, 8)); want[p, q] = 1.0
    np.testing.assert_allclose(c, want, atol=1e-13)
    ramp = np.tile(np.arange(8.0), (8, 1))                     # varies along x only -> only row p = 0 is non-zero
    c = oracle.block_dct8(ramp)
    assert np.max(np.abs(c[1:, :])) < 1e-13 and abs(c[0, 1]) > 1.0


def test_D4_projection_properties():
    g = _rng(4)
    y = 50 * g.standard_normal((16, 24))
    lo = 20 * g.standard_normal((16, 24)); hi = lo + g.uniform(0, 30, size=lo.shape)
    u = oracle.qcs_project(y, lo, hi)
    z = oracle.block_dct8(u)
    assert np.all(z >= lo - 1e-10) and np.all(z <= hi + 1e-10)          # result lies in the QCS
    np.testing.assert_allclose(oracle.qcs_project(u, lo, hi), u, atol=1e-10)   # idempotent
    np.testing.assert_allclose(z, np.clip(oracle.block_dct8(y), lo, hi), atol=1e-10)   # eta, Supp. Eq. 26
    big = np.full_like(y, 1e30)
    np.testing.assert_allclose(oracle.qcs_project(y, -big, big), y, atol=1e-10)        # infinite box: identity
    c0 = g.standard_normal(y.shape)
    np.testing.assert_allclose(oracle.qcs_project(y, c0, c0), oracle.block_dct8(c0, inverse=True), atol=1e-12)
    # orthogonal projection: no point of the box is closer to y (spot check with random feasible points)
    for _ in range(5):
        other = oracle.block_dct8(g.uniform(lo, hi), inverse=True)
        assert np.sum((u - y) ** 2) <= np.sum((other - y) ** 2) + 1e-9


def test_D5_infinite_box_reduces_to_denoising_stage_with_lambda_zero():
    c = tnrd_gen.make_deblock(1, 2, 16, 24, 2, 5, 5)
    big = np.full(c["u0"].shape, 1e30)
    got = oracle.deblock_diffuse(c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], -big, big)
    want = oracle.diffuse(c["u0"], c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], np.zeros(2))
    np.testing.assert_allclose(got, want, atol=1e-9)


def test_D6_stage_by_stage_and_scipy_composition():
    c = tnrd_gen.make_deblock(2, 1, 24, 32, 2, 4, 3)
    got = oracle.deblock_diffuse(c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["qcs_lo"],
                                 c["qcs_hi"])
    u = c["u0"][0].astype(np.float64)
    for t in range(2):                                         # Supp. Eq. 29 with scipy's DCT for D
        y = oracle.stage(u, u, c["filters"][t], c["rbf_w"][t], c["rbf_mu"], c["rbf_gamma"], 0.0)
        z = sfft.dctn(_blocks(y), type=2, norm="ortho", axes=(2, 3))
        v = np.clip(z, _blocks(c["qcs_lo"][0].astype(np.float64)), _blocks(c["qcs_hi"][0].astype(np.float64)))
        u = sfft.idctn(v, type=2, norm="ortho", axes=(2, 3)).transpose(0, 2, 1, 3).reshape(24, 32)
    np.testing.assert_allclose(got[0], u, atol=1e-10)
    assert np.max(np.abs(got[0] - c["u0"][0])) > 1e-3          # the stage does something


def test_D7_generator_qcs_contains_the_clean_image_and_the_decoded_one():
    c = tnrd_gen.make_deblock(3, 1, 32, 32, 1, 4, 3, strength=8.0)
    for img in (c["clean"][0], c["u0"][0]):
        z = oracle.block_dct8(img)
        assert np.all(z >= c["qcs_lo"][0] - 1e-3) and np.all(z <= c["qcs_hi"][0] + 1e-3)
    assert np.max(np.abs(c["clean"][0] - c["u0"][0])) > 1.0    # compression lost something


def test_D8_bad_shapes_rejected():
    with pytest.raises(ValueError):
        oracle.block_dct8(np.zeros((12, 16)))
    c = tnrd_gen.make_deblock(4, 1, 16, 16, 1, 3, 3)
    with pytest.raises(ValueError):
        oracle.deblock_diffuse(c["u0"][:, :12], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                               c["qcs_lo"][:, :12], c["qcs_hi"][:, :12])
