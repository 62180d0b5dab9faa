"""Pins of the BACKWARD-pass oracle (oracle/tnrd_oracle_bwd.c) -- no GPU.

The gradient formulas of the supplement (Supp. Eq. 7, 10, 19 and the stage Jacobian at PAPER.md:612-616) are
pinned against things other than themselves:
  BP1  each transposed loop is the adjoint of the PINNED forward loop (<A x, y> = <x, A^T y>)
  BP2  closed form of phi' for a single non-zero weight
  BP3  central finite differences of the PINNED forward oracle (oracle.stage; loss 1/2 ||u_t - u_gt||^2)
  BP4  dense-matrix Jacobian on tiny images, matrices built here by brute force
  BP5  degenerate parameters
  BP6  T-stage back-propagation (Supp. Eq. 21) against finite differences of oracle.diffuse
"""
import math

import numpy as np
import pytest

import oracle
import tnrd_gen

MU = tnrd_gen.rbf_centres()
GAMMA = tnrd_gen.RBF_GAMMA
M = tnrd_gen.NUM_RBF


def _rng(n):
    return np.random.default_rng([20150305, 7, n])


def _problem(seed, B, H, W, n_k, K, w_std=0.3):
    """Small problem with O(1) influence-function slopes (w_std larger than the configs' so that every term of
    the gradients is well above rounding)."""
    r = _rng(seed)
    k = tnrd_gen.dct_filters(K, n_k, r)
    w = w_std * r.standard_normal((n_k, M))
    lam = float(r.uniform(0.05, 0.2))
    u = 255.0 * r.random((B, H, W))
    f = u + 20.0 * r.standard_normal((B, H, W))
    gt = u + 5.0 * r.standard_normal((B, H, W))
    return f, u, gt, k, w, lam


def _loss(f, u, gt, k, w, lam):
    ut = oracle.stage(f, u, k, w, MU, GAMMA, lam)
    return 0.5 * float(np.sum((ut - gt) ** 2))


# ---- BP1: adjoint identities against the pinned forward loops -----------------------------------------------------
@pytest.mark.parametrize("K", [3, 5, 7])
def test_BP1_transposed_loops_are_adjoints(K):
    r = _rng(K)
    H, W = 9, 12
    k = r.standard_normal((K, K))
    x = r.standard_normal((H + K - 1, W + K - 1))
    y = r.standard_normal((H, W))
    assert math.isclose(np.sum(oracle.conv_valid(x, k) * y), np.sum(x * oracle.conv_valid_T(y, k)), rel_tol=1e-12)
    assert math.isclose(np.sum(oracle.corr_valid(x, k) * y), np.sum(x * oracle.corr_valid_T(y, k)), rel_tol=1e-12)
    p = K - 1
    u = r.standard_normal((H, W))
    up = r.standard_normal((H + 2 * p, W + 2 * p))
    assert math.isclose(np.sum(oracle.pad(u, p) * up), np.sum(u * oracle.pad_T(up, H, W, p)), rel_tol=1e-12)
    # the two transposes are NOT interchangeable for a non-symmetric kernel (catches a swapped operand)
    assert not np.allclose(oracle.conv_valid_T(y, k), oracle.corr_valid_T(y, k))


def test_BP1_pad_T_counts_preimages():
    # folding an all-ones padded image counts how often each pixel is seen: 1 in the interior, 2 on edges, 4 at corners
    H, W, p = 6, 7, 2
    cnt = oracle.pad_T(np.ones((H + 2 * p, W + 2 * p)), H, W, p)
    assert cnt[3, 3] == 1 and cnt[0, 3] == 2 and cnt[3, 0] == 2 and cnt[0, 0] == 4 and cnt[1, 1] == 4
    assert cnt[2, 2] == 1 and cnt.sum() == (H + 2 * p) * (W + 2 * p)


# ---- BP2: closed form of phi' (reading BR2: derivative of PAPER.md:553) -------------------------------------------
def test_BP2_dphi_closed_form_single_weight():
    j, wj = 31, 0.7
    w = np.zeros(M); w[j] = wj
    z = MU[j] + GAMMA * np.array([0.0, 1.0, -1.0, 2.0, -0.5])
    got = oracle.dphi(z, w, MU, GAMMA)
    # phi(z) = w exp(-d^2 / 2 gamma^2)  =>  phi'(z) = -w (d / gamma^2) exp(-d^2 / 2 gamma^2),  d = z - mu_j
    want = [0.0, -wj / GAMMA * math.exp(-0.5), wj / GAMMA * math.exp(-0.5), -2 * wj / GAMMA * math.exp(-2.0),
            0.5 * wj / GAMMA * math.exp(-0.125)]
    assert np.allclose(got, want, rtol=1e-14, atol=1e-16)


def test_BP2_dphi_is_derivative_of_pinned_phi():
    r = _rng(2)
    w = 0.3 * r.standard_normal(M)
    z = r.uniform(-330, 330, size=200)
    h = 1e-4
    fd = (oracle.phi(z + h, w, MU, GAMMA) - oracle.phi(z - h, w, MU, GAMMA)) / (2 * h)
    assert np.allclose(oracle.dphi(z, w, MU, GAMMA), fd, rtol=1e-6, atol=1e-9)


# ---- BP3: finite differences of the pinned forward oracle ----------------------------------------------------------
@pytest.mark.parametrize("B,H,W,n_k,K", [(1, 9, 11, 3, 3), (2, 10, 8, 4, 5), (1, 12, 13, 3, 7), (1, 6, 6, 2, 7)])
def test_BP3_finite_differences(B, H, W, n_k, K):
    f, u, gt, k, w, lam = _problem(10 * K + B, B, H, W, n_k, K)
    e = oracle.stage(f, u, k, w, MU, GAMMA, lam) - gt                      # dl/du_t (reading BR3)
    g = oracle.stage_backward(f, u, e, k, w, MU, GAMMA, lam)
    r = _rng(99)

    def fd(fun, eps):
        return (fun(+eps) - fun(-eps)) / (2 * eps)

    for trial in range(3):
        d = r.standard_normal(u.shape)
        num = fd(lambda s: _loss(f, u + s * d, gt, k, w, lam), 1e-4)
        assert math.isclose(np.sum(g["g_u"] * d), num, rel_tol=2e-6, abs_tol=1e-6), "dl/du"
        dk = r.standard_normal(k.shape)
        num = fd(lambda s: _loss(f, u, gt, k + s * dk, w, lam), 1e-6)
        assert math.isclose(np.sum(g["g_k"] * dk), num, rel_tol=2e-6, abs_tol=1e-5), "dl/dk (Supp. Eq. 10)"
        dw = r.standard_normal(w.shape)
        num = fd(lambda s: _loss(f, u, gt, k, w + s * dw, lam), 1e-4)
        assert math.isclose(np.sum(g["g_w"] * dw), num, rel_tol=2e-6, abs_tol=1e-6), "dl/dw (Supp. Eq. 19)"
    num = fd(lambda s: _loss(f, u, gt, k, w, lam + s), 1e-5)
    assert math.isclose(g["g_lambda"], num, rel_tol=1e-7), "dl/dlambda (Supp. Eq. 7, reading BR1)"
    # single entries too (a permuted gradient passes random-direction tests only by accident, but be explicit)
    for (i, a, b) in [(0, 0, 0), (n_k - 1, K - 1, 0), (1, 1, K - 1)]:
        dk = np.zeros_like(k); dk[i, a, b] = 1.0
        num = fd(lambda s: _loss(f, u, gt, k + s * dk, w, lam), 1e-6)
        assert math.isclose(g["g_k"][i, a, b], num, rel_tol=5e-6, abs_tol=1e-4)
    for (i, j) in [(0, 0), (n_k - 1, 31), (1, 40)]:
        dw = np.zeros_like(w); dw[i, j] = 1.0
        num = fd(lambda s: _loss(f, u, gt, k, w + s * dw, lam), 1e-3)      # the loss is quadratic in w: exact
        assert math.isclose(g["g_w"][i, j], num, rel_tol=1e-7, abs_tol=1e-7)


# ---- BP4: dense-matrix Jacobian, matrices built by brute force -----------------------------------------------------
def _dense_ops(H, W, K, k):
    """P2r (mirror extension by 2r), K_i (valid convolution), Kbar_i (valid correlation) as dense matrices, built by
    applying the textbook index formulas to unit vectors (PAPER.md:70 'K_i u <=> k_i * u', :383)."""
    r = (K - 1) // 2
    Hu, Wu, Hz, Wz = H + 4 * r, W + 4 * r, H + 2 * r, W + 2 * r

    def mir(q, n):
        return -1 - q if q < 0 else (2 * n - 1 - q if q >= n else q)

    P = np.zeros((Hu * Wu, H * W))
    for y in range(Hu):
        for x in range(Wu):
            P[y * Wu + x, mir(y - 2 * r, H) * W + mir(x - 2 * r, W)] = 1.0
    Kc = np.zeros((Hz * Wz, Hu * Wu))
    for y in range(Hz):
        for x in range(Wz):
            for a in range(K):
                for b in range(K):
                    Kc[y * Wz + x, (y + K - 1 - a) * Wu + (x + K - 1 - b)] += k[a, b]
    Kb = np.zeros((H * W, Hz * Wz))
    for y in range(H):
        for x in range(W):
            for a in range(K):
                for b in range(K):
                    Kb[y * W + x, (y + a) * Wz + (x + b)] += k[a, b]
    return P, Kc, Kb


@pytest.mark.parametrize("H,W,K", [(8, 8, 3), (7, 9, 5), (6, 7, 7)])
def test_BP4_dense_matrix_jacobian(H, W, K):
    n_k = 3
    f, u, gt, k, w, lam = _problem(40 + K, 1, H, W, n_k, K)
    e = _rng(5).standard_normal((1, H, W))
    # J = (1 - lambda) I - sum_i Kbar_i diag(phi_i'(K_i P u)) K_i P     (crop built in)
    J = (1.0 - lam) * np.eye(H * W)
    for i in range(n_k):
        P, Kc, Kb = _dense_ops(H, W, K, k[i])
        z = Kc @ (P @ u.ravel())
        d = z[:, None] - MU[None, :]
        dphi = np.sum(-w[i][None, :] * d / GAMMA ** 2 * np.exp(-d ** 2 / (2 * GAMMA ** 2)), axis=1)
        J -= Kb @ (dphi[:, None] * (Kc @ P))
    g = oracle.stage_backward(f, u, e, k, w, MU, GAMMA, lam)
    assert np.allclose(g["g_u"].ravel(), J.T @ e.ravel(), rtol=1e-11, atol=1e-11)


# ---- BP5: degenerate parameters ---------------------------------------------------------------------------------------
def test_BP5_zero_weights_and_batch_sum():
    f, u, gt, k, w, lam = _problem(50, 2, 9, 10, 3, 5)
    e = _rng(6).standard_normal(u.shape)
    g0 = oracle.stage_backward(f, u, e, k, 0.0 * w, MU, GAMMA, lam)
    assert np.allclose(g0["g_u"], (1.0 - lam) * e, atol=1e-15)            # phi = phi' = 0: J = (1 - lambda) I
    assert np.allclose(g0["g_k"], 0.0, atol=1e-15)
    assert np.abs(g0["g_w"]).max() > 1e-3                                  # dl/dw does not depend on w
    assert math.isclose(g0["g_lambda"], -np.sum((u - f) * e), rel_tol=1e-13)
    # reading BR4: parameter gradients of a batch are the sum over its images
    g = oracle.stage_backward(f, u, e, k, w, MU, GAMMA, lam)
    parts = [oracle.stage_backward(f[b], u[b], e[b], k, w, MU, GAMMA, lam) for b in range(2)]
    for key in ("g_k", "g_w"):
        assert np.allclose(g[key], parts[0][key] + parts[1][key], rtol=1e-12, atol=1e-12)
    assert math.isclose(g["g_lambda"], parts[0]["g_lambda"] + parts[1]["g_lambda"], rel_tol=1e-12)
    assert np.array_equal(g["g_u"][1], parts[1]["g_u"])


# ---- BP6: back-propagation through T stages (Supp. Eq. 20-21) ------------------------------------------------------
def test_BP6_joint_backprop_finite_differences():
    T, n_k, K, H, W = 3, 3, 5, 11, 9
    r = _rng(60)
    k = np.stack([tnrd_gen.dct_filters(K, n_k, r) for _ in range(T)])
    w = 0.3 * r.standard_normal((T, n_k, M))
    lam = r.uniform(0.05, 0.2, size=T)
    u0 = 255.0 * r.random((1, H, W))
    f = u0 + 20.0 * r.standard_normal((1, H, W))
    gt = u0 + 5.0 * r.standard_normal((1, H, W))

    def loss(k_, w_, lam_, u0_):
        return 0.5 * float(np.sum((oracle.diffuse(f, u0_, k_, w_, MU, GAMMA, lam_) - gt) ** 2))

    g = oracle.diffuse_backward(f, u0, k, w, MU, GAMMA, lam, u_gt=gt)
    assert np.allclose(g["u_T"], oracle.diffuse(f, u0, k, w, MU, GAMMA, lam), rtol=0, atol=0)
    for name, base, eps in (("g_k", k, 1e-6), ("g_w", w, 1e-4), ("g_lambda", lam, 1e-5), ("g_u0", u0, 1e-4)):
        for trial in range(2):
            d = r.standard_normal(base.shape)
            args = {"g_k": lambda s: (k + s * d, w, lam, u0), "g_w": lambda s: (k, w + s * d, lam, u0),
                    "g_lambda": lambda s: (k, w, lam + s * d, u0), "g_u0": lambda s: (k, w, lam, u0 + s * d)}[name]
            num = (loss(*args(eps)) - loss(*args(-eps))) / (2 * eps)
            assert math.isclose(np.sum(g[name] * d), num, rel_tol=5e-6, abs_tol=1e-5), name
    # every stage's gradient is non-trivial (a recurrence that stopped early would leave zeros)
    assert all(np.abs(g["g_w"][t]).max() > 0 for t in range(T))
