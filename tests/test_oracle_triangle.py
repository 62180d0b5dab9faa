"""Pins of the triangular-shaped radial basis phi_t of the oracle (Supp. Fig. 2) -- no GPU.

  PT1  with equidistant centres and gamma = spacing, sum_j w_j phi_t is the linear interpolant of the weights at the
       centres ("any input z only involves two basis functions")  -> numpy.interp
  PT2  closed forms of one basis function; partition of unity inside the range of the centres
  PT3  the stage with the triangular basis equals the stage assembled from pinned pieces (pad, conv_valid, corr_valid)
       with numpy.interp as phi; the Gaussian default is untouched by the switch
"""
import numpy as np

import oracle
import tnrd_gen

MU = tnrd_gen.rbf_centres()
DELTA = float(MU[1] - MU[0])
M = tnrd_gen.NUM_RBF


def _rng(n):
    return np.random.default_rng([20150305, 9, n])


def test_PT1_linear_interpolant_of_the_weights():
    r = _rng(1)
    w = r.standard_normal(M)
    z = r.uniform(MU[0] - 2.5 * DELTA, MU[-1] + 2.5 * DELTA, size=4000)
    with oracle.basis(oracle.TRIANGLE):
        got = oracle.phi(z, w, MU, DELTA)
    # numpy.interp on the centres extended by one zero node on either side (phi_t vanishes beyond mu +- gamma)
    xp = np.concatenate([[MU[0] - DELTA], MU, [MU[-1] + DELTA]])
    fp = np.concatenate([[0.0], w, [0.0]])
    want = np.interp(z, xp, fp, left=0.0, right=0.0)
    assert np.allclose(got, want, rtol=1e-12, atol=1e-12)


def test_PT2_closed_forms_and_partition_of_unity():
    j, wj, g = 20, 0.8, 7.5
    w = np.zeros(M); w[j] = wj
    z = MU[j] + g * np.array([0.0, 0.25, -0.5, 1.0, -1.0, 1.5, -3.0])
    with oracle.basis(oracle.TRIANGLE):
        got = oracle.phi(z, w, MU, g)
        ones = oracle.phi(_rng(2).uniform(MU[0], MU[-1], 500), np.ones(M), MU, DELTA)
    assert np.allclose(got, wj * np.array([1.0, 0.75, 0.5, 0.0, 0.0, 0.0, 0.0]), rtol=0, atol=1e-15)
    assert np.allclose(ones, 1.0, rtol=0, atol=1e-12)          # sum_j phi_t((z - mu_j) / delta) = 1 between the centres
    # the switch is restored: the default basis is the Gaussian one (P3's closed form)
    assert abs(oracle.phi(np.array([MU[j] + g]), w, MU, g)[0] - wj * np.exp(-0.5)) < 1e-15


def test_PT3_stage_with_triangular_basis():
    r = _rng(3)
    K, n_k, H, W = 5, 4, 11, 13
    k = tnrd_gen.dct_filters(K, n_k, r)
    w = 0.3 * r.standard_normal((n_k, M))
    lam = 0.13
    u = 255.0 * r.random((H, W))
    f = u + 20.0 * r.standard_normal((H, W))
    with oracle.basis(oracle.TRIANGLE):
        got = oracle.stage(f, u, k, w, MU, DELTA, lam)
    xp = np.concatenate([[MU[0] - DELTA], MU, [MU[-1] + DELTA]])
    up = oracle.pad(u, K - 1)
    s = np.zeros((H, W))
    for i in range(n_k):
        zi = oracle.conv_valid(up, k[i])
        vi = np.interp(zi, xp, np.concatenate([[0.0], w[i], [0.0]]), left=0.0, right=0.0)
        s += oracle.corr_valid(vi, k[i])
    assert np.allclose(got, u - (s + lam * (u - f)), rtol=1e-12, atol=1e-10)
    assert not np.allclose(got, oracle.stage(f, u, k, w, MU, DELTA, lam))      # the Gaussian stage differs
