"""GPU parity of the small-image kernel (tnrd_set_kernel(4), csrc/tnrd_small.cu: all T stages of an image that fits a
thread-block cluster in one launch) against the double-precision CPU oracle."""
import numpy as np
import pytest

import tnrd_gen
from test_gpu_parity import check, dev, run_gpu, run_oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tnrd():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1503_05768_b200 as t
    t.build()
    t.lib()
    t.tnrd_set_kernel(0)
    t.tnrd_set_phi_mode(t.PHI_FACTORED)
    return t


# seed, B, H, W, T, N_k, ksize: every ksize, odd / even T, fewer rows than CTAs in the cluster, ragged bands, batches
SMALL_CASES = [
    (301, 1, 64, 64, 2, 8, 3), (302, 2, 13, 29, 3, 8, 3), (303, 1, 4, 4, 2, 4, 5), (304, 3, 37, 23, 2, 6, 5),
    (305, 1, 6, 6, 1, 5, 7), (306, 2, 70, 50, 2, 7, 7), (307, 1, 8, 8, 1, 2, 9), (308, 1, 45, 61, 2, 4, 9),
    (309, 1, 2, 300, 1, 3, 3), (310, 1, 100, 2, 4, 3, 3), (311, 1, 64, 64, 1, 48, 7), (312, 5, 33, 47, 5, 12, 5),
]


@pytest.mark.parametrize("case", SMALL_CASES, ids=[f"m{c[0]}" for c in SMALL_CASES])
def test_small_kernel_matches_oracle(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    check(run_gpu(tnrd, c, kernel=4), run_oracle(c), f"small-image kernel {case}", tight=True)


def test_config1_one_launch_and_direct_mode(tnrd):
    """BASELINE.json configs[0] (64 x 64, T = 2, 8 filters 3x3): the automatic choice is the small-image kernel, one launch
    per call; the direct evaluator (one ex2 per Gaussian) runs on it too."""
    c = tnrd_gen.make_config(1)
    want = run_oracle(c)
    tnrd.tnrd_reset_launch_count()
    got = run_gpu(tnrd, c)
    assert tnrd.tnrd_launch_count() == 1
    check(got, want, "C1 small-image kernel", tight=True)
    assert np.max(np.abs(got - run_gpu(tnrd, c, kernel=2))) <= 2e-4          # the tile kernel agrees to fp32 rounding
    tnrd.tnrd_set_phi_mode(tnrd.PHI_DENSE)
    try:
        check(run_gpu(tnrd, c, kernel=4), want, "C1 small-image kernel, direct phi", tight=True)
    finally:
        tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)


def test_small_kernel_inplace_stage_and_determinism(tnrd):
    for T in (1, 2, 3):
        c = tnrd_gen.make_small(320 + T, 2, 40, 52, T, 6, 5)
        ref = run_gpu(tnrd, c, kernel=4)
        assert np.array_equal(run_gpu(tnrd, c, kernel=4), ref)                       # run to run
        u0 = dev(c["u0"])
        assert np.array_equal(run_gpu(tnrd, c, kernel=4, out=u0, u0=u0), ref), f"T={T}: in place"
        tnrd.tnrd_set_kernel(4)
        try:
            f, u = dev(c["f"]), dev(c["u0"])
            k, w, mu = dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"])
            for t in range(T):                                                       # T x tnrd_stage, in place
                tnrd.tnrd_stage(f, u, 2, 40, 52, 6, 5, k[t], w[t], mu, c["rbf_gamma"], float(c["lambda"][t]), u)
            torch.cuda.synchronize()
        finally:
            tnrd.tnrd_set_kernel(0)
        assert np.array_equal(u.cpu().numpy().astype(np.float64), ref), f"T={T}: diffuse != T x stage"


@pytest.mark.parametrize("change", ["jitter", "narrow", "wide"])
def test_small_kernel_other_centres_and_widths(tnrd, change):
    c = tnrd_gen.make_small(330, 2, 50, 61, 2, 5, 7)
    d = dict(c)
    if change == "jitter":
        mu = c["rbf_mu"].copy(); mu[10] += 2.0; d["rbf_mu"] = mu
    else:
        d["rbf_gamma"] = {"narrow": 8.0, "wide": 14.0}[change]
    check(run_gpu(tnrd, d, kernel=4), run_oracle(d), f"small-image kernel {change}", tight=True)


def test_small_kernel_extremes_nan_and_unsupported(tnrd):
    c = tnrd_gen.make_small(331, 1, 40, 44, 1, 6, 5)
    c["f"] = (c["f"] * 6.0 - 400.0).astype(np.float32); c["u0"] = c["f"].copy()     # z up to ~ +-1000
    w = c["rbf_w"].copy(); w[..., :3] = 0.5; w[..., -3:] = -0.5; c["rbf_w"] = w
    check(run_gpu(tnrd, c, kernel=4), run_oracle(c), "small-image kernel, extreme responses")
    c = tnrd_gen.make_small(332, 1, 40, 40, 1, 3, 5)
    c["f"][0, 20, 20] = np.nan; c["u0"] = c["f"].copy()
    got = run_gpu(tnrd, c, kernel=4)[0]
    assert np.isnan(got[16:25, 16:25]).all() and np.isfinite(got[:12, :]).all() and np.isfinite(got[:, 29:]).all()
    big = tnrd_gen.make_small(333, 1, 300, 300, 1, 4, 3)                             # does not fit a cluster
    with pytest.raises(tnrd.TnrdError) as ei:
        run_gpu(tnrd, big, kernel=4)
    assert ei.value.status == tnrd.ERR_UNSUPPORTED
    tnrd.tnrd_set_kernel(0)
    check(run_gpu(tnrd, big), run_oracle(big), "automatic choice for a larger image")
