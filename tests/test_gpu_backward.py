"""GPU parity of the backward pass (tnrd_stage_backward / tnrd_diffuse_backward, through the C ABI binding) against the
double-precision oracle of oracle/tnrd_oracle_bwd.c on the same seeded inputs.

Tolerance: every gradient array within REL * max|oracle gradient| element by element.
The kernels work in fp32 with ex2.approx (2^-22 relative) and sum up to ~1e5 products per parameter in fp32; the
measured distance is ~1e-6 .. 2e-5 of the array's largest entry, REL = 2e-4 leaves a factor of ten."""
import numpy as np
import pytest

import oracle
import tnrd_gen

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

REL = 2e-4


@pytest.fixture(scope="module")
def tnrd():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1503_05768_b200 as t
    t.build()
    t.lib()
    t.tnrd_set_kernel(0)
    return t


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def close(got, want, what):
    got = np.asarray(got, dtype=np.float64)
    scale = float(np.max(np.abs(want)))
    err = float(np.max(np.abs(got - want)))
    assert np.all(np.isfinite(got)), what
    assert err <= REL * scale + 1e-30, f"{what}: max-abs error {err:.3e} against scale {scale:.3e} ({err / scale:.2e})"
    return err / max(scale, 1e-300)


def problem(seed, B, H, W, T, n_k, K):
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    c["u0"] = (0.5 * (c["f"] + c["clean"])).astype(np.float32)        # u_{t-1} != f, so that dl/dlambda is not trivially 0
    r = np.random.default_rng([150305768, 77, seed])
    e = r.standard_normal(c["f"].shape).astype(np.float32)
    gt = (c["f"] - 10.0 * r.standard_normal(c["f"].shape)).astype(np.float32)
    return c, e, gt


def gpu_stage_backward(tnrd, c, e, t=0, want=("u", "k", "w", "l")):
    B, H, W, n_k, K = c["B"], c["H"], c["W"], c["N_k"], c["ksize"]
    g_u = torch.full((B, H, W), float("nan"), device="cuda") if "u" in want else None
    g_k = torch.full((n_k, K, K), float("nan"), device="cuda") if "k" in want else None
    g_w = torch.full((n_k, 63), float("nan"), device="cuda") if "w" in want else None
    g_l = torch.full((1,), float("nan"), device="cuda") if "l" in want else None
    tnrd.tnrd_stage_backward(dev(c["f"]), dev(c["u0"]), dev(e), B, H, W, n_k, K, dev(c["filters"][t]), dev(c["rbf_w"][t]),
                             dev(c["rbf_mu"]), c["rbf_gamma"], float(c["lambda"][t]), g_u, g_k, g_w, g_l)
    torch.cuda.synchronize()
    return {k: (None if v is None else v.cpu().numpy()) for k, v in (("g_u", g_u), ("g_k", g_k), ("g_w", g_w), ("g_l", g_l))}


CASES = [  # seed, B, H, W, n_k, K : single tile, several tiles with ragged tails, tiny images (both mirrors hit a pixel)
    (1, 1, 8, 8, 3, 3), (2, 2, 13, 29, 5, 3), (3, 1, 4, 4, 2, 5), (4, 2, 37, 23, 6, 5), (5, 1, 6, 6, 3, 7),
    (6, 2, 70, 50, 7, 7), (7, 1, 8, 8, 2, 9), (8, 1, 45, 61, 4, 9), (9, 1, 131, 140, 5, 7), (10, 1, 2, 200, 3, 3),
    (11, 1, 118, 59, 4, 7),
]


@pytest.mark.parametrize("case", CASES, ids=[f"b{c[0]}" for c in CASES])
def test_stage_backward_matches_oracle(tnrd, case):
    seed, B, H, W, n_k, K = case
    c, e, _ = problem(seed, B, H, W, 1, n_k, K)
    want = oracle.stage_backward(c["f"], c["u0"], e, c["filters"][0], c["rbf_w"][0], c["rbf_mu"], c["rbf_gamma"],
                                 float(c["lambda"][0]))
    got = gpu_stage_backward(tnrd, c, e)
    close(got["g_u"], want["g_u"], f"{case} dl/du")
    close(got["g_w"], want["g_w"], f"{case} dl/dw (Supp. Eq. 19)")
    close(got["g_k"], want["g_k"], f"{case} dl/dk (Supp. Eq. 10)")
    close(got["g_l"], np.array([want["g_lambda"]]), f"{case} dl/dlambda (Supp. Eq. 7)")


def test_stage_backward_optional_outputs_and_determinism(tnrd):
    c, e, _ = problem(20, 2, 70, 90, 1, 6, 7)
    full = gpu_stage_backward(tnrd, c, e)
    again = gpu_stage_backward(tnrd, c, e)
    for k in full:
        assert np.array_equal(full[k], again[k]), f"{k} not deterministic"
    only_u = gpu_stage_backward(tnrd, c, e, want=("u",))
    assert np.array_equal(only_u["g_u"], full["g_u"]) and only_u["g_k"] is None
    only_w = gpu_stage_backward(tnrd, c, e, want=("w", "l"))
    assert np.array_equal(only_w["g_w"], full["g_w"]) and np.array_equal(only_w["g_l"], full["g_l"])


def test_stage_backward_paper_sized_image(tnrd):
    """BASELINE.json configs[2] geometry (321 x 481, 48 filters 7x7): many tiles, every border; the oracle needs ~20 s."""
    c = tnrd_gen.make_config(3)
    r = np.random.default_rng([150305768, 78])
    e = r.standard_normal(c["f"].shape).astype(np.float32)
    want = oracle.stage_backward(c["f"], c["u0"], e, c["filters"][0], c["rbf_w"][0], c["rbf_mu"], c["rbf_gamma"],
                                 float(c["lambda"][0]))
    got = gpu_stage_backward(tnrd, c, e)
    rel = {k: close(got[k], want[o], k) for k, o in (("g_u", "g_u"), ("g_w", "g_w"), ("g_k", "g_k"))}
    close(got["g_l"], np.array([want["g_lambda"]]), "dl/dlambda")
    print("C3 backward relative errors:", rel)


def test_stage_backward_errors(tnrd):
    c, e, _ = problem(21, 1, 16, 16, 1, 3, 3)
    f, u, ee = dev(c["f"]), dev(c["u0"]), dev(e)
    k, w, mu = dev(c["filters"][0]), dev(c["rbf_w"][0]), dev(c["rbf_mu"])
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_stage_backward(f, u, ee, 1, 16, 16, 3, 3, k, w, mu, 10.0, 0.1, grad_u=ee)
    assert ei.value.status == tnrd.ERR_ALIAS
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_stage_backward(f, u, None, 1, 16, 16, 3, 3, k, w, mu, 10.0, 0.1)
    assert ei.value.status == tnrd.ERR_NULL
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_stage_backward(f, u, ee, 1, 16, 16, 3, 4, k, w, mu, 10.0, 0.1)
    assert ei.value.status == tnrd.ERR_UNSUPPORTED


@pytest.mark.parametrize("case", [(30, 2, 40, 52, 3, 5, 5), (31, 1, 90, 77, 2, 6, 7)])
def test_diffuse_backward_matches_oracle(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c, e, gt = problem(seed, B, H, W, T, n_k, K)
    want = oracle.diffuse_backward(c["f"], c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"],
                                   u_gt=gt)
    u_T = torch.empty((B, H, W), device="cuda")
    g_u0, g_k = torch.empty((B, H, W), device="cuda"), torch.empty((T, n_k, K, K), device="cuda")
    g_w, g_l = torch.empty((T, n_k, 63), device="cuda"), torch.empty((T,), device="cuda")
    tnrd.tnrd_diffuse_backward(dev(c["f"]), dev(c["u0"]), dev(gt), None, B, H, W, T, n_k, K, dev(c["filters"]),
                               dev(c["rbf_w"]), dev(c["rbf_mu"]), c["rbf_gamma"], dev(c["lambda"]), u_T, g_u0, g_k, g_w, g_l)
    torch.cuda.synchronize()
    assert np.max(np.abs(u_T.cpu().numpy() - want["u_T"])) <= 1e-2
    close(g_u0.cpu().numpy(), want["g_u0"], "dl/du0")
    for t in range(T):
        close(g_k[t].cpu().numpy(), want["g_k"][t], f"stage {t} dl/dk")
        close(g_w[t].cpu().numpy(), want["g_w"][t], f"stage {t} dl/dw")
    close(g_l.cpu().numpy(), want["g_lambda"], "dl/dlambda")
    # the same gradients from a given e_T (= u_T - u_gt computed by the caller)
    eT = (want["u_T"] - gt).astype(np.float32)
    g_w2 = torch.empty_like(g_w)
    tnrd.tnrd_diffuse_backward(dev(c["f"]), dev(c["u0"]), None, dev(eT), B, H, W, T, n_k, K, dev(c["filters"]),
                               dev(c["rbf_w"]), dev(c["rbf_mu"]), c["rbf_gamma"], dev(c["lambda"]), None, None, None, g_w2,
                               None)
    torch.cuda.synchronize()
    close(g_w2.cpu().numpy(), want["g_w"], "dl/dw from e_T")


def _random_bwd_cases(n):
    r = np.random.default_rng([150305768, 98])
    out = []
    for i in range(n):
        K = int(r.choice([3, 5, 7, 9]))
        out.append((200 + i, int(r.integers(1, 3)), int(r.integers(K - 1, 140)), int(r.integers(K - 1, 200)),
                    int(r.integers(1, 7)), K))
    return out


@pytest.mark.parametrize("case", _random_bwd_cases(10), ids=lambda c: f"r{c[0]}-{c[1]}x{c[2]}x{c[3]}-k{c[5]}")
def test_stage_backward_random_shapes(tnrd, case):
    seed, B, H, W, n_k, K = case
    c, e, _ = problem(seed, B, H, W, 1, n_k, K)
    want = oracle.stage_backward(c["f"], c["u0"], e, c["filters"][0], c["rbf_w"][0], c["rbf_mu"], c["rbf_gamma"],
                                 float(c["lambda"][0]))
    got = gpu_stage_backward(tnrd, c, e)
    close(got["g_u"], want["g_u"], f"{case} dl/du")
    close(got["g_w"], want["g_w"], f"{case} dl/dw")
    close(got["g_k"], want["g_k"], f"{case} dl/dk")
    close(got["g_l"], np.array([want["g_lambda"]]), f"{case} dl/dlambda")
