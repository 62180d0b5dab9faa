"""GPU parity of the JPEG-deblocking path (tnrd_deblock_diffuse, tnrd_qcs_project) against the CPU oracle."""
import numpy as np
import pytest

import oracle
import tnrd_gen

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

MAX_ABS, RMS = 1e-2, 1e-3


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


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(tnrd, c, T=None, inplace=False):
    T = c["T"] if T is None else T
    u0 = dev(c["u0"])
    out = u0 if inplace else torch.empty_like(u0)
    tnrd.tnrd_deblock_diffuse(u0, c["B"], c["H"], c["W"], T, c["N_k"], c["ksize"], dev(c["filters"]), dev(c["rbf_w"]),
                              dev(c["rbf_mu"]), c["rbf_gamma"], dev(c["qcs_lo"]), dev(c["qcs_hi"]), out)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def run_oracle(c, T=None):
    T = c["T"] if T is None else T
    return oracle.deblock_diffuse(c["u0"], c["filters"][:T], c["rbf_w"][:T], c["rbf_mu"], c["rbf_gamma"], c["qcs_lo"],
                                  c["qcs_hi"])


def check(got, want, what):
    err = got - want
    mx, rms = float(np.max(np.abs(err))), float(np.sqrt(np.mean(err ** 2)))
    assert np.all(np.isfinite(got)) and mx <= MAX_ABS and rms <= RMS, f"{what}: max-abs {mx:.3e} rms {rms:.3e}"
    return mx, rms


CASES = [  # seed, B, H, W, T, N_k, ksize
    (1, 1, 8, 8, 1, 3, 3), (2, 2, 16, 40, 2, 6, 5), (3, 1, 72, 56, 3, 8, 7), (4, 3, 24, 136, 2, 5, 7),
    (5, 1, 160, 144, 4, 12, 7), (6, 1, 8, 264, 1, 4, 9),
]


@pytest.mark.parametrize("case", CASES, ids=[f"d{c[0]}" for c in CASES])
def test_deblock_cases_match_oracle(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_deblock(seed, B, H, W, T, n_k, K)
    want = run_oracle(c)
    check(run_gpu(tnrd, c), want, f"deblock {case}")
    check(run_gpu(tnrd, c, inplace=True), want, f"deblock in place {case}")
    assert np.array_equal(run_gpu(tnrd, c), run_gpu(tnrd, c, inplace=True))


def test_qcs_project_alone_and_in_the_box(tnrd):
    c = tnrd_gen.make_deblock(7, 2, 64, 96, 1, 4, 3, strength=10.0)
    g = np.random.default_rng(7)
    y = (c["u0"] + 20 * g.standard_normal(c["u0"].shape)).astype(np.float32)
    yd = dev(y); out = torch.empty_like(yd)
    tnrd.tnrd_qcs_project(yd, 2, 64, 96, dev(c["qcs_lo"]), dev(c["qcs_hi"]), out)
    got = out.cpu().numpy().astype(np.float64)
    want = np.stack([oracle.qcs_project(y[b], c["qcs_lo"][b], c["qcs_hi"][b]) for b in range(2)])
    assert np.max(np.abs(got - want)) <= 2e-4
    tnrd.tnrd_qcs_project(yd, 2, 64, 96, dev(c["qcs_lo"]), dev(c["qcs_hi"]), yd)          # in place
    assert np.array_equal(yd.cpu().numpy().astype(np.float64), got)
    z = np.stack([oracle.block_dct8(got[b]) for b in range(2)])                            # result lies in the QCS
    assert np.all(z >= c["qcs_lo"] - 1e-3) and np.all(z <= c["qcs_hi"] + 1e-3)
    # a misaligned view takes the scalar load path and gives the same numbers
    buf = torch.empty(2 * 64 * 96 + 1, device="cuda"); view = buf[1:].view(2, 64, 96); view.copy_(dev(y))
    out2 = torch.empty_like(view)
    tnrd.tnrd_qcs_project(view, 2, 64, 96, dev(c["qcs_lo"]), dev(c["qcs_hi"]), out2)
    assert np.array_equal(out2.cpu().numpy().astype(np.float64), got)


def test_deblock_infinite_box_equals_denoise_with_lambda_zero(tnrd):
    c = tnrd_gen.make_deblock(8, 1, 48, 64, 2, 6, 5)
    big = np.full(c["u0"].shape, 3e38, dtype=np.float32)
    d = dict(c, qcs_lo=-big, qcs_hi=big)
    got = run_gpu(tnrd, d)
    u0 = dev(c["u0"]); out = torch.empty_like(u0)
    tnrd.tnrd_diffuse(u0, u0, 1, 48, 64, 2, 6, 5, dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"]), c["rbf_gamma"],
                      dev(np.zeros(2, dtype=np.float32)), out)
    assert np.max(np.abs(got - out.cpu().numpy())) <= 5e-4       # D^T D = I up to fp32 rounding


def test_deblock_paper_workload_1024_sampled_blocks(tnrd):
    # TRD^4_{7x7} at 1024 x 1024, the size the paper times deblocking at
    c = tnrd_gen.make_deblock(9, 1, 1024, 1024, 4, 48, 7)
    got = run_gpu(tnrd, c)[0]
    assert np.all(np.isfinite(got))
    m = 6 * 4 + 8                                               # 2 r T, rounded up to whole blocks
    for (y0, x0) in [(0, 0), (1024 - 16, 1024 - 16), (504, 256), (0, 640)]:
        ya, yb, xa, xb = max(0, y0 - m), min(1024, y0 + 16 + m), max(0, x0 - m), min(1024, x0 + 16 + m)
        crop = lambda a: a[:, ya:yb, xa:xb]                     # noqa: E731  block-aligned crop with margin
        want = oracle.deblock_diffuse(crop(c["u0"]), c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                                      crop(c["qcs_lo"]), crop(c["qcs_hi"]))[0]
        check(got[y0:y0 + 16, x0:x0 + 16], want[y0 - ya:y0 - ya + 16, x0 - xa:x0 - xa + 16], f"deblock 1024 {(y0, x0)}")


def test_deblock_errors(tnrd):
    L = tnrd.lib()
    p = 0x1000
    assert L.tnrd_deblock_diffuse(p, 1, 12, 16, 1, 4, 3, p, p, p, 10.0, p, p, p + 64, None) == tnrd.ERR_SHAPE
    assert L.tnrd_deblock_diffuse(p, 1, 16, 16, 1, 4, 3, p, p, p, 10.0, None, p, p + 64, None) == tnrd.ERR_NULL
    assert L.tnrd_deblock_diffuse(p, 1, 16, 16, 1, 4, 3, p, p, p, 10.0, p + 64, p, p + 64, None) == tnrd.ERR_ALIAS
    assert L.tnrd_qcs_project(p, 1, 16, 20, p, p, p, None) == tnrd.ERR_SHAPE
