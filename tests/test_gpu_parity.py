"""GPU parity: libtnrd (through the C ABI binding) against the double-precision CPU oracle, element by
element on the same seeded inputs.  Tolerance (BASELINE.json north_star (d)): max-abs <= 1e-2 and
RMS <= 1e-3 on the 0..255 scale after all T stages."""
import numpy as np
import pytest

import oracle
import tnrd_gen

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

MAX_ABS, RMS = 1e-2, 1e-3
# Regression bound for the EXACT evaluators (factorised, direct, windowed; tile and tensor-core kernels): they sit at
# ~3e-5 / 6e-6 from the oracle (fp32 rounding + ex2.approx), so 10 x that catches a loss of accuracy that the north_star
# tolerance above would let through.
TIGHT_MAX_ABS, TIGHT_RMS = 3e-4, 5e-5


@pytest.fixture(scope="module")
def tnrd():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1503_05768_b200 as t
    t.build()                    # compiles libtnrd.so with nvcc if it is stale or absent (not a fallback)
    t.lib()                      # fails loudly if libtnrd.so is missing: no fallback
    t.tnrd_set_kernel(0)
    t.tnrd_set_phi_mode(t.PHI_FACTORED)     # the default evaluator (include/tnrd.h)
    return t


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_gpu(tnrd, c, kernel=0, T=None, out=None, u0=None):
    """tnrd_diffuse on config dict c; returns float64 numpy [B][H][W]."""
    tnrd.tnrd_set_kernel(kernel)
    T = c["T"] if T is None else T
    f = dev(c["f"]); u0 = dev(c["u0"]) if u0 is None else u0
    k, w, mu, lam = dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"]), dev(c["lambda"])
    out = torch.empty_like(f) if out is None else out
    tnrd.tnrd_diffuse(f, u0, c["B"], c["H"], c["W"], T, c["N_k"], c["ksize"], k, w, mu, c["rbf_gamma"], lam, out)
    torch.cuda.synchronize()
    tnrd.tnrd_set_kernel(0)
    return out.cpu().numpy().astype(np.float64)


def run_oracle(c, T=None):
    T = c["T"] if T is None else T
    return oracle.diffuse(c["f"], c["u0"], c["filters"][:T], c["rbf_w"][:T], c["rbf_mu"], c["rbf_gamma"],
                          c["lambda"][:T])


def check(got, want, what="", tight=False):
    err = got - want
    mx, rms = float(np.max(np.abs(err))), float(np.sqrt(np.mean(err ** 2)))
    assert np.all(np.isfinite(got)), what
    assert mx <= MAX_ABS and rms <= RMS, f"{what}: max-abs {mx:.3e} rms {rms:.3e}"
    if tight:
        assert mx <= TIGHT_MAX_ABS and rms <= TIGHT_RMS, f"{what}: max-abs {mx:.3e} rms {rms:.3e} (regression bound)"
    return mx, rms


# --- small and ragged shapes, every ksize, both kernels: element by element ---------------------------------
SMALL = [  # seed, B, H, W, T, N_k, ksize
    (1, 1, 8, 8, 1, 3, 3), (2, 2, 13, 29, 2, 8, 3), (3, 1, 4, 4, 2, 4, 5), (4, 3, 37, 23, 2, 6, 5),
    (5, 1, 6, 6, 1, 5, 7), (6, 2, 70, 50, 2, 7, 7), (7, 1, 8, 8, 1, 2, 9), (8, 1, 45, 61, 2, 4, 9),
    (9, 1, 131, 140, 1, 5, 7), (10, 1, 2, 300, 1, 3, 3), (11, 1, 300, 2, 1, 3, 3), (12, 1, 64, 64, 1, 128, 3),
]


@pytest.mark.parametrize("kernel", [1, 2])
@pytest.mark.parametrize("case", SMALL, ids=[f"s{c[0]}" for c in SMALL])
def test_small_cases_match_oracle(tnrd, case, kernel):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    check(run_gpu(tnrd, c, kernel=kernel), run_oracle(c), f"case {case} kernel {kernel}", tight=True)


# --- BASELINE.json configs 1-3 in full ------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_configs_1_to_3_full_image(tnrd, cfg):
    c = tnrd_gen.make_config(cfg)
    want = run_oracle(c)
    mx, rms = check(run_gpu(tnrd, c), want, f"config {cfg}", tight=True)
    print(f"config {cfg}: max-abs {mx:.3e} rms {rms:.3e}")
    if cfg == 2:   # transposed orientation of the stand-in image (reading S14)
        ct = dict(c, H=c["W"], W=c["H"], f=np.ascontiguousarray(c["f"].transpose(0, 2, 1)),
                  u0=np.ascontiguousarray(c["u0"].transpose(0, 2, 1)),
                  filters=np.ascontiguousarray(np.swapaxes(c["filters"], -1, -2)))
        check(run_gpu(tnrd, ct).transpose(0, 2, 1), want, "config 2 transposed")


# --- full sizes in the launch configuration bench.py times: sampled windows the oracle computes one by one --------
def _windows(H, W, size, n_random, seed):
    ys = [0, (H - size) // 2, H - size]
    xs = [0, (W - size) // 2, W - size]
    wins = [(y, x) for y in ys for x in xs]                      # 4 corners, 4 edge mid-points, centre
    r = np.random.default_rng([7, seed])
    wins += [(int(r.integers(0, H - size + 1)), int(r.integers(0, W - size + 1))) for _ in range(n_random)]
    return wins


def test_config4_4096_T5_sampled_windows(tnrd):
    c = tnrd_gen.make_config(4, size=4096, T=5)
    got = run_gpu(tnrd, c)[0]
    assert np.all(np.isfinite(got))
    worst = 0.0
    for (y0, x0) in _windows(4096, 4096, 24, 4, 4):
        want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"],
                                     c["rbf_gamma"], c["lambda"], y0, x0, 24, 24)
        mx, _ = check(got[y0:y0 + 24, x0:x0 + 24], want, f"C4 window {(y0, x0)}")
        worst = max(worst, mx)
    print(f"config 4 (4096^2, T=5): worst window max-abs {worst:.3e}")
    # tile seams: a window straddling the first tile boundaries in both directions
    for (y0, x0) in [(110, 110), (122 * 17 - 3 - 12, 122 * 5 - 3 - 12)]:
        want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"],
                                     c["rbf_gamma"], c["lambda"], y0, x0, 24, 24)
        check(got[y0:y0 + 24, x0:x0 + 24], want, f"C4 seam window {(y0, x0)}")


def test_config4_1024_T8_sampled_windows_and_T5_prefix(tnrd):
    c8 = tnrd_gen.make_config(4, size=1024, T=8)
    got8 = run_gpu(tnrd, c8)[0]
    got5 = run_gpu(tnrd, c8, T=5)[0]
    for (y0, x0) in _windows(1024, 1024, 20, 1, 8)[::3]:
        for T, got in ((8, got8), (5, got5)):
            want = oracle.diffuse_window(c8["f"][0], c8["u0"][0], c8["filters"][:T], c8["rbf_w"][:T], c8["rbf_mu"],
                                         c8["rbf_gamma"], c8["lambda"][:T], y0, x0, 20, 20)
            check(got[y0:y0 + 20, x0:x0 + 20], want, f"C4-1024 T={T} window {(y0, x0)}")


def test_config5_batch_sampled_and_independent(tnrd):
    c = tnrd_gen.make_config(5)
    got = run_gpu(tnrd, c)
    assert got.shape == (128, 321, 481) and np.all(np.isfinite(got))
    for b in (0, 63, 127):
        for (y0, x0) in [(0, 0), (321 - 24, 481 - 24), (150, 230)]:
            want = oracle.diffuse_window(c["f"][b], c["u0"][b], c["filters"], c["rbf_w"], c["rbf_mu"],
                                         c["rbf_gamma"], c["lambda"], y0, x0, 24, 24)
            check(got[b, y0:y0 + 24, x0:x0 + 24], want, f"C5 image {b} window {(y0, x0)}")
    # P10: images are independent.  Inside one plan (same B, same tiles) an image's result is bit-identical wherever it
    # sits in the batch; processed alone the planner tiles it differently (other partial-sum boundaries), and the result
    # agrees to fp32 rounding
    rev = dict(c, f=np.ascontiguousarray(c["f"][::-1]), u0=np.ascontiguousarray(c["u0"][::-1]))
    assert np.array_equal(run_gpu(tnrd, rev)[127 - 5], got[5])
    one = dict(c, B=1, f=c["f"][5:6], u0=c["u0"][5:6])
    assert np.max(np.abs(run_gpu(tnrd, one)[0] - got[5])) <= 2e-4


# --- properties that hold at any size ----------------------------------------------------------------------------
def test_P2_constant_image_gpu(tnrd):
    c = tnrd_gen.make_config(3)
    u0 = np.full_like(c["f"], 93.25)
    got = run_gpu(tnrd, dict(c, u0=u0), T=1)
    lam = float(c["lambda"][0])
    want = u0.astype(np.float64) - lam * (u0.astype(np.float64) - c["f"])
    assert np.max(np.abs(got - want)) <= 2e-4          # zero-mean DCT filters: sum_i kbar_i * const = O(eps)


def test_P12_degenerate_parameters_gpu(tnrd):
    c = tnrd_gen.make_small(21, 2, 40, 52, 2, 6, 5)
    z = dict(c, rbf_w=np.zeros_like(c["rbf_w"]))
    u, f = c["u0"].astype(np.float64), c["f"].astype(np.float64)
    want = u - float(c["lambda"][0]) * (u - f)
    assert np.max(np.abs(run_gpu(tnrd, z, T=1) - want)) <= 1e-4
    one = dict(z, **{"lambda": np.ones_like(c["lambda"])})
    assert np.max(np.abs(run_gpu(tnrd, one, T=1) - f)) <= 1e-4          # lambda = 1, w = 0 => u_1 = f
    assert np.array_equal(run_gpu(tnrd, c, T=0), u)                      # T = 0 copies u0


def test_P9_flip_equivariance_gpu(tnrd):
    c = tnrd_gen.make_small(22, 1, 150, 139, 2, 8, 7)
    base = run_gpu(tnrd, c)
    fl = dict(c, f=np.ascontiguousarray(c["f"][..., ::-1]), u0=np.ascontiguousarray(c["u0"][..., ::-1]),
              filters=np.ascontiguousarray(c["filters"][..., ::-1]))
    assert np.max(np.abs(run_gpu(tnrd, fl)[..., ::-1] - base)) <= 2e-3   # fp32 summation order differs


# --- API semantics (P11, aliasing, host entry point, determinism) -------------------------------------------------
@pytest.mark.parametrize("kernel", [1, 2])
def test_diffuse_equals_repeated_stage_and_inplace(tnrd, kernel):
    for T in (1, 2, 3, 4):
        c = tnrd_gen.make_small(30 + T, 2, 33, 47, T, 5, 5)
        ref = run_gpu(tnrd, c, kernel=kernel)
        tnrd.tnrd_set_kernel(kernel)
        f, u = dev(c["f"]), dev(c["u0"])
        k, w, mu = dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"])
        for t in range(T):
            nxt = torch.empty_like(u)
            tnrd.tnrd_stage(f, u, 2, 33, 47, 5, 5, k[t], w[t], mu, c["rbf_gamma"], float(c["lambda"][t]), nxt)
            u = nxt
        torch.cuda.synchronize()
        tnrd.tnrd_set_kernel(0)
        assert np.array_equal(u.cpu().numpy().astype(np.float64), ref), f"T={T}: diffuse != T x stage"
        u0 = dev(c["u0"])                                   # in place: out == u0
        assert np.array_equal(run_gpu(tnrd, c, kernel=kernel, out=u0, u0=u0), ref), f"T={T}: in-place differs"
        tnrd.tnrd_set_kernel(kernel)                        # tnrd_stage in place: u_out == u_in
        v = dev(c["u0"])
        for t in range(T):
            tnrd.tnrd_stage(f, v, 2, 33, 47, 5, 5, k[t], w[t], mu, c["rbf_gamma"], float(c["lambda"][t]), v)
        torch.cuda.synchronize()
        tnrd.tnrd_set_kernel(0)
        assert np.array_equal(v.cpu().numpy().astype(np.float64), ref), f"T={T}: in-place stage differs"


def test_host_entry_point_and_determinism(tnrd):
    c = tnrd_gen.make_small(40, 3, 90, 77, 3, 9, 7)
    ref = run_gpu(tnrd, c)
    assert np.array_equal(run_gpu(tnrd, c), ref)           # run-to-run deterministic
    f = torch.from_numpy(c["f"]).pin_memory()
    out = torch.empty_like(f).pin_memory()
    tnrd.tnrd_diffuse_host(f, f, 3, 90, 77, 3, 9, 7, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                           c["lambda"], out)
    assert np.array_equal(out.numpy().astype(np.float64), ref)
    out2 = np.empty_like(c["f"])                            # pageable numpy buffers work too
    tnrd.tnrd_diffuse_host(c["f"], c["u0"], 3, 90, 77, 3, 9, 7, c["filters"], c["rbf_w"], c["rbf_mu"],
                           c["rbf_gamma"], c["lambda"], out2)
    assert np.array_equal(out2.astype(np.float64), ref)


def test_side_stream_and_launch_count(tnrd):
    c = tnrd_gen.make_small(41, 1, 60, 60, 2, 4, 3)
    ref = run_gpu(tnrd, c)
    s = torch.cuda.Stream()
    tnrd.tnrd_reset_launch_count()
    with torch.cuda.stream(s):
        got = run_gpu(tnrd, c)
    assert np.array_equal(got, ref)
    assert tnrd.tnrd_launch_count() == 1                   # the small-image kernel: all stages in one launch
    tnrd.tnrd_reset_launch_count()
    assert np.max(np.abs(run_gpu(tnrd, c, kernel=2) - ref)) <= 2e-4
    assert tnrd.tnrd_launch_count() == 1 + 2 * c["T"]      # tile kernel: one staging kernel + (tile, update) per stage
    tnrd.tnrd_shutdown()
    assert np.array_equal(run_gpu(tnrd, c), ref)            # usable after shutdown


def test_microbench_rates_are_sane(tnrd):
    ffma, mufu, phi = (tnrd.tnrd_microbench(i) for i in range(3))
    print(f"FFMA {ffma / 1e12:.2f} T/s  MUFU.EX2 {mufu / 1e12:.2f} T/s  phi terms {phi / 1e12:.2f} T/s")
    assert 5e12 < ffma < 60e12 and 1e12 < mufu < 12e12 and 0.5e12 < phi <= mufu * 1.05
    disp = tnrd.tnrd_microbench(3)          # FFMA2 + FMNMX warp instructions per second (1.0 per clock per scheduler if the pipes issued side by side)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    print(f"FFMA2 + FMNMX mixed: {disp / 1e9:.0f} G warp-instr/s = {disp / (sms * 4 * 1.965e9):.2f} per clock per scheduler")
    assert 0.45 < disp / (sms * 4 * 1.965e9) < 1.05
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_microbench(4)
    assert ei.value.status == tnrd.ERR_UNSUPPORTED


# --- windowed phi evaluator (tnrd_set_phi_mode(1)): same oracle, same tolerance ------------------------------------
def run_gpu_window(tnrd, c, **kw):
    tnrd.tnrd_set_phi_mode(1)
    try:
        return run_gpu(tnrd, c, **kw)
    finally:
        tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)


@pytest.mark.parametrize("case", SMALL, ids=[f"s{c[0]}" for c in SMALL])
def test_window_phi_small_cases(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    check(run_gpu_window(tnrd, c), run_oracle(c), f"window case {case}")


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_window_phi_configs(tnrd, cfg):
    c = tnrd_gen.make_config(cfg)
    got = run_gpu_window(tnrd, c)
    mx, rms = check(got, run_oracle(c), f"window config {cfg}")
    dense = run_gpu(tnrd, c)
    print(f"window config {cfg}: max-abs {mx:.3e} rms {rms:.3e}; vs dense GPU {np.max(np.abs(got - dense)):.3e}")
    assert np.max(np.abs(got - dense)) <= 2e-4     # truncated mass < 1e-9 w: only fp32 rounding differs


def test_window_phi_extreme_responses(tnrd):
    # responses far outside [mu_1, mu_63] and large weights on the outermost centres: the clamped window must hold
    c = tnrd_gen.make_small(50, 1, 40, 44, 1, 6, 5)
    c["f"] = (c["f"] * 6.0 - 400.0).astype(np.float32); c["u0"] = c["f"].copy()     # z up to ~ +-1000
    w = c["rbf_w"].copy(); w[..., :3] = 0.5; w[..., -3:] = -0.5; c["rbf_w"] = w
    check(run_gpu_window(tnrd, c), run_oracle(c), "window extreme")


def test_window_phi_falls_back_to_dense(tnrd):
    c = tnrd_gen.make_small(51, 2, 50, 61, 2, 5, 7)
    for change in ("jitter", "gamma"):
        d = dict(c)
        if change == "jitter":                      # centres not equidistant
            mu = c["rbf_mu"].copy(); mu[10] += 2.0; d["rbf_mu"] = mu
        else:                                       # gamma > delta: 14 centres no longer cover 6.5 gamma
            d["rbf_gamma"] = 14.0
        dense = run_gpu_mode(tnrd, d, phi_mode=0, kernel=2)
        tnrd.tnrd_reset_launch_count()
        got = run_gpu_window(tnrd, d)
        assert tnrd.tnrd_launch_count() == 1 + 3 * d["T"]      # both fused kernels launched (one returns at once) + update
        assert np.array_equal(got, dense), change               # ... and the dense one did the work
        check(got, run_oracle(d), f"fallback {change}")


def test_window_phi_full_size_windows(tnrd):
    c = tnrd_gen.make_config(4, size=2048, T=5)
    got = run_gpu_window(tnrd, c)[0]
    for (y0, x0) in _windows(2048, 2048, 24, 2, 9)[::2]:
        want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"],
                                     c["rbf_gamma"], c["lambda"], y0, x0, 24, 24)
        check(got[y0:y0 + 24, x0:x0 + 24], want, f"window C4-2048 {(y0, x0)}")


# --- the two exact evaluators: TNRD_PHI_FACTORED (default; every test above ran it) and TNRD_PHI_DENSE (direct) -----------
@pytest.mark.parametrize("case", SMALL, ids=[f"s{c[0]}" for c in SMALL])
def test_direct_phi_small_cases(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    check(run_gpu_mode(tnrd, c, phi_mode=0), run_oracle(c), f"direct case {case}")


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_direct_and_factorised_phi_configs(tnrd, cfg):
    """Both exact evaluators against the oracle on BASELINE.json's configs, and against each other: the factorisation is an
    identity, the two differ by fp32 rounding only."""
    c = tnrd_gen.make_config(cfg)
    want = run_oracle(c)
    direct, fact = run_gpu_mode(tnrd, c, phi_mode=0), run_gpu_mode(tnrd, c, phi_mode=3)
    md, _ = check(direct, want, f"direct config {cfg}")
    mf, _ = check(fact, want, f"factorised config {cfg}")
    d = float(np.max(np.abs(direct - fact)))
    print(f"config {cfg}: direct {md:.3e}, factorised {mf:.3e} from the oracle; {d:.3e} from each other")
    assert d <= 2e-4 and mf <= 2.0 * md + 1e-4


def test_factorised_phi_extreme_responses(tnrd):
    """Responses far outside the centres (the clamp of the distance to a group's anchor is active for every group), large
    weights on the outermost centres, and a response exactly on a centre."""
    c = tnrd_gen.make_small(50, 1, 40, 44, 1, 6, 5)
    c["f"] = (c["f"] * 6.0 - 400.0).astype(np.float32); c["u0"] = c["f"].copy()     # z up to ~ +-1000
    w = c["rbf_w"].copy(); w[..., :3] = 0.5; w[..., -3:] = -0.5; c["rbf_w"] = w
    check(run_gpu_mode(tnrd, c, phi_mode=3), run_oracle(c), "factorised extreme")
    c = tnrd_gen.make_small(52, 1, 33, 35, 1, 4, 3)
    c["f"] = np.full_like(c["f"], 40.0); c["u0"] = c["f"].copy()                    # constant image
    k = np.zeros_like(c["filters"]); k[:, :, 1, 1] = np.array([1.0, -2.0, 0.25, 7.75])[None, :]   # z = 40, -80, 10, 310
    c["filters"] = k
    check(run_gpu_mode(tnrd, c, phi_mode=3), run_oracle(c), "factorised on-centre responses")


def test_factorised_phi_large_weights(tnrd):
    # weights 1e4 times the configs' (|w| ~ 2e3): the polynomials stay far inside the fp32 range
    c = tnrd_gen.make_small(53, 1, 48, 52, 1, 5, 7)
    c["rbf_w"] = (c["rbf_w"] * 1e4).astype(np.float32)
    want = run_oracle(c)
    got = run_gpu_mode(tnrd, c, phi_mode=3)
    assert np.all(np.isfinite(got))
    scale = float(np.max(np.abs(want - c["f"].astype(np.float64))))
    assert np.max(np.abs(got - want)) <= 2e-5 * scale, "relative to the size of the update"


@pytest.mark.parametrize("change", ["jitter", "narrow", "wide", "wider"])
def test_factorised_phi_other_centres_and_widths(tnrd, change):
    """jitter: centres not equidistant -> the kernel evaluates the direct form (same launch); narrow: gamma = 0.8 delta ->
    direct form as well (the powers of rho would overflow); wide / wider: gamma = 1.4 / 3 delta -> factorised."""
    c = tnrd_gen.make_small(51, 2, 50, 61, 2, 5, 7)
    d = dict(c)
    if change == "jitter":
        mu = c["rbf_mu"].copy(); mu[10] += 2.0; d["rbf_mu"] = mu
    else:
        d["rbf_gamma"] = {"narrow": 8.0, "wide": 14.0, "wider": 30.0}[change]
    want = run_oracle(d)
    tnrd.tnrd_reset_launch_count()
    got = run_gpu_mode(tnrd, d, phi_mode=3, kernel=2)
    assert tnrd.tnrd_launch_count() == 1 + 2 * d["T"]
    check(got, want, f"factorised {change}")
    direct = run_gpu_mode(tnrd, d, phi_mode=0, kernel=2)
    if change in ("jitter", "narrow"):
        assert np.array_equal(got, direct), "the direct form inside the factorised kernel is the direct kernel's"
    else:
        assert np.max(np.abs(got - direct)) <= 2e-4


def test_nan_input_propagates_in_both_exact_evaluators(tnrd):
    c = tnrd_gen.make_small(54, 1, 40, 40, 1, 3, 5)
    c["f"][0, 20, 20] = np.nan; c["u0"] = c["f"].copy()
    for mode in (0, 3):
        got = run_gpu_mode(tnrd, c, phi_mode=mode)[0]
        assert np.isnan(got[20, 20]) and np.isnan(got[18:23, 18:23]).all(), mode     # inside the 5x5 footprint
        assert np.isfinite(got[:10, :10]).all(), mode


# --- small-image path: the filter bank of a tile split over several CTAs (tnrd_fused.cu, nsplit > 1) ------------
@pytest.mark.parametrize("tile", [1, 2, 3])
@pytest.mark.parametrize("split", [1, 2, 3, 7])
def test_filter_split_matches_oracle_and_is_deterministic(tnrd, tile, split, monkeypatch):
    c = tnrd_gen.make_small(41, 2, 70, 150, 2, 7, 7)
    want = run_oracle(c)
    monkeypatch.setenv("TNRD_TILE", str(tile))
    monkeypatch.setenv("TNRD_SPLIT", str(split))
    a = run_gpu(tnrd, c, kernel=2)
    b = run_gpu(tnrd, c, kernel=2)
    check(a, want, f"tile {tile} split {split}")
    assert np.array_equal(a, b), "partial sums are added in fixed order: run-to-run identical"


def test_filter_split_auto_plan_on_single_paper_image(tnrd):
    """A single 321x481 image (C3) does not fill 148 SMs with whole-bank tiles: the planner splits the bank; the
    result must not depend on it (same tolerance against the oracle as the forced no-split plan)."""
    c = tnrd_gen.make_config(3)
    want = run_oracle(c, T=2)
    check(run_gpu(tnrd, c, T=2), want, "C3 auto plan")


# --- piecewise-linear table evaluator: lookup table of the Gaussian phi and the triangular basis ------
def run_gpu_mode(tnrd, c, phi_mode=3, basis=0, **kw):
    tnrd.tnrd_set_phi_mode(phi_mode)
    tnrd.tnrd_set_rbf_basis(basis)
    try:
        return run_gpu(tnrd, c, **kw)
    finally:
        tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)
        tnrd.tnrd_set_rbf_basis(0)


@pytest.mark.parametrize("case", [SMALL[1], SMALL[3], SMALL[5], SMALL[7], SMALL[8]], ids=lambda c: f"s{c[0]}")
def test_lut_phi_small_cases_within_tolerance(tnrd, case):
    """TNRD_PHI_LUT approximates Main Eq. 6 (4096 nodes, linear interpolation): same tolerance against the SAME oracle."""
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    check(run_gpu_mode(tnrd, c, phi_mode=2), run_oracle(c), f"lut {case}")


def test_lut_phi_config3_and_distance_from_dense(tnrd):
    c = tnrd_gen.make_config(3)
    want = run_oracle(c)
    lut = run_gpu_mode(tnrd, c, phi_mode=2)
    mx, rms = check(lut, want, "lut C3")
    d = np.max(np.abs(lut - run_gpu(tnrd, c)))
    print(f"C3 lookup-table phi: max-abs {mx:.3e} rms {rms:.3e} vs oracle; {d:.3e} from the dense GPU result")
    assert d <= 5e-3


def run_oracle_triangle(c, T=None):
    with oracle.basis(oracle.TRIANGLE):
        return run_oracle(c, T)


@pytest.mark.parametrize("case", [SMALL[0], SMALL[1], SMALL[3], SMALL[5], SMALL[7], SMALL[8], SMALL[11]],
                         ids=lambda c: f"s{c[0]}")
def test_triangular_basis_exact_table(tnrd, case):
    """gamma = spacing of the centres: phi_t is the linear interpolant of the weights, 65-node table."""
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    assert c["rbf_gamma"] == float(c["rbf_mu"][1] - c["rbf_mu"][0])
    check(run_gpu_mode(tnrd, c, basis=1), run_oracle_triangle(c), f"triangle {case}")


def test_triangular_basis_config3_and_other_gamma(tnrd):
    c = tnrd_gen.make_config(3)
    mx, rms = check(run_gpu_mode(tnrd, c, basis=1), run_oracle_triangle(c), "triangle C3")
    print(f"C3 triangular basis: max-abs {mx:.3e} rms {rms:.3e}")
    # gamma != spacing: tabulated on the fine grid (kinks between nodes: approximate, still inside the tolerance)
    d = dict(tnrd_gen.make_small(61, 1, 60, 70, 2, 6, 5), rbf_gamma=7.0)
    check(run_gpu_mode(tnrd, d, basis=1), run_oracle_triangle(d), "triangle gamma 7")
    # the Gaussian default is restored afterwards
    check(run_gpu(tnrd, d), run_oracle(d), "gaussian after triangle")


def test_triangular_basis_unsupported_paths(tnrd):
    c = tnrd_gen.make_small(62, 1, 20, 20, 1, 3, 3)
    with pytest.raises(tnrd.TnrdError) as ei:
        run_gpu_mode(tnrd, c, basis=1, kernel=1)
    assert ei.value.status == tnrd.ERR_UNSUPPORTED
    tnrd.tnrd_set_rbf_basis(1)
    try:
        f = dev(c["f"])
        with pytest.raises(tnrd.TnrdError) as ei:
            tnrd.tnrd_stage_backward(f, f, f, 1, 20, 20, 3, 3, dev(c["filters"][0]), dev(c["rbf_w"][0]), dev(c["rbf_mu"]),
                                     10.0, 0.1, grad_w=torch.empty((3, 63), device="cuda"))
        assert ei.value.status == tnrd.ERR_UNSUPPORTED
    finally:
        tnrd.tnrd_set_rbf_basis(0)
        tnrd.tnrd_set_kernel(0)


# --- extreme aspect ratios: more than 65535 rows in the batch (the update kernel folds rows over grid.y and grid.z) -----
def test_many_rows_tall_image_and_large_batch(tnrd):
    tall = tnrd_gen.make_small(71, 1, 70000, 8, 1, 3, 3)
    got = run_gpu(tnrd, tall)[0]
    assert np.all(np.isfinite(got))
    for y0 in (0, 33000, 65530, 70000 - 24):
        want = oracle.diffuse_window(tall["f"][0], tall["u0"][0], tall["filters"], tall["rbf_w"], tall["rbf_mu"],
                                     tall["rbf_gamma"], tall["lambda"], y0, 0, 24, 8)
        check(got[y0:y0 + 24, :], want, f"tall image rows {y0}")
    many = tnrd_gen.make_small(72, 1200, 60, 9, 1, 2, 5)           # 72000 rows in the batch
    gotb = run_gpu(tnrd, many)
    for b in (0, 1091, 1092, 1199):                                 # around row 65535 and the last image
        one = dict(many, B=1, f=many["f"][b:b + 1], u0=many["u0"][b:b + 1])
        check(gotb[b:b + 1], run_oracle(one), f"batch image {b}")


# --- seeded random shapes, every evaluator: ragged tiles, images smaller than a tile, images of a few tiles ------------
def _random_cases(n):
    r = np.random.default_rng([150305768, 99])
    out = []
    for i in range(n):
        K = int(r.choice([3, 5, 7, 9]))
        lo = K - 1
        H, W = int(r.integers(lo, 160)), int(r.integers(lo, 260))
        out.append((100 + i, int(r.integers(1, 4)), H, W, int(r.integers(1, 4)), int(r.integers(1, 11)), K))
    return out


@pytest.mark.parametrize("case", _random_cases(18), ids=lambda c: f"r{c[0]}-{c[1]}x{c[2]}x{c[3]}-k{c[6]}")
def test_random_shapes_all_evaluators(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    want = run_oracle(c)
    check(run_gpu(tnrd, c), want, f"dense {case}")
    check(run_gpu_mode(tnrd, c, phi_mode=1), want, f"window {case}")
    check(run_gpu_mode(tnrd, c, phi_mode=2), want, f"lut {case}")
    check(run_gpu_mode(tnrd, c, basis=1), run_oracle_triangle(c), f"triangle {case}")


# --- one image as row slabs with a 2 r T overlap (multi-GPU strong-scaling mode of bench.py, run here on one GPU) ------
def test_row_slabs_with_overlap_match_the_full_image(tnrd):
    from paper_1503_05768_b200.shard import slab_bounds
    c = tnrd_gen.make_config(4, size=1024, T=5)
    full = run_gpu(tnrd, c)[0]
    stitched = np.empty_like(full)
    for rank in range(3):
        lo, hi, s0, s1 = slab_bounds(1024, rank, 3, c["T"], c["ksize"])
        part = run_gpu(tnrd, dict(c, H=s1 - s0, f=np.ascontiguousarray(c["f"][:, s0:s1]),
                                  u0=np.ascontiguousarray(c["u0"][:, s0:s1])))[0]
        stitched[lo:hi] = part[lo - s0:hi - s0]
    assert np.max(np.abs(stitched - full)) <= 2e-4          # other tiles, other partial-sum boundaries: fp32 rounding
    y0 = slab_bounds(1024, 1, 3, c["T"], c["ksize"])[0] - 12  # a window across the first slab seam against the oracle
    want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"],
                                 y0, 500, 24, 24)
    check(stitched[y0:y0 + 24, 500:524], want, "slab seam")


# --- a large single image: 16384 x 16384 (2^28 pixels, 1 GiB per plane; the API limit is B*H*W < 2^31) --------------------
def test_large_image_16384_sampled_windows(tnrd):
    c = tnrd_gen.make_config(4, size=4096, T=5)
    T, n = 2, 16384
    f = np.tile(c["f"][0], (4, 4))
    f += np.random.default_rng(5).standard_normal(f.shape, dtype=np.float32)      # break the periodicity
    df = torch.from_numpy(f).cuda()
    out = torch.empty_like(df)
    tnrd.tnrd_diffuse(df, df, 1, n, n, T, c["N_k"], c["ksize"], dev(c["filters"][:T]), dev(c["rbf_w"][:T]), dev(c["rbf_mu"]),
                      c["rbf_gamma"], dev(c["lambda"][:T]), out)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all())
    for (y0, x0) in [(0, 0), (n - 24, n - 24), (n // 2, n // 2), (n - 24, 0), (12345, n - 24), (n - 3000, 7777)]:
        want = oracle.diffuse_window(f, f, c["filters"][:T], c["rbf_w"][:T], c["rbf_mu"], c["rbf_gamma"], c["lambda"][:T],
                                     y0, x0, 24, 24)
        check(out[y0:y0 + 24, x0:x0 + 24].cpu().numpy().astype(np.float64), want, f"16384^2 window {(y0, x0)}")
    del df, out
    torch.cuda.empty_cache()


# --- run-to-run determinism at a size with many tiles, a split wave tail and every evaluator (no float atomics anywhere;
# compute-sanitizer is not available on this pool, so a shared-memory race would have to show up here) -----------------
@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_bitwise_determinism_2048(tnrd, mode):
    c = tnrd_gen.make_config(4, size=2048, T=5)
    f = dev(c["f"])
    k, w, mu, lam = dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"]), dev(c["lambda"])
    outs = []
    tnrd.tnrd_set_phi_mode(mode)
    try:
        for _ in range(4):
            out = torch.empty_like(f)
            tnrd.tnrd_diffuse(f, f, 1, 2048, 2048, 5, c["N_k"], c["ksize"], k, w, mu, c["rbf_gamma"], lam, out)
            outs.append(out)
        torch.cuda.synchronize()
    finally:
        tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)
    assert all(torch.equal(outs[0], o) for o in outs[1:])


# --- the opt-in evaluators at the size bench.py times (4096^2, T = 5): sampled windows against the oracle --------------
@pytest.mark.parametrize("mode,basis", [(0, 0), (1, 0), (2, 0), (0, 1)], ids=["direct", "window", "lut", "triangle"])
def test_evaluators_4096_sampled_windows(tnrd, mode, basis):
    c = tnrd_gen.make_config(4, size=4096, T=5)
    got = run_gpu_mode(tnrd, c, phi_mode=mode, basis=basis)[0]
    assert np.all(np.isfinite(got))
    worst = 0.0
    for (y0, x0) in _windows(4096, 4096, 24, 2, 11)[::2] + [(122 * 17 - 3 - 12, 122 * 5 - 3 - 12)]:
        with oracle.basis(oracle.TRIANGLE if basis else oracle.GAUSSIAN):
            want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                                         c["lambda"], y0, x0, 24, 24)
        mx, _ = check(got[y0:y0 + 24, x0:x0 + 24], want, f"4096^2 mode {mode} basis {basis} window {(y0, x0)}")
        worst = max(worst, mx)
    print(f"4096^2 phi mode {mode} basis {basis}: worst window max-abs {worst:.3e}")
