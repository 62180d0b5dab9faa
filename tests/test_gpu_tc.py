"""GPU parity of the tensor-core stage kernel (tnrd_set_kernel(3), csrc/tnrd_tc.cu) against the double-precision CPU
oracle, and the full-size configs C4 / C5 of BASELINE.json in the launch configuration bench.py times (automatic kernel
choice).  Tolerance: north_star's max-abs <= 1e-2 / RMS <= 1e-3, plus the regression bound of the exact evaluators."""
import numpy as np
import pytest

import oracle
import tnrd_gen
from test_gpu_parity import check, dev, run_gpu, run_oracle, _windows

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


def num_sms():
    return torch.cuda.get_device_properties(0).multi_processor_count


# seed, B, H, W, T, N_k, ksize: one strip / several strips (250 resp. 252 output columns each), ragged last strip, images
# smaller than a strip, odd widths, filter counts that are not multiples of 8 (padded), the largest bank
TC_CASES = [
    (201, 1, 6, 6, 1, 5, 7), (202, 2, 70, 50, 2, 8, 7), (203, 1, 131, 140, 1, 5, 7), (204, 1, 97, 531, 2, 48, 7),
    (205, 1, 37, 600, 1, 24, 7), (206, 3, 37, 23, 2, 6, 5), (207, 1, 90, 300, 2, 24, 5), (208, 1, 4, 4, 2, 4, 5),
    (209, 1, 33, 251, 1, 9, 7), (210, 1, 40, 250, 1, 16, 7), (211, 1, 25, 253, 1, 3, 5), (212, 2, 61, 757, 1, 40, 7),
    (213, 1, 300, 8, 1, 1, 7),
]


@pytest.mark.parametrize("case", TC_CASES, ids=[f"t{c[0]}" for c in TC_CASES])
def test_tc_small_cases_match_oracle(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    check(run_gpu(tnrd, c, kernel=3), run_oracle(c), f"tc case {case}", tight=True)


@pytest.mark.parametrize("seg", [1, 2, 3, 7, 24])
def test_tc_row_segments_match_oracle_and_each_other(tnrd, seg, monkeypatch):
    """Row segments of every height (TNRD_TC_SEG), including one and two output rows per CTA: each CTA recomputes the 2r
    phi rows above and below its segment."""
    c = tnrd_gen.make_small(220, 2, 53, 280, 2, 8, 7)
    want = run_oracle(c)
    monkeypatch.setenv("TNRD_TC_SEG", str(seg))
    pl = tnrd.tnrd_tc_plan_query(2, 53, 280, 8, 7, num_sms())
    assert pl["seg_rows"] == seg and pl["nys"] == -(-53 // seg) and pl["nxs"] == 2
    a = run_gpu(tnrd, c, kernel=3)
    check(a, want, f"tc seg {seg}", tight=True)
    assert np.array_equal(a, run_gpu(tnrd, c, kernel=3)), "run-to-run identical"


def test_tc_agrees_with_the_tile_kernel(tnrd):
    c = tnrd_gen.make_config(3)
    a, b = run_gpu(tnrd, c, kernel=3), run_gpu(tnrd, c, kernel=2)
    assert np.max(np.abs(a - b)) <= 2e-4               # fp32 rounding: both are ~3e-5 from the oracle
    check(a, run_oracle(c), "tc C3", tight=True)
    c2 = tnrd_gen.make_config(2)                        # 24 filters 5x5
    check(run_gpu(tnrd, c2, kernel=3), run_oracle(c2), "tc C2", tight=True)


def test_tc_unsupported_shapes_and_modes(tnrd):
    for K, n_k in ((3, 8), (9, 4), (7, 49)):
        c = tnrd_gen.make_small(230, 1, 40, 40, 1, n_k, K)
        assert tnrd.tnrd_tc_plan_query(1, 40, 40, n_k, K)["applies"] == 0
        with pytest.raises(tnrd.TnrdError) as ei:
            run_gpu(tnrd, c, kernel=3)
        assert ei.value.status == tnrd.ERR_UNSUPPORTED
        tnrd.tnrd_set_kernel(0)
        check(run_gpu(tnrd, c), run_oracle(c), "automatic choice still works")
    c = tnrd_gen.make_small(231, 1, 40, 40, 1, 8, 7)
    for mode in (tnrd.PHI_DENSE, tnrd.PHI_WINDOW, tnrd.PHI_LUT):
        tnrd.tnrd_set_phi_mode(mode)
        try:
            with pytest.raises(tnrd.TnrdError) as ei:
                run_gpu(tnrd, c, kernel=3)
            assert ei.value.status == tnrd.ERR_UNSUPPORTED
        finally:
            tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)
            tnrd.tnrd_set_kernel(0)


def test_tc_diffuse_equals_repeated_stage_and_inplace(tnrd):
    for T in (1, 2, 3, 4):
        c = tnrd_gen.make_small(240 + T, 2, 33, 47, T, 8, 7)
        ref = run_gpu(tnrd, c, kernel=3)
        tnrd.tnrd_set_kernel(3)
        try:
            f, u = dev(c["f"]), dev(c["u0"])
            k, w, mu = dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"])
            for t in range(T):
                nxt = torch.empty_like(u)
                tnrd.tnrd_stage(f, u, 2, 33, 47, 8, 7, k[t], w[t], mu, c["rbf_gamma"], float(c["lambda"][t]), nxt)
                u = nxt
            torch.cuda.synchronize()
            assert np.array_equal(u.cpu().numpy().astype(np.float64), ref), f"T={T}: diffuse != T x stage"
            v = dev(c["u0"])                                    # tnrd_stage in place: u_out == u_in (ping-pong + copy)
            for t in range(T):
                tnrd.tnrd_stage(f, v, 2, 33, 47, 8, 7, k[t], w[t], mu, c["rbf_gamma"], float(c["lambda"][t]), v)
            torch.cuda.synchronize()
            assert np.array_equal(v.cpu().numpy().astype(np.float64), ref), f"T={T}: in-place stage differs"
        finally:
            tnrd.tnrd_set_kernel(0)
        u0 = dev(c["u0"])                                       # tnrd_diffuse in place: out == u0, odd and even T
        assert np.array_equal(run_gpu(tnrd, c, kernel=3, out=u0, u0=u0), ref), f"T={T}: in-place differs"


@pytest.mark.parametrize("change", ["jitter", "narrow", "wide"])
def test_tc_other_centres_and_widths(tnrd, change):
    """Centres that are not equidistant, or gamma < 0.96 delta: the tensor-core kernel evaluates the direct form (one ex2
    per Gaussian) in the same launch; gamma = 1.4 delta stays factorised."""
    c = tnrd_gen.make_small(251, 2, 50, 61, 2, 5, 7)
    d = dict(c)
    if change == "jitter":
        mu = c["rbf_mu"].copy(); mu[10] += 2.0; d["rbf_mu"] = mu
    else:
        d["rbf_gamma"] = {"narrow": 8.0, "wide": 14.0}[change]
    check(run_gpu(tnrd, d, kernel=3), run_oracle(d), f"tc {change}", tight=True)


def test_tc_extreme_responses_large_weights_and_nan(tnrd):
    c = tnrd_gen.make_small(250, 1, 40, 44, 1, 6, 5)
    c["f"] = (c["f"] * 6.0 - 400.0).astype(np.float32); c["u0"] = c["f"].copy()     # z up to ~ +-1000
    w = c["rbf_w"].copy(); w[..., :3] = 0.5; w[..., -3:] = -0.5; c["rbf_w"] = w
    check(run_gpu(tnrd, c, kernel=3), run_oracle(c), "tc extreme")
    c = tnrd_gen.make_small(253, 1, 48, 52, 1, 5, 7)
    c["rbf_w"] = (c["rbf_w"] * 1e4).astype(np.float32)
    want = run_oracle(c)
    got = run_gpu(tnrd, c, kernel=3)
    assert np.all(np.isfinite(got))
    scale = float(np.max(np.abs(want - c["f"].astype(np.float64))))
    assert np.max(np.abs(got - want)) <= 5e-5 * scale, "relative to the size of the update"
    c = tnrd_gen.make_small(254, 1, 40, 300, 1, 3, 5)
    c["f"][0, 20, 20] = np.nan; c["u0"] = c["f"].copy()
    got = run_gpu(tnrd, c, kernel=3)[0]
    assert np.isnan(got[20, 20]) and np.isnan(got[18:23, 18:23]).all()                # at least the 5x5 footprint ...
    assert np.isfinite(got[:8, :]).all() and np.isfinite(got[33:, :]).all()          # ... and nothing beyond 2r rows
    assert np.isfinite(got[:, :8]).all() and np.isfinite(got[:, 40:]).all()          # and the 8-column windows around it


def test_tc_deblocking_matches_oracle(tnrd):
    c = tnrd_gen.make_deblock(seed=5, B=2, H=64, W=264, T=3, n_k=8, ksize=7)
    want = oracle.deblock_diffuse(c["u0"], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["qcs_lo"], c["qcs_hi"])
    tnrd.tnrd_set_kernel(3)
    try:
        u0 = dev(c["u0"])
        for out in (torch.empty_like(u0), u0):                   # out of place, in place (T odd: u0 is copied first)
            tnrd.tnrd_deblock_diffuse(dev(c["u0"]) if out is not u0 else u0, 2, 64, 264, 3, 8, 7, dev(c["filters"]),
                                      dev(c["rbf_w"]), dev(c["rbf_mu"]), c["rbf_gamma"], dev(c["qcs_lo"]),
                                      dev(c["qcs_hi"]), out)
            torch.cuda.synchronize()
            check(out.cpu().numpy().astype(np.float64), want, "tc deblock")
    finally:
        tnrd.tnrd_set_kernel(0)


# --- BASELINE.json configs[3] and [4] at full size, automatic kernel choice (the tensor-core kernel) --------------------
def _seams(tnrd, size, T):
    """Windows across the first strip seam / row-segment seam of the plan the library uses for this shape."""
    pl = tnrd.tnrd_tc_plan_query(1, size, size, 48, 7, num_sms())
    assert pl["applies"] == 2, "the automatic choice at this size is the tensor-core kernel"
    xs, ys = pl["out_cols"], pl["seg_rows"]
    return [(ys - 12, xs - 12), (min(size - 24, 3 * ys - 12), min(size - 24, 5 * xs - 12)), (size - 24, xs - 12)]


@pytest.mark.parametrize("size,T", [(2048, 5), (2048, 8), (4096, 8)])
def test_config4_remaining_sizes_sampled_windows(tnrd, size, T):
    """BASELINE.json configs[3]: 2048^2 with the default evaluator at T = 5 and T = 8, 4096^2 at T = 8 (4096^2 T = 5 and
    1024^2 are in test_gpu_parity.py / below)."""
    c = tnrd_gen.make_config(4, size=size, T=T)
    got = run_gpu(tnrd, c)[0]
    assert np.all(np.isfinite(got))
    worst = 0.0
    for (y0, x0) in _windows(size, size, 24, 2, size + T)[::2] + _seams(tnrd, size, T):
        want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                                     c["lambda"], y0, x0, 24, 24)
        mx, _ = check(got[y0:y0 + 24, x0:x0 + 24], want, f"C4 {size}^2 T={T} window {(y0, x0)}", tight=True)
        worst = max(worst, mx)
    print(f"config 4 ({size}^2, T={T}): worst window max-abs {worst:.3e}")


def test_config4_4096_T5_seams_of_the_tc_plan(tnrd):
    c = tnrd_gen.make_config(4, size=4096, T=5)
    got = run_gpu(tnrd, c)[0]
    for (y0, x0) in _seams(tnrd, 4096, 5):
        want = oracle.diffuse_window(c["f"][0], c["u0"][0], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                                     c["lambda"], y0, x0, 24, 24)
        check(got[y0:y0 + 24, x0:x0 + 24], want, f"C4 4096^2 T=5 seam {(y0, x0)}", tight=True)


def test_config4_1024_full_image_T8_and_T5_prefix(tnrd):
    """full-image oracle parity is mandatory for C4-1024^2.  One oracle run gives u_5 (the T = 5 model is
    the first five stages of the T = 8 parameter set) and, continued in double precision, u_8."""
    c = tnrd_gen.make_config(4, size=1024, T=8)
    want5 = run_oracle(c, T=5)
    want8 = oracle.diffuse(c["f"], want5, c["filters"][5:], c["rbf_w"][5:], c["rbf_mu"], c["rbf_gamma"], c["lambda"][5:])
    m5, r5 = check(run_gpu(tnrd, c, T=5), want5, "C4 1024^2 T=5 full image", tight=True)
    m8, r8 = check(run_gpu(tnrd, c, T=8), want8, "C4 1024^2 T=8 full image", tight=True)
    print(f"config 4 (1024^2) full image: T=5 max-abs {m5:.3e} rms {r5:.3e}; T=8 max-abs {m8:.3e} rms {r8:.3e}")
    for kernel in (2, 3):                                        # both stage kernels at this size, full image
        check(run_gpu(tnrd, c, T=5, kernel=kernel), want5, f"C4 1024^2 T=5 kernel {kernel}", tight=True)


def test_config5_eight_full_images(tnrd):
    """>= 8 images of C5 compared in full (the batch is run as BASELINE.json configs[4] states it: 128
    images at once)."""
    c = tnrd_gen.make_config(5)
    got = run_gpu(tnrd, c)
    worst = 0.0
    for b in (0, 1, 17, 42, 63, 64, 100, 127):
        want = oracle.diffuse(c["f"][b], c["u0"][b], c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"])
        mx, _ = check(got[b], want, f"C5 image {b} in full", tight=True)
        worst = max(worst, mx)
    print(f"config 5: worst of 8 full images max-abs {worst:.3e}")


def test_automatic_kernel_choice(tnrd):
    n = num_sms()
    assert tnrd.tnrd_tc_plan_query(1, 4096, 4096, 48, 7, n)["applies"] == 2
    assert tnrd.tnrd_tc_plan_query(128, 321, 481, 48, 7, n)["applies"] == 2
    q = tnrd.tnrd_tc_plan_query(1, 321, 481, 48, 7, n)                          # one small image: the bank cut in chunks
    assert q["applies"] == 2 and q["nchunk"] > 1 and q["units"] == q["nxs"] * q["nys"] * q["nchunk"]
    assert tnrd.tnrd_tc_plan_query(1, 1024, 1024, 48, 7, n)["nchunk"] == 1
    assert tnrd.tnrd_tc_plan_query(1, 200, 150, 48, 7, n)["applies"] == 1       # narrower than a strip: the tile kernel
    assert tnrd.tnrd_tc_plan_query(1, 64, 64, 8, 3, n)["applies"] == 0
    # launch count: one staging kernel + the operand kernel + one stage kernel per stage
    c = tnrd_gen.make_config(4, size=1024, T=5)
    tnrd.tnrd_reset_launch_count()
    run_gpu(tnrd, c)
    assert tnrd.tnrd_launch_count() == 2 + c["T"]
    # with a split bank each stage is the tensor-core kernel plus the kernel that sums the chunks' partial updates
    c = tnrd_gen.make_small(262, 1, 321, 481, 3, 48, 7)
    tnrd.tnrd_reset_launch_count()
    run_gpu(tnrd, c)
    assert tnrd.tnrd_launch_count() == 2 + 2 * c["T"]


@pytest.mark.parametrize("nchunk,N_k,ksize", [(2, 48, 7), (3, 48, 7), (6, 48, 7), (3, 24, 5), (2, 16, 7)])
def test_filter_chunks(tnrd, monkeypatch, nchunk, N_k, ksize):
    """The filter bank cut into chunks (units = chunks x segments x strips, partial updates summed by a second kernel):
    same bound against the oracle as the whole bank, identical from run to run, equal to the whole bank up to the order
    of the sum over filters, and legal in place (the partial sums live in scratch)."""
    B, H, W, T = 2, 77, 300, 3
    c = tnrd_gen.make_small(263 + nchunk, B, H, W, T, N_k, ksize)
    want = run_oracle(c)
    monkeypatch.setenv("TNRD_TC_CHUNK", "1")
    whole = run_gpu(tnrd, c, kernel=3)
    monkeypatch.setenv("TNRD_TC_CHUNK", str(nchunk))
    got = run_gpu(tnrd, c, kernel=3)
    assert np.array_equal(got, run_gpu(tnrd, c, kernel=3))
    check(got, want, f"tc chunks {nchunk}", tight=True)
    assert np.max(np.abs(got - whole)) <= 6.2e-5          # 4 ulp at 255: only the order of the sum over filters differs
    tnrd.tnrd_set_kernel(3)
    try:
        f, v = dev(c["f"]), dev(c["u0"])
        k, w, mu = dev(c["filters"]), dev(c["rbf_w"]), dev(c["rbf_mu"])
        for t in range(T):
            tnrd.tnrd_stage(f, v, B, H, W, N_k, ksize, k[t], w[t], mu, c["rbf_gamma"], float(c["lambda"][t]), v)
        torch.cuda.synchronize()
        assert np.array_equal(v.cpu().numpy().astype(np.float64), got), "in-place stage with chunks differs"
    finally:
        tnrd.tnrd_set_kernel(0)


def test_nearly_equidistant_centres_take_the_direct_form(tnrd):
    """Centres jittered by 5e-5 of their spacing are NOT equidistant to rounding: both stage kernels must evaluate the
    direct form with the centres as given (the factorised identity would silently move them onto the ideal grid)."""
    c = tnrd_gen.make_small(260, 1, 60, 270, 2, 8, 7)
    r = np.random.default_rng(3)
    mu = (c["rbf_mu"].astype(np.float64) + 5e-5 * 10.0 * r.uniform(-1, 1, 63)).astype(np.float32)
    big = dict(c, rbf_mu=mu, rbf_w=(c["rbf_w"] * 40.0).astype(np.float32))      # large weights make a moved centre visible
    want = run_oracle(big)
    scale = float(np.max(np.abs(want - big["f"].astype(np.float64))))
    for kernel in (2, 3):
        got = run_gpu(tnrd, big, kernel=kernel)
        assert np.max(np.abs(got - want)) <= 1.5e-5 * scale, kernel         # fp32 level, relative to the update
    tnrd.tnrd_set_phi_mode(0)
    try:
        direct = run_gpu(tnrd, big, kernel=2)
    finally:
        tnrd.tnrd_set_phi_mode(tnrd.PHI_FACTORED)
    assert np.array_equal(run_gpu(tnrd, big, kernel=2), direct), "same launch, direct form"


def test_phi_statistics_counters(tnrd, monkeypatch):
    """tnrd_phi_stats: executed <= defined, defined = 5 groups x filters x warps x stages; results unchanged by counting;
    a constant image (z = 0) leaves 2 of 5 groups executed."""
    c = tnrd_gen.make_small(261, 1, 64, 500, 2, 16, 7)
    monkeypatch.setenv("TNRD_TC_SEG", "16")
    ref = run_gpu(tnrd, c, kernel=3)
    tnrd.tnrd_phi_stats(True)
    got = run_gpu(tnrd, c, kernel=3)
    ex, de = tnrd.tnrd_phi_stats(False)
    assert np.array_equal(got, ref)
    pl = tnrd.tnrd_tc_plan_query(1, 64, 500, 16, 7, num_sms())
    batches = (pl["seg_rows"] + 6 + 1) // 2                    # per unit (every segment has seg_rows rows here)
    assert 64 % pl["seg_rows"] == 0
    assert pl["units"] == pl["nxs"] * pl["nys"] * pl["nchunk"]      # a unit of a split bank counts its own filters only
    assert de == 5 * 16 * 4 * batches * pl["nxs"] * pl["nys"] * c["T"], "5 groups x filters x lane quarters x batches x strips x segments x stages"
    assert 0 < ex <= de
    flat = dict(c, f=np.full_like(c["f"], 100.0), u0=np.full_like(c["f"], 100.0))     # z = 0 everywhere
    tnrd.tnrd_phi_stats(True)
    run_gpu(tnrd, flat, kernel=3, T=1)
    ex, de = tnrd.tnrd_phi_stats(False)
    assert 5 * ex == 2 * de, "z = 0 is within reach (133) of the anchors at -110 and 20 only"
    run_gpu(tnrd, c, kernel=3)
    assert tnrd.tnrd_phi_stats(False) == (0, 0), "counting is off"


def test_non_finite_weights_are_unspecified_but_harmless(tnrd):
    """include/tnrd.h: rbf_w must be finite.  An infinite weight on a centre no response comes near is skipped with its
    group, so every output pixel is either non-finite or the result with that weight zeroed; nothing faults."""
    c = tnrd_gen.make_small(262, 1, 40, 260, 1, 8, 7)
    w = c["rbf_w"].copy(); w[:, :, 62] = np.inf
    w0 = c["rbf_w"].copy(); w0[:, :, 62] = 0.0
    for kernel in (2, 3):
        got = run_gpu(tnrd, dict(c, rbf_w=w), kernel=kernel)
        ref = run_gpu(tnrd, dict(c, rbf_w=w0), kernel=kernel)
        ok = ~np.isfinite(got) | (np.abs(got - ref) <= 1e-4)
        assert ok.all(), kernel


def test_two_devices_in_one_process(tnrd):
    """The opt-in shared-memory attribute is per device: the first call on a second GPU must work."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    c = tnrd_gen.make_small(263, 1, 80, 300, 2, 8, 7)
    want = run_oracle(c)
    for kernel in (2, 3):
        with torch.cuda.device(1):
            tnrd.tnrd_set_kernel(kernel)
            try:
                f = torch.from_numpy(c["f"]).cuda(1)
                out = torch.empty_like(f)
                d1 = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda(1)   # noqa: E731
                tnrd.tnrd_diffuse(f, f, 1, 80, 300, 2, 8, 7, d1(c["filters"]), d1(c["rbf_w"]), d1(c["rbf_mu"]),
                                  c["rbf_gamma"], d1(c["lambda"]), out)
                torch.cuda.synchronize()
            finally:
                tnrd.tnrd_set_kernel(0)
            check(out.cpu().numpy().astype(np.float64), want, f"device 1 kernel {kernel}", tight=True)


@pytest.mark.parametrize("shape", [(1, 600, 520), (1, 257, 300), (5, 130, 300), (2, 64, 512), (1, 1500, 700), (1, 1024, 1024)],
                         ids=lambda s: "x".join(map(str, s)))
@pytest.mark.parametrize("T,ksize,mode", [(1, 7, 0), (2, 7, 0), (3, 7, 0), (3, 5, 0), (2, 7, 1), (2, 7, 2), (2, 7, 3)])
def test_host_entry_point_pipelined_is_bit_identical(tnrd, shape, T, ksize, mode, monkeypatch):
    """tnrd_diffuse_host with the tensor-core kernel overlaps the copies with the first and the last stage: a batch is cut
    in two halves; a single image arrives in blocks of 32 rows that the first stage's loaders wait for (arrival words),
    and the last stage stores into pinned host memory itself.  The result must be bit-identical to the device call.
    TNRD_HOST_MODE selects the variants (1: halves for a single image, 2: no stores to host memory, 3: input top to
    bottom)."""
    B, H, W = shape
    monkeypatch.setenv("TNRD_HOST_PIPE_MIN", "0")                    # small images take the serial path otherwise
    if mode:
        monkeypatch.setenv("TNRD_HOST_MODE", str(mode))
    c = tnrd_gen.make_small(270 + T, B, H, W, T, 8, ksize)
    ref = run_gpu(tnrd, c, kernel=3)
    tnrd.tnrd_set_kernel(3)
    try:
        out = torch.empty(c["f"].shape).pin_memory()
        f = torch.from_numpy(c["f"]).pin_memory()
        for _ in range(2):                                           # the arrival words are reset by every call
            out.zero_()
            tnrd.tnrd_diffuse_host(f, f, B, H, W, T, 8, ksize, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"], out)
            assert np.array_equal(out.numpy().astype(np.float64), ref)
        g = f.clone().pin_memory()                                   # in place on the host: out is the input buffer
        tnrd.tnrd_diffuse_host(g, g, B, H, W, T, 8, ksize, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"], g)
        assert np.array_equal(g.numpy().astype(np.float64), ref)
        out2 = np.empty_like(c["f"])                                 # pageable buffers, u0 distinct from f
        u0 = c["u0"].copy()
        tnrd.tnrd_diffuse_host(c["f"], u0, B, H, W, T, 8, ksize, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                               c["lambda"], out2)
        assert np.array_equal(out2.astype(np.float64), ref)
    finally:
        tnrd.tnrd_set_kernel(0)


def test_host_entry_point_single_image_with_a_split_bank(tnrd, monkeypatch):
    """A single image small enough for the planner to cut the filter bank: the first stage of the host call must cut it
    the way the device call does (the order of the sum over filters), so the two stay bit-identical."""
    monkeypatch.setenv("TNRD_HOST_PIPE_MIN", "0")
    c = tnrd_gen.make_small(281, 1, 321, 481, 3, 48, 7)
    assert tnrd.tnrd_tc_plan_query(1, 321, 481, 48, 7, num_sms())["nchunk"] > 1
    ref = run_gpu(tnrd, c)
    out = torch.empty(c["f"].shape).pin_memory()
    f = torch.from_numpy(c["f"]).pin_memory()
    tnrd.tnrd_diffuse_host(f, f, 1, 321, 481, 3, 48, 7, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"], out)
    assert np.array_equal(out.numpy().astype(np.float64), ref)


@pytest.mark.parametrize("shape,T", [((1, 321, 481), 3), ((3, 100, 260), 1), ((1, 600, 520), 2)], ids=lambda v: str(v))
def test_host_entry_point_serial_path_stores_into_pinned_memory(tnrd, shape, T):
    """Below the pipelining threshold the host call uploads, runs the stages and -- with the tensor-core kernel and a pinned
    result buffer -- lets the last stage store u_T into host memory; pageable buffers get a copy.  Bit-identical."""
    B, H, W = shape
    c = tnrd_gen.make_small(290 + T, B, H, W, T, 16, 7)
    ref = run_gpu(tnrd, c, kernel=3)
    tnrd.tnrd_set_kernel(3)
    try:
        f = torch.from_numpy(c["f"]).pin_memory()
        out = torch.zeros(c["f"].shape).pin_memory()
        tnrd.tnrd_diffuse_host(f, f, B, H, W, T, 16, 7, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"], out)
        assert np.array_equal(out.numpy().astype(np.float64), ref)
        out2 = np.zeros_like(c["f"])
        tnrd.tnrd_diffuse_host(c["f"], c["u0"].copy(), B, H, W, T, 16, 7, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"],
                               c["lambda"], out2)
        assert np.array_equal(out2.astype(np.float64), ref)
        g = f.clone().pin_memory()                                   # in place on the host
        tnrd.tnrd_diffuse_host(g, g, B, H, W, T, 16, 7, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"], g)
        assert np.array_equal(g.numpy().astype(np.float64), ref)
    finally:
        tnrd.tnrd_set_kernel(0)


def test_host_entry_point_repeated_calls_of_changing_shapes(tnrd):
    """The pipelined host paths at their natural sizes (above the two-million-pixel threshold), called again and again with
    changing shapes: the arrival words, the pinned snapshots and the scratch planes are reused and regrown between calls, and
    every result must equal the device call's bit for bit."""
    shapes = [(1, 1500, 1500), (1, 1100, 2000), (2, 1024, 1100), (1, 2100, 1030), (6, 600, 640)]
    cases = []
    for k, (B, H, W) in enumerate(shapes):
        c = tnrd_gen.make_small(300 + k, B, H, W, 2, 8, 7)
        cases.append((c, run_gpu(tnrd, c, kernel=3)))
    tnrd.tnrd_set_kernel(3)
    try:
        for rep in range(3):
            for c, ref in cases:
                f = torch.from_numpy(c["f"]).pin_memory()
                out = torch.zeros(c["f"].shape).pin_memory()
                tnrd.tnrd_diffuse_host(f, f, c["B"], c["H"], c["W"], 2, 8, 7, c["filters"], c["rbf_w"], c["rbf_mu"],
                                       c["rbf_gamma"], c["lambda"], out)
                assert np.array_equal(out.numpy().astype(np.float64), ref), (rep, c["B"], c["H"], c["W"])
    finally:
        tnrd.tnrd_set_kernel(0)


@pytest.mark.parametrize("kernel", [0, 2], ids=["tensor-core", "tile"])
def test_billion_pixel_image_sampled_windows(tnrd, kernel):
    """The size limit B*H*W < 2^31: one 36000 x 32000 image (1.15 G pixels, 4.6 GB per plane -- byte offsets beyond 2^32), T = 2,
    8 filters 7x7, on the tensor-core kernel and on the tile kernel (8 GB of partial sums); windows at the corners, the centre and beyond the 2^32-byte offset against the
    oracle.  The image comes from tnrd_gen.hash_image in row chunks; the oracle gets crops of it with a 2rT margin."""
    H, W, T, n_k, K = 36000, 32000, 2, 8, 7
    free, _ = torch.cuda.mem_get_info()
    if free < 24 * (1 << 30):
        pytest.skip("needs 24 GB of device memory")
    p = tnrd_gen.make_small(320, 1, 16, 16, T, n_k, K)              # parameters only
    f = torch.empty((1, H, W), dtype=torch.float32, device="cuda")
    for r0 in range(0, H, 2000):
        f[0, r0:r0 + 2000] = torch.from_numpy(tnrd_gen.hash_image(H, W, r0, min(H, r0 + 2000))).cuda()
    out = torch.empty_like(f)
    k, w, mu, lam = dev(p["filters"]), dev(p["rbf_w"]), dev(p["rbf_mu"]), dev(p["lambda"])
    tnrd.tnrd_set_kernel(kernel)
    try:
        tnrd.tnrd_diffuse(f, f, 1, H, W, T, n_k, K, k, w, mu, p["rbf_gamma"], lam, out)
        torch.cuda.synchronize()
    finally:
        tnrd.tnrd_set_kernel(0)
        tnrd.tnrd_shutdown()                                        # give the scratch (planes, partial sums) back
    assert tnrd.tnrd_tc_plan_query(1, H, W, n_k, K, num_sms())["applies"] == 2
    m = 2 * (K // 2) * T + 4
    wins = _windows(H, W, 24, 2, 99) + [(H - 30, W // 2), (33555, 17000)]       # row 33555: byte offset 2^32 and a bit
    worst = 0.0
    for (y0, x0) in wins:
        cy0, cy1, cx0, cx1 = max(0, y0 - m), min(H, y0 + 24 + m), max(0, x0 - m), min(W, x0 + 24 + m)
        crop = tnrd_gen.hash_image(H, W, cy0, cy1)[:, cx0:cx1]
        # the crop's border is the image border exactly where the window is within the margin of it
        assert (cy0 == 0 or y0 - cy0 == m) and (cx0 == 0 or x0 - cx0 == m)
        assert (cy1 == H or cy1 - (y0 + 24) == m) and (cx1 == W or cx1 - (x0 + 24) == m)
        want = oracle.diffuse_window(crop, crop, p["filters"], p["rbf_w"], p["rbf_mu"], p["rbf_gamma"], p["lambda"],
                                     y0 - cy0, x0 - cx0, 24, 24)
        got = out[0, y0:y0 + 24, x0:x0 + 24].cpu().numpy().astype(np.float64)
        mx, _ = check(got, want, f"billion-pixel window {(y0, x0)}", tight=True)
        worst = max(worst, mx)
    print(f"36000 x 32000, T = 2: worst window max-abs {worst:.3e}")
