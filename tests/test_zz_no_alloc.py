"""tnrd_stage_static (include/tnrd.h): the stage entry point that allocates nothing -- its scratch is a fixed device array
inside libtnrd.so -- against tnrd_stage with the same kernel, on two calls in a row, and against the oracle.  This file is
collected last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the others."""
import numpy as np
import pytest

import tnrd_gen
from test_gpu_parity import check, dev, run_oracle

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


def _stage_args(c, t, d):
    return (d["f"], d["u"], c["B"], c["H"], c["W"], c["N_k"], c["ksize"], d["k"][t], d["w"][t], d["mu"], c["rbf_gamma"],
            float(c["lambda"][t]))


@pytest.mark.parametrize("case", [(301, 2, 77, 300, 2, 48, 7), (302, 1, 50, 61, 2, 24, 5), (303, 3, 33, 47, 2, 8, 3),
                                  (304, 1, 40, 44, 2, 6, 9)], ids=lambda c: f"n{c[0]}")
def test_static_scratch_stage_matches_the_existing_path_twice(tnrd, case):
    seed, B, H, W, T, n_k, K = case
    c = tnrd_gen.make_small(seed, B, H, W, T, n_k, K)
    want = run_oracle(c)
    d = {"f": dev(c["f"]), "u": dev(c["u0"]), "k": dev(c["filters"]), "w": dev(c["rbf_w"]), "mu": dev(c["rbf_mu"])}
    # the existing path with the same kernel (the tile kernel): T stages through tnrd_stage
    tnrd.tnrd_set_kernel(2)
    try:
        ref = d["u"]
        for t in range(T):
            nxt = torch.empty_like(ref)
            tnrd.tnrd_stage(*_stage_args(c, t, dict(d, u=ref)), nxt)
            ref = nxt
        torch.cuda.synchronize()
    finally:
        tnrd.tnrd_set_kernel(0)
    ref = ref.cpu().numpy().astype(np.float64)
    # two calls in a row per run (stage 1, stage 2: the second finds the first one's scratch contents), and the whole
    # run twice; between the runs a call of another shape dirties the array
    for rep in range(2):
        u = d["u"]
        for t in range(T):
            nxt = torch.empty_like(u)
            tnrd.tnrd_stage_static(*_stage_args(c, t, dict(d, u=u)), nxt)
            u = nxt
        torch.cuda.synchronize()
        got = u.cpu().numpy().astype(np.float64)
        assert np.array_equal(got, ref), f"run {rep}: same kernel, same arithmetic"
        check(got, want, f"static {case} run {rep}", tight=True)
        o = tnrd_gen.make_small(399, 1, 90, 130, 1, 16, 7)
        od = {"f": dev(o["f"]), "u": dev(o["u0"]), "k": dev(o["filters"]), "w": dev(o["rbf_w"]), "mu": dev(o["rbf_mu"])}
        tnrd.tnrd_stage_static(*_stage_args(o, 0, od), torch.empty_like(od["u"]))
    # in place (u_out == u_in), as tnrd_stage allows
    v = d["u"].clone()
    for t in range(T):
        tnrd.tnrd_stage_static(*_stage_args(c, t, dict(d, u=v)), v)
    torch.cuda.synchronize()
    assert np.array_equal(v.cpu().numpy().astype(np.float64), ref)


def test_static_scratch_stage_allocates_nothing_and_knows_its_limit(tnrd):
    c = tnrd_gen.make_small(310, 1, 128, 256, 1, 48, 7)
    d = {"f": dev(c["f"]), "u": dev(c["u0"]), "k": dev(c["filters"]), "w": dev(c["rbf_w"]), "mu": dev(c["rbf_mu"])}
    out = torch.empty_like(d["u"])
    tnrd.tnrd_set_kernel(2)                                          # what the same stage launches through tnrd_stage
    try:
        tnrd.tnrd_stage(*_stage_args(c, 0, d), out)
        tnrd.tnrd_reset_launch_count()
        tnrd.tnrd_stage(*_stage_args(c, 0, d), out)
        per_call = tnrd.tnrd_launch_count()
    finally:
        tnrd.tnrd_set_kernel(0)
    ref = out.cpu().numpy().copy()
    tnrd.tnrd_stage_static(*_stage_args(c, 0, d), out)               # the CUDA runtime loads the kernels' code on first use
    out.zero_()                                                      # (torch's fill kernel too)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    tnrd.tnrd_reset_launch_count()
    for _ in range(3):                                               # nothing but the entry point between the two readings
        tnrd.tnrd_stage_static(*_stage_args(c, 0, d), out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "device memory in use changed across the calls"
    assert tnrd.tnrd_launch_count() == 3 * per_call and per_call >= 2
    assert np.array_equal(out.cpu().numpy(), ref)
    # under stream capture: legal without a warm-up of the library scratch, which tnrd_stage needs
    cap = torch.zeros_like(d["u"])
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.graph(g, stream=s):
        tnrd.tnrd_stage_static(*_stage_args(c, 0, d), cap, stream=s)
    g.replay()
    torch.cuda.synchronize()
    assert np.array_equal(cap.cpu().numpy(), ref)
    check(ref.astype(np.float64), run_oracle(c), "static, one stage", tight=True)
    # the limit: 4096 x 4096 needs 1756 CTAs x 64 KiB of partial sums
    q = tnrd.tnrd_plan_query(1, 4096, 4096, 48, 7, torch.cuda.get_device_properties(0).multi_processor_count)
    assert 4 * q["part_floats"] > tnrd.STATIC_SCRATCH_BYTES - (1 << 20)
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_stage_static(0x1000, 0x2000, 1, 4096, 4096, 48, 7, 0x3000, 0x4000, 0x5000, 10.0, 0.1, 0x6000, stream=0)
    assert ei.value.status == tnrd.ERR_TOO_LARGE
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_stage_static(0x1000, 0x2000, 1, 64, 64, 8, 7, 0x3000, 0x4000, 0x5000, 10.0, 0.1, 0x1000, stream=0)
    assert ei.value.status == tnrd.ERR_ALIAS
