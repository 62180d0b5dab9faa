"""CUDA-graph capture of tnrd_diffuse (graph stage loop for launch-bound small images).

The device entry points never synchronise and allocate only on the first call of a shape (stream-ordered scratch), so
after one warm-up call on the capturing stream the whole T-stage call is capturable; replays must reproduce it bit for bit."""
import numpy as np
import pytest

import oracle
import tnrd_gen

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def test_diffuse_is_graph_capturable_and_replay_is_identical():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1503_05768_b200 as tnrd
    tnrd.build(); tnrd.lib()
    c = tnrd_gen.make_config(1)                         # 64 x 64, T = 2, 8 filters 3x3: launch-bound
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()   # noqa: E731
    f, k, w, mu, lam = d(c["f"]), d(c["filters"]), d(c["rbf_w"]), d(c["rbf_mu"]), d(c["lambda"])
    out = torch.empty_like(f)
    s = torch.cuda.Stream()
    args = (c["B"], c["H"], c["W"], c["T"], c["N_k"], c["ksize"])

    def call():
        tnrd.tnrd_diffuse(f, f, *args, k, w, mu, c["rbf_gamma"], lam, out, s)

    with torch.cuda.stream(s):
        call()                                          # sizes the scratch of this (device, stream)
        s.synchronize()
        ref = out.clone()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            call()
        out.zero_()
        g.replay()
        s.synchronize()
        assert torch.equal(out, ref)
        # replays follow the inputs: new image in the same buffers
        f.copy_(d(np.ascontiguousarray(c["f"][:, ::-1, :])))
        g.replay()
        s.synchronize()
        got = out.cpu().numpy().astype(np.float64)
        # timing, informational: graph replay against T + 1 individual launches
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record(s)
        for _ in range(50):
            g.replay()
        e1.record(s)
        for _ in range(50):
            call()
        e2.record(s)
        s.synchronize()
        print(f"C1 per call: graph replay {e0.elapsed_time(e1) * 20:.1f} us, direct launches {e1.elapsed_time(e2) * 20:.1f} us")
    flipped = np.ascontiguousarray(c["f"][:, ::-1, :])
    want = oracle.diffuse(flipped, flipped, c["filters"], c["rbf_w"], c["rbf_mu"], c["rbf_gamma"], c["lambda"])
    assert np.max(np.abs(got - want)) <= 1e-2


def test_scratch_growth_during_capture_is_refused():
    """include/tnrd.h: a call that would have to grow the library scratch while its stream is being captured returns
    TNRD_ERR_CUDA instead of caching a graph-owned allocation."""
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1503_05768_b200 as tnrd
    tnrd.build(); tnrd.lib()
    c = tnrd_gen.make_small(77, 1, 50, 60, 1, 4, 5)
    tnrd.tnrd_set_kernel(2)                             # the tile kernel keeps partial sums in the library scratch
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()   # noqa: E731
    f, k, w, mu, lam = d(c["f"]), d(c["filters"]), d(c["rbf_w"]), d(c["rbf_mu"]), d(c["lambda"])
    out = torch.empty_like(f)
    s = torch.cuda.Stream()                             # a fresh stream: no scratch yet for (device, stream)
    with torch.cuda.stream(s):
        g = torch.cuda.CUDAGraph()
        with pytest.raises(tnrd.TnrdError) as ei:
            with torch.cuda.graph(g, stream=s):
                tnrd.tnrd_diffuse(f, f, 1, 50, 60, 1, 4, 5, k, w, mu, c["rbf_gamma"], lam, out, s)
        assert ei.value.status == tnrd.ERR_CUDA and "capture" in str(ei.value)
    s.synchronize()
    tnrd.tnrd_set_kernel(0)
    tnrd.tnrd_diffuse(f, f, 1, 50, 60, 1, 4, 5, k, w, mu, c["rbf_gamma"], lam, out)     # the library is still usable
    torch.cuda.synchronize()
    assert bool(torch.isfinite(out).all())
