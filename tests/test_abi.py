"""C-ABI checks that need no GPU: the library loads, exports every symbol include/tnrd.h declares, and
rejects bad arguments before touching CUDA."""
import ctypes
import os
import re

import pytest

import paper_1503_05768_b200 as tnrd

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    tnrd.build()
    return tnrd.lib()


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "tnrd.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(tnrd_[a-z_]+)\s*\(", src)))


def test_header_declares_the_boundary():
    names = _declared_functions()
    for must in ("tnrd_stage", "tnrd_diffuse", "tnrd_diffuse_host", "tnrd_strerror", "tnrd_version",
                 "tnrd_shutdown", "tnrd_last_cuda_error"):
        assert must in names


def test_every_declared_symbol_is_exported(L):
    for name in _declared_functions():
        assert hasattr(L, name), f"{name} declared in include/tnrd.h but not exported by libtnrd.so"


def test_python_binding_has_the_same_names():
    for name in _declared_functions():
        assert hasattr(tnrd, name), f"binding lacks {name}"


def test_version_and_strerror(L):
    assert tnrd.tnrd_version() == 200
    assert tnrd.tnrd_strerror(0) == "ok"
    for code in range(-6, 0):
        assert tnrd.tnrd_strerror(code) not in ("", "unknown status")
    assert tnrd.tnrd_strerror(-99) == "unknown status"
    assert tnrd.tnrd_last_cuda_error() == ""


def test_argument_validation_without_gpu(L):
    p = 0x1000  # never dereferenced: validation fails first
    n = None
    st = ctypes.c_void_p(0)
    # NULL pointers
    assert L.tnrd_stage(n, p, 1, 8, 8, 4, 3, p, p, p, 10.0, 0.1, p, st) == tnrd.ERR_NULL
    assert L.tnrd_diffuse(p, p, 1, 8, 8, 2, 4, 3, p, p, p, 10.0, p, n, st) == tnrd.ERR_NULL
    assert L.tnrd_diffuse(p, p, 1, 8, 8, 2, 4, 3, n, p, p, 10.0, p, p + 64, st) == tnrd.ERR_NULL
    assert L.tnrd_diffuse_host(p, n, 1, 8, 8, 2, 4, 3, p, p, p, 10.0, p, p, st) == tnrd.ERR_NULL
    # shapes
    assert L.tnrd_stage(p, p, 0, 8, 8, 4, 3, p, p, p, 10.0, 0.1, p + 64, st) == tnrd.ERR_SHAPE
    assert L.tnrd_stage(p, p, 1, 8, 8, 0, 3, p, p, p, 10.0, 0.1, p + 64, st) == tnrd.ERR_SHAPE
    assert L.tnrd_stage(p, p, 1, 8, 8, 129, 3, p, p, p, 10.0, 0.1, p + 64, st) == tnrd.ERR_SHAPE
    assert L.tnrd_stage(p, p, 1, 5, 8, 4, 7, p, p, p, 10.0, 0.1, p + 64, st) == tnrd.ERR_SHAPE     # H < 2r
    assert L.tnrd_stage(p, p, 2, 32768, 32768, 4, 3, p, p, p, 10.0, 0.1, p + 64, st) == tnrd.ERR_SHAPE
    assert L.tnrd_diffuse(p, p, 1, 8, 8, -1, 4, 3, p, p, p, 10.0, p, p + 64, st) == tnrd.ERR_SHAPE
    # ksize
    for ks in (1, 2, 4, 6, 8, 11):
        assert L.tnrd_stage(p, p, 1, 16, 16, 4, ks, p, p, p, 10.0, 0.1, p + 64, st) == tnrd.ERR_UNSUPPORTED
    # gamma
    for g in (0.0, -1.0, float("inf"), float("nan")):
        assert L.tnrd_stage(p, p, 1, 8, 8, 4, 3, p, p, p, g, 0.1, p + 64, st) == tnrd.ERR_PARAM
    # aliasing
    assert L.tnrd_stage(p, p + 64, 1, 8, 8, 4, 3, p, p, p, 10.0, 0.1, p, st) == tnrd.ERR_ALIAS     # u_out == f
    assert L.tnrd_diffuse(p, p + 64, 1, 8, 8, 2, 4, 3, p, p, p, 10.0, p, p, st) == tnrd.ERR_ALIAS
    # deblocking: H, W multiples of 8; bounds may not be the output
    assert L.tnrd_deblock_diffuse(p, 1, 12, 16, 1, 4, 3, p, p, p, 10.0, p, p, p + 64, st) == tnrd.ERR_SHAPE
    assert L.tnrd_deblock_diffuse(p, 1, 16, 16, 1, 4, 3, p, p, p, 10.0, p, n, p + 64, st) == tnrd.ERR_NULL
    assert L.tnrd_deblock_diffuse(p, 1, 16, 16, 1, 4, 3, p, p, p, 10.0, p, p + 64, p + 64, st) == tnrd.ERR_ALIAS
    assert L.tnrd_qcs_project(p, 1, 16, 20, p, p, p + 64, st) == tnrd.ERR_SHAPE
    assert L.tnrd_qcs_project(p, 1, 16, 16, p + 64, p, p + 64, st) == tnrd.ERR_ALIAS
    assert L.tnrd_set_phi_mode(4) == tnrd.ERR_UNSUPPORTED and L.tnrd_set_phi_mode(0) == tnrd.OK
    assert L.tnrd_set_phi_mode(tnrd.PHI_FACTORED) == tnrd.OK
    # options
    assert L.tnrd_set_kernel(7) == tnrd.ERR_UNSUPPORTED
    assert L.tnrd_set_kernel(3) == tnrd.OK and L.tnrd_set_kernel(0) == tnrd.OK
    # backward pass: the forward result may not overwrite what the gradients are formed from
    bw = (1, 16, 16, 2, 4, 3, p, p, p, 10.0, p)
    assert L.tnrd_diffuse_backward(p, p + 64, p + 128, n, *bw, p + 128, n, n, n, n, st) == tnrd.ERR_ALIAS    # u_T == u_gt
    assert L.tnrd_diffuse_backward(p, p + 64, n, p + 128, *bw, p + 128, n, n, n, n, st) == tnrd.ERR_ALIAS    # u_T == e_T
    assert L.tnrd_diffuse_backward(p, p + 64, p + 128, n, *bw, p + 192, p + 192, n, n, n, st) == tnrd.ERR_ALIAS  # u_T == grad_u0
    assert L.tnrd_diffuse_backward(p, p + 64, p + 128, n, *bw, p + 64, n, n, n, n, st) == tnrd.ERR_ALIAS     # u_T == u0
    # tensor-core plan query: pure host logic
    q = (ctypes.c_longlong * 7)()
    assert L.tnrd_tc_plan_query(1, 4096, 4096, 48, 7, 148, q) == tnrd.OK and q[0] == 2 and q[1] == 17 and q[5] == 250
    assert q[4] == q[1] * q[2] * q[6] and q[3] % 2 == 0 and q[6] == 1
    assert L.tnrd_tc_plan_query(1, 64, 64, 8, 3, 148, q) == tnrd.OK and q[0] == 0
    assert L.tnrd_tc_plan_query(1, 64, 64, 8, 3, 148, None) == tnrd.ERR_NULL
    assert L.tnrd_microbench(0, None, st) == tnrd.ERR_NULL
    r = ctypes.c_double()
    assert L.tnrd_microbench(9, ctypes.byref(r), st) == tnrd.ERR_UNSUPPORTED


def test_binding_raises_on_error(L):
    with pytest.raises(tnrd.TnrdError) as ei:
        tnrd.tnrd_stage(0x1000, 0x1000, 1, 8, 8, 4, 4, 0x1000, 0x1000, 0x1000, 10.0, 0.1, 0x2000, stream=0)
    assert ei.value.status == tnrd.ERR_UNSUPPORTED


def test_no_cpu_fallback_when_library_is_missing(monkeypatch, tmp_path):
    monkeypatch.setattr(tnrd, "_lib", None)
    monkeypatch.setattr(tnrd, "LIB_PATH", str(tmp_path / "libtnrd.so"))
    with pytest.raises(FileNotFoundError):
        tnrd.lib()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1503_05768_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".h", ".cuh")):
                txt = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "oracle/" not in txt, fn
    otxt = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(
        os.path.join(ROOT, "oracle", "tnrd_oracle.c")).read()
    assert "import paper_1503_05768_b200" not in otxt and "tnrd.h" not in otxt
