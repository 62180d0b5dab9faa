"""Host logic of the tile planner (tnrd_plan_query: pure host code of libtnrd.so, no GPU): the plan must always cover the
phi region with tiles that fit a CTA, and its CTA / scratch arithmetic must be consistent."""
import itertools

import numpy as np
import pytest

import paper_1503_05768_b200 as tnrd

AREA = {1: (128, 128), 2: (64, 32), 3: (64, 64)}      # output area (RW, RH) of the kernel configurations


@pytest.fixture(scope="module")
def lib():
    tnrd.build()
    return tnrd.lib()


def check_plan(p, B, H, W, n_k, K, sms):
    r = (K - 1) // 2
    Wz, Hz = W + 2 * r, H + 2 * r
    rw, rh = AREA[p["cfg"]]
    assert 1 <= p["tw"] <= rw - 2 * r and 1 <= p["th"] <= rh - 2 * r            # tile + r ring fits the output area
    assert p["ntx"] * p["tw"] >= Wz > (p["ntx"] - 1) * p["tw"]                    # tiles cover the phi region, none empty
    assert p["nty"] * p["th"] >= Hz > (p["nty"] - 1) * p["th"]
    tiles = p["ntx"] * p["nty"] * B
    assert 1 <= p["nsplit"] <= max(1, n_k) and 0 <= p["n_full"] <= tiles
    assert p["ctas"] == p["n_full"] + (tiles - p["n_full"]) * p["nsplit"]
    assert p["cta_floats"] == rw * rh and p["part_floats"] == p["ctas"] * p["cta_floats"]
    if 0 < p["n_full"] < tiles:                                                   # tail split: whole waves first
        assert p["n_full"] % sms == 0 and p["nsplit"] >= 2


def test_plans_cover_every_shape(lib):
    rng = np.random.default_rng([150305768, 55])
    cases = [(1, 64, 64, 8, 3), (1, 321, 481, 24, 5), (1, 321, 481, 48, 7), (128, 321, 481, 48, 7), (1, 4096, 4096, 48, 7),
             (1, 2048, 2048, 48, 7), (1, 1024, 1024, 48, 7), (1, 8, 8, 1, 9), (1, 2, 300, 3, 3), (3, 70000, 8, 2, 3),
             (1, 16384, 16384, 48, 7), (1200, 60, 9, 2, 5), (1, 122, 122, 128, 3)]
    for _ in range(300):
        K = int(rng.choice([3, 5, 7, 9]))
        cases.append((int(rng.integers(1, 40)), int(rng.integers(K - 1, 3000)), int(rng.integers(K - 1, 3000)),
                      int(rng.integers(1, 129)), K))
    for (B, H, W, n_k, K), sms in itertools.product(cases, (148, 132, 1)):
        if B * H * W >= 2 ** 31:
            continue
        check_plan(tnrd.tnrd_plan_query(B, H, W, n_k, K, sms), B, H, W, n_k, K, sms)


def test_known_plans(lib):
    p = tnrd.tnrd_plan_query(1, 4096, 4096, 48, 7)          # headline: 34 x 34 tiles (33 of the largest size 122 and a
    assert (p["cfg"], p["ntx"], p["nty"], p["tw"], p["th"]) == (1, 34, 34, 122, 122)   # ragged one), 7 waves + a split tail
    assert p["n_full"] == 7 * 148 and p["nsplit"] > 1
    p = tnrd.tnrd_plan_query(128, 321, 481, 48, 7)          # C5: a 481-wide image needs 4 tile columns (487 <= 4 x 122)
    assert (p["ntx"], p["nty"]) == (4, 3)
    p = tnrd.tnrd_plan_query(1, 321, 481, 48, 7)            # C3: fewer tiles than SMs -> the filter bank is split
    assert p["n_full"] == 0 and p["nsplit"] > 1 and p["ctas"] <= 2 * 148


def test_plan_query_errors(lib):
    import ctypes
    buf = (ctypes.c_longlong * 10)()
    L = tnrd.lib()
    assert L.tnrd_plan_query(1, 64, 64, 8, 4, 148, buf) == tnrd.ERR_UNSUPPORTED
    assert L.tnrd_plan_query(1, 3, 64, 8, 7, 148, buf) == tnrd.ERR_SHAPE
    assert L.tnrd_plan_query(1, 64, 64, 8, 3, 0, buf) == tnrd.ERR_SHAPE
    assert L.tnrd_plan_query(1, 64, 64, 8, 3, 148, None) == tnrd.ERR_NULL
