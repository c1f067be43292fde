"""-m gpu: the CUDA path at BASELINE.json's FULL sizes, in the launch configuration bench.py times (AUTO lane
scheduling, default chunking, n_rays of the config), held against the oracle on what the oracle can compute one by one
(reading R26):

  * the tallies a full-size run adds for its LAST `w` ray indices -- tally(trace [0, n)) - tally(trace [0, n - w)) --
    equal the oracle's tallies of the window [n - w, n): N bit-exact, P and P2 within 1e-9 of the window's weight;
    this goes through the chunked, sorted path with its ragged last chunk, deep inside the index range;
  * per-ray records (mcx_trace_dump) of windows in the middle and at the end of the range equal the oracle's;
  * exact invariants at any size: ray accounting sums to n_rays, sum(N) = detected, 0 <= P2 <= P <= N per bin
    (every weight is in (0, 1]), no capacity overflow.
"""
import numpy as np
import pytest

from _parity import assert_dump_parity, tallies_from_dump

pytestmark = pytest.mark.gpu

WINDOW = 40_000


@pytest.fixture(scope="module")
def M():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_2410_08747_b200 as m
    m.lib()
    return m


def has_mesh(inst):
    return any(s["shape"] == "mesh" for c in inst["components"] if c["kind"] == "solids" for s in c["solids"])


def full_size(M, O, W, k, window=WINDOW):
    import torch
    inst = W.config(k)
    n = inst["n_rays"]
    accel = 1 if has_mesh(inst) else 0
    g = M.Instrument(inst)                                   # AUTO lane scheduling = what bench.py times
    nb = W.n_bins(W.detectors_of(inst)[-1])
    last = len(g.dets) - 1
    # (1) the run without its last window, then the window on top of it (mcx_trace accumulates)
    g.trace(n - window, first=0)
    N1, P1, P21 = (t.clone() for t in g.tally(last))
    c1 = g.counters()
    g.trace(window, first=n - window)
    N2, P2, P22 = g.tally(last)
    c2 = g.counters()
    # (3) invariants of the whole run
    total = int(c2["absorbed"].sum()) + c2["detected"] + c2["missed"] + c2["degenerate"]
    assert total == n and c2["overflows"] == 0
    assert int(N2.sum()) == c2["detected"]
    assert bool((P22 >= 0).all()) and bool((P22 <= P2 * (1 + 1e-12)).all()) and bool((P2 <= N2.double() * (1 + 1e-12)).all())
    dN = (N2 - N1).cpu().numpy()
    dP = (P2 - P1).cpu().numpy()
    dP2 = (P22 - P21).cpu().numpy()
    del N1, P1, P21, N2, P2, P22
    torch.cuda.empty_cache()
    o = O.trace(inst, first=n - window, n=window, dump=True, mesh_accel=accel)
    gd = g.trace_dump(n - window, window)
    st = assert_dump_parity(gd, o["dump"], strict=False)
    keep = np.ones(window, dtype=bool)
    keep[st["diff_idx"]] = False
    oN, oP, oP2 = tallies_from_dump(o["dump"], nb) if st["n_diff"] == 0 else tallies_from_dump(gd, nb)
    if st["n_diff"] == 0:
        assert np.array_equal(oN, o["N"][last]) and c2["detected"] - c1["detected"] == o["detected"]
    assert np.array_equal(dN.astype(np.uint64), oN), "integer ray counts of the last window differ"
    Wt, W2t = float(oP.sum()), float(oP2.sum())
    # the difference of two large sums: each bin holds <= ~1e2 rays of weight <= 1, so its rounding is ~1e-14 absolute
    assert float(np.abs(dP - oP).max()) <= 1e-9 * max(Wt, 1e-300)
    assert float(np.abs(dP2 - oP2).max()) <= 1e-9 * max(W2t, 1e-300)
    # (2) a window in the middle of the range, ray by ray
    mid = (n // 2 // 977) * 977 + 13
    om = O.trace(inst, first=mid, n=window // 2, dump=True, mesh_accel=accel)
    assert_dump_parity(g.trace_dump(mid, window // 2), om["dump"], strict=False)
    g.close()
    return st


def test_c1_full_size(M, O, W):
    full_size(M, O, W, 1)


def test_c2_full_size(M, O, W):
    full_size(M, O, W, 2, window=200_000)


def test_c3_full_size(M, O, W):
    full_size(M, O, W, 3)


def test_c4_full_size(M, O, W):
    full_size(M, O, W, 4, window=20_000)


def test_c5_basic_instrument_full_size(M, O, W):
    full_size(M, O, W, 5)


def test_c6_focusing_instrument_full_size(M, O, W):
    full_size(M, O, W, 6)


def test_c7_line_scanner_full_size(M, O, W):
    full_size(M, O, W, 7, window=20_000)


def test_c8_c9_scattering_full_size(M, O, W):
    full_size(M, O, W, 8, window=4_000)
    full_size(M, O, W, 9, window=8_000)
