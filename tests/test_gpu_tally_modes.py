"""-m gpu: the three tally update paths of step 14 (include/mcx.h mcx_tally_mode: one set of reductions per ray,
warp-aggregated, warp-aggregated into a block-private shared-memory cache) against the oracle: N bit-exact, p and p2
within the parity bar, in both lane schedules, plus the cases the aggregation exists for (every lane of a warp in one
bin; more bins than cache slots; two detectors sharing the cache; timing API)."""
import numpy as np
import pytest

from _parity import assert_tally_parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def M():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_2410_08747_b200 as m
    m.lib()
    return m


def tallies(M, inst, n, tally_mode, mode="auto", strict=False, first=0):
    g = M.Instrument(inst, strict=strict)
    g.set_exec(mode)
    g.set_tuning(tally_mode=tally_mode)
    g.trace(n, first=first)
    out = [tuple(t.cpu().numpy() for t in g.tally(d)) for d in range(len(g.dets))]
    cnt = g.counters()
    g.close()
    return out, cnt


@pytest.mark.parametrize("tally_mode", ["global", "warp", "block"])
@pytest.mark.parametrize("cfg", [0, 1, 2, 4])
def test_tally_modes_match_the_oracle(M, O, W, cfg, tally_mode):
    inst = W.config(cfg) if cfg == 0 else W.config(cfg, small=True)
    n = {0: 300_001, 1: 60_001, 2: 400_001, 4: 30_001}[cfg]
    o = O.trace(inst, first=0, n=n)
    for mode in ("direct", "sorted"):
        gt, cnt = tallies(M, inst, n, tally_mode, mode)
        assert cnt["detected"] == o["detected"]
        assert_tally_parity((gt[0][0].view(np.uint64), gt[0][1], gt[0][2]), (o["N"][0], o["P"][0], o["P2"][0]))


@pytest.mark.parametrize("tally_mode", ["warp", "block"])
def test_whole_warps_in_one_bin(M, O, W, tally_mode):
    # a one-pixel, one-energy-bin detector: every detected lane of every warp lands in the same record
    inst = W.config0()
    det = inst["components"][-1]
    det.update(nx=1, ny=1, nE=1)
    n = 200_003
    o = O.trace(inst, first=0, n=n)
    gt, cnt = tallies(M, inst, n, tally_mode)
    assert int(gt[0][0][0]) == int(o["N"][0][0]) == cnt["detected"]
    assert abs(gt[0][1][0] - o["P"][0][0]) <= 1e-9 * o["P"][0][0]
    assert abs(gt[0][2][0] - o["P2"][0][0]) <= 1e-9 * o["P2"][0][0]


def test_more_bins_than_cache_slots_and_two_detectors(M, O, W):
    # 512 x 512 illuminated bins against 2048 slots per block: most updates take the global path; a second detector
    # behind the first shares the cache (the key holds the detector)
    inst = W.config0()
    inst["components"][1].update(xw=40e-3, yh=40e-3)               # open the slit: the whole target is illuminated
    d0 = inst["components"][-1]
    d0.update(nx=512, ny=512)
    d1 = W.detector(-10e-3, 10e-3, -10e-3, 10e-3, 16, 16, 0.0, 40.0, 1, T=(0, 0, 1.2))
    inst["components"].append(d1)
    n = 500_000
    o = O.trace(inst, first=0, n=n)
    for tally_mode in ("block", "warp", "global"):
        gt, cnt = tallies(M, inst, n, tally_mode)
        for d in range(2):
            assert_tally_parity((gt[d][0].view(np.uint64), gt[d][1], gt[d][2]), (o["N"][d], o["P"][d], o["P2"][d]))


def test_timing_split_adds_up(M, W):
    import torch
    inst = W.config1(small=True)
    g = M.Instrument(inst)
    g.set_timing(True)
    g.set_tuning(chunk_log2=16)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.trace(300_000)
    e1.record()
    t = g.timing()
    assert t["launches"] == 5 and t["sort_ms"] > 0 and t["trace_ms"] > 0        # ceil(300000 / 65536) chunks
    assert t["sort_ms"] + t["trace_ms"] <= e0.elapsed_time(e1) * 1.05 + 0.05
    assert g.timing() == {"sort_ms": 0.0, "trace_ms": 0.0, "launches": 0}      # read clears
    g.close()
