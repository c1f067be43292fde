"""-m gpu: the CUDA path (through the C ABI) against the oracle, element by element, on the same seeded inputs.
Sizes: what the oracle finishes in seconds, still many blocks of 256 rays plus a ragged tail."""
import numpy as np
import pytest

from _parity import assert_dump_parity, assert_tally_parity, tallies_from_dump

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def M():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; there is no CPU fallback")
    import paper_2410_08747_b200 as m
    m.lib()
    return m


def run_gpu(M, inst, n, first, seed, strict, mode="auto", tuning=None):
    g = M.Instrument(inst, strict=strict)
    g.set_exec(mode)
    if tuning:
        g.set_tuning(**tuning)
    gdump = g.trace_dump(first, n, seed)
    g.trace(n, seed, first)
    gt = [tuple(t.cpu().numpy() for t in g.tally(d)) for d in range(len(g.dets))]
    gc = g.counters()
    assert g.launch_count() >= 2
    g.close()
    return gdump, gt, gc


def check(M, O, W, inst, n, exact_counts=False, first=0, seed=None, mesh_accel=0):
    """Traces rays [first, first+n) with the oracle and with both builds of the CUDA library (default, and
    -fmad=false = 'strict'), in both lane schedules (index order and detector-tile order),
    and holds each against the parity bar of _parity.py."""
    seed = inst["seed"] if seed is None else seed
    o = O.trace(inst, first=first, n=n, seed=seed, dump=True, mesh_accel=mesh_accel)
    out = {}
    for strict in (True, False):
        for mode in ("direct", "sorted"):
            out[strict] = check_one(M, W, inst, n, o, exact_counts, first, seed, strict, mode)
    return out[False]


def check_one(M, W, inst, n, o, exact_counts, first, seed, strict, mode="auto", tuning=None):
    gdump, gt, gc = run_gpu(M, inst, n, first, seed, strict, mode, tuning)
    st = assert_dump_parity(gdump, o["dump"], strict=strict)
    nb = [W.n_bins(d) for d in W.detectors_of(inst)]
    if st["n_diff"] == 0:
        # tallies of the two sides, bin by bin
        for d in range(len(nb)):
            assert_tally_parity((gt[d][0].view(np.uint64), gt[d][1], gt[d][2]), (o["N"][d], o["P"][d], o["P2"][d]))
        assert np.array_equal(gc["absorbed"].astype(np.uint64), o["absorbed"])
        assert (gc["detected"], gc["missed"], gc["degenerate"]) == (o["detected"], o["missed"], o["degenerate"])
    else:
        assert not exact_counts, "configs[0] must match bit-exactly"
        # remove the flagged rays on both sides (reading R25): compare what the GPU tallied with its own dump
        keep = np.ones(len(gdump), dtype=bool)
        keep[st["diff_idx"]] = False
        if len(nb) == 1:
            assert_tally_parity(tallies_from_dump(gdump[keep], nb[0]), tallies_from_dump(o["dump"][keep], nb[0]))
    # the GPU tallies are the sums of the GPU's own per-ray records (no lost or duplicated update)
    if len(nb) == 1:
        N, P, P2 = tallies_from_dump(gdump, nb[0])
        assert np.array_equal(gt[0][0].view(np.uint64), N)
        assert np.allclose(gt[0][1], P, rtol=1e-12, atol=1e-300) and np.allclose(gt[0][2], P2, rtol=1e-12, atol=1e-300)
    assert gc["overflows"] == 0
    total = int(gc["absorbed"].sum()) + gc["detected"] + gc["missed"] + gc["degenerate"]
    assert total == n                                                           # ray accounting (step 15)
    return st


def test_c0_full_size_bit_exact_counts(M, O, W):
    inst = W.config0()
    st = check(M, O, W, inst, inst["n_rays"], exact_counts=True)
    assert st["n_diff"] == 0


def test_c0_ragged_and_tiny_sizes(M, O, W):
    inst = W.config0()
    for n in (1, 31, 33, 255, 257, 1000):
        check(M, O, W, inst, n, exact_counts=True)


def test_c0_ray_window_beyond_32_bits(M, O, W):
    inst = W.config0()
    check(M, O, W, inst, 5000, first=(1 << 33) + 12345, exact_counts=True)
    check(M, O, W, inst, 5000, seed=0xDEADBEEFCAFEF00D, exact_counts=True)


def test_c1_primitives(M, O, W):
    check(M, O, W, W.config1(small=True), 100_003)


def test_c2_beamline_optics(M, O, W):
    check(M, O, W, W.config2(small=True), 500_009)


def test_c3_mesh_vs_brute_force_oracle(M, O, W):
    check(M, O, W, W.config3(small=True), 20_011, mesh_accel=0)


def test_c3_mesh_larger_prefix(M, O, W):
    check(M, O, W, W.config3(small=True), 200_000, mesh_accel=1)


def test_c4_voxels(M, O, W):
    check(M, O, W, W.config4(small=True), 100_001)
    check(M, O, W, W.config4(small=True, n_vox=96), 30_000)


def test_sorted_order_is_a_permutation_over_several_chunks(M, O, W):
    """Detector-tile order with chunks of 2^15 rays: 100 003 rays = three full chunks + a ragged one that is still
    sorted + (in the second case) a tail short enough to be traced in index order.  Every ray must be traced exactly
    once: the dump equals the oracle's ray by ray and the tallies equal the sums of the dump."""
    tuning = {"chunk_log2": 15}
    inst = W.config1(small=True)
    for n in (100_003, 3 * 32768 + 1000):
        o = O.trace(inst, first=7, n=n, dump=True)
        check_one(M, W, inst, n, o, False, 7, inst["seed"], True, "sorted", tuning)
    inst = W.config0()
    o = O.trace(inst, first=0, n=200_000, dump=True)
    st = check_one(M, W, inst, 200_000, o, True, 0, inst["seed"], False, "sorted", tuning)
    assert st["n_diff"] == 0
    # a forced bucket grid and the absorber gate switched off: the same rays again
    check_one(M, W, inst, 200_000, o, True, 0, inst["seed"], False, "sorted", {"chunk_log2": 16, "sort_grid_bits": 3, "absorber_gate": 2})


def test_exec_mode_and_tuning_arguments_are_checked(M, W):
    g = M.Instrument(W.config0())
    with pytest.raises(M.McxError):
        M.binding._check(g.L.mcx_instrument_set_exec(g.handle, 7), g.L)
    for bad in ({"chunk_log2": 13}, {"chunk_log2": 27}, {"sort_grid_bits": 12}, {"absorber_gate": 3}):
        with pytest.raises(M.McxError):
            g.set_tuning(**bad)
    g.set_tuning()                                                              # all zeros: nothing changes
    g.status()
    g.close()


def test_empty_trace_and_accumulation(M, O, W):
    inst = W.config0()
    g = M.Instrument(inst)
    g.trace(0)
    assert g.counters()["detected"] == 0
    g.trace(1000, first=0)
    g.trace(1000, first=1000)
    N2 = g.tally(0)[0].cpu().numpy().copy()
    g.reset()
    assert int(g.tally(0)[0].sum()) == 0
    g.trace(2000, first=0)
    assert np.array_equal(g.tally(0)[0].cpu().numpy(), N2)                      # prefix property (reading R2)
    g.close()
