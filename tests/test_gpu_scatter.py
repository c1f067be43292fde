"""-m gpu: step 17, scattering in voxel and solids samples, on the CUDA path
against the oracle: ray by ray (fate, bin, weight) and bin by bin, both builds, both lane schedules."""
import numpy as np
import pytest

from _parity import assert_dump_parity, assert_tally_parity
from test_gpu_parity import M, check, run_gpu  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("K", [1, 4])
def test_c4_voxels_with_scattering(M, O, W, K):
    check(M, O, W, W.config4(small=True, scatter_order=K), 80_003)


def test_c7_line_scanner_with_scattering(M, O, W):
    check(M, O, W, W.config7(small=True, scatter_order=3), 80_001)
    check(M, O, W, W.config7(scatter_order=2), 20_000)


def test_c1_primitives_with_scattering(M, O, W):
    check(M, O, W, W.config1(small=True, scatter_order=3), 60_001)


def test_c3_meshes_with_scattering(M, O, W):
    check(M, O, W, W.config3(small=True, scatter_order=2), 20_003, mesh_accel=1)


def test_scatter_order_without_scattering_tables_changes_nothing(M, O, W):
    for make in (lambda K: W.config4(small=True), lambda K: W.config1(small=True)):
        a, b = make(0), make(0)
        for c in b["components"]:
            if c["kind"] in ("solids", "voxels"):
                c["scatter_order"] = 5
        da = run_gpu(M, a, 30_000, 0, a["seed"], True)[0]
        db = run_gpu(M, b, 30_000, 0, b["seed"], True)[0]
        assert np.array_equal(da["fate"], db["fate"]) and np.array_equal(da["bin"], db["bin"])
        assert np.allclose(da["p"], db["p"], rtol=1e-13, atol=0)


def test_purely_scattering_block_keeps_the_weight(M, O, W):
    n, h, mu = 8, 2.5e-3, 80.0
    tab = {"E": np.array([1.0, 200.0]), "mu": np.array([mu, mu]), "mu_s": np.array([mu, mu])}
    L = n * h
    comps = [W.source("point", "target", "mono", target_w=4e-3, target_h=4e-3, target_dist=1.0, E0=30.0),
             W.voxels(np.ones((n, n, n), dtype=np.uint8), h, T=(-0.5 * L, -0.5 * L, 0.1), scatter_order=300),
             W.detector(-0.5, 0.5, -0.5, 0.5, 8, 8, 0.0, 60.0, 1, T=(0, 0, 1.0))]
    inst = W.instrument("scatter_block", comps, [None, tab], 50_000)
    gd = run_gpu(M, inst, 50_000, 0, 1, False)[0]
    assert np.all(np.abs(gd["p"] - 1.0) < 1e-12)
    o = O.trace(inst, n=50_000, dump=True)
    assert_dump_parity(gd, o["dump"], strict=False)


def test_scattering_and_plain_volumes_in_one_instrument(M, O, W):
    # the all-features kernel walks both: the scattering volume by its cube radii, the plain one by its runs
    rng = np.random.default_rng(8)
    mats = [None] + [W.with_scattering(rng, W.mu_table(rng, Emin=10.0, Emax=60.0, a_range=(20.0, 120.0))) for _ in range(3)]
    ids_a = rng.integers(1, 4, size=(10, 12, 14), dtype=np.uint8)
    ids_a[2:8, 3:9, 2:12] = 2
    ids_b = rng.integers(0, 4, size=(9, 9, 9), dtype=np.uint8)
    comps = [W.source("gauss", "target", "uniform", sigma_x=1e-4, sigma_y=1e-4, target_w=0.03, target_h=0.03, target_dist=1.0, E0=30.0,
                      dE_rel=0.5),
             W.voxels(ids_a, 2e-3, R=W.random_rotation(rng), T=(-0.01, -0.012, 0.4), scatter_order=3),
             W.solids([W.solid_sphere(0.006, 1, 0, T=(0.001, 0.0, 0.55))]),
             W.voxels(ids_b, 3e-3, T=(-0.0135, -0.0135, 0.7)),
             W.detector(-0.2, 0.2, -0.2, 0.2, 20, 20, 10.0, 50.0, 4, T=(0, 0, 1.0))]
    check(M, O, W, W.instrument("two_volumes", comps, mats, 40_000), 40_003)


def _both_ways(M, inst, n, first=0, **tuning):
    out = []
    for staged in (1, 2):
        g = M.Instrument(inst)
        g.set_tuning(staged_walk=staged, **tuning)
        assert g.get_tuning()["staged_walk"] == staged
        d = g.trace_dump(first, n)
        before = g.launch_count()
        g.trace(n, first=first)
        launches = g.launch_count() - before
        out.append((d, [tuple(t.cpu().numpy() for t in g.tally(k)) for k in range(len(g.dets))], g.counters(), launches))
        g.close()
    return out


def test_staged_walk_is_the_same_trace_ray_for_ray(M, O, W):
    # the walk stage (a lane takes the next ray of the pool when its own leaves the sample) against the whole chain in
    # one launch: same fate and bin, same counts, weights and sums to rounding; several chunks, a ragged tail; and every
    # setting of the two batch thresholds gives the same rays
    for inst, n, tuning in ((W.config8(small=True), 70_001, {}), (W.config9(small=True), 50_003, {"chunk_log2": 14}),
                            (W.config8(), 30_000, {}), (W.config8(small=True), 20_001, {"walk_batch_setup": 1, "walk_batch_settle": 1}),
                            (W.config9(small=True), 20_001, {"walk_batch_setup": 32, "walk_batch_settle": 32})):
        (ds, ts, cs, ls), (dw, tw, cw, lw) = _both_ways(M, inst, n, **tuning)
        assert np.array_equal(ds["fate"], dw["fate"]) and np.array_equal(ds["bin"], dw["bin"])
        assert np.allclose(ds["p"], dw["p"], rtol=1e-11, atol=0)                # (two compilations of the same expressions)
        for (Ns, Ps, P2s), (Nw, Pw, P2w) in zip(ts, tw):
            assert np.array_equal(Ns, Nw)
            assert np.allclose(Ps, Pw, rtol=1e-11, atol=1e-300) and np.allclose(P2s, P2w, rtol=1e-11, atol=1e-300)
        assert np.array_equal(cs["absorbed"], cw["absorbed"])
        assert (cs["detected"], cs["missed"], cs["degenerate"]) == (cw["detected"], cw["missed"], cw["degenerate"])


def test_staged_walk_with_components_on_both_sides_of_the_sample(M, O, W):
    # a slit that absorbs and a monitor in front of the sample (stage 1), a second scattering volume, a slit and two
    # detectors behind it (stage 2); checked against the oracle in every build and order, and staged against unstaged
    rng = np.random.default_rng(11)
    mats = [None] + [W.with_scattering(rng, W.mu_table(rng, Emin=10.0, Emax=60.0, a_range=(20.0, 120.0))) for _ in range(3)]
    ids_a = np.kron(rng.integers(1, 4, size=(4, 3, 5), dtype=np.uint8), np.ones((4, 4, 4), dtype=np.uint8))  # blocks of 4^3 voxels
    ids_a[5:11, 2:10, 6:14] = 1
    ids_b = np.kron(rng.integers(0, 4, size=(4, 4, 4), dtype=np.uint8), np.ones((2, 2, 2), dtype=np.uint8))
    comps = [W.source("gauss", "target", "uniform", sigma_x=1e-4, sigma_y=1e-4, target_w=0.04, target_h=0.04, target_dist=1.0, E0=30.0,
                      dE_rel=0.5),
             W.slit_rect(0.012, 0.02, T=(0, 0, 0.3)),
             W.detector(-0.02, 0.02, -0.02, 0.02, 8, 8, 10.0, 50.0, 2, T=(0, 0, 0.35)),
             W.voxels(ids_a, 2e-3, R=W.random_rotation(rng), T=(-0.016, -0.012, 0.4), scatter_order=4),
             W.voxels(ids_b, 3e-3, T=(-0.012, -0.012, 0.6), scatter_order=2),
             W.slit_circ(0.15, T=(0, 0, 0.8)),
             W.detector(-0.2, 0.2, -0.2, 0.2, 20, 20, 10.0, 50.0, 4, T=(0, 0, 1.0)),
             W.detector(-0.3, 0.3, -0.3, 0.3, 5, 5, 10.0, 50.0, 1, T=(0, 0, 1.2))]
    inst = W.instrument("staged_both_sides", comps, mats, 60_000)
    check(M, O, W, inst, 60_003)
    (ds, ts, cs, _), (dw, tw, cw, _) = _both_ways(M, inst, 60_003, chunk_log2=14)
    assert np.array_equal(ds["fate"], dw["fate"]) and np.array_equal(ds["bin"], dw["bin"])
    assert np.allclose(ds["p"], dw["p"], rtol=1e-11, atol=0)
    assert np.array_equal(cs["absorbed"], cw["absorbed"]) and 0 < int(cs["absorbed"][1]) < 60_003
    for (Ns, _, _), (Nw, _, _) in zip(ts, tw):
        assert np.array_equal(Ns, Nw)


def test_staged_walk_on_the_four_byte_cells(M, O, W):
    # more than 16 materials: no one-byte cells (DVoxels::cmap), the walk stage reads the cells the trace kernel reads
    inst = W.config9(small=True)
    inst["materials"] = list(inst["materials"]) + [inst["materials"][k] for k in (1, 2, 3, 4)]
    assert len(inst["materials"]) > 16
    check(M, O, W, inst, 40_003)
    (ds, ts, cs, _), (dw, tw, cw, _) = _both_ways(M, inst, 40_003)
    assert np.array_equal(ds["fate"], dw["fate"]) and np.array_equal(ds["bin"], dw["bin"])
    assert np.allclose(ds["p"], dw["p"], rtol=1e-11, atol=0)


def test_staged_walk_only_where_the_chain_allows_it(M, O, W):
    for inst, want in ((W.config8(small=True), 1), (W.config4(small=True), 2), (W.config1(small=True, scatter_order=2), 2)):
        g = M.Instrument(inst)
        assert g.get_tuning()["staged_walk"] == want
        g.set_tuning(staged_walk=1)
        assert g.get_tuning()["staged_walk"] == want
        g.close()


def test_staged_line_scan_with_set_pose(M, O, W):
    inst = W.config8(small=True)
    g = M.Instrument(inst)
    assert g.get_tuning()["staged_walk"] == 1
    comp = inst["sample_component"]
    n = 20_000
    for line, T in enumerate(inst["scan"][1:8:3]):
        g.set_pose(comp, T=T)
        g.reset()
        g.trace(n, first=line * n)
        moved = dict(inst)
        moved["components"] = [dict(c) for c in inst["components"]]
        moved["components"][comp]["T"] = np.array(T)
        o = O.trace(moved, first=line * n, n=n)
        for d in range(len(g.dets)):
            gt = tuple(t.cpu().numpy() for t in g.tally(d))
            assert_tally_parity((gt[0].view(np.uint64), gt[1], gt[2]), (o["N"][d], o["P"][d], o["P2"][d]))
    g.close()
