"""-m gpu: step 17, scattering in voxel and solids samples, on the CUDA path
against the oracle: ray by ray (fate, bin, weight) and bin by bin, both builds, both lane schedules."""
import numpy as np
import pytest

from _parity import assert_dump_parity
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
