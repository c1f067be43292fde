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
