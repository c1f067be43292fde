"""-m gpu: the voxel walk (step 11) against the oracle on the cases its structure could get wrong: volumes whose
fast axis is not the beam axis or runs against it (no run-length skipping, negative address steps), rays oblique to
all three axes (the walk axis differs from ray to ray), a source inside the volume, non-cubic and one-cell-thick
grids, and per-voxel random IDs (a run ends at nearly every face)."""
import numpy as np
import pytest

from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


def rot_axis(axis, angle):
    c, s = np.cos(angle), np.sin(angle)
    R = np.eye(3)
    i, j = [(1, 2), (2, 0), (0, 1)][axis]
    R[i, i], R[i, j], R[j, i], R[j, j] = c, -s, s, c
    return R


def voxel_instrument(W, ids, h, R, centre, n_rays=60_000, target=0.30, src_z=0.0, det_z=2.5, seed_k=0):
    """Point source at (0, 0, src_z) aimed at a target x target rectangle at det_z; the volume (ids[z][y][x], cell h)
    with pose rotation R (lab -> local) and its centre at lab point `centre`."""
    rng = np.random.default_rng(777 + seed_k)
    nz, ny, nx = ids.shape
    half = 0.5 * h * np.array([nx, ny, nz])
    T = np.asarray(centre, dtype=float) - R.T @ half          # local = R (lab - T)
    n_ids = int(ids.max()) + 1
    mats = [None] + [W.mu_table(rng, Emin=20.0, Emax=150.0, a_range=(5.0, 300.0)) for _ in range(n_ids - 1)]
    spec = W.bremsstrahlung_spectrum(rng, 300, 20.0, 150.0, 150.0)
    comps = [
        W.source("point", "target", "spectrum", target_w=target, target_h=target, target_dist=det_z - src_z, spec_Emin=20.0,
                 spec_Emax=150.0, spectrum=spec, T=(0, 0, src_z)),
        W.voxels(ids, h, R=R, T=tuple(T)),
        W.detector(-target / 2, target / 2, -target / 2, target / 2, 32, 32, 20.0, 150.0, 8, T=(0, 0, det_z)),
    ]
    return W.instrument("voxel_edges", comps, mats, n_rays)


def blobs(rng, shape, n_ids=6):
    """a few axis-aligned blocks of material in vacuum: long runs with sharp ends"""
    ids = np.zeros(shape, dtype=np.uint8)
    for _ in range(12):
        lo = [rng.integers(0, s) for s in shape]
        hi = [min(s, l + rng.integers(1, max(2, s // 2))) for s, l in zip(shape, lo)]
        ids[lo[0]:hi[0], lo[1]:hi[1], lo[2]:hi[2]] = rng.integers(1, n_ids)
    return ids


@pytest.mark.parametrize("case", ["beam_along_minus_x", "beam_along_y", "beam_against_z", "oblique", "oblique2"])
def test_rotated_volumes(M, O, W, case):
    rng = np.random.default_rng(11)
    ids = blobs(rng, (40, 48, 56))
    R = {"beam_along_minus_x": rot_axis(1, np.pi / 2), "beam_along_y": rot_axis(0, np.pi / 2),
         "beam_against_z": rot_axis(0, np.pi), "oblique": rot_axis(0, 0.7) @ rot_axis(1, 0.6) @ rot_axis(2, 0.5),
         "oblique2": rot_axis(2, 2.1) @ rot_axis(0, -0.9)}[case]
    check(M, O, W, voxel_instrument(W, ids, 2.0e-3, R, (0.0, 0.0, 1.5)), 60_000)


def test_source_inside_the_volume(M, O, W):
    rng = np.random.default_rng(12)
    ids = blobs(rng, (64, 64, 64))
    ids[ids == 0] = 1                                          # no vacuum: the first run starts at t = 0
    check(M, O, W, voxel_instrument(W, ids, 4.0e-3, np.eye(3), (0.0, 0.0, 0.05), src_z=0.0), 60_000)
    check(M, O, W, voxel_instrument(W, ids, 4.0e-3, rot_axis(1, 0.8), (0.01, -0.02, 0.03), src_z=0.0), 60_000)


def test_random_ids_every_face_ends_a_run(M, O, W):
    rng = np.random.default_rng(13)
    ids = rng.integers(0, 8, size=(24, 24, 24), dtype=np.uint8)
    check(M, O, W, voxel_instrument(W, ids, 5.0e-3, np.eye(3), (0.0, 0.0, 1.0)), 40_000)
    check(M, O, W, voxel_instrument(W, ids, 5.0e-3, rot_axis(0, 0.4) @ rot_axis(1, 1.1), (0.0, 0.0, 1.0)), 40_000)


def test_thin_and_tiny_grids(M, O, W):
    rng = np.random.default_rng(14)
    for shape in ((1, 1, 1), (1, 30, 30), (30, 1, 30), (30, 30, 1), (3, 2, 300)):
        ids = rng.integers(1, 4, size=shape, dtype=np.uint8)
        check(M, O, W, voxel_instrument(W, ids, 3.0e-3, np.eye(3), (0.0, 0.0, 1.2), target=0.25), 30_000)
        check(M, O, W, voxel_instrument(W, ids, 3.0e-3, rot_axis(1, np.pi / 2), (0.0, 0.0, 1.2), target=0.25), 30_000)


def test_long_runs_beyond_the_run_cap(M, O, W):
    """a homogeneous 600-cell row is longer than the 255-cell run cap: several skips per run"""
    ids = np.full((4, 4, 600), 2, dtype=np.uint8)
    ids[:, :, 300:310] = 1
    check(M, O, W, voxel_instrument(W, ids, 1.0e-3, np.eye(3), (0.0, 0.0, 1.0), target=0.02), 30_000)


def test_ids_beyond_the_materials_are_vacuum(M, O, W):
    """include/mcx.h: a voxel value >= n_materials is traced as material 0.  The GPU gets the raw volume, the oracle
    the volume with those values replaced."""
    rng = np.random.default_rng(15)
    ids = blobs(rng, (32, 32, 32))
    raw = ids.copy()
    raw[4:9, 10:20, 3:30] = 200
    raw[20:25, 5:9, 8:12] = 254
    clean = np.where(raw >= 6, 0, raw).astype(np.uint8)       # blobs() uses IDs 0..5 -> 6 materials
    inst_clean = voxel_instrument(W, clean, 4.0e-3, np.eye(3), (0.0, 0.0, 1.0))
    assert len(inst_clean["materials"]) == 6
    inst_raw = dict(inst_clean)                                # same source, tables and detector; only the volume differs
    inst_raw["components"] = [dict(c) for c in inst_clean["components"]]
    inst_raw["components"][1]["ids"] = np.ascontiguousarray(raw)
    n = 30_000
    o = O.trace(inst_clean, first=0, n=n, dump=True)
    g = M.Instrument(inst_raw)
    d = g.trace_dump(0, n)
    g.close()
    assert np.array_equal(d["fate"], o["dump"]["fate"]) and np.array_equal(d["bin"], o["dump"]["bin"])
    assert np.allclose(d["p"], o["dump"]["p"], rtol=1e-9, atol=0)
