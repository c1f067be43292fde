"""-m gpu: steps 8-10 (solids) against the oracle where the end-point sweep and the stackless BVH could go wrong:
the maximum number of solids with tied priorities, a source inside overlapping solids, rays through shared mesh
edges and vertices (duplicate hits), nested meshes mixed with primitives, and a mesh whose every triangle is hit by
some ray of a dense fan (every BVH leaf is reached)."""
import numpy as np
import pytest

from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


def solids_instrument(W, solid_list, n_mats, n_rays=60_000, target=0.12, src=(0.0, 0.0, 0.0), det_z=1.0, seed_k=0):
    rng = np.random.default_rng(4242 + seed_k)
    mats = [None] + [W.mu_table(rng, Emin=20.0, Emax=100.0, a_range=(20.0, 400.0)) for _ in range(n_mats)]
    spec = W.bremsstrahlung_spectrum(rng, 200, 20.0, 100.0, 100.0)
    comps = [
        W.source("point", "target", "spectrum", target_w=target, target_h=target, target_dist=det_z - src[2], spec_Emin=20.0,
                 spec_Emax=100.0, spectrum=spec, T=src),
        W.solids(solid_list),
        W.detector(-0.1, 0.1, -0.1, 0.1, 32, 32, 20.0, 100.0, 8, T=(0, 0, det_z)),
    ]
    return W.instrument("solids_edges", comps, mats, n_rays)


def random_primitives(W, rng, n, priorities):
    out = []
    for k in range(n):
        T = (rng.uniform(-0.03, 0.03), rng.uniform(-0.03, 0.03), 0.5 + rng.uniform(-0.03, 0.03))
        R = W.random_rotation(rng)
        mat, pr = int(rng.integers(1, 5)), int(priorities[k])
        kind = k % 3
        if kind == 0:
            out.append(W.solid_box(rng.uniform(0.005, 0.03, size=3), mat, pr, R=R, T=T))
        elif kind == 1:
            out.append(W.solid_cylinder(rng.uniform(0.005, 0.025), rng.uniform(0.005, 0.03), mat, pr, R=R, T=T))
        else:
            out.append(W.solid_sphere(rng.uniform(0.005, 0.03), mat, pr, T=T))
    return out


def test_sixteen_solids_tied_priorities(M, O, W):
    rng = np.random.default_rng(1)
    for prios in (np.zeros(16), rng.integers(0, 3, size=16), np.arange(16)[::-1]):
        check(M, O, W, solids_instrument(W, random_primitives(W, rng, 16, prios), 4), 60_000)


def test_source_inside_overlapping_solids(M, O, W):
    rng = np.random.default_rng(2)
    sl = [W.solid_sphere(0.2, 1, 0, T=(0, 0, 0.05)), W.solid_box((0.05, 0.05, 0.3), 2, 1, T=(0, 0, 0.1)),
          W.solid_cylinder(0.03, 0.5, 3, 1, R=W.random_rotation(rng), T=(0.0, 0.0, 0.2))]
    check(M, O, W, solids_instrument(W, sl, 3), 60_000)


def test_rays_through_shared_edges_and_vertices(M, O, W):
    """target of zero width: every ray runs down the axis, through the diagonal edge of two cube faces (cube_mesh
    splits a face along its diagonal) or, for the rotated cube, through two opposite vertices"""
    V, F = W.cube_mesh(0.02, 0.02, 0.02)
    check(M, O, W, solids_instrument(W, [W.solid_mesh(V, F, 1, 0, T=(0, 0, 0.5))], 1, n_rays=2_000, target=0.0), 2_000)
    # body diagonal along z: rotation taking (1,1,1)/sqrt(3) to z
    a = np.array([1.0, 1.0, 1.0]) / np.sqrt(3.0)
    b = np.cross(a, [0.0, 0.0, 1.0]); b /= np.linalg.norm(b)
    R = np.stack([b, np.cross(a, b), a])                      # rows: local axes in lab... local = R (lab - T)
    check(M, O, W, solids_instrument(W, [W.solid_mesh(V, F, 1, 0, R=R.T, T=(0, 0, 0.5))], 1, n_rays=2_000, target=0.0), 2_000)
    # an edge-on sheet of rays: target of zero height sweeps the plane y = 0, which holds cube edges when rotated by 45 deg
    c, s = np.cos(np.pi / 4), np.sin(np.pi / 4)
    Rz = np.array([[c, -s, 0], [s, c, 0], [0, 0, 1.0]])
    inst = solids_instrument(W, [W.solid_mesh(V, F, 1, 0, R=Rz, T=(0, 0, 0.5))], 1, n_rays=20_000)
    inst["components"][0]["target_h"] = 0.0
    check(M, O, W, inst, 20_000)


def test_nested_meshes_with_primitives(M, O, W):
    rng = np.random.default_rng(3)
    Vo, Fo = W.bumpy_sphere(rng, 3, 0.03)
    Vi, Fi = W.bumpy_sphere(rng, 2, 0.012)
    Vc, Fc = W.cube_mesh(0.01, 0.02, 0.015)
    sl = [W.solid_mesh(Vo, Fo, 1, 0, T=(0, 0, 0.5)), W.solid_mesh(Vi, Fi, 2, 2, T=(0.005, 0, 0.5)),
          W.solid_mesh(Vc, Fc, 3, 1, R=W.random_rotation(rng), T=(-0.01, 0.01, 0.5)),
          W.solid_sphere(0.02, 4, 1, T=(0.02, -0.01, 0.47)), W.solid_box((0.04, 0.002, 0.04), 2, 3, T=(0, 0.0, 0.5))]
    check(M, O, W, solids_instrument(W, sl, 4), 40_000, mesh_accel=0)


def test_dense_fan_reaches_every_leaf(M, O, W):
    rng = np.random.default_rng(4)
    V, F = W.bumpy_sphere(rng, 4, 0.04)                        # 5120 triangles
    inst = solids_instrument(W, [W.solid_mesh(V, F, 1, 0, T=(0, 0, 0.5))], 1, n_rays=300_000, target=0.2)
    check(M, O, W, inst, 300_000, mesh_accel=1)
