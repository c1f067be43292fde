"""-m gpu: seeded random instruments (random chains of slits, solids groups of primitives and meshes, voxel volumes,
monitors; random poses, sizes, materials, source modes), each traced by the oracle and by the CUDA path and compared
ray by ray.  Differential testing: whatever the generator happens to produce -- solids behind the source, volumes the
beam misses, overlapping everything -- must come out the same on both sides."""
import numpy as np
import pytest

from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


def small_rotation(rng, scale):
    a = rng.normal(size=3) * scale
    cx, sx, cy, sy, cz, sz = np.cos(a[0]), np.sin(a[0]), np.cos(a[1]), np.sin(a[1]), np.cos(a[2]), np.sin(a[2])
    Rx = np.array([[1, 0, 0], [0, cx, -sx], [0, sx, cx]])
    Ry = np.array([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]])
    Rz = np.array([[cz, -sz, 0], [sz, cz, 0], [0, 0, 1]])
    return Rx @ Ry @ Rz


def random_instrument(W, seed, n_rays):
    rng = np.random.default_rng(31_000 + seed)
    n_mats = int(rng.integers(2, 7))
    mats = [None] + [W.mu_table(rng, n=int(rng.integers(2, 60)), Emin=8.0, Emax=90.0, a_range=(5.0, 200.0)) for _ in range(n_mats)]
    spec = W.bremsstrahlung_spectrum(rng, int(rng.integers(3, 400)), 10.0, 80.0, 80.0)
    pos = ("point", "disk", "gauss")[rng.integers(0, 3)]
    em = ("mono", "uniform", "spectrum")[rng.integers(0, 3)]
    span = float(rng.uniform(0.02, 0.12))
    comps = [W.source(pos, "target", em, radius=rng.uniform(0, 3e-3), sigma_x=rng.uniform(0, 2e-3), sigma_y=rng.uniform(0, 2e-3),
                      target_w=span, target_h=span * rng.uniform(0.5, 1.5), target_dist=1.0, E0=rng.uniform(15.0, 60.0),
                      dE_rel=rng.uniform(0.0, 0.2), spec_Emin=10.0, spec_Emax=80.0, spectrum=spec)]
    z = 0.15
    for _ in range(int(rng.integers(1, 5))):
        kind = rng.choice(5, p=[0.12, 0.08, 0.4, 0.3, 0.1])
        z += rng.uniform(0.05, 0.15)
        T = (rng.normal() * 3e-3, rng.normal() * 3e-3, z)
        if kind == 0:
            comps.append(W.slit_rect(span * z * rng.uniform(0.3, 1.2), span * z * rng.uniform(0.3, 1.2), R=small_rotation(rng, 0.05), T=T))
        elif kind == 1:
            comps.append(W.slit_circ(span * z * rng.uniform(0.2, 0.7), R=small_rotation(rng, 0.05), T=T))
        elif kind == 2:
            sl = []
            for _ in range(int(rng.integers(1, 7))):
                c = (T[0] + rng.normal() * span * z * 0.3, T[1] + rng.normal() * span * z * 0.3, z + rng.normal() * 0.01)
                m, pr, s = int(rng.integers(0, n_mats + 1)), int(rng.integers(0, 3)), span * z * rng.uniform(0.05, 0.4)
                shape = rng.integers(0, 4)
                if shape == 0:
                    sl.append(W.solid_box(s * rng.uniform(0.3, 1.0, size=3), m, pr, R=W.random_rotation(rng), T=c))
                elif shape == 1:
                    sl.append(W.solid_cylinder(s * rng.uniform(0.3, 1.0), s * rng.uniform(0.3, 1.5), m, pr, R=W.random_rotation(rng), T=c))
                elif shape == 2:
                    sl.append(W.solid_sphere(s, m, pr, T=c))
                else:
                    V, F = W.bumpy_sphere(rng, int(rng.integers(0, 3)), s) if rng.random() < 0.7 else W.cube_mesh(s, s * 0.7, s * 1.2)
                    sl.append(W.solid_mesh(V, F, m, pr, R=W.random_rotation(rng), T=c))
            comps.append(W.solids(sl))
        elif kind == 3:
            shape = tuple(int(x) for x in rng.integers(1, 24, size=3))
            ids = rng.integers(0, n_mats + 1, size=shape, dtype=np.uint8)
            if rng.random() < 0.5:
                ids[: shape[0] // 2 + 1] = ids.flat[0]                      # a homogeneous half: long runs
            h = span * z / max(shape) * rng.uniform(0.5, 1.5)
            R = W.random_rotation(rng) if rng.random() < 0.5 else small_rotation(rng, 0.1)
            half = 0.5 * h * np.array(shape[::-1], dtype=float)
            comps.append(W.voxels(ids, h, R=R, T=tuple(np.array(T) - R.T @ half)))
        else:
            comps.append(W.detector(-span, span, -span, span, int(rng.integers(1, 20)), int(rng.integers(1, 20)), 5.0, 70.0,
                                    int(rng.integers(1, 6)), R=small_rotation(rng, 0.05), T=(0, 0, z)))
    n_det = sum(1 for c in comps if c["kind"] == "detector")
    if n_det >= 4:                                                      # MCX_MAX_DETECTORS
        comps = [c for c in comps if c["kind"] != "detector"]
    comps.append(W.detector(-span * 0.8, span * 0.8, -span * 0.8, span * 0.8, 16, 12, 9.0, 85.0, 5, T=(0, 0, 1.0)))
    return W.instrument(f"fuzz{seed}", comps, mats, n_rays)


@pytest.mark.parametrize("seed", range(24))
def test_random_instrument(M, O, W, seed):
    n = 25_000
    check(M, O, W, random_instrument(W, seed, n), n)
