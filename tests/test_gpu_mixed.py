"""-m gpu: chains that mix component kinds, so that the all-features instantiation of the kernel (every scratch area
of shared memory in use at once), two solids groups, two detectors (a monitor in mid-chain does not absorb) and the
absorber gate in front of heavy components are all exercised against the oracle."""
import numpy as np
import pytest

from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


def mixed_instrument(W, n_rays, with_mirror):
    rng = np.random.default_rng(99)
    mats = [None] + [W.mu_table(rng, Emin=10.0, Emax=60.0, a_range=(5.0, 80.0)) for _ in range(5)]
    spec = W.bremsstrahlung_spectrum(rng, 200, 10.0, 60.0, 60.0)
    ids = rng.integers(0, 6, size=(12, 14, 16), dtype=np.uint8)
    ids[3:9, 4:10, :] = 2
    Vc, Fc = W.cube_mesh(0.004, 0.006, 0.005)
    Vs, Fs = W.bumpy_sphere(rng, 2, 0.006)
    comps = [
        W.source("gauss", "target", "spectrum", sigma_x=1e-4, sigma_y=2e-4, target_w=0.05, target_h=0.05, target_dist=1.0,
                 spec_Emin=10.0, spec_Emax=60.0, spectrum=spec),
        W.slit_rect(0.004, 0.005, T=(0, 0, 0.3)),                                   # absorbs ~90 %: the gate engages
        W.solids([W.solid_box((0.003, 0.004, 0.002), 1, 0, R=W.random_rotation(rng), T=(0.001, 0, 0.40)),
                  W.solid_mesh(Vc, Fc, 3, 1, R=W.random_rotation(rng), T=(-0.002, 0.001, 0.402)),
                  W.solid_sphere(0.004, 2, 2, T=(0.0, -0.002, 0.399))]),
        W.detector(-0.02, 0.02, -0.02, 0.02, 16, 16, 10.0, 60.0, 4, T=(0, 0, 0.5)),  # monitor: rays go on
        W.voxels(ids, 1.0e-3, R=W.random_rotation(rng), T=(-0.006, -0.007, 0.6)),
        W.solids([W.solid_mesh(Vs, Fs, 4, 0, T=(0.002, 0.001, 0.7)), W.solid_cylinder(0.003, 0.01, 5, 1, T=(-0.003, 0, 0.7))]),
    ]
    if with_mirror:  # optics at the end of the chain: every feature bit set
        tab = W.reflectivity_table(rng, n_theta=20, n_E=30, theta_max=0.2, Emin=5.0, Emax=70.0)
        c, s = np.cos(0.05), np.sin(0.05)
        R = np.array([[1, 0, 0], [0, c, -s], [0, s, c]], dtype=float)              # mirror tilted by 50 mrad about x
        comps.append(W.mirror_elliptic(0.9, 0.3, 0.05, 0.2, 0.1, tab, R=R, T=(0, -0.002, 0.9)))
        comps.append(W.detector(-0.3, 0.3, -0.3, 0.3, 24, 24, 10.0, 60.0, 4, R=rot_x(0.1), T=(0, 0.0, 1.2)))
    else:
        comps.append(W.detector(-0.05, 0.05, -0.05, 0.05, 32, 32, 10.0, 60.0, 8, T=(0, 0, 1.0)))
    return W.instrument("mixed", comps, mats, n_rays)


def rot_x(a):
    c, s = np.cos(a), np.sin(a)
    return np.array([[1, 0, 0], [0, c, -s], [0, s, c]], dtype=float)


def test_mixed_chain_two_detectors(M, O, W):
    check(M, O, W, mixed_instrument(W, 120_000, with_mirror=False), 120_000)


def test_all_feature_bits(M, O, W):
    check(M, O, W, mixed_instrument(W, 120_000, with_mirror=True), 120_000)
