"""-m gpu: every combination of the source's position / direction / energy modes (step 3), a circular slit, a tilted
detector whose energy range cuts the spectrum (rays outside are MISSED, not absorbed), and a chain the rays leave
backwards -- against the oracle, ray by ray."""
import itertools

import numpy as np
import pytest

from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


def rot_y(a):
    c, s = np.cos(a), np.sin(a)
    return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]], dtype=float)


@pytest.mark.parametrize("pos,dirm,em", list(itertools.product(("point", "disk", "gauss"), ("target", "gauss"),
                                                               ("mono", "uniform", "spectrum"))))
def test_source_modes(M, O, W, pos, dirm, em):
    rng = np.random.default_rng(5)
    spec = W.bremsstrahlung_spectrum(rng, 97, 8.0, 40.0, 40.0)
    comps = [
        W.source(pos, dirm, em, radius=2e-3, sigma_x=1e-3, sigma_y=5e-4, target_w=0.04, target_h=0.03, target_dist=0.8,
                 div_x=0.02, div_y=0.01, E0=20.0, dE_rel=0.3, spec_Emin=8.0, spec_Emax=40.0, spectrum=spec,
                 R=rot_y(0.01), T=(1e-3, -2e-3, 0.0)),
        W.slit_circ(0.012, T=(0, 0, 0.4)),
        # tilted detector; its energy window (12-30 keV) is narrower than any of the three spectra
        W.detector(-0.03, 0.03, -0.02, 0.02, 24, 16, 12.0, 30.0, 6, R=rot_y(0.2), T=(0.002, 0, 0.8)),
    ]
    check(M, O, W, W.instrument("source_modes", comps, [None], 40_000), 40_000)


def test_rays_leaving_backwards(M, O, W):
    """second slit faces the other way (its local z points back at the source): every ray that reaches it is absorbed
    there (d'_z <= 0, step 5); the detector behind it sees nothing"""
    comps = [
        W.source("disk", "target", "mono", radius=1e-3, target_w=0.02, target_h=0.02, target_dist=1.0, E0=15.0),
        W.slit_rect(0.01, 0.01, T=(0, 0, 0.3)),
        W.slit_rect(0.05, 0.05, R=rot_y(np.pi), T=(0, 0, 0.6)),
        W.detector(-0.02, 0.02, -0.02, 0.02, 8, 8, 10.0, 20.0, 1, T=(0, 0, 1.0)),
    ]
    check(M, O, W, W.instrument("backwards", comps, [None], 20_000), 20_000)
