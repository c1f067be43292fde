"""-m gpu: the SURVEY.md 8(f) rows on the CUDA path against the oracle: the paper's three instruments (basic instrument
with an L_monitor; focusing instrument with a compound refractive lens; EDXCT line
scanner with five tilted line detectors), the Darwin-Prins curve, the line scan with
mcx_instrument_set_pose and the CNR of Eq. (1)."""
import numpy as np
import pytest

from _parity import assert_tally_parity
from test_gpu_parity import M, check  # noqa: F401  (M is a fixture)

pytestmark = pytest.mark.gpu


def test_c5_basic_instrument_wavelength_monitor(M, O, W):
    st = check(M, O, W, W.config5(small=True), 150_003)
    assert st["n_diff"] == 0
    check(M, O, W, W.config5(), 40_000)


def test_c6_focusing_instrument_lens(M, O, W):
    check(M, O, W, W.config6(small=True), 200_001)
    check(M, O, W, W.config6(), 50_000)


def test_lens_edge_cases(M, O, W):
    rng = np.random.default_rng(5)
    tab = W.delta_table(rng, Emin=5.0, Emax=60.0, A=0.5)                # huge delta (2e-2 .. 1e-3): strong refraction, total reflection
    mu = {"E": np.array([1.0, 100.0]), "mu": np.array([300.0, 80.0])}
    c, s = np.cos(0.02), np.sin(0.02)
    tilt = np.array([[1, 0, 0], [0, c, -s], [0, s, c]], dtype=float)
    for n_lenses, R in ((1, None), (7, tilt), (40, None)):
        comps = [W.source("disk", "target", "uniform", radius=2e-4, target_w=2.4e-3, target_h=2.4e-3, target_dist=0.5, E0=20.0,
                          dE_rel=0.6),
                 W.lens_parab(1e-3, 1e-4, 1.4e-3, 1.1e-3, n_lenses, 1, tab, R=R, T=(1e-5, -2e-5, 0.5)),
                 W.detector(-0.02, 0.02, -0.02, 0.02, 40, 40, 5.0, 40.0, 8, T=(0, 0, 1.0))]
        inst = W.instrument("lens_edges", comps, [None, mu], 60_000)
        st = check(M, O, W, inst, 60_001)
        o = O.trace(inst, n=60_001)
        assert 0 < int(o["absorbed"][1]) < 60_001                       # some rays miss the aperture or reflect totally


def test_c7_edxct_line_detectors(M, O, W):
    check(M, O, W, W.config7(small=True), 120_007)


def test_c7_full_size_prefix(M, O, W):
    inst = W.config7()
    check(M, O, W, inst, 30_000)


def test_darwin_prins_crystals_in_the_beamline(M, O, W):
    inst = W.config2(small=True)
    for c in inst["components"]:
        if c["kind"] == "crystal":
            c.update(g=0.08, kappa=0.015)
    check(M, O, W, inst, 400_003)


def test_line_scan_with_set_pose(M, O, W):
    # the sample moves between traces (one simulation per imaged line); per line the tallies must equal the
    # oracle's for an instrument built with the sample at that position
    inst = W.config7(small=True)
    g = M.Instrument(inst)
    n = 30_000
    comp = inst["sample_component"]
    for line, T in enumerate(inst["scan"][2:9:3]):
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
    # a pose that would turn the volume's fast axis is refused, as is the source or a solids group
    flip = np.array([[0, 0, 1.0], [0, 1.0, 0], [-1.0, 0, 0]])
    with pytest.raises(M.McxError):
        g.set_pose(comp, R=flip, T=(0.3, 0, 1.8))
    with pytest.raises(M.McxError):
        g.set_pose(0, T=(0, 0, 0))
    g.close()


def test_cnr_matches_the_oracle(M, O, W):
    inst = W.config4(small=True)
    g = M.Instrument(inst)
    g.trace(3_000_000)
    N, P, P2 = g.tally(0)
    d = g.dets[0]
    for rm, rr, efit in (((10, 20, 10, 20), (40, 50, 30, 40), 80.0), ((0, 64, 0, 1), (3, 4, 5, 64), 20.0), ((5, 6, 5, 6), (7, 9, 7, 8), 149.0)):
        c, fit = g.cnr(0, rm, rr, efit, tallies=(N, P, P2))
        oc, oa, ob = O.cnr(N.cpu().numpy().view(np.uint64), P.cpu().numpy(), P2.cpu().numpy(), d["ny"], d["nx"], d["nE"], rm, rr,
                           d["Emin"], d["Emax"], efit)
        c, fit = c.cpu().numpy(), fit.cpu().numpy()
        assert np.allclose(c, oc, rtol=1e-11, atol=1e-300)
        assert abs(fit[0] - oa) <= 1e-9 * max(1.0, abs(oa)) and abs(fit[1] - ob) <= 1e-9 * max(1.0, abs(ob))
    with pytest.raises(M.McxError):
        g.cnr(0, (0, 65, 0, 1), (0, 1, 0, 1), 80.0, tallies=(N, P, P2))
    g.close()
