"""Pins on whole chains (SURVEY.md 8(c) "Pins": slab, slit, weight conservation, ray accounting, prefix)."""
import numpy as np


def test_c0_slit_acceptance_is_0p16(O, W):
    # acceptance = (4 mm / 10 mm)^2 exactly, independent of the source disk (north_star closed form)
    inst = W.config0()
    r = O.trace(inst)
    n = inst["n_rays"]
    assert abs(r["detected"] - 0.16 * n) < 5 * np.sqrt(n * 0.16 * 0.84)
    assert r["detected"] + r["missed"] + r["degenerate"] + int(r["absorbed"].sum()) == n
    assert int(r["absorbed"][1]) == n - r["detected"]            # everything else dies on the slit
    N = r["N"][0].reshape(128, 128)
    assert int(N.sum()) == r["detected"]
    ys, xs = np.nonzero(N)
    # slit shadow at the detector = 4x4 mm -> pixels 51..76 (+-2 mm at 0.15625 mm/pixel), all inside 48..79
    assert xs.min() >= 48 and xs.max() <= 79 and ys.min() >= 48 and ys.max() <= 79
    assert xs.min() <= 52 and xs.max() >= 75


def test_c0_slab_transmission_per_ray(O, W):
    # every slit-passing ray crosses both box faces: p = exp(-mu L / |d_z|), mu L = 0.6
    inst = W.config0(n_rays=20000)
    r = O.trace(inst, dump=True)
    src = inst["components"][0]
    det = np.nonzero(r["dump"]["fate"] == O.F_DETECTED)[0]
    assert len(det) > 2500
    for i in det[:400]:
        dz = O.source_ray(src, inst["seed"], int(i))[5]
        # chord = difference of two t ~ 0.8 m: cancellation leaves ~1e-16/5e-3 relative on the chord
        assert abs(r["dump"]["p"][i] - np.exp(-120.0 * 5e-3 / dz)) < 5e-14
    pm = r["P"][0].sum() / r["detected"]
    assert abs(pm - np.exp(-0.6)) < 1e-5                         # 0.54881, d_z within 1e-5 of 1
    assert abs(r["P2"][0].sum() / r["detected"] - np.exp(-1.2)) < 1e-5


def test_weight_conserved_without_absorbers(O, W):
    src = W.config0()["components"][0]
    det = W.detector(-10e-3, 10e-3, -10e-3, 10e-3, 16, 16, 0, 40, 1, T=(0, 0, 1.0))
    inst = W.instrument("free", [src, det], [None], 50_000)
    r = O.trace(inst)
    assert r["detected"] == 50_000 and int(r["N"][0].sum()) == 50_000
    assert r["P"][0].sum() == 50_000.0 and r["P2"][0].sum() == 50_000.0      # sums of ones: exact
    # uniform on the 10x10 mm target = the middle 8x8 pixels of this detector
    N = r["N"][0].reshape(16, 16)
    assert N[4:12, 4:12].sum() == 50_000
    assert abs(N[4:12, 4:12] / (50_000 / 64) - 1).max() < 0.2


def test_prefix_property_and_accumulation(O, W):
    # rays are pure functions of (seed, i); tallies are additive (reading R2)
    inst = W.config1(small=True)
    a = O.trace(inst, first=0, n=3000)
    b = O.trace(inst, first=0, n=1000)
    b = O.trace(inst, first=1000, n=2000, tallies=b)
    assert np.array_equal(a["N"][0], b["N"][0])
    assert np.allclose(a["P"][0], b["P"][0], rtol=0, atol=1e-12)
    assert a["detected"] == b["detected"]
    c = O.trace(inst, first=0, n=3000, seed=2)
    assert not np.array_equal(a["N"][0], c["N"][0])


def test_ray_accounting_all_configs(O, W):
    for k, n in ((1, 5000), (2, 20000), (3, 500), (4, 2000)):
        inst = W.config(k, small=True)
        r = O.trace(inst, n=n, dump=True)
        assert r["detected"] + r["missed"] + r["degenerate"] + int(r["absorbed"].sum()) == n
        assert int(r["N"][0].sum()) == r["detected"]
        d = r["dump"]
        assert (d["fate"] == O.F_DETECTED).sum() == r["detected"]
        assert np.all((d["bin"] >= 0) == (d["fate"] == O.F_DETECTED))
        # tallies rebuilt from the per-ray dump agree with the accumulated ones
        sel = d["fate"] == O.F_DETECTED
        P = np.bincount(d["bin"][sel], weights=d["p"][sel], minlength=len(r["P"][0]))
        assert np.allclose(P, r["P"][0], rtol=1e-13, atol=1e-300)
        assert np.all(d["p"] > 0) and np.all(d["p"] <= 1.0)


def test_detector_binning_centres_and_edges(O, W):
    det = W.detector(-4e-3, 4e-3, -2e-3, 2e-3, 8, 4, 10.0, 50.0, 4, T=(0, 0, 1.0))
    for ix in range(8):
        for iy in range(4):
            for ie in range(4):
                x, y, E = -4e-3 + (ix + 0.5) * 1e-3, -2e-3 + (iy + 0.5) * 1e-3, 10 + (ie + 0.5) * 10
                _, _, b = O.apply(det, [x, y, 0, 0, 0, 1, E, 1.0])
                assert b == (iy * 8 + ix) * 4 + ie
    # half-open: lower edge belongs to the bin, upper edge of the last bin is outside
    assert O.apply(det, [-4e-3, -2e-3, 0, 0, 0, 1, 10.0, 1.0])[2] == 0
    assert O.apply(det, [4e-3, 0, 0, 0, 0, 1, 20.0, 1.0])[2] == -1
    assert O.apply(det, [0, 2e-3, 0, 0, 0, 1, 20.0, 1.0])[2] == -1
    assert O.apply(det, [0, 0, 0, 0, 0, 1, 50.0, 1.0])[2] == -1
    assert O.apply(det, [0, 0, 0, 0, 0, 1, 9.999, 1.0])[2] == -1
    # backwards ray, ray behind the plane: missed
    assert O.apply(det, [0, 0, 0, 0, 0, -1, 20.0, 1.0])[2] == -1
    assert O.apply(det, [0, 0, 2.0, 0, 0, 1, 20.0, 1.0])[2] == -1
    # oblique ray: lands where the line meets the plane
    d = np.array([1e-3, 0.5e-3, 1.0]); d /= np.linalg.norm(d)
    assert O.apply(det, [0, 0, 0, *d, 20.0, 1.0])[2] == (2 * 8 + 5) * 4 + 1
    # rotated / translated detector: pose is honoured
    Rz = np.array([[0, 1.0, 0], [-1.0, 0, 0], [0, 0, 1.0]])      # local x = lab y
    det2 = W.detector(-4e-3, 4e-3, -2e-3, 2e-3, 8, 4, 10.0, 50.0, 4, R=Rz, T=(1e-3, 0, 1.0))
    # lab point (1e-3 + 0.5e-3 ... ) -> local x = lab y = 2.5e-3 (ix 6), local y = -(lab x - 1e-3) = -0.5e-3 (iy 1)
    assert O.apply(det2, [1.5e-3, 2.5e-3, 0, 0, 0, 1, 20.0, 1.0])[2] == (1 * 8 + 6) * 4 + 1


def test_slits(O, W):
    s = W.slit_rect(2e-3, 1e-3, T=(0, 0, 0.5))
    assert O.apply(s, [0.999e-3, -0.499e-3, 0, 0, 0, 1, 20, 1])[0] == 1
    assert O.apply(s, [1e-3, 0.5e-3, 0, 0, 0, 1, 20, 1])[0] == 1          # edge inclusive (R10)
    assert O.apply(s, [1.001e-3, 0, 0, 0, 0, 1, 20, 1])[0] == 0
    assert O.apply(s, [0, 0.501e-3, 0, 0, 0, 1, 20, 1])[0] == 0
    assert O.apply(s, [0, 0, 0, 0, 0, -1, 20, 1])[0] == 0                 # backwards
    assert O.apply(s, [0, 0, 1.0, 0, 0, 1, 20, 1])[0] == 0                # already past it
    c = W.slit_circ(1e-3, T=(0, 0, 0.5))
    assert O.apply(c, [0.7e-3, 0.7e-3, 0, 0, 0, 1, 20, 1])[0] == 1
    assert O.apply(c, [0.72e-3, 0.72e-3, 0, 0, 0, 1, 20, 1])[0] == 0
    # the slit does not change the ray
    rc, st, _ = O.apply(s, [0.1e-3, 0.2e-3, 0, 0, 0, 1, 20, 0.7])
    assert rc == 1 and np.array_equal(st, [0.1e-3, 0.2e-3, 0, 0, 0, 1, 20, 0.7])


def test_fate_with_several_detectors_is_what_the_last_component_said(O, W):
    """DESIGN.md section 2, step 14 (a reading; the paper only says monitors measure "at given points"):
    a monitor never ends a ray, every monitor the ray crosses tallies it, and the ray's FATE is decided by where the
    chain ends for it -- absorbed at component c, else DETECTED / MISSED by the LAST component of the chain (MISSED if
    that is not a detector).  Pinned against plain plane geometry written out here in numpy."""
    src = W.source("point", "target", "mono", target_w=20e-3, target_h=20e-3, target_dist=1.0, E0=20.0)
    detA = W.detector(-3e-3, 3e-3, -3e-3, 3e-3, 6, 6, 0.0, 40.0, 1, T=(0, 0, 0.4))
    slit = W.slit_rect(8e-3, 8e-3, T=(0, 0, 0.6))
    detB = W.detector(-5e-3, 5e-3, -5e-3, 5e-3, 10, 10, 0.0, 40.0, 1, T=(0, 0, 1.0))
    n = 6000
    inst = W.instrument("two_monitors", [src, detA, slit, detB], [None], n)
    r = O.trace(inst, dump=True)
    rays = np.array([O.source_ray(src, inst["seed"], i) for i in range(n)])
    at = lambda z: rays[:, 3:5] / rays[:, 5:6] * z                     # (x, y) where the line meets the plane z
    a, s, b = at(0.4), at(0.6), at(1.0)
    inA = np.all((a >= -3e-3) & (a < 3e-3), axis=1)
    passes = np.all(np.abs(s) <= 4e-3, axis=1)
    inB = np.all((b >= -5e-3) & (b < 5e-3), axis=1)
    expect = np.where(~passes, 2, np.where(inB, O.F_DETECTED, O.F_MISSED))
    assert np.array_equal(r["dump"]["fate"], expect)
    assert (inA & ~passes).sum() > 100 and (inA & passes & inB).sum() > 100 and (~passes).sum() > 100 and (passes & ~inB).sum() > 100
    # both monitors tally every ray that crosses them, whatever happens to it afterwards
    assert int(r["N"][0].sum()) == inA.sum() and int(r["N"][1].sum()) == (passes & inB).sum() == r["detected"]
    binB = (np.floor((b[:, 1] + 5e-3) / 1e-3) * 10 + np.floor((b[:, 0] + 5e-3) / 1e-3)).astype(np.int64)
    sel = expect == O.F_DETECTED
    assert np.array_equal(r["dump"]["bin"][sel], binB[sel]) and np.all(r["dump"]["bin"][~sel] == -1)
    # a slit AFTER the first monitor that absorbs rays the monitor has already counted
    tight = W.slit_rect(2e-3, 2e-3, T=(0, 0, 0.6))
    r2 = O.trace(W.instrument("monitor_then_slit", [src, detA, tight, detB], [None], n), dump=True)
    passes2 = np.all(np.abs(s) <= 1e-3, axis=1)
    assert (inA & ~passes2).sum() > 100
    assert np.array_equal(r2["dump"]["fate"], np.where(~passes2, 2, O.F_DETECTED))      # a passing ray always lands in B
    assert int(r2["N"][0].sum()) == inA.sum() and int(r2["absorbed"][2]) == (~passes2).sum()
    # a chain that ENDS with a non-detector: nobody is DETECTED although monitor A has counted its rays
    r3 = O.trace(W.instrument("monitor_not_last", [src, detA, slit], [None], n), dump=True)
    assert np.array_equal(r3["dump"]["fate"], np.where(passes, O.F_MISSED, 2))
    assert r3["detected"] == 0 and r3["missed"] == passes.sum() and int(r3["N"][0].sum()) == inA.sum()
    assert np.all(r3["dump"]["bin"] == -1)


def test_closed_meshes_never_degenerate_over_a_million_rays(O, W):
    # SURVEY.md 8(c) "Pins", mesh row: an even, alternating crossing count for every ray of a closed outward-wound mesh
    inst = W.config3(small=True)
    r = O.trace(inst, n=1_000_000, mesh_accel=1)
    assert r["degenerate"] == 0 and r["detected"] + r["missed"] == 1_000_000
