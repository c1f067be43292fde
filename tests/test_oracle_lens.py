"""Pins for the oracle's SURVEY.md 8(f) steps: the compound refractive lens (step 16), the
Darwin-Prins curve (step 13b) and wavelength bins (step 14b).  Each pin is something the mathematics
fixes outside the oracle: thin-lens optics, Snell's law on a plane-parallel plate, Beer-Lambert on a known thickness
profile, time reversal, closed forms and numpy's complex arithmetic."""
import numpy as np

HC = 12.398419843
RNG = np.random.default_rng(16)


def unit(v):
    v = np.asarray(v, dtype=float)
    return v / np.linalg.norm(v)


def flat_delta(delta):
    return {"E": np.array([1.0, 100.0]), "delta": np.array([delta, delta])}


def flat_mu(mu):
    return {"E": np.array([1.0, 100.0]), "mu": np.array([mu, mu])}


def test_thin_lens_deflection_and_focal_length(O, W):
    # paraxial ray parallel to the axis at height x: N thin lenses deflect it by 2 N delta x / R towards the axis
    # (lens maker: 1/f = 2 delta / R per double-sided lens).  R = 0.1 m, x <= 1e-4 m: (x / R)^2 <= 1e-6.
    Rc, delta = 0.1, 3e-6
    for N in (1, 4):
        L = W.lens_parab(Rc, 1e-5, 2e-5, 5e-4, N, 1, flat_delta(delta))
        for x, y in ((1e-4, 0.0), (0.0, -5e-5), (3e-5, 4e-5)):
            rc, st, _ = O.apply(L, [x, y, -1.0, 0, 0, 1, 20.0, 1.0], materials=(None, flat_mu(1e-9)))
            assert rc == 1
            dx, dy = st[3] / st[5], st[4] / st[5]
            for got, h in ((dx, x), (dy, y)):
                want = -2 * N * delta * h / Rc
                assert abs(got - want) <= 2e-5 * abs(want) + 1e-18
            assert abs(np.linalg.norm(st[3:6]) - 1) < 1e-15


def test_thick_stack_focal_length(O, W):
    # the paper's lens (N = 16, R = 200 um) with delta of Be near 23 keV: a parallel paraxial ray crosses
    # the axis at f = R / (2 N delta) + L / 6 behind the centre of the stack (thick-CRL correction, L = N pitch)
    Rc, N, pitch, delta = 200e-6, 16, 1.3e-3, 6.27e-7
    L = W.lens_parab(Rc, 50e-6, pitch, 0.5e-3, N, 1, flat_delta(delta))
    f0 = Rc / (2 * N * delta)
    for x in (2e-6, 5e-6):
        rc, st, _ = O.apply(L, [x, 0, -0.1, 0, 0, 1, 23.32, 1.0], materials=(None, flat_mu(1e-9)))
        assert rc == 1
        z_cross = st[2] - st[0] * st[5] / st[3]
        assert abs(z_cross - (f0 + N * pitch / 6)) < 2e-4 * f0          # (x / R)^2 ~ 6e-4 at x = 5 um; f0 = 9.97 m
        assert abs(z_cross - f0) > 1e-3                                 # the L / 6 term (3.5 mm) is resolved


def test_plane_parallel_plate_is_snells_law(O, W):
    # R -> infinity: one lens is a plate of thickness d.  An oblique ray leaves parallel to itself, displaced sideways by
    # d sin(tt - ti) / cos(tt) with sin(ti) = n sin(tt), n = 1 - delta (delta = 0.3 makes the law visible), and its
    # path inside is d / cos(tt)
    d_web, delta, mu = 2e-3, 0.3, 40.0
    L = W.lens_parab(1e12, d_web, 1e-2, 1.0, 1, 1, flat_delta(delta))
    n = 1 - delta
    for ti in (0.05, 0.3, 0.6):                                         # sin(0.6) / 0.7 = 0.807 < 1: no total reflection
        d = np.array([np.sin(ti), 0.0, np.cos(ti)])
        o = np.array([0.0, 0.0, -1e-3 - d_web / 2]) - 0.0 * d
        rc, st, _ = O.apply(L, [*o, *d, 20.0, 1.0], materials=(None, flat_mu(mu)))
        assert rc == 1
        assert np.allclose(st[3:6], d, atol=1e-15)
        tt = np.arcsin(np.sin(ti) / n)
        # exit point on the back face z = +d/2
        assert abs(st[2] - d_web / 2) < 1e-12
        x_straight = o[0] + (st[2] - o[2]) * np.tan(ti)
        shift = d_web * np.sin(tt - ti) / np.cos(tt)                    # = d (tan tt - tan ti) cos ti > 0: n < 1 bends away from the normal
        assert abs((st[0] - x_straight) * np.cos(ti) - shift) < 1e-13
        assert abs(st[7] - np.exp(-mu * d_web / np.cos(tt))) < 1e-14
    # beyond the critical angle of the entrance face there is no transmitted ray: absorbed
    ti = np.arcsin(n) + 0.01
    rc, _, _ = O.apply(L, [0, 0, -1e-3, np.sin(ti), 0, np.cos(ti), 20.0, 1.0], materials=(None, flat_mu(mu)))
    assert rc == 0


def test_on_axis_and_thickness_profile(O, W):
    # no refraction to speak of (delta = 1e-15: the focusing moves the ray by 1e-16 m): the ray is straight and sees N (d + rho^2 / R) of material
    Rc, N, d_web, mu = 200e-6, 16, 50e-6, 150.0
    L = W.lens_parab(Rc, d_web, 1.3e-3, 0.5e-3, N, 1, flat_delta(1e-15))
    rc, st, _ = O.apply(L, [0, 0, -1.0, 0, 0, 1, 23.0, 1.0], materials=(None, flat_mu(mu)))
    assert rc == 1 and np.allclose(st[3:6], [0, 0, 1], atol=0) and abs(st[7] - np.exp(-mu * N * d_web)) < 1e-12
    for _ in range(50):
        x, y = RNG.uniform(-3e-4, 3e-4, size=2)
        rc, st, _ = O.apply(L, [x, y, -1.0, 0, 0, 1, 23.0, 1.0], materials=(None, flat_mu(mu)))
        assert rc == 1
        assert abs(st[7] - np.exp(-mu * N * (d_web + (x * x + y * y) / Rc))) < 1e-12
    # the holder absorbs what falls outside the aperture; a ray travelling backwards never enters
    assert O.apply(L, [0.5001e-3, 0, -1.0, 0, 0, 1, 23.0, 1.0], materials=(None, flat_mu(mu)))[0] == 0
    assert O.apply(L, [0.4999e-3, 0, -1.0, 0, 0, 1, 23.0, 1.0], materials=(None, flat_mu(mu)))[0] == 1
    assert O.apply(L, [0, 0, 1.0, 0, 0, -1, 23.0, 1.0], materials=(None, flat_mu(mu)))[0] == 0


def test_delta_is_interpolated_like_mu(O, W):
    # delta(E) = A E^-2 is a power law: log-log interpolation reproduces it, so the deflection scales as E^-2
    E = np.exp(np.linspace(np.log(5.0), np.log(50.0), 40))
    tab = {"E": E, "delta": 3.4e-4 / E ** 2}
    L = W.lens_parab(0.1, 1e-5, 2e-5, 5e-4, 1, 1, tab)
    x = 1e-4
    for Eq in (7.3, 23.32, 41.0):
        rc, st, _ = O.apply(L, [x, 0, -1.0, 0, 0, 1, Eq, 1.0], materials=(None, flat_mu(1e-9)))
        want = -2 * (3.4e-4 / Eq ** 2) * x / 0.1
        assert abs(st[3] / st[5] - want) < 2e-5 * abs(want)


def test_reversibility(O, W):
    # the stack is symmetric under z -> -z, so the same lens turned by 180 degrees about x takes the reversed exit ray
    # back onto the entrance ray
    Rc, N = 200e-6, 16
    tab = flat_delta(5e-6)
    fwd = W.lens_parab(Rc, 50e-6, 1.3e-3, 0.5e-3, N, 1, tab)
    back = W.lens_parab(Rc, 50e-6, 1.3e-3, 0.5e-3, N, 1, tab, R=np.diag([1.0, -1.0, -1.0]))
    mats = (None, flat_mu(30.0))
    n = 0
    for _ in range(40):
        o = np.array([*RNG.uniform(-2e-4, 2e-4, size=2), -0.05])
        d = unit([*RNG.uniform(-2e-4, 2e-4, size=2), 1.0])
        rc, st, _ = O.apply(fwd, [*o, *d, 20.0, 1.0], materials=mats)
        if rc != 1:
            continue
        start = st[0:3] + 1e-3 * st[3:6]                                # a millimetre behind the last surface
        rc2, st2, _ = O.apply(back, [*start, *(-st[3:6]), 20.0, 1.0], materials=mats)
        assert rc2 == 1
        n += 1
        assert np.allclose(st2[3:6], -d, atol=1e-14)
        assert np.linalg.norm(np.cross(st2[0:3] - o, d)) < 1e-15 + 1e-13 * 0.05
        assert abs(st2[7] - st[7]) < 1e-14                              # same chords both ways
    assert n > 30


def test_lens_in_a_chain_counts_and_images(O, W):
    # point source on the axis at p, lens, detector at the image distance q with 1/p + 1/q = 1/f (thick correction as
    # above): all rays that pass the aperture land within a spot far smaller than the aperture
    Rc, N, pitch, delta = 200e-6, 16, 1.3e-3, 6.27e-7
    f = Rc / (2 * N * delta) + N * pitch / 6
    p = 31.5
    q = 1 / (1 / f - 1 / p)
    comps = [W.source("point", "target", "mono", target_w=1e-3, target_h=1e-3, target_dist=p, E0=23.32),
             W.lens_parab(Rc, 50e-6, pitch, 0.5e-3, N, 1, flat_delta(delta), T=(0, 0, p)),
             W.detector(-5e-6, 5e-6, -5e-6, 5e-6, 10, 10, 0.0, 40.0, 1, T=(0, 0, p + q))]
    inst = W.instrument("lens_chain", comps, [None, flat_mu(1e-6)], 20000)
    o = O.trace(inst, n=20000)
    frac = np.pi / 4                                                    # circular aperture in the square window
    assert abs(int(o["absorbed"][1]) / 20000 - (1 - frac)) < 4 * np.sqrt(frac * (1 - frac) / 20000)
    assert o["detected"] == 20000 - int(o["absorbed"][1])               # a 10 um detector catches every focused ray
    img = o["N"][0].reshape(10, 10)
    assert img[4:6, 4:6].sum() > 0.9 * o["detected"]                    # spherical aberration ~ x^3 / R^2-scale: microns


def test_darwin_prins_closed_forms(O):
    # g = kappa = 0 is the Darwin curve; eta = 0, kappa = 0: R = (sqrt(1 + g^2) - g)^2; anywhere: numpy complex arithmetic
    for eta in (-3.0, -1.0, -0.3, 0.0, 0.9, 1.0, 1.5, 20.0):
        assert O.darwin_prins(eta, 0.0, 0.0) == O.darwin(eta)
        assert abs(O.darwin_prins(eta, 1e-12, 0.0) - O.darwin(eta)) < 3e-6      # continuity in g (sqrt(g) at |eta| = 1)
    for g in (0.01, 0.1, 1.0):
        assert abs(O.darwin_prins(0.0, g, 0.0) - (np.sqrt(1 + g * g) - g) ** 2) < 1e-15
    for eta in np.linspace(-6, 6, 97):
        for g, kappa in ((0.05, 0.0), (0.1, 0.02), (0.3, -0.1)):
            ec = (eta + 1j * g) / (1 + 1j * kappa)
            s = np.sqrt(ec * ec - 1 + 0j)
            want = min(abs(ec - s) ** 2, abs(ec + s) ** 2)
            got = O.darwin_prins(eta, g, kappa)
            assert abs(got - want) < 1e-13 and got <= 1.0
    # absorption lowers the plateau; the curve stays even in eta for kappa = 0 and is skewed by kappa != 0
    # (R(eta_c) = R(-conj(eta_c))); tails ~ 1 / (4 eta^2)
    assert O.darwin_prins(0.5, 0.1, 0.0) < 1.0
    assert abs(O.darwin_prins(-0.9, 0.1, 0.0) - O.darwin_prins(0.9, 0.1, 0.0)) < 1e-15
    assert abs(O.darwin_prins(-0.9, 0.1, 0.05) - O.darwin_prins(0.9, 0.1, 0.05)) > 1e-3
    assert abs(O.darwin_prins(50.0, 0.1, 0.0) * 4 * 50.0 ** 2 - 1) < 2e-3


def test_crystal_uses_the_prins_curve(O, W):
    d_hkl, zeta, E = 3.135601154, 1.33e-4, 12.0
    thB = np.arcsin(HC / E / (2 * d_hkl))
    for g, kappa in ((0.0, 0.0), (0.08, 0.01)):
        X = W.crystal_bragg(0.05, 0.02, d_hkl, zeta, g=g, kappa=kappa)
        for eta in (-2.0, 0.0, 0.5, 3.0):
            th = thB + eta * 0.5 * zeta * np.tan(thB)
            rc, st, _ = O.apply(X, [0, 0.01 * np.sin(th), -0.01 * np.cos(th), 0, -np.sin(th), np.cos(th), E, 1.0])
            assert rc == 1
            eta_eff = (np.arcsin(np.sin(th)) - thB) / (0.5 * zeta * np.tan(thB))
            assert abs(st[7] - O.darwin_prins(eta_eff, g, kappa)) < 1e-9   # d R / d eta <= ~1 near |eta| = 1, asin roundings 1e-12


def test_wavelength_bins(O, W):
    # an L_monitor bins lambda = hc / E: E = hc / lambda_centre of bin k lands in bin k; half-open edges
    nL, lmin, lmax = 20, 2.0, 3.2
    det = W.detector(-0.01, 0.01, -0.01, 0.01, 1, 1, lmin, lmax, nL, T=(0, 0, 1.0), mode="wavelength")
    for k in range(nL):
        lam = lmin + (k + 0.5) * (lmax - lmin) / nL
        rc, _, b = O.apply(det, [0, 0, 0, 0, 0, 1, HC / lam, 1.0])
        assert b == k
    assert O.apply(det, [0, 0, 0, 0, 0, 1, HC / 1.99, 1.0])[2] == -1
    assert O.apply(det, [0, 0, 0, 0, 0, 1, HC / 3.21, 1.0])[2] == -1
    # the same detector in energy mode reads the range as keV
    det_e = W.detector(-0.01, 0.01, -0.01, 0.01, 1, 1, lmin, lmax, nL, T=(0, 0, 1.0))
    assert O.apply(det_e, [0, 0, 0, 0, 0, 1, 2.03, 1.0])[2] == 0
