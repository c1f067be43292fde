"""Pins for oracle steps 12-13: elliptic mirror (focal property, bilinear table) and Darwin-curve crystal."""
import numpy as np
from scipy import integrate

RNG = np.random.default_rng(77)


def unit(v):
    v = np.asarray(v, dtype=float)
    return v / np.linalg.norm(v)


def const_table(val=1.0, n_theta=5, n_E=4):
    return {"theta_min": 0.0, "theta_max": 8e-3, "n_theta": n_theta, "E_min": 5.0, "E_max": 25.0, "n_E": n_E,
            "R": np.full((n_theta, n_E), val)}


def test_mirror_constants(O):
    p, q, th = 30.0, 10.4, 3e-3
    m = O.mirror_prep(p, q, th)
    assert abs(m["a"] - 20.2) < 1e-14 and abs(m["b"] - np.sqrt(p * q) * np.sin(th)) < 1e-16
    c = np.sqrt(m["a"] ** 2 - m["b"] ** 2)
    assert abs(m["Z0"] ** 2 / m["a"] ** 2 + m["Y0"] ** 2 / m["b"] ** 2 - 1) < 1e-12       # pole on the ellipse
    assert abs(np.hypot(m["Z0"] + c, m["Y0"]) - p) < 1e-11 and abs(np.hypot(m["Z0"] - c, m["Y0"]) - q) < 1e-11
    assert abs(m["nZ"] ** 2 + m["nY"] ** 2 - 1) < 1e-15 and m["nY"] > 0 and m["tZ"] > 0
    assert abs(m["nZ"] * m["tZ"] + m["nY"] * m["tY"]) < 1e-16
    # grazing angle of the F1 -> pole ray against the tangent is theta
    v = unit([m["Z0"] + c, m["Y0"]])
    assert abs(np.arcsin(-(v[0] * m["nZ"] + v[1] * m["nY"])) - th) < 1e-12


def test_ellipse_focal_property(O, W):
    # every ray from focus F1 that hits the arc passes through F2 after reflection; path F1->P->F2 = 2a
    p, q, th, L, Wd = 30.0, 10.4, 3e-3, 0.1, 10e-3
    mir = W.mirror_elliptic(p, q, th, L, Wd, const_table(1.0))
    F1 = np.array([0.0, p * np.sin(th), -p * np.cos(th)])
    F2 = np.array([0.0, q * np.sin(th), q * np.cos(th)])
    n = 0
    for _ in range(300):
        aim = np.array([0.0, 0.0, RNG.uniform(-0.6 * L, 0.6 * L)])      # meridional rays: the 2-D focal property
        d = unit(aim - F1)
        rc, st, _ = O.apply(mir, [*F1, *d, 12.0, 1.0])
        if abs(aim[2]) > 0.5 * L + 2e-4:
            assert rc == 0
            continue
        if rc == 0:
            continue
        n += 1
        P, dr = st[0:3], st[3:6]
        assert abs(np.linalg.norm(dr) - 1) < 1e-14 and st[7] == 1.0
        miss = np.linalg.norm(np.cross(F2 - P, dr))
        assert miss < 1e-10                                            # metres; fp64 at a = 20 m, 1/theta = 333
        assert abs(np.linalg.norm(P - F1) + np.linalg.norm(F2 - P) - (p + q)) < 1e-12
        # on the arc: concave towards +y with the pole's radius of curvature 2pq / ((p+q) sin theta)
        Rc = 2 * p * q / ((p + q) * np.sin(th))
        assert abs(P[2]) <= 0.5 * L and abs(P[1] - P[2] ** 2 / (2 * Rc)) < 2e-3 * P[2] ** 2 / (2 * Rc) + 1e-13
    assert n > 150
    # sagittal offset: a cylinder focuses in its meridional plane only -- the (y,z) projection still focuses
    aim = np.array([3e-3, 0.0, 0.02])
    rc, st, _ = O.apply(mir, [*F1, *unit(aim - F1), 12.0, 1.0])
    assert rc == 1
    P, dr = st[0:3], st[3:6]
    s = (F2[2] - P[2]) / dr[2]
    assert abs(P[1] + s * dr[1] - F2[1]) < 1e-9


def test_mirror_absorbs_misses_and_back_side(O, W):
    p, q, th, L, Wd = 30.0, 10.4, 3e-3, 0.1, 10e-3
    mir = W.mirror_elliptic(p, q, th, L, Wd, const_table(0.5))
    F1 = np.array([0.0, p * np.sin(th), -p * np.cos(th)])
    assert O.apply(mir, [*F1, *unit(np.array([0, 0, 0.02]) - F1), 12.0, 1.0])[1][7] == 0.5
    assert O.apply(mir, [*F1, *unit(np.array([0, 0, 0.051]) - F1), 12.0, 1.0])[0] == 0          # beyond the length
    assert O.apply(mir, [*F1, *unit(np.array([5.1e-3, 0, 0.0]) - F1), 12.0, 1.0])[0] == 0        # beyond the width
    assert O.apply(mir, [0, -1.0, -1.0, *unit([0, 1, 1]), 12.0, 1.0])[0] == 0                    # from behind
    assert O.apply(mir, [0, 1e-3, -1.0, 0, 0, 1.0, 12.0, 1.0])[0] == 0                           # passes above it
    # grazing angle above the table range -> absorbed
    steep = np.array([0.0, 1.0 * np.sin(20e-3), -1.0 * np.cos(20e-3)])
    assert O.apply(mir, [*steep, *unit(-steep), 12.0, 1.0])[0] == 0


def test_bilinear_table(O, W):
    nt, nE = 7, 9
    th = np.linspace(1e-3, 8e-3, nt); E = np.linspace(5.0, 25.0, nE)
    al, be, ga, de = 0.3, 40.0, 0.01, -2.0
    tab = {"theta_min": 1e-3, "theta_max": 8e-3, "n_theta": nt, "E_min": 5.0, "E_max": 25.0, "n_E": nE,
           "R": al + be * th[:, None] + ga * E[None, :] + de * th[:, None] * E[None, :]}
    mir = W.mirror_elliptic(30, 10, 3e-3, 0.1, 0.01, tab)
    for i in range(nt):
        for j in range(nE):
            assert abs(O.bilinear(mir, th[i], E[j]) - tab["R"][i, j]) < 1e-15                    # exact at nodes
    for _ in range(200):
        t, e = RNG.uniform(1e-3, 8e-3), RNG.uniform(5, 25)
        assert abs(O.bilinear(mir, t, e) - (al + be * t + ga * e + de * t * e)) < 1e-14          # exact for bilinear f
    # clamping: below theta range and outside the energy range
    assert abs(O.bilinear(mir, 0.0, 10.0) - O.bilinear(mir, 1e-3, 10.0)) < 1e-16
    assert abs(O.bilinear(mir, 4e-3, 30.0) - O.bilinear(mir, 4e-3, 25.0)) < 1e-16
    assert abs(O.bilinear(mir, 4e-3, 1.0) - O.bilinear(mir, 4e-3, 5.0)) < 1e-16
    # a non-bilinear table is NOT reproduced between nodes but stays within the cell's corner values
    tab2 = dict(tab); tab2["R"] = RNG.random((nt, nE))
    mir2 = W.mirror_elliptic(30, 10, 3e-3, 0.1, 0.01, tab2)
    v = O.bilinear(mir2, 0.5 * (th[2] + th[3]), 0.5 * (E[4] + E[5]))
    assert abs(v - tab2["R"][2:4, 4:6].mean()) < 1e-15


def test_darwin_curve_closed_forms(O):
    for eta in (-1.0, -0.3, 0.0, 0.99, 1.0):
        assert O.darwin(eta) == 1.0
    assert abs(O.darwin(np.sqrt(2)) - (np.sqrt(2) - 1) ** 2) < 1e-15      # 0.1715728753 (rhs cancels: 1 ulp)
    assert abs(O.darwin(np.sqrt(2)) - 0.1715728753) < 1e-10
    assert O.darwin(-3.0) == O.darwin(3.0)
    assert abs(O.darwin(1e6) * 4e12 - 1) < 1e-6                             # tail 1/(4 eta^2), no cancellation
    tail, _ = integrate.quad(O.darwin, 1.0, np.inf, epsabs=1e-12, epsrel=1e-12)
    assert abs(tail - 1 / 3) < 1e-9                                         # so the full integral is 2 + 2/3 = 8/3


def test_crystal_bragg_reflection(O, W):
    d111, zeta = W.SI_D111, 1.33e-4
    xt = W.crystal_bragg(0.05, 0.02, d111, zeta)
    E = 12.0
    thB = np.arcsin(12.398419843 / E / (2 * d111))
    assert abs(thB - 0.16550795) < 1e-8                                     # SURVEY 8(c) pins
    wD = zeta * np.tan(thB)
    assert abs(wD - 22.2e-6) < 0.1e-6

    def shoot(theta, E=E, x=0.0, z=0.0):
        d = np.array([0.0, -np.sin(theta), np.cos(theta)])
        o = np.array([x, 0.0, z]) - 0.1 * d
        return O.apply(xt, [*o, *d, E, 1.0])

    rc, st, _ = shoot(thB)
    assert rc == 1 and st[7] == 1.0
    assert np.allclose(st[3:6], [0, np.sin(thB), np.cos(thB)], atol=1e-15)  # specular
    assert np.allclose(st[0:3], [0, 0, 0], atol=1e-15)
    assert shoot(thB + 0.49 * wD)[1][7] == 1.0 and shoot(thB - 0.49 * wD)[1][7] == 1.0
    assert abs(shoot(thB + 0.5 * wD * np.sqrt(2))[1][7] - (np.sqrt(2) - 1) ** 2) < 1e-6
    assert shoot(thB + 100 * wD)[1][7] < 1e-4
    # energy detuning moves the Bragg angle: d(theta_B) = tan(theta_B) dE/E
    rc, st, _ = shoot(thB, E=E * (1 + 1e-3))
    eta = (thB - np.arcsin(12.398419843 / (E * 1.001) / (2 * d111))) / (0.5 * zeta * np.tan(np.arcsin(12.398419843 / (E * 1.001) / (2 * d111))))
    assert abs(st[7] - 1 / (abs(eta) + np.sqrt(eta * eta - 1)) ** 2) < 1e-12
    # aperture, back side, unreachable wavelength
    assert shoot(thB, z=0.0251)[0] == 0 and shoot(thB, x=0.0101)[0] == 0 and shoot(thB, z=0.0249)[0] == 1
    assert O.apply(xt, [0, -0.1, -0.1, *unit([0, 1, 1]), E, 1.0])[0] == 0
    assert shoot(thB, E=1.9)[0] == 0                                        # lambda / 2d >= 1


def test_c2_central_ray_reaches_the_focus(O, W):
    inst = W.config2(small=True)
    comps = inst["components"]
    st = np.array([0, 0, 0, 0, 0, 1.0, 12.0, 1.0])
    for c in comps[1:-1]:
        rc, st, _ = O.apply(c, list(st))
        assert rc == 1, c["kind"]
    det = comps[-1]
    rc, st2, b = O.apply(det, list(st))
    local = det["R"] @ (st[0:3] - det["T"])
    dloc = det["R"] @ st[3:6]
    hit = local + (-local[2] / dloc[2]) * dloc
    assert np.abs(hit[:2]).max() < 1e-8                                     # centre of the PSD
    # the hit is the pixel corner shared by the four central pixels, up to rounding
    assert b in {iy * 128 + ix for iy in (63, 64) for ix in (63, 64)}
    # weight = product of the two mirror reflectivities at (3 mrad, 12 keV); crystals sit on the Bragg peak
    RV = O.bilinear(comps[1], 3e-3, 12.0); RH = O.bilinear(comps[2], 3e-3, 12.0)
    assert abs(st[7] / (RV * RH) - 1) < 1e-6
    # off-axis source rays converge to the same spot (KB pair images the source point)
    for ang in ((2e-6, 0), (0, 2e-6), (-3e-6, 1e-6)):
        s = np.array([0, 0, 0, *unit([ang[0], ang[1], 1.0]), 12.0, 1.0])
        for c in comps[1:-1]:
            rc, s, _ = O.apply(c, list(s))
            assert rc == 1
        local = det["R"] @ (s[0:3] - det["T"]); dloc = det["R"] @ s[3:6]
        hit = local + (-local[2] / dloc[2]) * dloc
        assert np.abs(hit[:2]).max() < 2e-7
