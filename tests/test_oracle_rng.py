"""Pins for oracle steps 1-3: Philox4x32-10, u32->double, Box-Muller, source sampling."""
import os

import numpy as np

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers(O):
    rows = [l.split() for l in open(GOLD) if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert O.philox(v[0:4], v[4:6]) == tuple(v[6:10])


def test_philox_is_a_bijection_on_a_small_counter_range(O):
    outs = {O.philox((i, 0, 0, 0), (7, 9)) for i in range(2000)}
    assert len(outs) == 2000


def test_u01_end_points_and_exactness(O):
    assert O.u01(0, 0) == 2.0 ** -53
    assert O.u01(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    # bits below the top 52 are dropped
    assert O.u01(0, 0xFFF) == O.u01(0, 0)
    assert O.u01(0, 0x1000) == 2.0 ** -53 + 2.0 ** -52
    assert O.u01(0x80000000, 0) == 0.5 + 2.0 ** -53


def test_u01_mean_and_variance(O):
    n = 200_000
    u = np.array([O.draw2(1, i, 0, 0) for i in range(n // 2)]).ravel()
    assert abs(u.mean() - 0.5) < 4.0 / np.sqrt(12 * n)
    assert abs(u.var() - 1 / 12) < 5e-4
    assert u.min() > 0.0 and u.max() < 1.0


def test_draws_are_slot_addressed(O):
    # counter = (i lo, i hi, slot, component); key = (seed lo, seed hi)
    i, seed = (5 << 32) | 17, (3 << 32) | 11
    w = O.philox((17, 5, 2, 4), (11, 3))
    ua, ub = O.draw2(seed, i, 2, 4)
    assert ua == O.u01(w[0], w[1]) and ub == O.u01(w[2], w[3])
    assert O.draw2(seed, i, 1, 4) != (ua, ub)
    assert O.draw2(seed, i, 2, 3) != (ua, ub)


def test_box_muller_identity_and_moments(O):
    g0, g1 = O.gauss_pair(0.3, 0.125)
    r = np.sqrt(-2 * np.log(0.3))
    assert abs(g0 - r * np.cos(np.pi / 4)) < 1e-15 and abs(g1 - r * np.sin(np.pi / 4)) < 1e-15
    g = np.array([O.gauss_pair(*O.draw2(9, i, 0, 0)) for i in range(50_000)]).ravel()
    assert abs(g.mean()) < 0.02 and abs(g.var() - 1.0) < 0.02
    assert abs(np.mean(g ** 4) - 3.0) < 0.15  # kurtosis of a normal


def test_source_disk_target(O, W):
    src = W.config0()["components"][0]
    s = np.array([O.source_ray(src, 1, i) for i in range(40_000)])
    r, d, E, p = s[:, 0:3], s[:, 3:6], s[:, 6], s[:, 7]
    assert np.all(E == 20.0) and np.all(p == 1.0) and np.all(r[:, 2] == 0.0)
    rr = r[:, 0] ** 2 + r[:, 1] ** 2
    assert rr.max() <= (0.5e-3) ** 2
    assert abs(rr.mean() / (0.5e-3) ** 2 - 0.5) < 0.01          # uniform in area: <r^2> = R^2/2
    assert np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-15)
    hit = r + d * ((1.0 - r[:, 2]) / d[:, 2])[:, None]          # where the ray meets the target plane
    assert np.abs(hit[:, :2]).max() <= 5e-3 + 1e-15
    assert abs(hit[:, 0].var() / (10e-3) ** 2 - 1 / 12) < 0.002  # uniform on the rectangle
    assert abs(hit[:, 1].var() / (10e-3) ** 2 - 1 / 12) < 0.002


def test_source_gauss_divergent_uniform_energy(O, W):
    src = W.config2(small=True)["components"][0]
    s = np.array([O.source_ray(src, 1, i) for i in range(40_000)])
    assert abs(s[:, 0].std() / 50e-6 - 1) < 0.02 and abs(s[:, 1].std() / 10e-6 - 1) < 0.02
    tx, ty = s[:, 3] / s[:, 5], s[:, 4] / s[:, 5]
    assert abs(tx.std() / 20e-6 - 1) < 0.02 and abs(ty.std() / 5e-6 - 1) < 0.02
    E = s[:, 6]
    assert E.min() >= 12 * 0.99 and E.max() <= 12 * 1.01
    assert abs(E.var() - (0.24 ** 2) / 12) < 2e-4


def test_source_spectrum_inverse_cdf(O, W):
    # a two-level spectrum: bins 0..9 have weight 1, bins 10..19 weight 3 -> 25% / 75%, flat inside each half
    spec = np.array([1.0] * 10 + [3.0] * 10)
    src = W.source("point", "target", "spectrum", target_w=0.01, target_h=0.01, target_dist=1.0, spec_Emin=10.0,
                   spec_Emax=30.0, spectrum=spec)
    E = np.array([O.source_ray(src, 3, i)[6] for i in range(40_000)])
    assert E.min() >= 10.0 and E.max() < 30.0
    assert abs((E < 20.0).mean() - 0.25) < 0.01
    lo = E[E < 20.0]
    assert abs(lo.mean() - 15.0) < 0.1
    # direct check of the formula on one ray: E = Emin + (j + frac) dE with v = u * C[n]
    ue, _ = O.draw2(3, 5, 2, 0)
    v = ue * 40.0
    Eexp = 10.0 + v if v < 10.0 else 10.0 + (10 + (v - 10.0) / 3.0)
    assert abs(O.source_ray(src, 3, 5)[6] - Eexp) < 1e-12
