"""Pins for the oracle's step 17, scattering in samples: what the mathematics
fixes outside the oracle -- the Thomson distribution's inverse CDF and moments, Beer-Lambert limits, the exponential law
of the first event, weight conservation in a purely scattering medium, and a fine-step marching of the same draws (the
paper's own stepping) written out in numpy."""
import numpy as np

RNG = np.random.default_rng(17)


def flat(mu, mu_s=None):
    t = {"E": np.array([1.0, 200.0]), "mu": np.array([mu, mu])}
    if mu_s:                                                            # a table holds positive values; none = no scattering
        t["mu_s"] = np.array([mu_s, mu_s])
    return t


def unit(v):
    v = np.asarray(v, dtype=float)
    return v / np.linalg.norm(v)


def test_thomson_inverse_cdf_and_frame(O):
    # cos(theta) solves F(x) = u with F(x) = 1/2 + (3/8)(x + x^3/3); the new direction is unit, at that angle to the old
    # one, and its azimuth about the old one advances with u_phi
    for d in (unit([0, 0, 1]), unit([1, 0, 0]), unit([0.3, -0.5, 0.8]), unit([-0.7, 0.7, 1e-9]), unit([1, 1, 1])):
        prev = None
        for u in (1e-12, 0.01, 0.25, 0.5, 0.77, 1 - 1e-12):
            for uphi in (0.0, 0.125, 0.6):
                n = O.scatter_direction(d, u, uphi)
                assert abs(np.linalg.norm(n) - 1) < 4e-16
                x = float(n @ d)
                assert abs(0.5 + 0.375 * (x + x ** 3 / 3) - u) < 1e-14
        a, b = O.scatter_direction(d, 0.3, 0.0), O.scatter_direction(d, 0.3, 0.25)
        pa, pb = a - (a @ d) * d, b - (b @ d) * d                     # quarter turn of the azimuth
        assert abs(pa @ pb) < 1e-15 and abs(np.linalg.norm(pa) - np.linalg.norm(pb)) < 1e-15
        assert np.cross(pa, pb) @ d > 0                                 # right-handed about d
    # moments of the sampled distribution: E[x] = 0, E[x^2] = (3/8)(2/3 + 2/5) = 0.4
    u = (np.arange(200000) + 0.5) / 200000
    xs = np.array([O.scatter_direction([0, 0, 1.0], ui, 0.3)[2] for ui in u[::40]])
    assert abs(xs.mean()) < 1e-3 and abs((xs ** 2).mean() - 0.4) < 1e-3


def homogeneous(W, n, h, mat=1, K=0):
    return W.voxels(np.full((n, n, n), mat, dtype=np.uint8), h, T=(-0.5 * n * h, -0.5 * n * h, 0.0), scatter_order=K)


def test_no_scattering_limits_are_beer_lambert_bit_for_bit(O, W):
    rng = np.random.default_rng(3)
    ids = rng.integers(0, 4, size=(9, 8, 7), dtype=np.uint8)
    mats = [None, flat(30.0), flat(55.0), flat(12.0)]
    mats_s0 = [None, flat(30.0), flat(55.0), flat(12.0)]              # K > 0 but no material scatters
    for _ in range(60):
        o = np.array([*rng.uniform(-3e-3, 10e-3, size=2), -0.01])
        d = unit([*rng.uniform(-0.4, 0.4, size=2), 1.0])
        ray = [*o, *d, 40.0, 1.0]
        ref = O.apply(W.voxels(ids, 1e-3), ray, materials=mats)[1]
        got = O.apply(W.voxels(ids, 1e-3, scatter_order=3), ray, materials=mats_s0)[1]
        assert np.array_equal(ref, got)
    # the same for a solids group
    grp = [W.solid_box((2e-3, 3e-3, 1e-3), 1, 0, T=(0, 0, 0.01)), W.solid_sphere(2.5e-3, 2, 1, T=(1e-3, 0, 0.011))]
    for _ in range(60):
        o = np.array([*rng.uniform(-3e-3, 3e-3, size=2), 0.0])
        d = unit([*rng.uniform(-0.2, 0.2, size=2), 1.0])
        ray = [*o, *d, 40.0, 1.0]
        assert np.array_equal(O.apply(W.solids(grp), ray, materials=mats)[1],
                              O.apply(W.solids(grp, scatter_order=2), ray, materials=mats_s0)[1])


def test_first_event_depth_is_minus_log_u_over_mu_s(O, W):
    # homogeneous block, K = 1: the event lies at depth -ln(u_f) / mu_s along the ray (u_f = first draw of slot 0 of the
    # component's stream), the weight up to there carries exp(-(mu - mu_s) depth), and the leg after the event carries the
    # full mu over what is left of the block
    n, h, mu, mu_s = 10, 2e-3, 90.0, 60.0
    vol = homogeneous(W, n, h, K=1)
    L = n * h
    seen = 0
    for i in range(200):
        u_f, u_mu = O.draw2(7, i, 0, 1)
        u_phi, _ = O.draw2(7, i, 1, 1)
        depth = -np.log(u_f) / mu_s
        rc, st, _ = O.apply(vol, [1e-4, -2e-4, -0.05, 0, 0, 1, 30.0, 1.0], materials=[None, flat(mu, mu_s)], seed=7, ray_index=i)
        if depth >= L:                                                  # left the block unscattered
            assert np.array_equal(st[0:6], [1e-4, -2e-4, -0.05, 0, 0, 1]) and abs(st[7] - np.exp(-(mu - mu_s) * L)) < 1e-14
            continue
        seen += 1
        assert np.allclose(st[0:3], [1e-4, -2e-4, depth], atol=1e-15)
        nd = O.scatter_direction([0, 0, 1.0], u_mu, u_phi)
        assert np.allclose(st[3:6], nd, atol=1e-15)
        # exit chord from the event point along nd inside the box |x|, |y| <= L/2, 0 <= z <= L
        p0 = np.array([1e-4, -2e-4, depth])
        lo, hi = np.array([-L / 2, -L / 2, 0.0]), np.array([L / 2, L / 2, L])
        with np.errstate(divide="ignore"):
            t_exit = np.min(np.where(nd > 0, (hi - p0) / nd, np.where(nd < 0, (lo - p0) / nd, np.inf)))
        assert abs(st[7] - np.exp(-(mu - mu_s) * depth - mu * t_exit)) < 1e-13
    assert 100 < seen < 200                                             # 1 - exp(-1.2) = 70 % scatter


def test_unscattered_fraction_and_weight_conservation(O, W):
    # purely scattering medium (mu_s = mu): no weight is ever lost while events remain (K large); the rays that cross the
    # block without an event are exp(-mu_s L) of all, and they alone reach a small detector on the axis
    n, h, mu = 8, 2.5e-3, 80.0
    L = n * h
    comps = [W.source("point", "target", "mono", target_w=1e-6, target_h=1e-6, target_dist=1.0, E0=30.0),
             homogeneous(W, n, h, K=200),
             W.detector(-1e-4, 1e-4, -1e-4, 1e-4, 1, 1, 0.0, 60.0, 1, T=(0, 0, 1.0))]
    comps[1]["T"] = np.array([-0.5 * L, -0.5 * L, 0.1])
    inst = W.instrument("scatter_block", comps, [None, flat(mu, mu)], 40000)
    o = O.trace(inst, n=40000, dump=True)
    assert np.all(np.abs(o["dump"]["p"] - 1.0) < 1e-13)                 # exp(-0) on every ray
    frac = o["detected"] / 40000
    want = np.exp(-mu * L)
    assert abs(frac - want) < 4 * np.sqrt(want * (1 - want) / 40000)
    # with absorption the direct beam carries exp(-mu L) per ray whatever K is
    inst2 = W.instrument("scatter_block", comps, [None, flat(mu, 0.5 * mu)], 4000)
    o2 = O.trace(inst2, n=4000, dump=True)
    det = o2["dump"]["fate"] == -1
    assert det.sum() > 100 and np.all(np.abs(o2["dump"]["p"][det] - np.exp(-0.5 * mu * L)) < 1e-13)


def test_heterogeneous_volume_against_fine_marching(O, W):
    # the paper's own scheme (small steps, look up the voxel, update weight and direction) written out in
    # numpy with the same draws: the event positions agree to the step length, the directions exactly
    rng = np.random.default_rng(5)
    n, h = 6, 2e-3
    ids = rng.integers(1, 4, size=(n, n, n), dtype=np.uint8)
    mu = {1: (40.0, 25.0), 2: (150.0, 100.0), 3: (15.0, 0.0)}
    mats = [None] + [flat(*mu[m]) for m in (1, 2, 3)]
    vol = W.voxels(ids, h, T=(0, 0, 0), scatter_order=2)
    step = h / 400
    checked = 0
    for i in range(40):
        o = np.array([*rng.uniform(1e-3, 11e-3, size=2), -1e-3])
        d = unit([*rng.uniform(-0.3, 0.3, size=2), 1.0])
        rc, st, _ = O.apply(vol, [*o, *d, 50.0, 1.0], materials=mats, seed=11, ray_index=i)
        # marching
        pos, dirn, tau, k = o.copy(), d.copy(), 0.0, 0
        events, gap = [], np.inf
        while k <= 2:
            tau_s = -np.log(O.draw2(11, i, 2 * k, 1)[0]) if k < 2 else np.inf
            cum, t, scattered = 0.0, 0.0, False
            while t < 0.05:
                q = pos + (t + 0.5 * step) * dirn
                idx = np.floor(q / h).astype(int)
                if np.all(idx >= 0) and np.all(idx < n):
                    mt, ms = mu[int(ids[idx[2], idx[1], idx[0]])]
                    if k == 2:
                        ms_eff = 0.0
                    else:
                        ms_eff = ms
                    if cum + ms_eff * step >= tau_s:
                        l = (tau_s - cum) / ms_eff
                        tau += (mt - ms_eff) * l
                        pos = pos + (t + l) * dirn
                        dirn = O.scatter_direction(dirn, O.draw2(11, i, 2 * k, 1)[1], O.draw2(11, i, 2 * k + 1, 1)[0])
                        events.append(pos.copy())
                        scattered = True
                        break
                    cum += ms_eff * step
                    tau += (mt - ms_eff) * step
                t += step
            if not scattered:
                gap = tau_s - cum                                       # how far the leg was from an event
                break
            k += 1
        if events:
            assert np.linalg.norm(st[0:3] - events[-1]) < 50 * step     # marching error accumulates over two legs
            checked += 1
            assert abs(-np.log(st[7]) - tau) < 0.02 * max(tau, 1e-3) + 1e-3
        elif not np.array_equal(st[0:3], o):
            assert gap < 2e-3                                           # borderline: the marching's own error (mu_s step / 2 per face)
        else:
            assert np.array_equal(st[3:6], d)
    assert checked > 10


def test_scattering_solids_group(O, W):
    # a sphere of a purely scattering material: weights stay 1, the unscattered fraction through the centre is
    # exp(-mu_s 2R), and a ray can re-enter the sphere's neighbour after an event (segments are recomputed per leg)
    R, mu = 5e-3, 120.0
    grp = W.solids([W.solid_sphere(R, 1, 0, T=(0, 0, 0.1)), W.solid_box((2e-3, 2e-3, 2e-3), 2, 1, T=(9e-3, 0, 0.1))], scatter_order=50)
    comps = [W.source("point", "target", "mono", target_w=1e-7, target_h=1e-7, target_dist=1.0, E0=30.0), grp,
             W.detector(-1e-5, 1e-5, -1e-5, 1e-5, 1, 1, 0.0, 60.0, 1, T=(0, 0, 1.0))]
    inst = W.instrument("scatter_sphere", comps, [None, flat(mu, mu), flat(400.0)], 30000)
    o = O.trace(inst, n=30000, dump=True)
    want = np.exp(-mu * 2 * R)
    assert abs(o["detected"] / 30000 - want) < 4 * np.sqrt(want * (1 - want) / 30000)
    p = o["dump"]["p"]
    assert np.all(p <= 1.0 + 1e-13)
    hit_box = p < 1.0 - 1e-9                                            # only the absorbing box takes weight
    assert 0.001 < hit_box.mean() < 0.2
    assert np.all(np.abs(p[~hit_box] - 1.0) < 1e-13)
