"""Pins for oracle steps 8-10: primitive intervals, priority resolution, Beer-Lambert; mesh pins for step 9."""
import numpy as np
import pytest

RNG = np.random.default_rng(42)


def unit(v):
    v = np.asarray(v, dtype=float)
    return v / np.linalg.norm(v)


def test_sphere_chord(O):
    R = 7e-3
    for _ in range(200):
        d = unit(RNG.normal(size=3))
        o = RNG.uniform(-0.05, 0.05, size=3)
        b = np.linalg.norm(np.cross(o, d))                      # impact parameter
        iv = O.primitive_interval("sphere", o, d, [R])
        if b >= R:
            assert iv is None
        else:
            assert abs((iv[1] - iv[0]) - 2 * np.sqrt(R * R - b * b)) < 1e-15 + 1e-12 * R
            assert abs(0.5 * (iv[0] + iv[1]) + np.dot(o, d)) < 1e-15


def test_box_hand_values(O):
    h = [1e-2, 2e-2, 3e-2]
    assert O.primitive_interval("box", [0, 0, -1], [0, 0, 1], h) == pytest.approx((0.97, 1.03), abs=1e-15)
    assert O.primitive_interval("box", [-1, 0, 0], [1, 0, 0], h) == pytest.approx((0.99, 1.01), abs=1e-15)
    assert O.primitive_interval("box", [0, 0.0201, -1], [0, 0, 1], h) is None
    d = unit([1, 1, 0])                                          # diagonal through the x-y rectangle
    a, b = O.primitive_interval("box", [-0.5, -0.5, 0], d, h)
    assert abs((b - a) - 2e-2 * np.sqrt(2)) < 1e-14              # limited by the x slab, |x|<=1e-2
    # origin inside: tin < 0 < tout, chord is the full chord
    a, b = O.primitive_interval("box", [0, 0, 0], [0, 0, 1], h)
    assert (a, b) == (-0.03, 0.03)
    # ray parallel to a face and outside / inside that slab
    assert O.primitive_interval("box", [0.011, 0, -1], [0, 0, 1], h) is None
    assert O.primitive_interval("box", [0.009, 0, -1], [0, 0, 1], h) is not None


def test_cylinder_analytic(O):
    Rc, H = 5e-3, 8e-3                                           # axis = local y (R13)
    a, b = O.primitive_interval("cyl", [0, 0, -1], [0, 0, 1], [Rc, H])
    # origin 1 m away: b^2 - a c cancels to ~1e-16 / R^2 relative, so ~1e-14 m on the roots
    assert (a, b) == pytest.approx((1 - Rc, 1 + Rc), abs=1e-13)
    a, b = O.primitive_interval("cyl", [3e-3, 0, -1], [0, 0, 1], [Rc, H])
    assert abs((b - a) - 2 * 4e-3) < 1e-13                       # 3-4-5 triangle
    assert O.primitive_interval("cyl", [0, 8.1e-3, -1], [0, 0, 1], [Rc, H]) is None
    a, b = O.primitive_interval("cyl", [1e-3, -1, 1e-3], [0, 1, 0], [Rc, H])   # along the axis
    assert (a, b) == pytest.approx((1 - H, 1 + H), abs=1e-15)
    assert O.primitive_interval("cyl", [5.1e-3, -1, 0], [0, 1, 0], [Rc, H]) is None
    # oblique ray cut by an end cap: enters through the barrel, leaves through the cap y = +H
    d = unit([0, 1, 1])
    a, b = O.primitive_interval("cyl", [0, 0, -Rc], d, [Rc, H])
    assert abs(a) < 1e-15 and abs(b - H * np.sqrt(2)) < 1e-15
    # random rays against brute-force point sampling
    for _ in range(30):
        d = unit(RNG.normal(size=3)); o = RNG.uniform(-0.01, 0.01, size=3) - 0.05 * d
        t = np.linspace(0, 0.1, 200001)
        P = o[None, :] + t[:, None] * d[None, :]
        inside = (P[:, 0] ** 2 + P[:, 2] ** 2 < Rc * Rc) & (np.abs(P[:, 1]) < H)
        iv = O.primitive_interval("cyl", o, d, [Rc, H])
        L = 0.0 if iv is None else max(0.0, min(iv[1], 0.1) - max(iv[0], 0.0))
        assert abs(inside.mean() * 0.1 - L) < 2e-6


def _tau(O, W, solids, ray, mats):
    rc, st, _ = O.apply(W.solids(solids), ray, materials=mats)
    assert rc == 1
    return -np.log(st[7] / ray[7])


def _flat(mu):
    return {"E": np.array([1.0, 1000.0]), "mu": np.array([mu, mu])}


def test_disjoint_solids_add_and_overlap_rules(O, W):
    mats = [None, _flat(100.0), _flat(300.0)]
    ray = [0, 0, 0, 0, 0, 1, 50.0, 1.0]
    TOL = 2e-12   # quadratics seen from 0.3-0.5 m cancel to ~1e-14 m; times mu = 300 1/m
    A = W.solid_box((1e-2, 1e-2, 1e-2), 1, 0, T=(0, 0, 0.3))
    B = W.solid_sphere(1e-2, 2, 1, T=(0, 0, 0.5))
    assert abs(_tau(O, W, [A, B], ray, mats) - (100 * 2e-2 + 300 * 2e-2)) < TOL
    # same-material overlap = union chord
    A2 = W.solid_box((1e-2, 1e-2, 1e-2), 1, 1, T=(0, 0, 0.31))
    assert abs(_tau(O, W, [A, A2], ray, mats) - 100 * 3e-2) < TOL
    # different materials: the higher priority owns the overlap, whatever the list order
    B2 = W.solid_box((1e-2, 1e-2, 1e-2), 2, 5, T=(0, 0, 0.31))
    expect = 100 * 1e-2 + 300 * 2e-2
    assert abs(_tau(O, W, [A, B2], ray, mats) - expect) < TOL
    assert abs(_tau(O, W, [B2, A], ray, mats) - expect) < TOL
    # nested: inner sphere of higher priority inside a box
    inner = W.solid_sphere(0.4e-2, 2, 9, T=(0, 0, 0.3))
    assert abs(_tau(O, W, [A, inner], ray, mats) - (100 * 1.2e-2 + 300 * 0.8e-2)) < TOL
    # ... and of LOWER priority: invisible
    inner_lo = W.solid_sphere(0.4e-2, 2, -1, T=(0, 0, 0.3))
    assert abs(_tau(O, W, [A, inner_lo], ray, mats) - 100 * 2e-2) < TOL
    # ray starting inside a solid: only the part ahead of it counts (clip to t >= 0)
    assert abs(_tau(O, W, [A], [0, 0, 0.3, 0, 0, 1, 50.0, 1.0], mats) - 100 * 1e-2) < TOL
    # solid behind the ray: nothing
    assert _tau(O, W, [A], [0, 0, 0.4, 0, 0, 1, 50.0, 1.0], mats) == 0.0
    # the ray itself is untouched
    rc, st, _ = O.apply(W.solids([A]), ray, materials=mats)
    assert np.array_equal(st[:7], ray[:7])


def _inside(s, P):
    """Point-in-solid, written independently of the oracle (lab points P [n,3])."""
    L = (P - s["T"]) @ s["R"].T
    if s["shape"] == "box":
        return np.all(np.abs(L) < np.array(s["half"]), axis=1)
    if s["shape"] == "cyl":
        return (L[:, 0] ** 2 + L[:, 2] ** 2 < s["radius"] ** 2) & (np.abs(L[:, 1]) < s["half_height"])
    return np.sum(L * L, axis=1) < s["radius"] ** 2


def test_c1_solids_against_brute_force_point_sampling(O, W):
    # tau = integral of mu_owner along the ray, by classifying 4e5 sample points with an independent
    # point-in-solid test and the priority rule (R12)
    inst = W.config1(small=True)
    comp = inst["components"][1]
    sl = comp["solids"]
    mats = inst["materials"]
    E = 60.0
    mus = np.array([0.0] + [O.mu(m, E) for m in mats[1:]])
    checked = 0
    for i in range(40):
        ray = O.source_ray(inst["components"][0], 1, i)
        ray[6] = E
        t = (np.arange(400000) + 0.5) * (1.0 / 400000)
        P = ray[None, 0:3] + t[:, None] * ray[None, 3:6]
        owner_mu = np.zeros(len(t))
        best = np.full(len(t), -10 ** 9)
        for s in sl:
            ins = _inside(s, P) & (s["priority"] > best)
            owner_mu[ins] = mus[s["material"]]
            best[ins] = s["priority"]
        tau_bf = owner_mu.mean() * 1.0
        tau = _tau(O, W, sl, list(ray), mats)
        assert abs(tau - tau_bf) < 2e-5 * max(mus) + 1e-12
        checked += tau > 0
    assert checked >= 10


# ---------------------------------------------------------------------------------- meshes (step 9)
def test_ray_triangle_orientation_and_t(O):
    v0, v1, v2 = [0, 0, 1.0], [1, 0, 1.0], [0, 1, 1.0]        # normal = +z
    r, t = O.ray_triangle([0.2, 0.2, 0], [0, 0, 1], v0, v1, v2)
    assert (r, t) == (-1, 1.0)                                 # d.n > 0: exiting
    r, t = O.ray_triangle([0.2, 0.2, 2], [0, 0, -1], v0, v1, v2)
    assert (r, t) == (+1, 1.0)                                 # entering
    assert O.ray_triangle([0.2, 0.2, 0], [0, 0, 1], v0, v2, v1)[0] == +1   # flipped winding
    assert O.ray_triangle([0.8, 0.8, 0], [0, 0, 1], v0, v1, v2)[0] == 0
    # hit behind the origin is still reported (t < 0): the whole line is intersected
    assert O.ray_triangle([0.2, 0.2, 2], [0, 0, 1], v0, v1, v2) == (-1, -1.0)
    # all six dominant-axis / sign cases against a plain Moller-Trumbore
    rng = np.random.default_rng(1)
    for _ in range(300):
        tri = rng.normal(size=(3, 3))
        o = rng.normal(size=3) * 3
        target = tri.T @ rng.dirichlet([1, 1, 1]) if rng.random() < 0.7 else rng.normal(size=3) * 2
        d = unit(target - o)
        e1, e2 = tri[1] - tri[0], tri[2] - tri[0]
        pv = np.cross(d, e2); det = e1 @ pv
        tv = o - tri[0]; u = (tv @ pv) / det
        qv = np.cross(tv, e1); v = (d @ qv) / det
        t_mt = (e2 @ qv) / det
        hit_mt = (u > 1e-9) and (v > 1e-9) and (u + v < 1 - 1e-9)
        miss_mt = (u < -1e-9) or (v < -1e-9) or (u + v > 1 + 1e-9)
        r, t = O.ray_triangle(o, d, *tri)
        if hit_mt:
            assert r == (+1 if d @ np.cross(e1, e2) < 0 else -1)
            assert abs(t - t_mt) < 1e-11
        if miss_mt:
            assert r == 0


def test_shared_edge_is_watertight(O):
    # a ray aimed exactly at points of the shared edge of two triangles hits at least one of them, never zero
    a, b, c, d4 = np.array([0, 0, 1.0]), np.array([1, 0.3, 1.2]), np.array([0.1, 1, 0.9]), np.array([1.1, 1.2, 1.4])
    rng = np.random.default_rng(2)
    for _ in range(500):
        s = rng.random()
        p = b + s * (c - b)                                    # on the shared edge b-c
        o = rng.normal(size=3) * 0.3 - np.array([0, 0, 2.0])
        d = unit(p - o)
        h1 = O.ray_triangle(o, d, a, b, c)[0]
        h2 = O.ray_triangle(o, d, c, b, d4)[0]
        assert h1 != 0 or h2 != 0


def test_cube_mesh_equals_box_primitive(O, W):
    h = (1e-2, 1.5e-2, 0.7e-2)
    V, F = W.cube_mesh(*h)
    mats = [None, _flat(80.0)]
    Rm = W.random_rotation(np.random.default_rng(7))
    mesh = W.solid_mesh(V, F, 1, 0, R=Rm, T=(1e-3, -2e-3, 0.5))
    box = W.solid_box(h, 1, 0, R=Rm, T=(1e-3, -2e-3, 0.5))
    rng = np.random.default_rng(8)
    nhit = 0
    for _ in range(300):
        o = np.array([rng.uniform(-5e-3, 5e-3), rng.uniform(-5e-3, 5e-3), 0.0])
        tgt = np.array([rng.uniform(-2e-2, 2e-2), rng.uniform(-2e-2, 2e-2), 0.5])
        ray = [*o, *unit(tgt - o), 30.0, 1.0]
        tm, tb = _tau(O, W, [mesh], ray, mats), _tau(O, W, [box], ray, mats)
        assert abs(tm - tb) < 1e-13
        nhit += tb > 0
    assert nhit > 100
    # origin inside the mesh: hits behind the origin close the interval, clip keeps the forward half
    ray = [1e-3, -2e-3, 0.5, *unit([0.1, 0.2, 1.0]), 30.0, 1.0]
    assert abs(_tau(O, W, [mesh], ray, mats) - _tau(O, W, [box], ray, mats)) < 1e-13
    assert _tau(O, W, [mesh], ray, mats) > 0


def test_icosphere_chord_matches_analytic_sphere(O, W):
    # inscribed polyhedron: chord within 1e-4 R + facet sag of the analytic chord away from grazing
    R = 20e-3
    V, F = W.icosphere(5)
    # closedness (generator check): oriented area vectors sum to 0, divergence-theorem volume -> 4/3 pi
    nrm = np.cross(V[F[:, 1]] - V[F[:, 0]], V[F[:, 2]] - V[F[:, 0]])
    assert np.abs(nrm.sum(axis=0)).max() < 1e-12
    vol = np.einsum("ij,ij->i", V[F[:, 0]], nrm).sum() / 6.0
    assert 0.995 * 4 / 3 * np.pi < vol < 4 / 3 * np.pi
    mesh = W.solid_mesh(V * R, F, 1, 0, T=(0, 0, 0.5))
    rng = np.random.default_rng(9)
    for _ in range(60):
        o = np.zeros(3)
        tgt = np.array([rng.uniform(-10e-3, 10e-3), rng.uniform(-10e-3, 10e-3), 0.5])
        d = unit(tgt - o)
        t, orient, ntest = O.mesh_hits(mesh, o - np.array([0, 0, 0.5]), d)
        assert ntest == len(F)
        assert len(t) >= 2 and orient[0] == +1 and orient[-1] == -1
        b = np.linalg.norm(np.cross(np.array([0, 0, 0.5]), d))
        chord = 2 * np.sqrt(R * R - b * b)
        assert 0 <= chord - (t[-1] - t[0]) < 4e-3 * R           # level 5: sag 2e-4 R per side, amplified near grazing


def test_grid_accelerator_equals_brute_force(O, W):
    rng = np.random.default_rng(11)
    V, F = W.bumpy_sphere(rng, 4, 20e-3)
    mesh = W.solid_mesh(V, F, 1, 0)
    total_bf = total_grid = 0
    for k in range(400):
        if k % 2:
            o = rng.normal(size=3) * 0.05; d = unit(rng.normal(size=3))
        else:                                                   # through the body
            o = unit(rng.normal(size=3)) * 0.1; d = unit(rng.normal(size=3) * 0.01 - o)
        t0, o0, n0 = O.mesh_hits(mesh, o, d, use_grid=False)
        t1, o1, n1 = O.mesh_hits(mesh, o, d, use_grid=True)
        assert np.array_equal(t0, t1) and np.array_equal(o0, o1)  # bitwise: same test, same operands
        assert len(t0) % 2 == 0
        total_bf += n0; total_grid += n1
    assert total_grid < total_bf / 20
    # and through the whole solids component
    inst = W.config3(small=True)
    a = O.trace(inst, n=3000, dump=True, mesh_accel=0)
    b = O.trace(inst, n=3000, dump=True, mesh_accel=1)
    assert np.array_equal(a["dump"], b["dump"])
    assert a["degenerate"] == 0


def test_nested_meshes_priority(O, W):
    V, F = W.icosphere(3)
    mats = [None, _flat(50.0), _flat(400.0)]
    outer = W.solid_mesh(V * 20e-3, F, 1, 0, T=(0, 0, 0.5))
    inner = W.solid_mesh(V * 10e-3, F, 2, 1, T=(0, 0, 0.5))
    ray = [0, 0, 0, 0, 0, 1, 30.0, 1.0]
    t_out, _, _ = O.mesh_hits(outer, [0, 0, -0.5], [0, 0, 1])
    t_in, _, _ = O.mesh_hits(inner, [0, 0, -0.5], [0, 0, 1])
    Lo, Li = t_out[-1] - t_out[0], t_in[-1] - t_in[0]
    assert abs(_tau(O, W, [outer, inner], ray, mats) - (50 * (Lo - Li) + 400 * Li)) < 1e-12
    assert 0.039 < Lo <= 0.04 + 1e-15 and 0.0195 < Li <= 0.02 + 1e-15


# ------------------------------------------------------------------ step 9, second half: hits -> intervals
# Coordinates below are dyadic (exact in fp64) and the direction ratios are +-1 or 0, so the rays go EXACTLY through
# the shared diagonal of a cube face, through a cube edge or through a cube vertex: every edge function that
# should vanish is an exact zero, and the duplicate hits really occur.  What the mathematics fixes is the chord of
# the box, which the box primitive pins independently (test_box_hand_values).
H_DYADIC = (1 / 64, 3 / 128, 1 / 128)


def _tau_rc(O, W, solids, ray, mats):
    rc, st, _ = O.apply(W.solids(solids), ray, materials=mats)
    return rc, (-np.log(st[7] / ray[7]) if rc == 1 else None)


def test_mesh_duplicate_hits_on_diagonal_edge_vertex_collapse_to_box_chord(O, W):
    mats = [None, _flat(80.0)]
    hx, hy, hz = H_DYADIC
    V, F = W.cube_mesh(hx, hy, hz)
    mesh, box = W.solid_mesh(V, F, 1, 0), W.solid_box(H_DYADIC, 1, 0)
    s2 = np.sqrt(2.0)
    cases = [
        # (origin, direction, hits of the full line: t-multiplicities (enter, exit), chord)
        ([0, 0, -1], [0, 0, 1], (2, 2), 2 * hz),                          # both face diagonals (shared edge of 2 triangles)
        ([1 / 256, 3 / 512, -1], [0, 0, 1], (2, 2), 2 * hz),              # another point of the same diagonals
        ([2 * hx, 1 / 256, -hz - hx], [-1, 0, 1], (2, 1), 2 * hz * s2),   # in through the edge x = hx, z = -hz
    ]
    for o, d, mult, chord in cases:
        d = unit(d)
        t, orient, _ = O.mesh_hits(mesh, o, d)
        assert (int((orient == 1).sum()), int((orient == -1).sum())) == mult, (o, orient)   # the duplicates are there
        ray = [*o, *d, 30.0, 1.0]
        rc_m, tau_m = _tau_rc(O, W, [mesh], ray, mats)
        rc_b, tau_b = _tau_rc(O, W, [box], ray, mats)
        assert rc_m == 1 and rc_b == 1
        assert abs(tau_m - 80.0 * chord) < 1e-13 and abs(tau_m - tau_b) < 1e-13
    # through two opposite vertices of a cube (six triangles meet the ray at either end)
    hc = 1 / 64
    Vc, Fc = W.cube_mesh(hc, hc, hc)
    o, d = [-2 * hc] * 3, unit([1, 1, 1])
    t, orient, _ = O.mesh_hits(W.solid_mesh(Vc, Fc, 1, 0), o, d)
    assert (orient == 1).sum() >= 3 and (orient == -1).sum() >= 3
    rc, tau = _tau_rc(O, W, [W.solid_mesh(Vc, Fc, 1, 0)], [*o, *d, 30.0, 1.0], mats)
    assert rc == 1 and abs(tau - 80.0 * 2 * hc * np.sqrt(3.0)) < 1e-13
    # the same rays against a rotated and shifted cube (not exact any more, still the box chord)
    Rm = W.random_rotation(np.random.default_rng(70))
    T = np.array([1e-3, -2e-3, 0.5])
    mesh_r, box_r = W.solid_mesh(V, F, 1, 0, R=Rm, T=T), W.solid_box(H_DYADIC, 1, 0, R=Rm, T=T)
    for o, d, _, chord in cases:
        ol, dl = Rm.T @ np.asarray(o, float) + T, Rm.T @ unit(d)
        ray = [*ol, *dl, 30.0, 1.0]
        rc_m, tau_m = _tau_rc(O, W, [mesh_r], ray, mats)
        rc_b, tau_b = _tau_rc(O, W, [box_r], ray, mats)
        assert rc_m == 1 and abs(tau_m - tau_b) < 1e-12 and abs(tau_b - 80.0 * chord) < 1e-11


def test_mesh_grazing_edge_and_vertex_enter_sorts_before_exit(O, W):
    # A ray that only touches a cube edge (or vertex) from outside hits an entering and an exiting face at the SAME t.
    # With "enter before exit on ties" that is an interval of zero length (tau = 0, as for the box, whose chord is
    # empty); the opposite tie order would start the sequence with an exit and call the mesh degenerate.
    mats = [None, _flat(80.0)]
    hx, hy, hz = H_DYADIC
    V, F = W.cube_mesh(hx, hy, hz)
    mesh, box = W.solid_mesh(V, F, 1, 0), W.solid_box(H_DYADIC, 1, 0)
    for o, d in (([0, 1 / 256, -hz - hx], [1, 0, 1]),              # touches the edge x = hx, z = -hz
                 ([0, hy - hx, -hz - hx], [1, 1, 1])):             # touches the vertex (hx, hy, -hz)
        d = unit(d)
        t, orient, _ = O.mesh_hits(mesh, o, d)
        assert len(t) >= 2 and (orient == 1).any() and (orient == -1).any() and np.ptp(t) == 0.0
        ray = [*o, *d, 30.0, 1.0]
        assert _tau_rc(O, W, [mesh], ray, mats) == (1, 0.0)
        assert _tau_rc(O, W, [box], ray, mats) == (1, 0.0)


def test_open_or_inward_wound_mesh_is_degenerate(O, W):
    # step 9: a hit sequence that does not alternate enter, exit, ... starting with enter drops the ray (rc -3)
    mats = [None, _flat(80.0)]
    V, F = W.cube_mesh(*H_DYADIC)
    top = np.array([all(V[v][2] > 0 for v in f) for f in F])
    assert top.sum() == 2
    opened = W.solid_mesh(V, F[~top], 1, 0)                        # cube without its face z = +hz
    through_hole = [1e-3, 2e-3, -1, 0, 0, 1, 30.0, 1.0]            # in through z = -hz, out through the hole: 1 hit
    sideways = [-1, 2e-3, 1e-3, 1, 0, 0, 30.0, 1.0]                # in and out through the x faces: still closed there
    assert _tau_rc(O, W, [opened], through_hole, mats) == (-3, None)
    rc, tau = _tau_rc(O, W, [opened], sideways, mats)
    assert rc == 1 and abs(tau - 80.0 * 2 * H_DYADIC[0]) < 1e-13
    assert _tau_rc(O, W, [opened], [0.1, 0, -1, 0, 0, 1, 30.0, 1.0], mats) == (1, 0.0)       # misses it altogether
    inward = W.solid_mesh(V, F[:, [0, 2, 1]], 1, 0)                # every triangle flipped: the first hit is an exit
    assert _tau_rc(O, W, [inward], through_hole, mats) == (-3, None)
    assert _tau_rc(O, W, [inward], sideways, mats) == (-3, None)
    assert _tau_rc(O, W, [inward], [0.1, 0, -1, 0, 0, 1, 30.0, 1.0], mats) == (1, 0.0)
    # a closed, outward-wound mesh never is: 2000 random lines through a bumpy sphere, and whole chains count them
    rng = np.random.default_rng(12)
    Vb, Fb = W.bumpy_sphere(rng, 3, 20e-3)
    closed = W.solid_mesh(Vb, Fb, 1, 0)
    for _ in range(2000):
        o = unit(rng.normal(size=3)) * 0.1
        d = unit(rng.normal(size=3) * 0.012 - o)
        assert O.apply(W.solids([closed]), [*o, *d, 30.0, 1.0], materials=mats)[0] == 1
    # in a chain the ray is dropped and counted: fate -3, no tally, counters still add up
    src = W.source("point", "target", "mono", target_w=0.2, target_h=0.2, target_dist=1.0, E0=30.0)
    det = W.detector(-0.1, 0.1, -0.1, 0.1, 8, 8, 0.0, 60.0, 1, T=(0, 0, 1.0))
    opened_at = W.solid_mesh(V, F[~top], 1, 0, T=(0, 0, 0.5))
    r = O.trace(W.instrument("open", [src, W.solids([opened_at]), det], mats, 4000), dump=True)
    # degenerate = the rays through the missing face (2 hx x 2 hy at z = 0.5 + hz), seen from the point source
    zf = 0.5 + H_DYADIC[2]
    frac = (2 * H_DYADIC[0] / zf) * (2 * H_DYADIC[1] / zf) / 0.2 ** 2
    assert abs(r["degenerate"] / 4000 - frac) < 4 * np.sqrt(frac * (1 - frac) / 4000)
    assert r["degenerate"] + r["detected"] + r["missed"] + int(r["absorbed"].sum()) == 4000
    assert int(r["N"][0].sum()) == r["detected"] == int((r["dump"]["fate"] == O.F_DETECTED).sum())
    assert np.all(r["dump"]["p"][r["dump"]["fate"] == O.F_DEGENERATE] == 1.0)      # dropped before any attenuation


def test_icosphere_level6_chord_vs_analytic_sphere(O, W):
    # SURVEY.md 8(c) "Pins", mesh row: the unperturbed level-6 icosphere (the outer mesh of configs[3]) is inscribed in
    # the sphere.  Its faces lie 5.6e-5 R .. 7.1e-5 R below the sphere at their centres (computed here from the
    # generator's vertices; the survey's "5.0e-5 R" was an estimate), so away from grazing (impact parameter <= R/4,
    # incidence <= 14.5 deg) a chord is SHORT of the analytic 2 sqrt(R^2 - b^2) by at most 2 x 7.2e-5 R / cos(14.5 deg)
    # = 1.5e-4 R, and never longer.
    R = 20e-3
    V, F = W.icosphere(6)
    assert len(F) == 81920
    ctr = (V[F[:, 0]] + V[F[:, 1]] + V[F[:, 2]]) / 3.0
    sag = 1.0 - np.linalg.norm(ctr, axis=1)
    assert 5.5e-5 < sag.min() and sag.max() < 7.2e-5
    mesh = W.solid_mesh(V * R, F, 1, 0)
    rng = np.random.default_rng(90)
    worst = 0.0
    for _ in range(25):
        n = unit(rng.normal(size=3))
        e = unit(np.cross(n, rng.normal(size=3)))
        b = rng.uniform(0.0, 0.25) * R
        o = b * e - 0.5 * n
        t, orient, ntest = O.mesh_hits(mesh, o, n, use_grid=False)
        assert ntest == len(F) and len(t) >= 2 and orient[0] == +1 and orient[-1] == -1
        deficit = 2 * np.sqrt(R * R - b * b) - (t[-1] - t[0])
        assert 0.0 <= deficit < 1.5e-4 * R
        worst = max(worst, deficit)
    assert worst > 1e-5 * R                                        # it IS a polyhedron, not the sphere
