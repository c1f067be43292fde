"""Pins for oracle step 11 (exact voxel traversal, Amanatides-Woo; readings R15/R16)."""
import numpy as np

RNG = np.random.default_rng(123)


def unit(v):
    v = np.asarray(v, dtype=float)
    return v / np.linalg.norm(v)


def flat(mu):
    return {"E": np.array([1.0, 1000.0]), "mu": np.array([mu, mu])}


MUS = [0.0, 35.0, 120.0, 7.5, 260.0]
MATS = [None] + [flat(m) for m in MUS[1:]]


def tau(O, comp, ray, mats=MATS):
    rc, st, _ = O.apply(comp, ray, materials=mats)
    assert rc == 1
    assert np.array_equal(st[:7], np.asarray(ray, dtype=float)[:7])      # ray untouched, only the weight changes
    return -np.log(st[7] / ray[7])


def random_ray(n, h, origin):
    """A ray through the volume's neighbourhood (hits most of the time)."""
    L = n * h
    a = origin + RNG.uniform(0, L, 3)
    b = origin + RNG.uniform(-0.5 * L, 1.5 * L, 3)
    d = unit(b - a)
    return [*(a - 2 * L * d), *d, 50.0, 1.0]


def test_by_hand_4x4x4_diagonal_with_corner_ties(O, W):
    ids = np.zeros((4, 4, 4), dtype=np.uint8)
    for k in range(4):
        ids[0, k, k] = 1 + k                                    # [iz][iy][ix]: the x-y diagonal of slice z=0
    ids[0, 1, 0] = ids[0, 0, 1] = 4                             # off-diagonal neighbours must contribute nothing
    h = 1e-3
    vol = W.voxels(ids, h)
    d = unit([1, 1, 0])
    ray = [-1e-3, -1e-3, 0.5e-3, *d, 50.0, 1.0]                 # passes exactly through the voxel corners
    expect = (MUS[1] + MUS[2] + MUS[3] + MUS[4]) * h * np.sqrt(2)
    assert abs(tau(O, vol, ray) - expect) < 1e-15 * 500


def test_axis_parallel_ray_is_the_exact_sum(O, W):
    ids = RNG.integers(0, 5, size=(6, 5, 7)).astype(np.uint8)
    h = 2e-3
    vol = W.voxels(ids, h, T=(0.1, -0.2, 0.3))
    for (iy, iz) in ((0, 0), (4, 5), (2, 3)):
        ray = [0.0, -0.2 + (iy + 0.37) * h, 0.3 + (iz + 0.81) * h, 1, 0, 0, 50.0, 1.0]
        expect = sum(MUS[i] for i in ids[iz, iy, :]) * h
        assert abs(tau(O, vol, ray) - expect) < 1e-13
        ray_rev = [1.0, ray[1], ray[2], -1, 0, 0, 50.0, 1.0]
        assert abs(tau(O, vol, ray_rev) - expect) < 1e-13
    ray = [0.1 + 3.5 * h, -0.2 + 1.5 * h, 0.0, 0, 0, 1, 50.0, 1.0]
    assert abs(tau(O, vol, ray) - sum(MUS[i] for i in ids[:, 1, 3]) * h) < 1e-13


def test_homogeneous_volume_equals_box_chord(O, W):
    n, h = 16, 1.5e-3
    ids = np.full((n, n, n), 2, dtype=np.uint8)
    org = np.array([-0.01, 0.02, 0.4])
    Rm = W.random_rotation(np.random.default_rng(5))
    # voxel pose: T is the corner; the equivalent box primitive is centred at corner + R^T (L/2, L/2, L/2)
    vol = W.voxels(ids, h, R=Rm, T=org)
    half = 0.5 * n * h
    box = W.solids([W.solid_box((half,) * 3, 2, 0, R=Rm, T=org + Rm.T @ np.full(3, half))])
    hits = 0
    for _ in range(200):
        ray = random_ray(n, h, org)
        ray[0:3] = list(org + Rm.T @ (np.array(ray[0:3]) - org)); ray[3:6] = list(Rm.T @ np.array(ray[3:6]))
        a, b = tau(O, vol, ray), tau(O, box, ray)
        assert abs(a - b) < 1e-12
        hits += b > 0
    assert hits > 100


def test_box_phantom_on_voxel_faces_equals_box_primitive(O, W):
    n, h = 20, 1e-3
    ids = np.zeros((n, n, n), dtype=np.uint8)
    ids[4:15, 6:12, 3:17] = 3                                   # z 4..15, y 6..12, x 3..17
    vol = W.voxels(ids, h)
    box = W.solids([W.solid_box((7e-3, 3e-3, 5.5e-3), 3, 0, T=(10e-3, 9e-3, 9.5e-3))])
    for _ in range(200):
        ray = random_ray(n, h, np.zeros(3))
        assert abs(tau(O, vol, ray) - tau(O, box, ray)) < 1e-13


def test_reversed_ray_and_upsampled_phantom(O, W):
    n, h = 12, 2e-3
    ids = RNG.integers(0, 5, size=(n, n, n)).astype(np.uint8)
    vol = W.voxels(ids, h)
    up = W.voxels(np.repeat(np.repeat(np.repeat(ids, 2, 0), 2, 1), 2, 2), h / 2)
    nz = 0
    for _ in range(150):
        ray = random_ray(n, h, np.zeros(3))
        t = tau(O, vol, ray)
        o, d = np.array(ray[0:3]), np.array(ray[3:6])
        rev = [*(o + 10 * n * h * d), *(-d), 50.0, 1.0]
        assert abs(tau(O, vol, rev) - t) < 1e-12
        assert abs(tau(O, up, ray) - t) < 1e-12
        nz += t > 0
    assert nz > 75


def test_origin_inside_and_misses(O, W):
    n, h = 8, 1e-3
    ids = np.full((n, n, n), 1, dtype=np.uint8)
    vol = W.voxels(ids, h)
    assert abs(tau(O, vol, [4e-3, 4e-3, 4e-3, 0, 0, 1, 50.0, 1.0]) - MUS[1] * 4e-3) < 1e-15   # starts inside
    assert tau(O, vol, [4e-3, 4e-3, 9e-3, 0, 0, 1, 50.0, 1.0]) == 0.0                           # behind the ray
    assert tau(O, vol, [9e-3, 4e-3, -1e-3, 0, 0, 1, 50.0, 1.0]) == 0.0                          # passes beside
    assert tau(O, vol, [8e-3, 4e-3, -1e-3, 0, 0, 1, 50.0, 1.0]) == 0.0                          # on the boundary plane


def marching_tau(ids, h, mus, o, d, step, t_end):
    """The paper's own scheme: advance by a small increment, find the voxel, attenuate."""
    t = (np.arange(int(t_end / step)) + 0.5) * step
    P = o[None, :] + t[:, None] * d[None, :]
    idx = np.floor(P / h).astype(np.int64)
    nz, ny, nx = ids.shape
    ok = np.all(idx >= 0, axis=1) & (idx[:, 0] < nx) & (idx[:, 1] < ny) & (idx[:, 2] < nz)
    m = np.zeros(len(t))
    m[ok] = np.asarray(mus)[ids[idx[ok, 2], idx[ok, 1], idx[ok, 0]]]
    return m.sum() * step


def test_paper_fixed_step_marching_converges_to_the_exact_traversal(O, W):
    inst = W.config4(small=True, n_vox=32)
    vol = inst["components"][1]
    ids, h = vol["ids"], vol["h"]
    E = 60.0
    mus = [0.0] + [O.mu(m, E) for m in inst["materials"][1:]]
    src = inst["components"][0]
    for i in range(6):
        ray = O.source_ray(src, 1, i)
        ray[6] = E
        exact = tau(O, vol, list(ray), mats=inst["materials"])
        o = ray[0:3] - vol["T"]
        errs = [abs(marching_tau(ids, h, mus, o, ray[3:6], h / k, 3.0) - exact) for k in (3, 30, 300)]
        assert errs[2] < 2e-3 * max(exact, 1.0)
        assert errs[2] < errs[0] or errs[0] < 1e-3 * max(exact, 1.0)
        assert exact > 0
