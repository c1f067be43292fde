"""Seeded synthetic instruments for BASELINE.json configs[0..4].

This module serves BOTH the oracle (oracle/oracle.py) and the CUDA binding
(paper_2410_08747_b200/binding.py).  It only *describes* instruments: plain dicts holding numbers and
numpy arrays (poses, sizes, tables, meshes, voxel volumes).  It contains none of the method's
arithmetic: no Philox, no sampling, no intersection, no attenuation, no binning.  The paper's own
inputs (W-anode spectrum, water/Fe/Pb tables, the suitcase volume) are not available,
so every table here is generated from `workload_seed = 20241008 + k` with the shapes, sizes and value
distributions the paper and BASELINE.json describe; DESIGN.md "Input recipe" lists them.

Units: metres, keV, 1/m, radians.  Pose: r_local = R (r_lab - T); rows of R are the local axes in lab
coordinates.  Chain order = list order; component 0 is always the source.
"""
from __future__ import annotations

import numpy as np

WORKLOAD_SEED0 = 20241008
RAY_SEED = 1

I3 = np.eye(3)


def _pose(R=None, T=(0.0, 0.0, 0.0)):
    return {"R": np.array(I3 if R is None else R, dtype=np.float64), "T": np.array(T, dtype=np.float64)}


def source(pos_mode="point", dir_mode="target", e_mode="mono", *, radius=0.0, sigma_x=0.0, sigma_y=0.0,
           target_w=0.0, target_h=0.0, target_dist=1.0, div_x=0.0, div_y=0.0, E0=0.0, dE_rel=0.0,
           spec_Emin=0.0, spec_Emax=0.0, spectrum=None, R=None, T=(0, 0, 0)):
    d = {"kind": "source", "pos_mode": pos_mode, "dir_mode": dir_mode, "e_mode": e_mode, "radius": radius,
         "sigma_x": sigma_x, "sigma_y": sigma_y, "target_w": target_w, "target_h": target_h,
         "target_dist": target_dist, "div_x": div_x, "div_y": div_y, "E0": E0, "dE_rel": dE_rel,
         "spec_Emin": spec_Emin, "spec_Emax": spec_Emax,
         "spectrum": None if spectrum is None else np.ascontiguousarray(spectrum, dtype=np.float64)}
    d.update(_pose(R, T))
    return d


def slit_rect(xw, yh, R=None, T=(0, 0, 0)):
    d = {"kind": "slit_rect", "xw": xw, "yh": yh}
    d.update(_pose(R, T))
    return d


def slit_circ(radius, R=None, T=(0, 0, 0)):
    d = {"kind": "slit_circ", "radius": radius}
    d.update(_pose(R, T))
    return d


def solid_box(half, material, priority, R=None, T=(0, 0, 0)):
    d = {"shape": "box", "half": tuple(float(x) for x in half), "material": int(material), "priority": int(priority)}
    d.update(_pose(R, T))
    return d


def solid_cylinder(radius, half_height, material, priority, R=None, T=(0, 0, 0)):
    d = {"shape": "cyl", "radius": float(radius), "half_height": float(half_height), "material": int(material),
         "priority": int(priority)}
    d.update(_pose(R, T))
    return d


def solid_sphere(radius, material, priority, T=(0, 0, 0)):
    d = {"shape": "sphere", "radius": float(radius), "material": int(material), "priority": int(priority)}
    d.update(_pose(None, T))
    return d


def solid_mesh(verts, tris, material, priority, R=None, T=(0, 0, 0)):
    d = {"shape": "mesh", "verts": np.ascontiguousarray(verts, dtype=np.float64),
         "tris": np.ascontiguousarray(tris, dtype=np.int32), "material": int(material), "priority": int(priority)}
    d.update(_pose(R, T))
    return d


def solids(solid_list, scatter_order=0):
    """scatter_order: at most this many direction changes per ray in the group (materials with a "mu_s" table scatter)."""
    d = {"kind": "solids", "solids": list(solid_list), "scatter_order": int(scatter_order)}
    d.update(_pose())
    return d


def voxels(ids, h, R=None, T=(0, 0, 0), scatter_order=0):
    """ids: uint8 [nz][ny][nx] (x fastest); T = lab position of the corner of voxel (0,0,0); scatter_order: at most this
    many direction changes per ray in the volume (materials with a "mu_s" table scatter)."""
    d = {"kind": "voxels", "ids": np.ascontiguousarray(ids, dtype=np.uint8), "h": float(h), "scatter_order": int(scatter_order)}
    d.update(_pose(R, T))
    return d


def mirror_elliptic(p, q, theta, length, width, table, R=None, T=(0, 0, 0)):
    d = {"kind": "mirror", "p": float(p), "q": float(q), "theta": float(theta), "length": float(length),
         "width": float(width), "table": table}
    d.update(_pose(R, T))
    return d


def crystal_bragg(length, width, d_hkl, zeta, delta0=0.0, g=0.0, kappa=0.0, R=None, T=(0, 0, 0)):
    """g, kappa: absorption ratios of the Darwin-Prins curve (0, 0 = the non-absorbing Darwin curve)."""
    d = {"kind": "crystal", "length": float(length), "width": float(width), "d_hkl": float(d_hkl),
         "zeta": float(zeta), "delta0": float(delta0), "g": float(g), "kappa": float(kappa)}
    d.update(_pose(R, T))
    return d


def lens_parab(radius, web, pitch, aperture, n_lenses, material, delta_table, R=None, T=(0, 0, 0)):
    """Stack of n_lenses double-sided parabolic lenses along the local z axis, centred on the component origin
    (PAPER.md:134, 138).  radius: apex radius of curvature; web: thickness on the axis; pitch: lens-to-lens distance;
    aperture: radius of the circular opening; delta_table: {"E": array, "delta": array}, n = 1 - delta(E)."""
    d = {"kind": "lens", "radius": float(radius), "web": float(web), "pitch": float(pitch), "aperture": float(aperture),
         "n_lenses": int(n_lenses), "material": int(material), "delta_table": delta_table}
    d.update(_pose(R, T))
    return d


def detector(xmin, xmax, ymin, ymax, nx, ny, Emin, Emax, nE, R=None, T=(0, 0, 0), mode="energy"):
    """mode "energy": the third axis bins E [keV] over [Emin, Emax); mode "wavelength" (an L_monitor): it
    bins lambda = hc / E [Angstrom] over [Emin, Emax) read as wavelengths."""
    d = {"kind": "detector", "xmin": float(xmin), "xmax": float(xmax), "ymin": float(ymin), "ymax": float(ymax),
         "nx": int(nx), "ny": int(ny), "Emin": float(Emin), "Emax": float(Emax), "nE": int(nE), "mode": mode}
    d.update(_pose(R, T))
    return d


def instrument(name, components, materials, n_rays, seed=RAY_SEED, **extra):
    """materials[0] must be None (vacuum); others are {"E": array, "mu": array}."""
    assert components[0]["kind"] == "source"
    assert materials[0] is None
    d = {"name": name, "components": components, "materials": materials, "n_rays": int(n_rays), "seed": int(seed)}
    d.update(extra)
    return d


def n_bins(det):
    return det["nx"] * det["ny"] * det["nE"]


def detectors_of(inst):
    return [c for c in inst["components"] if c["kind"] == "detector"]


# ------------------------------------------------------------------------------------------------
# seeded tables
# ------------------------------------------------------------------------------------------------
def random_rotation(rng):
    """Uniform random rotation matrix from a seeded unit quaternion."""
    q = rng.normal(size=4)
    q /= np.linalg.norm(q)
    w, x, y, z = q
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
                     [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
                     [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)]])


def bremsstrahlung_spectrum(rng, n, Emin, Emax, E0):
    """Kramers-like continuum with low-energy filtration, 2% seeded ripple and two characteristic lines
    (stand-in for the tungsten-anode spectrum of PAPER.md:159)."""
    dE = (Emax - Emin) / n
    E = Emin + (np.arange(n) + 0.5) * dE
    Ef = rng.uniform(18.0, 25.0)
    xi = rng.uniform(-1.0, 1.0, size=n)
    S = np.maximum(E0 / E - 1.0, 0.0) * np.exp(-(Ef / E) ** 3) * (1.0 + 0.02 * xi)
    span = Emax - Emin
    for frac, amp in ((0.35, 0.6), (0.42, 0.25)):
        Eline = Emin + frac * span
        S += amp * S.max() * np.exp(-0.5 * ((E - Eline) / (0.004 * span)) ** 2)
    return np.ascontiguousarray(S)


def mu_table(rng, n=1000, Emin=10.0, Emax=150.0, a_range=(20.0, 400.0)):
    """mu(E) = a (E/30)^-b with 1-2 absorption-edge jumps (x J above the edge); n points, uniform in ln E except
    that the two grid points nearest to an edge are moved to E_edge (1 -/+ 1e-6) so the jump is sharp."""
    a = rng.uniform(*a_range)
    b = rng.uniform(2.6, 3.1)
    n_edges = int(rng.integers(1, 3))
    edges = np.sort(rng.uniform(15.0, 90.0, size=n_edges))
    jumps = rng.uniform(3.0, 6.0, size=n_edges)
    E = np.exp(np.linspace(np.log(Emin), np.log(Emax), n))
    E[0], E[-1] = Emin, Emax
    for Ee in edges:
        if not (E[1] < Ee < E[-3]):
            continue
        j = int(np.searchsorted(E, Ee))  # E[j-1] < Ee <= E[j]
        E[j - 1] = Ee * (1.0 - 1e-6)
        E[j] = Ee * (1.0 + 1e-6)
    assert np.all(np.diff(E) > 0)
    mu = a * (E / 30.0) ** (-b)
    for Ee, J in zip(edges, jumps):
        mu = np.where(E > Ee, mu * J, mu)
    return {"E": np.ascontiguousarray(E), "mu": np.ascontiguousarray(mu)}


def with_scattering(rng, table, frac_range=(0.2, 0.9)):
    """Adds the scattering part mu_s(E) = f(E) mu(E) to a mu table: the fraction rises smoothly with energy from about
    frac_range[0] to frac_range[1] (photo-absorption dominates at low energy, scattering at high), seeded midpoint."""
    E = table["E"]
    x = (np.log(E) - np.log(E[0])) / (np.log(E[-1]) - np.log(E[0]))
    mid, width = rng.uniform(0.3, 0.6), rng.uniform(0.1, 0.2)
    f = frac_range[0] + (frac_range[1] - frac_range[0]) / (1.0 + np.exp(-(x - mid) / width))
    out = dict(table)
    out["mu_s"] = np.ascontiguousarray(f * table["mu"])
    return out


def reflectivity_table(rng, n_theta=200, n_E=500, theta_max=8e-3, Emin=5.0, Emax=25.0):
    """Smooth total-external-reflection falloff: R = (1 - eps(E)) / (1 + exp((theta - theta_c(E)) / w))."""
    theta = np.linspace(0.0, theta_max, n_theta)
    E = np.linspace(Emin, Emax, n_E)
    w = rng.uniform(0.15e-3, 0.3e-3)
    eps = rng.uniform(0.02, 0.08) * (E / Emax) ** 0.5
    theta_c = 30e-3 / E
    Rtab = (1.0 - eps)[None, :] / (1.0 + np.exp((theta[:, None] - theta_c[None, :]) / w))
    return {"theta_min": 0.0, "theta_max": float(theta_max), "n_theta": int(n_theta), "E_min": float(Emin),
            "E_max": float(Emax), "n_E": int(n_E), "R": np.ascontiguousarray(Rtab)}


def icosphere(level):
    """Unit icosphere, outward-wound.  level 5 -> 20480, level 6 -> 81920 triangles."""
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = [(-1, t, 0), (1, t, 0), (-1, -t, 0), (1, -t, 0), (0, -1, t), (0, 1, t), (0, -1, -t), (0, 1, -t),
         (t, 0, -1), (t, 0, 1), (-t, 0, -1), (-t, 0, 1)]
    verts = [np.array(p, dtype=np.float64) / np.linalg.norm(p) for p in v]
    faces = [(0, 11, 5), (0, 5, 1), (0, 1, 7), (0, 7, 10), (0, 10, 11), (1, 5, 9), (5, 11, 4), (11, 10, 2),
             (10, 7, 6), (7, 1, 8), (3, 9, 4), (3, 4, 2), (3, 2, 6), (3, 6, 8), (3, 8, 9), (4, 9, 5), (2, 4, 11),
             (6, 2, 10), (8, 6, 7), (9, 8, 1)]
    for _ in range(level):
        cache = {}

        def mid(a, b):
            key = (a, b) if a < b else (b, a)
            if key not in cache:
                m = verts[a] + verts[b]
                verts.append(m / np.linalg.norm(m))
                cache[key] = len(verts) - 1
            return cache[key]

        nf = []
        for (a, b, c) in faces:
            ab, bc, ca = mid(a, b), mid(b, c), mid(c, a)
            nf += [(a, ab, ca), (b, bc, ab), (c, ca, bc), (ab, bc, ca)]
        faces = nf
    V = np.array(verts)
    F = np.array(faces, dtype=np.int32)
    # make sure the winding is outward
    n = np.cross(V[F[:, 1]] - V[F[:, 0]], V[F[:, 2]] - V[F[:, 0]])
    flip = np.einsum("ij,ij->i", n, V[F[:, 0]]) < 0
    F[flip] = F[flip][:, [0, 2, 1]]
    return V, F


def bumpy_sphere(rng, level, radius, amplitude=0.08, n_bumps=6):
    """Star-shaped closed mesh: icosphere with vertex radii x (1 + amplitude * f), |f| <= 1."""
    V, F = icosphere(level)
    f = np.zeros(len(V))
    for _ in range(n_bumps):
        axis = rng.normal(size=3)
        axis /= np.linalg.norm(axis)
        m = int(rng.integers(2, 6))
        c = rng.uniform(-1.0, 1.0)
        f += c * np.cos(m * np.arccos(np.clip(V @ axis, -1.0, 1.0)))
    f /= n_bumps
    return V * (radius * (1.0 + amplitude * f))[:, None], F


def cube_mesh(hx, hy, hz):
    """12-triangle box, outward-wound (used by the mesh == box pin)."""
    V = np.array([[sx * hx, sy * hy, sz * hz] for sz in (-1, 1) for sy in (-1, 1) for sx in (-1, 1)], dtype=np.float64)
    quads = [(0, 2, 3, 1), (4, 5, 7, 6), (0, 1, 5, 4), (2, 6, 7, 3), (0, 4, 6, 2), (1, 3, 7, 5)]
    F = []
    for (a, b, c, d) in quads:
        F += [(a, b, c), (a, c, d)]
    F = np.array(F, dtype=np.int32)
    n = np.cross(V[F[:, 1]] - V[F[:, 0]], V[F[:, 2]] - V[F[:, 0]])
    ctr = (V[F[:, 0]] + V[F[:, 1]] + V[F[:, 2]]) / 3.0
    flip = np.einsum("ij,ij->i", n, ctr) < 0
    F[flip] = F[flip][:, [0, 2, 1]]
    return V, F


def ellipsoid_phantom(rng, n=512, h=1.0e-3, n_ellipsoids=64, n_ids=15, semi=(15e-3, 120e-3)):
    """uint8 [n][n][n] material-ID volume painted with seeded random ellipsoids (suitcase-like contents,
    PAPER.md:184, 188); background 0 = vacuum.  Sizes are in metres and scale with the physical box n*h."""
    ids = np.zeros((n, n, n), dtype=np.uint8)
    L = n * h
    scale = L / 0.512
    coords = (np.arange(n) + 0.5) * h - 0.5 * L
    for e in range(n_ellipsoids):
        ctr = rng.uniform(-150e-3, 150e-3, size=3) * scale
        ax = rng.uniform(semi[0], semi[1], size=3) * scale
        Rm = random_rotation(rng)
        mat_id = 1 + (e % n_ids)
        A = Rm.T @ np.diag(1.0 / ax ** 2) @ Rm  # (x-c)^T A (x-c) <= 1
        rmax = ax.max()
        sl = []
        for a in range(3):
            lo = int(np.searchsorted(coords, ctr[a] - rmax))
            hi = int(np.searchsorted(coords, ctr[a] + rmax))
            sl.append(slice(max(lo, 0), min(hi, n)))
        x = (coords[sl[0]] - ctr[0]).astype(np.float32)
        y = (coords[sl[1]] - ctr[1]).astype(np.float32)
        z = (coords[sl[2]] - ctr[2]).astype(np.float32)
        if len(x) == 0 or len(y) == 0 or len(z) == 0:
            continue
        A32 = A.astype(np.float32)
        X, Y, Z = x[None, None, :], y[None, :, None], z[:, None, None]
        qf = (A32[0, 0] * X * X + A32[1, 1] * Y * Y + A32[2, 2] * Z * Z
              + 2 * A32[0, 1] * X * Y + 2 * A32[0, 2] * X * Z + 2 * A32[1, 2] * Y * Z)
        sub = ids[sl[2], sl[1], sl[0]]
        sub[qf <= 1.0] = mat_id
    return ids


# ------------------------------------------------------------------------------------------------
# optical-axis "turtle" for folded beamlines (placement only: rigid frames, like AT ... RELATIVE)
# ------------------------------------------------------------------------------------------------
class Axis:
    """A running frame (x, y, z unit vectors in lab coordinates) at a lab position; z = beam direction."""

    def __init__(self):
        self.x, self.y, self.z = np.array([1.0, 0, 0]), np.array([0, 1.0, 0]), np.array([0, 0, 1.0])
        self.pos = np.zeros(3)

    def advance(self, dist):
        self.pos = self.pos + dist * self.z

    def roll90(self):
        """Rotate the frame by 90 degrees about the beam, so 'up' becomes horizontal."""
        self.x, self.y = self.y, -self.x

    def pose_normal(self):
        """Pose of a plane component facing the beam."""
        return np.array([self.x, self.y, self.z]), self.pos.copy()

    def reflector(self, theta, sign=+1):
        """Pose of a reflecting surface whose normal (local y) faces the beam at grazing angle theta, deflecting
        towards sign * y; afterwards the frame is turned by 2 theta so z follows the reflected beam."""
        s, c = np.sin(theta), np.cos(theta)
        yy = sign * self.y
        zc = c * self.z + s * yy      # surface tangent
        yc = -s * self.z + c * yy     # surface normal
        xc = np.cross(yc, zc)
        R, T = np.array([xc, yc, zc]), self.pos.copy()
        s2, c2 = np.sin(2 * theta), np.cos(2 * theta)
        z_new = c2 * self.z + s2 * yy
        y_new = sign * (-s2 * self.z + c2 * yy)
        self.z, self.y = z_new, y_new
        self.x = np.cross(self.y, self.z)
        return R, T


# ------------------------------------------------------------------------------------------------
# the five configs
# ------------------------------------------------------------------------------------------------
def config0(n_rays=1_000_000):
    """BASELINE.json configs[0]: monochromatic minimal instrument (shape of paper problem 1)."""
    comps = [
        source("disk", "target", "mono", radius=0.5e-3, target_w=10e-3, target_h=10e-3, target_dist=1.0, E0=20.0),
        slit_rect(2e-3, 2e-3, T=(0, 0, 0.5)),
        solids([solid_box((2.5e-3, 2.5e-3, 2.5e-3), material=1, priority=0, T=(0, 0, 0.8))]),
        detector(-10e-3, 10e-3, -10e-3, 10e-3, 128, 128, 0.0, 40.0, 1, T=(0, 0, 1.0)),
    ]
    mats = [None, {"E": np.array([1.0, 100.0]), "mu": np.array([120.0, 120.0])}]
    return instrument("c0_minimal", comps, mats, n_rays)


def _scattering(rng_seed, mats, comps, scatter_order):
    """gives every material a scattering part (seeded) and lets every sample scatter up to
    scatter_order times per ray."""
    rng = np.random.default_rng(rng_seed)
    mats = [None if m is None else with_scattering(rng, m) for m in mats]
    for c in comps:
        if c["kind"] in ("solids", "voxels"):
            c["scatter_order"] = int(scatter_order)
    return mats


def config1(n_rays=100_000_000, small=False, scatter_order=0):
    """configs[1]: polychromatic energy-dispersive instrument, 8 overlapping primitives, 8 materials."""
    rng = np.random.default_rng(WORKLOAD_SEED0 + 1)
    npx, nE = (64, 32) if small else (256, 128)
    width = 102.4e-3
    spec = bremsstrahlung_spectrum(rng, 1500, 10.0, 150.0, 150.0)
    sl = []
    shapes = ["box", "box", "box", "cyl", "cyl", "cyl", "sphere", "sphere"]
    for s, shape in enumerate(shapes):
        ctr = np.array([rng.uniform(-30e-3, 30e-3), rng.uniform(-30e-3, 30e-3), 0.5 + rng.uniform(-30e-3, 30e-3)])
        size = rng.uniform(5e-3, 50e-3, size=3)
        Rm = random_rotation(rng)
        if shape == "box":
            sl.append(solid_box(0.5 * size, material=s + 1, priority=s, R=Rm, T=ctr))
        elif shape == "cyl":
            sl.append(solid_cylinder(0.5 * size[0], 0.5 * size[1], material=s + 1, priority=s, R=Rm, T=ctr))
        else:
            sl.append(solid_sphere(0.5 * size[0], material=s + 1, priority=s, T=ctr))
    mats = [None] + [mu_table(rng) for _ in range(8)]
    comps = [
        source("gauss", "target", "spectrum", sigma_x=0.1e-3, sigma_y=0.1e-3, target_w=width, target_h=width,
               target_dist=1.0, spec_Emin=10.0, spec_Emax=150.0, spectrum=spec),
        solids(sl),
        detector(-width / 2, width / 2, -width / 2, width / 2, npx, npx, 10.0, 150.0, nE, T=(0, 0, 1.0)),
    ]
    if scatter_order:
        mats = _scattering(WORKLOAD_SEED0 + 101, mats, comps, scatter_order)
    return instrument("c1_polychromatic" + ("_scatter" if scatter_order else ""), comps, mats, n_rays)


SI_D111 = 3.135601154      # Angstrom
HC_KEV_A = 12.398419843    # keV Angstrom (placement of the monochromator only)


def config2(n_rays=500_000_000, small=False):
    """configs[2]: synchrotron beamline: KB mirror pair, Si(111) double crystal, slit, PSD (reading R23)."""
    rng = np.random.default_rng(WORKLOAD_SEED0 + 2)
    theta = 3e-3
    tabV = reflectivity_table(rng)
    tabH = reflectivity_table(rng)
    ax = Axis()
    comps = [source("gauss", "gauss", "uniform", sigma_x=50e-6, sigma_y=10e-6, div_x=20e-6, div_y=5e-6, E0=12.0,
                    dE_rel=0.01)]
    p1, gap, q2 = 30.0, 0.4, 10.0
    ax.advance(p1)
    R, T = ax.reflector(theta, +1)                      # KB-V deflects up
    comps.append(mirror_elliptic(p1, gap + q2, theta, 0.1, 10e-3, tabV, R=R, T=T))
    ax.advance(gap)
    ax.roll90()
    R, T = ax.reflector(theta, +1)                      # KB-H deflects sideways
    comps.append(mirror_elliptic(p1 + gap, q2, theta, 0.1, 10e-3, tabH, R=R, T=T))
    ax.roll90(); ax.roll90(); ax.roll90()
    thetaB = float(np.arcsin(HC_KEV_A / 12.0 / (2 * SI_D111)))
    ax.advance(2.0)
    R, T = ax.reflector(thetaB, +1)
    comps.append(crystal_bragg(0.05, 0.02, SI_D111, 1.33e-4, R=R, T=T))
    ax.advance(0.02)
    R, T = ax.reflector(thetaB, -1)
    comps.append(crystal_bragg(0.05, 0.02, SI_D111, 1.33e-4, R=R, T=T))
    ax.advance(q2 - 2.0 - 0.02)                         # slit at the focus
    R, T = ax.pose_normal()
    comps.append(slit_rect(50e-6, 50e-6, R=R, T=T))
    ax.advance(1e-3)
    R, T = ax.pose_normal()
    npx = 128 if small else 1024
    half = 51.2e-6
    comps.append(detector(-half, half, -half, half, npx, npx, 11.0, 13.0, 1, R=R, T=T))
    return instrument("c2_beamline", comps, [None], n_rays)


def config3(n_rays=100_000_000, small=False, scatter_order=0):
    """configs[3]: two nested closed triangle meshes (bumpy icospheres), polychromatic 20-100 keV."""
    rng = np.random.default_rng(WORKLOAD_SEED0 + 3)
    lv_out, lv_in = (3, 2) if small else (6, 5)
    npx, nE = (64, 16) if small else (512, 64)
    Vo, Fo = bumpy_sphere(rng, lv_out, 20e-3)
    Vi, Fi = bumpy_sphere(rng, lv_in, 10e-3)
    mats = [None] + [mu_table(rng, Emin=20.0, Emax=100.0) for _ in range(2)]
    spec = bremsstrahlung_spectrum(rng, 1500, 20.0, 100.0, 100.0)
    width = 102.4e-3
    comps = [
        source("point", "target", "spectrum", target_w=width, target_h=width, target_dist=1.0, spec_Emin=20.0,
               spec_Emax=100.0, spectrum=spec),
        solids([solid_mesh(Vo, Fo, material=1, priority=0, T=(0, 0, 0.5)),
                solid_mesh(Vi, Fi, material=2, priority=1, T=(0, 0, 0.5))]),
        detector(-width / 2, width / 2, -width / 2, width / 2, npx, npx, 20.0, 100.0, nE, T=(0, 0, 1.0)),
    ]
    if scatter_order:
        mats = _scattering(WORKLOAD_SEED0 + 103, mats, comps, scatter_order)
    return instrument("c3_mesh" + ("_scatter" if scatter_order else ""), comps, mats, n_rays)


def config4(n_rays=1_000_000_000, small=False, n_vox=None, scatter_order=0):
    """configs[4]: energy-dispersive CT projection through a uint8 voxel phantom (paper problem 3)."""
    rng = np.random.default_rng(WORKLOAD_SEED0 + 4)
    if n_vox is None:
        n_vox = 64 if small else 512
    h = 0.512 / n_vox
    npx, nE = (64, 16) if small else (512, 128)
    spec = bremsstrahlung_spectrum(rng, 1500, 20.0, 150.0, 150.0)
    mats = [None] + [mu_table(rng, Emin=20.0, Emax=150.0, a_range=(5.0, 300.0)) for _ in range(15)]
    ids = ellipsoid_phantom(rng, n=n_vox, h=h)
    width = 409.6e-3
    comps = [
        source("point", "target", "spectrum", target_w=width, target_h=width, target_dist=2.5, spec_Emin=20.0,
               spec_Emax=150.0, spectrum=spec),
        voxels(ids, h, T=(-0.256, -0.256, 2.0 - 0.256)),
        detector(-width / 2, width / 2, -width / 2, width / 2, npx, npx, 20.0, 150.0, nE, T=(0, 0, 2.5)),
    ]
    if scatter_order:
        mats = _scattering(WORKLOAD_SEED0 + 104, mats, comps, scatter_order)
    return instrument("c4_edxct" + ("_scatter" if scatter_order else ""), comps, mats, n_rays)


def delta_table(rng, n=200, Emin=15.0, Emax=35.0, A=3.41e-4):
    """Refractive-index decrement delta(E) = A / E^2 (free-electron form; A = 3.41e-4 keV^2 is beryllium, delta = 6.27e-7 at
    23.32 keV) with a smooth seeded ripple of 0.5 %, n points uniform in ln E."""
    E = np.exp(np.linspace(np.log(Emin), np.log(Emax), n))
    E[0], E[-1] = Emin, Emax
    phase, period = rng.uniform(0, 2 * np.pi), rng.uniform(0.15, 0.4)
    delta = A / E ** 2 * (1.0 + 0.005 * np.sin(phase + np.log(E) / period))
    return {"E": np.ascontiguousarray(E), "delta": np.ascontiguousarray(delta)}


def config5(n_rays=100_000_000, small=False):
    """The paper's basic instrument (problem 1): Source_pt, a point source with a flat spectrum of
    5 +- 1 keV, cropped to the 20 mm x 20 mm L_monitor 1 m away, which histograms the wavelength."""
    nL = 32 if small else 128
    comps = [
        source("point", "target", "uniform", target_w=20e-3, target_h=20e-3, target_dist=1.0, E0=5.0, dE_rel=0.2),
        detector(-10e-3, 10e-3, -10e-3, 10e-3, 1, 1, 2.0, 3.2, nL, T=(0, 0, 1.0), mode="wavelength"),
    ]
    return instrument("c5_basic_lmonitor", comps, [None], n_rays)


def config6(n_rays=200_000_000, small=False):
    """The paper's focusing instrument (problem 2, Table 1): undulator-like Gaussian source cropped to
    a 1 mm x 1 mm window at the lens 31.5 m away, a stack of sixteen double-sided parabolic Be lenses (R = 200 um), a
    0.1 mm circular slit 14 m behind the lens centre, then a PSD_monitor and an E_monitor."""
    rng = np.random.default_rng(WORKLOAD_SEED0 + 6)
    p, q = 31.5, 14.0
    be = mu_table(rng, n=400, Emin=15.0, Emax=35.0, a_range=(18.0, 22.0))     # ~ 40 / m at 23 keV, like Be
    dtab = delta_table(rng)
    npx, nE = (64, 32) if small else (256, 128)
    comps = [
        source("gauss", "target", "uniform", sigma_x=48.2e-6, sigma_y=9.5e-6, target_w=1e-3, target_h=1e-3, target_dist=p,
               E0=23.32, dE_rel=1.0 / 23.32),
        lens_parab(200e-6, 50e-6, 1.3e-3, 0.5e-3, 16, 1, dtab, T=(0, 0, p)),
        slit_circ(0.05e-3, T=(0, 0, p + q)),
        detector(-0.1e-3, 0.1e-3, -0.1e-3, 0.1e-3, npx, npx, 0.0, 50.0, 1, T=(0, 0, p + q + 1e-3)),          # PSD_monitor
        detector(-0.1e-3, 0.1e-3, -0.1e-3, 0.1e-3, 1, 1, 22.0, 24.7, nE, T=(0, 0, p + q + 2e-3)),            # E_monitor
    ]
    return instrument("c6_focusing_crl", comps, [None, be], n_rays)


EDXCT_N_DET, EDXCT_PIX, EDXCT_DIST = 5, 0.8e-3, 2.5


def edxct_line_detectors(n_pix, nE, Emin=20.0, Emax=160.0, pix=EDXCT_PIX, dist=EDXCT_DIST):
    """Five 1 x n_pix line detectors stacked vertically on a circle of radius `dist` about the source, each tilted so
    that the line from the source to its centre is perpendicular to its plane (Fig. 3)."""
    half = 0.5 * n_pix * pix
    step = 2.0 * np.arctan(half / dist)
    out = []
    for k in range(EDXCT_N_DET):
        al = (k - (EDXCT_N_DET - 1) / 2) * step
        zax = np.array([0.0, np.sin(al), np.cos(al)])
        yax = np.array([0.0, np.cos(al), -np.sin(al)])
        xax = np.array([1.0, 0.0, 0.0])
        out.append(detector(-0.5 * pix, 0.5 * pix, -half, half, 1, n_pix, Emin, Emax, nE, R=np.array([xax, yax, zax]),
                            T=dist * zax))
    return out


def config7(n_rays=10_000_000, small=False, water=True, scatter_order=0):
    """The paper's EDXCT in-line instrument (problem 3, Table 2, Fig. 3): polychromatic fan beam, a
    voxel sample (a solid block of water, 1 mm voxels, 550 (scan) x 400 (up) x 300 (beam) mm; small: 10 mm voxels with the
    seeded ellipsoid phantom painted in), five tilted 1 x 128 line detectors of 0.8 mm pixels and 128 energy bins over
    20-160 keV.  One trace = one line; extra["scan"] gives the sample's x positions of the 550 lines of a projection."""
    rng = np.random.default_rng(WORKLOAD_SEED0 + 7)
    spec = bremsstrahlung_spectrum(rng, 1500, 20.0, 160.0, 160.0)
    n_mat = 1 if (water and not small) else 15
    mats = [None] + [mu_table(rng, Emin=20.0, Emax=160.0, a_range=(25.0, 45.0) if m == 0 else (5.0, 300.0)) for m in range(n_mat)]
    if small:
        h, shape = 10e-3, (30, 40, 55)                                  # (nz, ny, nx)
        cube = ellipsoid_phantom(rng, n=64, h=0.512 / 64)
        ids = np.ascontiguousarray(cube[:30, 12:52, 4:59])
        ids[ids == 0] = 1                                               # water between the objects
        n_pix, nE = 32, 16
        pix = EDXCT_PIX * 4
    else:
        h, shape = 1e-3, (300, 400, 550)
        ids = np.ones(shape, dtype=np.uint8)
        n_pix, nE = 128, 128
        pix = EDXCT_PIX
    nz, ny, nx = shape
    corner = (-0.5 * nx * h, -0.5 * ny * h, 1.8 - 0.5 * nz * h)
    dets = edxct_line_detectors(n_pix, nE, pix=pix)
    fan_h = 2.0 * EDXCT_DIST * np.tan(0.5 * EDXCT_N_DET * 2.0 * np.arctan(0.5 * n_pix * pix / EDXCT_DIST)) * 1.01
    comps = [source("point", "target", "spectrum", target_w=pix, target_h=fan_h, target_dist=EDXCT_DIST, spec_Emin=20.0,
                    spec_Emax=160.0, spectrum=spec),
             voxels(ids, h, T=corner)] + dets
    n_lines = nx if not small else 11
    scan = [(corner[0] + (line - (n_lines - 1) / 2) * (h if not small else 5 * h), corner[1], corner[2]) for line in range(n_lines)]
    if scatter_order:
        mats = _scattering(WORKLOAD_SEED0 + 107, mats, comps, scatter_order)
    return instrument("c7_edxct_lines" + ("_scatter" if scatter_order else ""), comps, mats, n_rays, scan=scan, sample_component=1)


def config8(n_rays=10_000_000, small=False):
    """The EDXCT line scanner with the sample physics the paper describes (absorption AND scattering):
    config7 whose water scatters, up to 8 events per ray."""
    return config7(n_rays=n_rays, small=small, scatter_order=8)


def config9(n_rays=10_000_000, small=False):
    """configs[4]'s phantom and detector with scattering materials, up to 4 events per ray: the case where a ray's pixel is
    no longer known at birth."""
    return config4(n_rays=n_rays, small=small, scatter_order=4)


def config(k, **kw):
    return (config0, config1, config2, config3, config4, config5, config6, config7, config8, config9)[k](**kw)
