"""ctypes binding of the CPU oracle (oracle/mcx_oracle.cpp).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It shares nothing with paper_2410_08747_b200/ and never imports it; the only common module is the
seeded input generator `workloads`, which holds none of the method's arithmetic.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mcx_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle_mcx.so")

KIND = {"source": 0, "slit_rect": 1, "slit_circ": 2, "solids": 3, "voxels": 4, "mirror": 5, "crystal": 6, "detector": 7,
        "lens": 8}
DET_MODE = {"energy": 0, "wavelength": 1}
POS = {"point": 0, "disk": 1, "gauss": 2}
DIR = {"target": 0, "gauss": 1}
EMODE = {"mono": 0, "uniform": 1, "spectrum": 2}
SHAPE = {"box": 0, "cyl": 1, "sphere": 2, "mesh": 3}
F_DETECTED, F_MISSED, F_DEGENERATE = -1, -2, -3

_dp = C.POINTER(C.c_double)


class OrcMaterial(C.Structure):
    _fields_ = [("n", C.c_int64), ("E", _dp), ("mu", _dp), ("mu_s", _dp)]


class OrcSolid(C.Structure):
    _fields_ = [("shape", C.c_int32), ("material", C.c_int32), ("priority", C.c_int32), ("pad", C.c_int32),
                ("R", C.c_double * 9), ("T", C.c_double * 3),
                ("hx", C.c_double), ("hy", C.c_double), ("hz", C.c_double), ("radius", C.c_double),
                ("half_height", C.c_double), ("n_verts", C.c_int64), ("n_tris", C.c_int64),
                ("verts", _dp), ("tris", C.POINTER(C.c_int32))]


class OrcComponent(C.Structure):
    _fields_ = [("kind", C.c_int32), ("pos_mode", C.c_int32), ("dir_mode", C.c_int32), ("e_mode", C.c_int32),
                ("R", C.c_double * 9), ("T", C.c_double * 3),
                ("radius", C.c_double), ("sigma_x", C.c_double), ("sigma_y", C.c_double),
                ("target_w", C.c_double), ("target_h", C.c_double), ("target_dist", C.c_double),
                ("div_x", C.c_double), ("div_y", C.c_double),
                ("E0", C.c_double), ("dE_rel", C.c_double), ("spec_Emin", C.c_double), ("spec_Emax", C.c_double),
                ("spec_n", C.c_int64), ("spectrum", _dp),
                ("xw", C.c_double), ("yh", C.c_double), ("slit_radius", C.c_double),
                ("n_solids", C.c_int64), ("solids", C.POINTER(OrcSolid)),
                ("vox_h", C.c_double), ("vnx", C.c_int64), ("vny", C.c_int64), ("vnz", C.c_int64),
                ("vox_ids", C.POINTER(C.c_uint8)),
                ("mir_p", C.c_double), ("mir_q", C.c_double), ("mir_theta", C.c_double), ("mir_length", C.c_double),
                ("mir_width", C.c_double),
                ("tab_theta_min", C.c_double), ("tab_theta_max", C.c_double), ("tab_E_min", C.c_double),
                ("tab_E_max", C.c_double), ("tab_n_theta", C.c_int64), ("tab_n_E", C.c_int64), ("tab_R", _dp),
                ("xtal_length", C.c_double), ("xtal_width", C.c_double), ("xtal_d", C.c_double),
                ("xtal_zeta", C.c_double), ("xtal_delta0", C.c_double),
                ("det_xmin", C.c_double), ("det_xmax", C.c_double), ("det_ymin", C.c_double), ("det_ymax", C.c_double),
                ("det_Emin", C.c_double), ("det_Emax", C.c_double),
                ("det_nx", C.c_int64), ("det_ny", C.c_int64), ("det_nE", C.c_int64),
                ("det_mode", C.c_int64), ("xtal_g", C.c_double), ("xtal_kappa", C.c_double),
                ("lens_R", C.c_double), ("lens_d", C.c_double), ("lens_pitch", C.c_double), ("lens_ra", C.c_double),
                ("lens_N", C.c_int64), ("lens_material", C.c_int64), ("lens_nd", C.c_int64), ("lens_dE", _dp),
                ("lens_delta", _dp), ("scatter_order", C.c_int64)]


class OrcRayFate(C.Structure):
    _fields_ = [("fate", C.c_int32), ("pad", C.c_int32), ("bin", C.c_int64), ("p", C.c_double)]


FATE_DTYPE = np.dtype([("fate", np.int32), ("pad", np.int32), ("bin", np.int64), ("p", np.float64)])


def build(force=False):
    """Compile the oracle with g++ (-O2, no FMA contraction; reading R20).  Building is not using."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        L = _lib
        L.orc_u01.restype = C.c_double
        L.orc_u01.argtypes = [C.c_uint32, C.c_uint32]
        L.orc_mu.restype = C.c_double
        L.orc_mu.argtypes = [_dp, _dp, C.c_int64, C.c_double]
        L.orc_darwin.restype = C.c_double
        L.orc_darwin.argtypes = [C.c_double]
        L.orc_darwin_prins.restype = C.c_double
        L.orc_darwin_prins.argtypes = [C.c_double, C.c_double, C.c_double]
        L.orc_bilinear.restype = C.c_double
        L.orc_bilinear.argtypes = [C.POINTER(OrcComponent), C.c_double, C.c_double]
        L.orc_draw2.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, _dp, _dp]
        L.orc_mesh_hits.restype = C.c_int64
        L.orc_sizeof_component.restype = C.c_int64
        L.orc_sizeof_solid.restype = C.c_int64
        L.orc_trace.restype = C.c_int
        assert L.orc_sizeof_component() == C.sizeof(OrcComponent)
        assert L.orc_sizeof_solid() == C.sizeof(OrcSolid)
    return _lib


def _ptr(a, typ=_dp):
    return a.ctypes.data_as(typ)


def _set_pose(s, d):
    R = np.ascontiguousarray(d["R"], dtype=np.float64).reshape(9)
    T = np.ascontiguousarray(d["T"], dtype=np.float64).reshape(3)
    for k in range(9):
        s.R[k] = R[k]
    for k in range(3):
        s.T[k] = T[k]


def marshal_solid(sd, keep):
    s = OrcSolid()
    s.shape = SHAPE[sd["shape"]]
    s.material, s.priority = sd["material"], sd["priority"]
    _set_pose(s, sd)
    if sd["shape"] == "box":
        s.hx, s.hy, s.hz = sd["half"]
    elif sd["shape"] == "cyl":
        s.radius, s.half_height = sd["radius"], sd["half_height"]
    elif sd["shape"] == "sphere":
        s.radius = sd["radius"]
    else:
        v = np.ascontiguousarray(sd["verts"], dtype=np.float64)
        t = np.ascontiguousarray(sd["tris"], dtype=np.int32)
        keep += [v, t]
        s.n_verts, s.n_tris = len(v), len(t)
        s.verts, s.tris = _ptr(v), _ptr(t, C.POINTER(C.c_int32))
    return s


def marshal_component(cd, keep):
    c = OrcComponent()
    c.kind = KIND[cd["kind"]]
    _set_pose(c, cd)
    k = cd["kind"]
    if k == "source":
        c.pos_mode, c.dir_mode, c.e_mode = POS[cd["pos_mode"]], DIR[cd["dir_mode"]], EMODE[cd["e_mode"]]
        for f in ("radius", "sigma_x", "sigma_y", "target_w", "target_h", "target_dist", "div_x", "div_y", "E0",
                  "dE_rel", "spec_Emin", "spec_Emax"):
            setattr(c, f, cd[f])
        if cd["spectrum"] is not None:
            sp = np.ascontiguousarray(cd["spectrum"], dtype=np.float64)
            keep.append(sp)
            c.spec_n, c.spectrum = len(sp), _ptr(sp)
    elif k == "slit_rect":
        c.xw, c.yh = cd["xw"], cd["yh"]
    elif k == "slit_circ":
        c.slit_radius = cd["radius"]
    elif k == "solids":
        arr = (OrcSolid * len(cd["solids"]))(*[marshal_solid(s, keep) for s in cd["solids"]])
        keep.append(arr)
        c.n_solids, c.solids = len(cd["solids"]), arr
        c.scatter_order = cd.get("scatter_order", 0)
    elif k == "voxels":
        ids = np.ascontiguousarray(cd["ids"], dtype=np.uint8)
        keep.append(ids)
        c.vox_h = cd["h"]
        c.vnz, c.vny, c.vnx = ids.shape
        c.vox_ids = _ptr(ids, C.POINTER(C.c_uint8))
        c.scatter_order = cd.get("scatter_order", 0)
    elif k == "mirror":
        c.mir_p, c.mir_q, c.mir_theta = cd["p"], cd["q"], cd["theta"]
        c.mir_length, c.mir_width = cd["length"], cd["width"]
        t = cd["table"]
        Rt = np.ascontiguousarray(t["R"], dtype=np.float64)
        keep.append(Rt)
        c.tab_theta_min, c.tab_theta_max, c.tab_E_min, c.tab_E_max = t["theta_min"], t["theta_max"], t["E_min"], t["E_max"]
        c.tab_n_theta, c.tab_n_E, c.tab_R = t["n_theta"], t["n_E"], _ptr(Rt)
    elif k == "crystal":
        c.xtal_length, c.xtal_width, c.xtal_d = cd["length"], cd["width"], cd["d_hkl"]
        c.xtal_zeta, c.xtal_delta0 = cd["zeta"], cd["delta0"]
        c.xtal_g, c.xtal_kappa = cd.get("g", 0.0), cd.get("kappa", 0.0)
    elif k == "lens":
        c.lens_R, c.lens_d, c.lens_pitch, c.lens_ra = cd["radius"], cd["web"], cd["pitch"], cd["aperture"]
        c.lens_N, c.lens_material = cd["n_lenses"], cd["material"]
        dE = np.ascontiguousarray(cd["delta_table"]["E"], dtype=np.float64)
        dl = np.ascontiguousarray(cd["delta_table"]["delta"], dtype=np.float64)
        keep += [dE, dl]
        c.lens_nd, c.lens_dE, c.lens_delta = len(dE), _ptr(dE), _ptr(dl)
    elif k == "detector":
        c.det_xmin, c.det_xmax, c.det_ymin, c.det_ymax = cd["xmin"], cd["xmax"], cd["ymin"], cd["ymax"]
        c.det_Emin, c.det_Emax = cd["Emin"], cd["Emax"]
        c.det_nx, c.det_ny, c.det_nE = cd["nx"], cd["ny"], cd["nE"]
        c.det_mode = DET_MODE[cd.get("mode", "energy")]
    else:
        raise ValueError(k)
    return c


def marshal_materials(mats, keep):
    arr = (OrcMaterial * max(1, len(mats)))()
    for m, md in enumerate(mats):
        if md is None:
            arr[m].n = 0
            continue
        E = np.ascontiguousarray(md["E"], dtype=np.float64)
        mu = np.ascontiguousarray(md["mu"], dtype=np.float64)
        keep += [E, mu]
        arr[m].n, arr[m].E, arr[m].mu = len(E), _ptr(E), _ptr(mu)
        if md.get("mu_s") is not None:
            mus = np.ascontiguousarray(md["mu_s"], dtype=np.float64)
            keep.append(mus)
            arr[m].mu_s = _ptr(mus)
    return arr


class Instrument:
    """Marshalled instrument; keeps every numpy buffer alive."""

    def __init__(self, inst):
        self.keep = []
        self.inst = inst
        comps = [marshal_component(cd, self.keep) for cd in inst["components"]]
        self.n_comps = len(comps)
        self.comps = (OrcComponent * len(comps))(*comps)
        self.mats = marshal_materials(inst["materials"], self.keep)
        self.n_mats = len(inst["materials"])
        self.dets = [cd for cd in inst["components"] if cd["kind"] == "detector"]


def trace(inst, first=0, n=None, seed=None, dump=False, mesh_accel=0, tallies=None):
    """Trace rays [first, first+n).  Returns dict(N, P, P2 (lists per detector), absorbed, detected, missed,
    degenerate, dump, work).  Pass `tallies` (a previous result) to accumulate into it."""
    oi = inst if isinstance(inst, Instrument) else Instrument(inst)
    n = oi.inst["n_rays"] if n is None else int(n)
    seed = oi.inst["seed"] if seed is None else int(seed)
    nd = len(oi.dets)
    if tallies is None:
        nb = [d["nx"] * d["ny"] * d["nE"] for d in oi.dets]
        res = {"N": [np.zeros(b, dtype=np.uint64) for b in nb], "P": [np.zeros(b) for b in nb],
               "P2": [np.zeros(b) for b in nb], "absorbed": np.zeros(oi.n_comps, dtype=np.uint64),
               "fates": np.zeros(3, dtype=np.uint64), "work": np.zeros(4, dtype=np.uint64)}
    else:
        res = tallies
    u64p = C.POINTER(C.c_uint64)
    Np = (u64p * max(1, nd))(*[_ptr(a, u64p) for a in res["N"]])
    Pp = (_dp * max(1, nd))(*[_ptr(a) for a in res["P"]])
    P2p = (_dp * max(1, nd))(*[_ptr(a) for a in res["P2"]])
    dump_arr = np.zeros(n, dtype=FATE_DTYPE) if dump else None
    rc = lib().orc_trace(oi.comps, C.c_int(oi.n_comps), oi.mats, C.c_int(oi.n_mats), C.c_uint64(first), C.c_uint64(n),
                         C.c_uint64(seed), Np, Pp, P2p, _ptr(res["absorbed"], u64p), _ptr(res["fates"], u64p),
                         dump_arr.ctypes.data_as(C.POINTER(OrcRayFate)) if dump else None,
                         _ptr(res["work"], u64p), C.c_int(mesh_accel))
    if rc != 0:
        raise RuntimeError(f"orc_trace failed: {rc}")
    res["detected"], res["missed"], res["degenerate"] = (int(x) for x in res["fates"])
    res["dump"] = dump_arr
    return res


# ---- thin wrappers over the single-purpose entry points (used by the pin tests) ----
def philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().orc_philox(c, k, o)
    return tuple(int(x) for x in o)


def u01(wa, wb):
    return lib().orc_u01(wa, wb)


def draw2(seed, i, slot, comp):
    a, b = C.c_double(), C.c_double()
    lib().orc_draw2(seed, i, slot, comp, C.byref(a), C.byref(b))
    return a.value, b.value


def gauss_pair(ua, ub):
    g = (C.c_double * 2)()
    lib().orc_gauss_pair(C.c_double(ua), C.c_double(ub), g)
    return g[0], g[1]


def mu(table, E):
    Ea = np.ascontiguousarray(table["E"], dtype=np.float64)
    ma = np.ascontiguousarray(table["mu"], dtype=np.float64)
    return lib().orc_mu(_ptr(Ea), _ptr(ma), len(Ea), float(E))


def source_ray(src, seed, i):
    keep = []
    c = marshal_component(src, keep)
    out = (C.c_double * 8)()
    lib().orc_source(C.byref(c), C.c_uint64(seed), C.c_uint64(i), out)
    return np.array(out[:])


def primitive_interval(shape, o, d, dims):
    oo = (C.c_double * 3)(*o)
    dd = (C.c_double * 3)(*d)
    dm = (C.c_double * 3)(*(list(dims) + [0, 0, 0])[:3])
    ab = (C.c_double * 2)()
    hit = lib().orc_primitive_interval(SHAPE[shape], oo, dd, dm, ab)
    return (ab[0], ab[1]) if hit else None


def ray_triangle(o, d, v0, v1, v2):
    t = C.c_double()
    arrs = [(C.c_double * 3)(*x) for x in (o, d, v0, v1, v2)]
    r = lib().orc_ray_triangle(*arrs, C.byref(t))
    return r, t.value


def mesh_hits(solid, o, d, use_grid=False, cap=4096):
    keep = []
    s = marshal_solid(solid, keep)
    t = np.zeros(cap)
    orient = np.zeros(cap, dtype=np.int32)
    nt = C.c_uint64()
    oo = (C.c_double * 3)(*o)
    dd = (C.c_double * 3)(*d)
    n = lib().orc_mesh_hits(C.byref(s), oo, dd, C.c_int(int(use_grid)), _ptr(t), _ptr(orient, C.POINTER(C.c_int32)),
                            C.c_int64(cap), C.byref(nt))
    return t[:n].copy(), orient[:n].copy(), int(nt.value)


def apply(comp, ray8, materials=(None,), mesh_accel=0, seed=1, ray_index=0):
    """Apply one non-source component to a ray state (r, d, E, p).  Returns (rc, state, bin).  A scattering sample draws
    from the Philox stream of (seed, ray_index) as component 1."""
    keep = []
    c = marshal_component(comp, keep)
    mats = marshal_materials(list(materials), keep)
    io = (C.c_double * 8)(*ray8)
    b = C.c_int64(-1)
    rc = lib().orc_apply_seeded(C.byref(c), mats, C.c_int(len(materials)), io, C.byref(b), C.c_int(mesh_accel),
                                C.c_uint64(seed), C.c_uint64(ray_index))
    return rc, np.array(io[:]), int(b.value)


def scatter_direction(d, u_mu, u_phi):
    dd = (C.c_double * 3)(*d)
    out = (C.c_double * 3)()
    lib().orc_scatter_direction(dd, C.c_double(u_mu), C.c_double(u_phi), out)
    return np.array(out[:])


def darwin(eta):
    return lib().orc_darwin(float(eta))


def darwin_prins(eta, g, kappa):
    return lib().orc_darwin_prins(float(eta), float(g), float(kappa))


def bilinear(mirror_comp, theta, E):
    keep = []
    c = marshal_component(mirror_comp, keep)
    return lib().orc_bilinear(C.byref(c), float(theta), float(E))


def mirror_prep(p, q, theta):
    out = (C.c_double * 8)()
    lib().orc_mirror_prep(C.c_double(p), C.c_double(q), C.c_double(theta), out)
    return dict(zip(("a", "b", "Z0", "Y0", "nZ", "nY", "tZ", "tY"), out[:]))


def cnr(N, P, P2, ny, nx, nE, region_mat, region_ref, Emin, Emax, E_fit_min):
    """Contrast-to-noise ratio of PAPER.md:257 Eq. (1), CNR = |I_mat - I_ref| / sqrt(sigma_mat^2 + sigma_ref^2), per
    energy bin of one detector's tallies (arrays of ny*nx*nE, bin = (iy*nx + ix)*nE + iE), and its least-squares line
    above E_fit_min ("A least-squares-fit was used to fit the CNR's for energies above the 80 keV").
    Plain definition, numpy.  Readings: a region is a pixel rectangle (x0, x1, y0, y1), half-open; I = mean
    over the region's pixels of the bin's weight sum P; the noise of a region is "the summed squared standard deviations
    of the means": sigma_region^2 = sum_pixels sigma_bin^2 / n_pixels^2, with the McXtrace error estimate of a monitor
    bin, sigma_bin^2 = N/(N-1) |P2 - (P/N)^2| for N > 1 and sigma_bin = P for N <= 1 (sqrt(N) for unit weights).
    Returns (cnr[nE], intercept, slope); cnr = 0 where the noise is 0; the fit uses the bins whose centre energy is
    >= E_fit_min (intercept = slope = 0 with fewer than two such bins)."""
    N = np.asarray(N, dtype=np.float64).reshape(ny, nx, nE)
    P = np.asarray(P, dtype=np.float64).reshape(ny, nx, nE)
    P2 = np.asarray(P2, dtype=np.float64).reshape(ny, nx, nE)
    Ns = np.where(N > 1, N, 2.0)
    var = np.where(N > 1, Ns / (Ns - 1.0) * np.abs(P2 - (P / Ns) ** 2), P * P)

    def region(r):
        x0, x1, y0, y1 = r
        n = (x1 - x0) * (y1 - y0)
        return P[y0:y1, x0:x1, :].sum(axis=(0, 1)) / n, var[y0:y1, x0:x1, :].sum(axis=(0, 1)) / (n * n)

    Im, vm = region(region_mat)
    Ir, vr = region(region_ref)
    noise = np.sqrt(vm + vr)
    out = np.where(noise > 0, np.abs(Im - Ir) / np.where(noise > 0, noise, 1.0), 0.0)
    Ec = Emin + (np.arange(nE) + 0.5) * (Emax - Emin) / nE
    sel = Ec >= E_fit_min
    a = b = 0.0
    if sel.sum() >= 2:
        x, y = Ec[sel], out[sel]
        xm, ym = x.mean(), y.mean()
        b = float(((x - xm) * (y - ym)).sum() / ((x - xm) ** 2).sum())
        a = float(ym - b * xm)
    return out, a, b
