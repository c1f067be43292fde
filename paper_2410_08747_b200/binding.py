"""ctypes binding of libmcx_b200.so (include/mcx.h).  Argument marshalling only: every step of the hot path runs
in the CUDA kernels.  PyTorch is used for device memory and streams, nothing else.

The instrument descriptions come from the `workloads` module (plain dicts of numbers and numpy arrays).
There is no CPU fallback: if the library is missing or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MCX_OK = 0
STATUS_NAMES = {0: "MCX_OK", 1: "MCX_ERR_INVALID_ARG", 2: "MCX_ERR_UNSUPPORTED", 3: "MCX_ERR_RANGE", 4: "MCX_ERR_WORKSPACE",
                5: "MCX_ERR_CUDA", 6: "MCX_ERR_CAPACITY"}
KIND = {"source": 0, "slit_rect": 1, "slit_circ": 2, "solids": 3, "voxels": 4, "mirror": 5, "crystal": 6, "detector": 7,
        "lens": 8}
DET_MODE = {"energy": 0, "wavelength": 1}
POS_MODE = {"point": 0, "disk": 1, "gauss": 2}
DIR_MODE = {"target": 0, "gauss": 1}
ENERGY_MODE = {"mono": 0, "uniform": 1, "spectrum": 2}
SHAPE = {"box": 0, "cyl": 1, "sphere": 2, "mesh": 3}
EXEC_MODE = {"auto": 0, "direct": 1, "sorted": 2}
TALLY_MODE = {"auto": 0, "global": 1, "warp": 2, "block": 3}
FATE_DETECTED, FATE_MISSED, FATE_DEGENERATE = -1, -2, -3

EXPORTS = ["mcx_instrument_workspace_size", "mcx_instrument_create", "mcx_trace", "mcx_trace_range", "mcx_tally_read",
           "mcx_tally_read_host", "mcx_instrument_set_exec", "mcx_instrument_set_tuning", "mcx_upload_bytes", "mcx_tally_reset",
           "mcx_counters_read", "mcx_trace_status", "mcx_trace_dump", "mcx_launch_count", "mcx_instrument_set_timing", "mcx_timing_read", "mcx_instrument_get_tuning", "mcx_instrument_set_pose", "mcx_cnr", "mcx_cnr_static", "mcx_probe_dfma", "mcx_probe_tally",
           "mcx_probe_l2", "mcx_probe_latency", "mcx_instrument_destroy", "mcx_last_error"]
MCX_ERR_CAPACITY = 6
CNR_STATIC_MAX_BINS, CNR_STATIC_MAX_NE = 1 << 18, 4096  # include/mcx.h, mcx_cnr_static

_dp = C.POINTER(C.c_double)
_u64p = C.POINTER(C.c_uint64)


class McxPose(C.Structure):
    _fields_ = [("rot", C.c_double * 9), ("origin", C.c_double * 3)]


class McxMaterial(C.Structure):
    _fields_ = [("n_points", C.c_int64), ("energy_keV", _dp), ("mu_per_m", _dp), ("mu_scatter_per_m", _dp)]


class McxSolid(C.Structure):
    _fields_ = [("shape", C.c_int32), ("material", C.c_int32), ("priority", C.c_int32), ("reserved", C.c_int32),
                ("pose", McxPose), ("dims", C.c_double * 3), ("n_vertices", C.c_int64), ("n_triangles", C.c_int64),
                ("vertices", _dp), ("triangles", C.POINTER(C.c_int32))]


class McxSourceParams(C.Structure):
    _fields_ = [("pos_mode", C.c_int32), ("dir_mode", C.c_int32), ("energy_mode", C.c_int32), ("reserved", C.c_int32),
                ("radius", C.c_double), ("sigma_x", C.c_double), ("sigma_y", C.c_double),
                ("target_w", C.c_double), ("target_h", C.c_double), ("target_dist", C.c_double),
                ("div_x", C.c_double), ("div_y", C.c_double), ("e0", C.c_double), ("de_rel", C.c_double),
                ("spec_emin", C.c_double), ("spec_emax", C.c_double), ("spec_n", C.c_int64), ("spectrum", _dp)]


class McxSlitParams(C.Structure):
    _fields_ = [("xw", C.c_double), ("yh", C.c_double), ("radius", C.c_double)]


class McxSolidsParams(C.Structure):
    _fields_ = [("n_solids", C.c_int64), ("solids", C.POINTER(McxSolid)), ("scatter_order", C.c_int64)]


class McxVoxelsParams(C.Structure):
    _fields_ = [("h", C.c_double), ("nx", C.c_int64), ("ny", C.c_int64), ("nz", C.c_int64), ("ids", C.c_void_p),
                ("scatter_order", C.c_int64)]


class McxMirrorParams(C.Structure):
    _fields_ = [("p", C.c_double), ("q", C.c_double), ("theta", C.c_double), ("length", C.c_double), ("width", C.c_double),
                ("theta_min", C.c_double), ("theta_max", C.c_double), ("e_min", C.c_double), ("e_max", C.c_double),
                ("n_theta", C.c_int64), ("n_e", C.c_int64), ("reflectivity", _dp)]


class McxCrystalParams(C.Structure):
    _fields_ = [("length", C.c_double), ("width", C.c_double), ("d_hkl", C.c_double), ("zeta", C.c_double),
                ("delta0", C.c_double), ("g", C.c_double), ("kappa", C.c_double)]


class McxLensParams(C.Structure):
    _fields_ = [("radius", C.c_double), ("web", C.c_double), ("pitch", C.c_double), ("aperture", C.c_double),
                ("n_lenses", C.c_int64), ("material", C.c_int64), ("n_delta", C.c_int64), ("delta_energy_keV", _dp),
                ("delta", _dp)]


class McxDetectorParams(C.Structure):
    _fields_ = [("xmin", C.c_double), ("xmax", C.c_double), ("ymin", C.c_double), ("ymax", C.c_double),
                ("emin", C.c_double), ("emax", C.c_double), ("nx", C.c_int64), ("ny", C.c_int64), ("ne", C.c_int64),
                ("mode", C.c_int64)]


class McxParamsUnion(C.Union):
    _fields_ = [("source", McxSourceParams), ("slit", McxSlitParams), ("solids", McxSolidsParams),
                ("voxels", McxVoxelsParams), ("mirror", McxMirrorParams), ("crystal", McxCrystalParams),
                ("detector", McxDetectorParams), ("lens", McxLensParams)]


class McxComponent(C.Structure):
    _fields_ = [("kind", C.c_int32), ("reserved", C.c_int32), ("pose", McxPose), ("u", McxParamsUnion)]


class McxTuning(C.Structure):
    _fields_ = [("chunk_log2", C.c_int32), ("sort_grid_bits", C.c_int32), ("absorber_gate", C.c_int32), ("tally_mode", C.c_int32),
                ("staged_walk", C.c_int32), ("walk_batch_setup", C.c_int32), ("walk_batch_settle", C.c_int32)]


FATE_DTYPE = np.dtype([("fate", np.int32), ("reserved", np.int32), ("bin", np.int64), ("p", np.float64)])

_libs = {}


def lib(strict=False):
    """Loads (building first if needed) libmcx_b200.so and declares the prototypes of include/mcx.h.
    strict=True loads the -fmad=false build of the same sources (parity diagnostics, reading R20)."""
    if strict in _libs:
        return _libs[strict]
    path = _build.build(strict=strict)
    if not os.path.exists(path):
        raise RuntimeError("libmcx_b200.so is missing and could not be built; there is no CPU fallback")
    L = C.CDLL(path)
    cp, vp = C.POINTER(McxComponent), C.c_void_p
    mp = C.POINTER(McxMaterial)
    L.mcx_instrument_workspace_size.argtypes = [cp, C.c_int, mp, C.c_int, C.POINTER(C.c_size_t)]
    L.mcx_instrument_create.argtypes = [cp, C.c_int, mp, C.c_int, vp, C.c_size_t, vp, C.POINTER(vp)]
    L.mcx_trace.argtypes = [vp, C.c_uint64, C.c_uint64, vp]
    L.mcx_trace_range.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, vp]
    L.mcx_tally_read.argtypes = [vp, C.c_int, vp, vp, vp, C.c_size_t, vp]
    L.mcx_tally_read_host.argtypes = [vp, C.c_int, vp, vp, vp, C.c_size_t, vp]
    L.mcx_instrument_set_exec.argtypes = [vp, C.c_int]
    L.mcx_instrument_set_exec.restype = C.c_int
    L.mcx_instrument_set_tuning.argtypes = [vp, C.POINTER(McxTuning)]
    L.mcx_instrument_set_tuning.restype = C.c_int
    L.mcx_instrument_get_tuning.argtypes = [vp, C.POINTER(McxTuning)]
    L.mcx_instrument_get_tuning.restype = C.c_int
    L.mcx_trace_status.argtypes = [vp, vp]
    L.mcx_trace_status.restype = C.c_int
    L.mcx_probe_l2.argtypes = [vp, C.c_uint64, vp, C.c_int, C.c_int64, vp]
    L.mcx_probe_l2.restype = C.c_int
    L.mcx_probe_latency.argtypes = [vp, C.c_uint64, vp, C.c_int, C.c_int, C.c_int64, vp]
    L.mcx_probe_latency.restype = C.c_int
    L.mcx_instrument_set_timing.argtypes = [vp, C.c_int]
    L.mcx_instrument_set_timing.restype = C.c_int
    L.mcx_timing_read.argtypes = [vp, _dp, _dp, C.POINTER(C.c_int64)]
    L.mcx_timing_read.restype = C.c_int
    L.mcx_instrument_set_pose.argtypes = [vp, C.c_int, C.POINTER(McxPose), vp]
    L.mcx_instrument_set_pose.restype = C.c_int
    L.mcx_cnr.argtypes = [vp, vp, vp, C.c_int64, C.c_int64, C.c_int64, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_double,
                          C.c_double, C.c_double, vp, vp, vp]
    L.mcx_cnr.restype = C.c_int
    L.mcx_cnr_static.argtypes = [vp, C.c_int, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.c_double, vp, vp, vp]
    L.mcx_cnr_static.restype = C.c_int
    L.mcx_upload_bytes.argtypes = [vp]
    L.mcx_upload_bytes.restype = C.c_uint64
    L.mcx_tally_reset.argtypes = [vp, vp]
    L.mcx_counters_read.argtypes = [vp, vp, C.c_int, vp]
    L.mcx_trace_dump.argtypes = [vp, C.c_uint64, C.c_uint64, C.c_uint64, vp, vp]
    L.mcx_launch_count.argtypes = [vp]
    L.mcx_launch_count.restype = C.c_uint64
    L.mcx_probe_dfma.argtypes = [vp, C.c_int, C.c_int64, vp]
    L.mcx_probe_tally.argtypes = [vp, C.c_uint64, C.c_int, C.c_int64, vp]
    L.mcx_instrument_destroy.argtypes = [vp]
    L.mcx_instrument_destroy.restype = None
    L.mcx_last_error.restype = C.c_char_p
    for name in ("mcx_instrument_workspace_size", "mcx_instrument_create", "mcx_trace", "mcx_trace_range",
                 "mcx_tally_read", "mcx_tally_read_host", "mcx_tally_reset", "mcx_counters_read", "mcx_trace_dump", "mcx_probe_dfma", "mcx_probe_tally"):
        getattr(L, name).restype = C.c_int
    _libs[strict] = L
    return L


class McxError(RuntimeError):
    def __init__(self, status, message):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


def _check(status, L=None):
    if status != MCX_OK:
        raise McxError(status, (L or lib()).mcx_last_error().decode("utf-8", "replace"))


def _set_pose(pose, d):
    R = np.ascontiguousarray(d["R"], dtype=np.float64).reshape(9)
    T = np.ascontiguousarray(d["T"], dtype=np.float64).reshape(3)
    pose.rot[:] = R.tolist()
    pose.origin[:] = T.tolist()


def _ptr(a, typ=_dp):
    return a.ctypes.data_as(typ)


def marshal(inst, keep, device_voxels):
    """workloads dict -> (McxComponent array, McxMaterial array).  `keep` collects the host buffers that must live
    until create returns; `device_voxels(ids_numpy)` uploads a voxel volume and returns its device pointer."""
    comps = (McxComponent * len(inst["components"]))()
    for c, cd in zip(comps, inst["components"]):
        k = cd["kind"]
        c.kind = KIND[k]
        _set_pose(c.pose, cd)
        if k == "source":
            s = c.u.source
            s.pos_mode, s.dir_mode, s.energy_mode = POS_MODE[cd["pos_mode"]], DIR_MODE[cd["dir_mode"]], ENERGY_MODE[cd["e_mode"]]
            s.radius, s.sigma_x, s.sigma_y = cd["radius"], cd["sigma_x"], cd["sigma_y"]
            s.target_w, s.target_h, s.target_dist = cd["target_w"], cd["target_h"], cd["target_dist"]
            s.div_x, s.div_y, s.e0, s.de_rel = cd["div_x"], cd["div_y"], cd["E0"], cd["dE_rel"]
            s.spec_emin, s.spec_emax = cd["spec_Emin"], cd["spec_Emax"]
            if cd["spectrum"] is not None:
                sp = np.ascontiguousarray(cd["spectrum"], dtype=np.float64)
                keep.append(sp)
                s.spec_n, s.spectrum = len(sp), _ptr(sp)
        elif k == "slit_rect":
            c.u.slit.xw, c.u.slit.yh = cd["xw"], cd["yh"]
        elif k == "slit_circ":
            c.u.slit.radius = cd["radius"]
        elif k == "solids":
            arr = (McxSolid * max(1, len(cd["solids"])))()
            for s, sd in zip(arr, cd["solids"]):
                s.shape, s.material, s.priority = SHAPE[sd["shape"]], sd["material"], sd["priority"]
                _set_pose(s.pose, sd)
                if sd["shape"] == "box":
                    s.dims[:] = list(sd["half"])
                elif sd["shape"] == "cyl":
                    s.dims[:] = [sd["radius"], sd["half_height"], 0.0]
                elif sd["shape"] == "sphere":
                    s.dims[:] = [sd["radius"], 0.0, 0.0]
                else:
                    v = np.ascontiguousarray(sd["verts"], dtype=np.float64)
                    t = np.ascontiguousarray(sd["tris"], dtype=np.int32)
                    keep += [v, t]
                    s.n_vertices, s.n_triangles = len(v), len(t)
                    s.vertices, s.triangles = _ptr(v), _ptr(t, C.POINTER(C.c_int32))
            keep.append(arr)
            c.u.solids.n_solids, c.u.solids.solids = len(cd["solids"]), arr
            c.u.solids.scatter_order = cd.get("scatter_order", 0)
        elif k == "voxels":
            ids = np.ascontiguousarray(cd["ids"], dtype=np.uint8)
            v = c.u.voxels
            v.h = cd["h"]
            v.nz, v.ny, v.nx = ids.shape
            v.ids = device_voxels(ids)
            v.scatter_order = cd.get("scatter_order", 0)
        elif k == "mirror":
            m, t = c.u.mirror, cd["table"]
            m.p, m.q, m.theta, m.length, m.width = cd["p"], cd["q"], cd["theta"], cd["length"], cd["width"]
            m.theta_min, m.theta_max, m.e_min, m.e_max = t["theta_min"], t["theta_max"], t["E_min"], t["E_max"]
            Rt = np.ascontiguousarray(t["R"], dtype=np.float64)
            keep.append(Rt)
            m.n_theta, m.n_e, m.reflectivity = t["n_theta"], t["n_E"], _ptr(Rt)
        elif k == "crystal":
            x = c.u.crystal
            x.length, x.width, x.d_hkl, x.zeta, x.delta0 = cd["length"], cd["width"], cd["d_hkl"], cd["zeta"], cd["delta0"]
            x.g, x.kappa = cd.get("g", 0.0), cd.get("kappa", 0.0)
        elif k == "lens":
            l = c.u.lens
            l.radius, l.web, l.pitch, l.aperture = cd["radius"], cd["web"], cd["pitch"], cd["aperture"]
            l.n_lenses, l.material = cd["n_lenses"], cd["material"]
            dE = np.ascontiguousarray(cd["delta_table"]["E"], dtype=np.float64)
            dl = np.ascontiguousarray(cd["delta_table"]["delta"], dtype=np.float64)
            keep += [dE, dl]
            l.n_delta, l.delta_energy_keV, l.delta = len(dE), _ptr(dE), _ptr(dl)
        elif k == "detector":
            d = c.u.detector
            d.xmin, d.xmax, d.ymin, d.ymax = cd["xmin"], cd["xmax"], cd["ymin"], cd["ymax"]
            d.emin, d.emax, d.nx, d.ny, d.ne = cd["Emin"], cd["Emax"], cd["nx"], cd["ny"], cd["nE"]
            d.mode = DET_MODE[cd.get("mode", "energy")]
        else:
            raise ValueError(f"unknown component kind {k!r}")
    mats = (McxMaterial * max(1, len(inst["materials"])))()
    for m, md in zip(mats, inst["materials"]):
        if md is None:
            m.n_points = 0
            continue
        E = np.ascontiguousarray(md["E"], dtype=np.float64)
        mu = np.ascontiguousarray(md["mu"], dtype=np.float64)
        keep += [E, mu]
        m.n_points, m.energy_keV, m.mu_per_m = len(E), _ptr(E), _ptr(mu)
        if md.get("mu_s") is not None:
            mus = np.ascontiguousarray(md["mu_s"], dtype=np.float64)
            keep.append(mus)
            m.mu_scatter_per_m = _ptr(mus)
    return comps, mats


class Instrument:
    """A device-resident instrument (mcx_instrument handle + the torch buffers it lives in)."""

    def __init__(self, inst, device="cuda:0", strict=False, voxels_pinned=None, sync=True):
        """voxels_pinned: optional pinned uint8 torch tensor holding the voxel volume (copied asynchronously instead
        of inst's numpy array); sync=False leaves the create enqueued on the current stream."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the mcx hot path has no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.inst = inst
        self.n_rays, self.seed = inst["n_rays"], inst["seed"]
        self.dets = [c for c in inst["components"] if c["kind"] == "detector"]
        self.n_comps, self.n_mats = len(inst["components"]), len(inst["materials"])
        self._keep, self._dev = [], []
        self.handle = None
        L = self.L = lib(strict)

        self.voxel_upload_bytes = 0

        def device_voxels(ids):
            src = voxels_pinned if voxels_pinned is not None else torch.from_numpy(ids)
            t = src.to(self.device, non_blocking=voxels_pinned is not None)
            self._dev.append(t)
            self.voxel_upload_bytes += t.numel()
            return t.data_ptr()

        with torch.cuda.device(self.device):
            comps, mats = marshal(inst, self._keep, device_voxels)
            nbytes = C.c_size_t()
            _check(L.mcx_instrument_workspace_size(comps, self.n_comps, mats, self.n_mats, C.byref(nbytes)), L)
            self.workspace_bytes = nbytes.value
            self.workspace = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
            base = (self.workspace.data_ptr() + 255) // 256 * 256
            h = C.c_void_p()
            _check(L.mcx_instrument_create(comps, self.n_comps, mats, self.n_mats, base, self.workspace_bytes,
                                           self._stream(), C.byref(h)), L)
            self.handle = h
            if sync:
                torch.cuda.current_stream().synchronize()
                self._dev.clear()    # the voxel volume was copied into the workspace
        self._keep.clear()   # HOST inputs are consumed by create

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def trace(self, n_rays=None, seed=None, first=0):
        """mcx_trace_range: enqueue rays [first, first+n_rays) on the current stream (asynchronous)."""
        n = self.n_rays if n_rays is None else int(n_rays)
        s = self.seed if seed is None else int(seed)
        _check(self.L.mcx_trace_range(self.handle, int(first), n, s, self._stream()), self.L)

    def tally(self, detector=0, out=None):
        """mcx_tally_read -> (N uint64-as-int64, p, p2) device tensors of n_bins."""
        torch = self.torch
        d = self.dets[detector]
        nb = d["nx"] * d["ny"] * d["nE"]
        if out is None:
            out = (torch.empty(nb, dtype=torch.int64, device=self.device), torch.empty(nb, dtype=torch.float64, device=self.device),
                   torch.empty(nb, dtype=torch.float64, device=self.device))
        N, P, P2 = out
        _check(self.L.mcx_tally_read(self.handle, detector, N.data_ptr(), P.data_ptr(), P2.data_ptr(), nb, self._stream()), self.L)
        return N, P, P2

    def tally_host(self, out, detector=0):
        """mcx_tally_read_host into (N int64, p, p2) pinned host tensors; asynchronous on the current stream."""
        N, P, P2 = out
        _check(self.L.mcx_tally_read_host(self.handle, detector, N.data_ptr(), P.data_ptr(), P2.data_ptr(), N.numel(),
                                          self._stream()), self.L)
        return out

    def set_exec(self, mode):
        """mcx_instrument_set_exec: "auto" | "direct" | "sorted" (lane scheduling, row a13)."""
        _check(self.L.mcx_instrument_set_exec(self.handle, EXEC_MODE[mode]), self.L)

    def set_tuning(self, chunk_log2=0, sort_grid_bits=0, absorber_gate=0, tally_mode="auto", staged_walk=0, walk_batch_setup=0,
                   walk_batch_settle=0):
        """mcx_instrument_set_tuning; 0 / "auto" = keep the library's choice."""
        t = McxTuning(int(chunk_log2), int(sort_grid_bits), int(absorber_gate), TALLY_MODE[tally_mode], int(staged_walk),
                      int(walk_batch_setup), int(walk_batch_settle))
        _check(self.L.mcx_instrument_set_tuning(self.handle, C.byref(t)), self.L)

    def get_tuning(self):
        """mcx_instrument_get_tuning -> dict of the settings in effect (tally_mode by name)."""
        t = McxTuning()
        _check(self.L.mcx_instrument_get_tuning(self.handle, C.byref(t)), self.L)
        names = {v: k for k, v in TALLY_MODE.items()}
        return {"chunk_log2": t.chunk_log2, "sort_grid_bits": t.sort_grid_bits, "absorber_gate": t.absorber_gate,
                "tally_mode": names[t.tally_mode], "staged_walk": t.staged_walk, "walk_batch_setup": t.walk_batch_setup,
                "walk_batch_settle": t.walk_batch_settle}

    def status(self):
        """mcx_trace_status: synchronises the current stream; raises McxError (MCX_ERR_CAPACITY / MCX_ERR_CUDA) if a
        trace since the last reset went wrong."""
        _check(self.L.mcx_trace_status(self.handle, self._stream()), self.L)

    def set_timing(self, on=True):
        """mcx_instrument_set_timing: CUDA events around the ray sort and trace_kernel of every chunk."""
        _check(self.L.mcx_instrument_set_timing(self.handle, int(bool(on))), self.L)

    def timing(self):
        """mcx_timing_read -> dict(sort_ms, trace_ms, launches) summed since the last read; waits for the last event."""
        a, b, n = C.c_double(), C.c_double(), C.c_int64()
        _check(self.L.mcx_timing_read(self.handle, C.byref(a), C.byref(b), C.byref(n)), self.L)
        return {"sort_ms": a.value, "trace_ms": b.value, "launches": int(n.value)}

    def set_pose(self, component, R=None, T=(0.0, 0.0, 0.0)):
        """mcx_instrument_set_pose: new pose (rotation rows R, origin T) of a component for the traces enqueued next."""
        pose = McxPose()
        _set_pose(pose, {"R": np.eye(3) if R is None else R, "T": T})
        _check(self.L.mcx_instrument_set_pose(self.handle, int(component), C.byref(pose), self._stream()), self.L)

    def cnr(self, detector, region_mat, region_ref, e_fit_min, tallies=None):
        """mcx_cnr on the tallies of `detector` (read with mcx_tally_read unless given): (cnr[nE], fit[2]) device tensors."""
        torch = self.torch
        d = self.dets[detector]
        N, P, P2 = self.tally(detector) if tallies is None else tallies
        out = torch.empty(d["nE"], dtype=torch.float64, device=self.device)
        fit = torch.empty(2, dtype=torch.float64, device=self.device)
        rm, rr = (C.c_int32 * 4)(*region_mat), (C.c_int32 * 4)(*region_ref)
        _check(self.L.mcx_cnr(N.data_ptr(), P.data_ptr(), P2.data_ptr(), d["nx"], d["ny"], d["nE"], rm, rr, d["Emin"], d["Emax"],
                              float(e_fit_min), out.data_ptr(), fit.data_ptr(), self._stream()), self.L)
        return out, fit

    def cnr_static(self, detector, region_mat, region_ref, e_fit_min, cnr_out, fit_out):
        """mcx_cnr_static: the same numbers as cnr() into the caller's own tensors (pinned host or device, float64 [nE] and [2]),
        with every intermediate array in the library's static device scratch: no allocation on the way."""
        torch = self.torch
        d = self.dets[detector]
        for t, n in ((cnr_out, d["nE"]), (fit_out, 2)):
            assert t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n and (t.is_cuda or t.is_pinned())
        rm, rr = (C.c_int32 * 4)(*region_mat), (C.c_int32 * 4)(*region_ref)
        _check(self.L.mcx_cnr_static(self.handle, int(detector), rm, rr, float(e_fit_min), cnr_out.data_ptr(), fit_out.data_ptr(),
                                     self._stream()), self.L)

    def upload_bytes(self):
        """host -> device bytes moved to build this instrument (tables by create + the voxel volume)."""
        return int(self.L.mcx_upload_bytes(self.handle)) + self.voxel_upload_bytes

    def reset(self):
        _check(self.L.mcx_tally_reset(self.handle, self._stream()), self.L)

    def counters(self, allow_capacity=False):
        """mcx_counters_read -> dict(absorbed=[n_comps], detected, missed, degenerate, overflows); synchronises.
        allow_capacity: return the counters even if the call reports MCX_ERR_CAPACITY (overflows > 0 says so)."""
        torch = self.torch
        n = self.n_comps + 4
        buf = torch.empty(n, dtype=torch.int64, device=self.device)
        st = self.L.mcx_counters_read(self.handle, buf.data_ptr(), n, self._stream())
        if not (allow_capacity and st == MCX_ERR_CAPACITY):
            _check(st, self.L)
        v = buf.cpu().numpy()
        return {"absorbed": v[:self.n_comps].copy(), "detected": int(v[self.n_comps]), "missed": int(v[self.n_comps + 1]),
                "degenerate": int(v[self.n_comps + 2]), "overflows": int(v[self.n_comps + 3])}

    def trace_dump(self, first, n_rays, seed=None):
        """mcx_trace_dump -> numpy structured array (fate, bin, p) per ray; synchronises."""
        torch = self.torch
        s = self.seed if seed is None else int(seed)
        buf = torch.empty(max(1, int(n_rays)) * FATE_DTYPE.itemsize, dtype=torch.uint8, device=self.device)
        _check(self.L.mcx_trace_dump(self.handle, int(first), int(n_rays), s, buf.data_ptr(), self._stream()), self.L)
        return buf.cpu().numpy()[:int(n_rays) * FATE_DTYPE.itemsize].view(FATE_DTYPE)

    def launch_count(self):
        return int(self.L.mcx_launch_count(self.handle))

    def close(self):
        if self.handle is not None:
            self.torch.cuda.synchronize(self.device)
            self.L.mcx_instrument_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def probe_tally(n_records, n_blocks, n_iters, device="cuda:0"):
    """mcx_probe_tally: returns tally records updated per second (3 reductions each) into a table of n_records x 32 B."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        table = torch.zeros(n_records * 4, dtype=torch.int64, device=dev)
        st = C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
        _check(lib().mcx_probe_tally(table.data_ptr(), n_records, n_blocks, max(1, n_iters // 4), st))
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _check(lib().mcx_probe_tally(table.data_ptr(), n_records, n_blocks, n_iters, st))
        e1.record()
        torch.cuda.synchronize(dev)
        return n_blocks * 256 * n_iters / (e0.elapsed_time(e1) * 1e-3)


def probe_dfma(n_blocks, n_iters, device="cuda:0"):
    """mcx_probe_dfma: returns the sustained FP64 rate in lane-ops (DFMA) per second, CUDA-event timed."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        sink = torch.empty(n_blocks * 256, dtype=torch.float64, device=dev)
        st = C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
        _check(lib().mcx_probe_dfma(sink.data_ptr(), n_blocks, n_iters // 4, st))
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _check(lib().mcx_probe_dfma(sink.data_ptr(), n_blocks, n_iters, st))
        e1.record()
        torch.cuda.synchronize(dev)
        return n_blocks * 256 * n_iters * 8 / (e0.elapsed_time(e1) * 1e-3)


def probe_l2(n_bytes, n_blocks, n_iters, device="cuda:0"):
    """mcx_probe_l2: returns random 32-byte sectors read per second from a table of n_bytes (CUDA-event timed)."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        table = torch.zeros(n_bytes // 8, dtype=torch.int64, device=dev)
        sink = torch.empty(n_blocks * 256, dtype=torch.int32, device=dev)
        st = C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
        _check(lib().mcx_probe_l2(table.data_ptr(), n_bytes, sink.data_ptr(), n_blocks, max(4, n_iters // 4), st))
        torch.cuda.synchronize(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _check(lib().mcx_probe_l2(table.data_ptr(), n_bytes, sink.data_ptr(), n_blocks, n_iters, st))
        e1.record()
        torch.cuda.synchronize(dev)
        return n_blocks * 256 * n_iters / (e0.elapsed_time(e1) * 1e-3)


def probe_latency(n_bytes, n_blocks, n_threads, n_iters, device="cuda:0"):
    """mcx_probe_latency: returns seconds per dependent load (one chain per thread) in a table of n_bytes."""
    import torch
    dev = torch.device(device)
    with torch.cuda.device(dev):
        table = torch.zeros(n_bytes // 8, dtype=torch.int64, device=dev)
        sink = torch.empty(n_blocks * 256, dtype=torch.int32, device=dev)
        st = C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
        _check(lib().mcx_probe_latency(table.data_ptr(), n_bytes, sink.data_ptr(), n_blocks, n_threads, max(1, n_iters // 4), st))
        torch.cuda.synchronize(dev)
        # the init launch of the second call is timed too: one pass over the table, small against n_iters dependent loads
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        _check(lib().mcx_probe_latency(table.data_ptr(), n_bytes, sink.data_ptr(), n_blocks, n_threads, n_iters, st))
        e1.record()
        torch.cuda.synchronize(dev)
        return e0.elapsed_time(e1) * 1e-3 / n_iters
