#!/usr/bin/env python
"""bench.py -- rays/s of the mcx hot path on B200 (BASELINE.json: "rays/sec on 1 B200 per instrument; achieved % of
binding roofline").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--instruments 0,1,2,3,4] [--impl reference]

A step = one pass of the whole hot path over one batch of synthetic rays: mcx_trace(n_rays) + mcx_tally_read.
The headline line is BASELINE.json configs[1] (polychromatic energy-dispersive instrument, 1e8 rays: the config the
task names for the N=1 line); every instrument, the headline included, is measured the same way and reported under
"instruments" in the same JSON line with its own roofline (the binding one of several candidates, each against a peak
measured in this run), e2e and cpu_baseline (north_star: "all five configs ... each reported in rays/s with its
achieved fraction of the binding roofline").  DESIGN.md "Measurement" states the algorithmic work model.
The CPU baselines (the oracle on one core and on all cores, as independent processes over disjoint ray windows,
PAPER.md:77) run first, before CUDA is initialised, so that the worker processes can be forked.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC, UNIT = "rays_per_second", "rays/s"
L2_NOTE = "CUDA arm: L2 flushed between timed steps (256 MiB memset, untimed); reference arm: host cores only"
FLUSH_BYTES = 256 << 20          # > the 126 MB L2

# ---------------------------------------------------------------------------------------------------------------
# Algorithmic work model: fp64-pipe lane-operations the method itself needs per unit.
# One DFMA / DADD / DMUL / compare = 1; library functions at the length of a correctly rounded-to-1-ulp fp64
# evaluation (sqrt, div ~ 12; exp ~ 25; log, asin ~ 35; sincos ~ 45; tan ~ 50).  Philox is integer work (not counted).
# ---------------------------------------------------------------------------------------------------------------
OPS_SOURCE = {("disk", "target", "mono"): 120, ("gauss", "target", "spectrum"): 250, ("point", "target", "spectrum"): 150,
              ("gauss", "gauss", "uniform"): 330, ("point", "target", "uniform"): 50, ("gauss", "target", "uniform"): 160}
OPS_LENS_ENTRY, OPS_LENS_SURFACE = 35 + 35 + 25, 110   # log E + delta(E) + final exp; quadratic, 3 sqrt, 3 div, Snell per surface
OPS_SLIT, OPS_DETECTOR, OPS_MIRROR, OPS_CRYSTAL = 35, 80, 250, 180
OPS_SOLIDS_ENTRY, OPS_PRIMITIVE_TEST, OPS_SEGMENT, OPS_MU, OPS_EXP = 35, 45, 10, 35, 25
OPS_VOXEL_ENTRY, OPS_VOXEL_STEP = 100, 6
OPS_TRI_TEST, OPS_BVH_NODE = 45, 14
NOMINAL_FP64_LANES_PER_SM, N_SM = 64, 148
# roofline.traffic (DRAM bytes of the dominant kernel) needs a profiler and is therefore null in this line; the ncu
# captures of the same command are summarised under profiles/ (TRAFFIC_NOTE names the file).
TRAFFIC_NOTE = "not measurable inside bench.py (needs ncu); see profiles/r02_README.md for dram__bytes of this command"


def reached_per_component(n_rays, absorbed):
    """reached[c] = rays that arrive at component c = n_rays - absorbed by components before c."""
    out, alive = [], int(n_rays)
    for a in absorbed:
        out.append(alive)
        alive -= int(a)
    return out


def algorithmic_ops(inst, n_rays, counters, work_per_ray):
    """fp64 lane-ops one trace of n_rays needs, from the ray-accounting counters (rays reaching each component) and the
    per-ray unit counts of the oracle sample (primitive tests, voxel steps, elementary segments, triangle hits)."""
    reach = reached_per_component(n_rays, counters["absorbed"])
    ops = 0.0
    for c, cd in enumerate(inst["components"]):
        k, r = cd["kind"], reach[c]
        if k == "source":
            ops += r * OPS_SOURCE.get((cd["pos_mode"], cd["dir_mode"], cd["e_mode"]), 250)
        elif k in ("slit_rect", "slit_circ"):
            ops += r * OPS_SLIT
        elif k == "detector":
            ops += r * OPS_DETECTOR
        elif k == "mirror":
            ops += r * OPS_MIRROR
        elif k == "crystal":
            ops += r * OPS_CRYSTAL
        elif k == "lens":
            ops += r * (OPS_LENS_ENTRY + 2 * cd["n_lenses"] * OPS_LENS_SURFACE)
        elif k == "solids":
            n_prim = sum(1 for s in cd["solids"] if s["shape"] != "mesh")
            n_mesh = len(cd["solids"]) - n_prim
            ops += r * (OPS_SOLIDS_ENTRY + n_prim * OPS_PRIMITIVE_TEST + OPS_EXP)
            ops += r * work_per_ray["segments"] * (OPS_SEGMENT + OPS_MU)
            if n_mesh:
                # per surface crossing: one exact triangle test and a root-to-leaf walk of a balanced BVH2
                depth = sum(np.log2(max(len(s["tris"]) / 4.0, 2.0)) for s in cd["solids"] if s["shape"] == "mesh") / n_mesh
                ops += r * work_per_ray["tri_hits"] * (OPS_TRI_TEST + 2.0 * depth * OPS_BVH_NODE)
        elif k == "voxels":
            n_mats = sum(1 for m in inst["materials"] if m is not None)
            ops += r * (OPS_VOXEL_ENTRY + n_mats * OPS_MU + OPS_EXP) + r * work_per_ray["voxel_steps"] * OPS_VOXEL_STEP
    return ops


def algorithmic_bytes(inst, n_rays, counters, work_per_ray):
    """HBM bytes the method itself must move per trace: one 32-byte tally sector read + written per detected ray when
    the tally array exceeds L2, one byte per voxel crossed."""
    b = 0.0
    for cd in inst["components"]:
        if cd["kind"] == "detector" and 32 * cd["nx"] * cd["ny"] * cd["nE"] > (126 << 20):
            b += 64.0 * counters["detected"]
        if cd["kind"] == "voxels":
            b += float(n_rays) * work_per_ray["voxel_steps"]
    return b


def mesh_l2(inst, n_rays, counters, work_per_ray):
    """Mesh instruments (L2 sector traffic binds the BVH walk).  Algorithmic 32-byte L2 sectors
    per trace: per surface crossing a root-to-leaf path of the balanced BVH2 (both 32-byte children of every node on
    the path) plus the 72-byte fp64 triangle (3 sectors).  Returns (sectors, bytes of BVH + triangles) or None."""
    reach = reached_per_component(n_rays, counters["absorbed"])
    sectors, footprint = 0.0, 0
    for c, cd in enumerate(inst["components"]):
        if cd["kind"] != "solids":
            continue
        meshes = [s for s in cd["solids"] if s["shape"] == "mesh"]
        if not meshes:
            continue
        depth = float(np.mean([np.ceil(np.log2(max(len(s["tris"]), 2))) for s in meshes]))
        sectors += reach[c] * work_per_ray["tri_hits"] * (2.0 * depth + 3.0)
        for s in meshes:
            d = int(np.ceil(np.log2(max(len(s["tris"]), 2))))
            footprint += (2 << d) * 32 + (1 << d) * 72
    return (sectors, footprint) if footprint else None


# ---------------------------------------------------------------------------------------------------------------
def oracle_work_per_ray(inst, n=20000):
    """Unit counts per ray from a small oracle sample (the oracle counts voxel steps, primitive tests, elementary
    segments and triangle tests exactly)."""
    from oracle import oracle as O
    has_mesh = any(s["shape"] == "mesh" for c in inst["components"] if c["kind"] == "solids" for s in c["solids"])
    o = O.trace(inst, first=0, n=n, dump=False, mesh_accel=1 if has_mesh else 0)
    w = o["work"].astype(np.float64) / n
    out = {"voxel_steps": float(w[0]), "solid_tests": float(w[1]), "tri_tests": float(w[2]), "segments": float(w[3])}
    # surface crossings per ray: every elementary segment inside a mesh has two end points on a surface
    out["tri_hits"] = 2.0 * out["segments"] if has_mesh else 0.0
    return out


def time_oracle(inst, budget_s=15.0, first=0):
    """The oracle as it stands, one host thread, on a bounded prefix of the workload's ray indices."""
    from oracle import oracle as O
    has_mesh = any(s["shape"] == "mesh" for c in inst["components"] if c["kind"] == "solids" for s in c["solids"])
    accel = 1 if has_mesh else 0
    oi = O.Instrument(inst)
    O.trace(oi, first=first, n=100, mesh_accel=accel)           # one-off set-up (the oracle's mesh grid) stays untimed
    n, dt = 1000, 0.0
    while dt < 0.3 and n < inst["n_rays"]:                       # probe until the rate estimate is stable
        n *= 4
        t0 = time.perf_counter()
        O.trace(oi, first=first, n=n, mesh_accel=accel)
        dt = max(time.perf_counter() - t0, 1e-6)
    n_big = int(min(inst["n_rays"], max(n, budget_s * n / dt)))
    t0 = time.perf_counter()
    O.trace(oi, first=first, n=n_big, mesh_accel=accel)
    dt = time.perf_counter() - t0
    return n_big / dt, n_big, dt


def _oracle_worker(oi, first, n, accel, barrier, q):
    from oracle import oracle as O
    barrier.wait()
    t0 = time.time()
    O.trace(oi, first=first, n=n, mesh_accel=accel)
    q.put((t0, time.time()))


def cpu_baseline(inst, budget_s=4.0):
    """The oracle as it stands on the host cores of this box: one thread over a bounded prefix of the workload's ray
    indices, then os.cpu_count() independent processes over disjoint windows of the same length (the paper's own
    scatter-gather scheme), all started together; rate = rays of all windows / (last end - first start).
    Must run before CUDA is initialised (the workers are forked)."""
    import multiprocessing as mp
    from oracle import oracle as O
    has_mesh = any(s["shape"] == "mesh" for c in inst["components"] if c["kind"] == "solids" for s in c["solids"])
    accel = 1 if has_mesh else 0
    rate1, n1, dt1 = time_oracle(inst, budget_s=budget_s)
    cores = os.cpu_count() or 1
    n_w = int(max(1000, rate1 * 0.75 * budget_s))   # windows may lie beyond n_rays: ray indices are just counters
    ctx = mp.get_context("fork")
    oi = O.Instrument(inst)
    barrier, q = ctx.Barrier(cores), ctx.Queue()
    procs = [ctx.Process(target=_oracle_worker, args=(oi, w * n_w, n_w, accel, barrier, q)) for w in range(cores)]
    for p_ in procs:
        p_.start()
    spans = [q.get(timeout=600) for _ in procs]
    for p_ in procs:
        p_.join(timeout=60)
    span = max(e for _, e in spans) - min(b for b, _ in spans)
    rate_all = cores * n_w / span
    cpu_model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                cpu_model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"value": rate_all, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{cores} processes x {n_w} consecutive ray indices of {inst['name']} ({span:.1f} s wall)",
            "one_core": {"value": rate1, "cores": 1, "sample": f"first {n1} ray indices ({dt1:.1f} s)"},
            "cpu_model": cpu_model}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz, self.stop_flag = index, [], set(), None, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.002)

    def result(self):
        self.stop_flag = True
        if self.is_alive():
            self.join(timeout=1.0)
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


# ---------------------------------------------------------------------------------------------------------------
EXEC_MODE = "auto"   # lane scheduling (mcx_instrument_set_exec); --exec overrides for experiments


def bench_instrument(M, torch, inst, n_rays, first, steps, warmup, device, probes, peaks, with_e2e=True, local_rank=0):
    """Times `steps` steps of mcx_trace + mcx_tally_read for one instrument on the current stream.  Returns a dict.
    probes: dict(dfma=lane-ops/s, l2=callable(bytes)->sectors/s, tally=callable(records)->records/s)."""
    g = M.Instrument(inst, device=device)
    g.set_exec(EXEC_MODE)
    tuning = g.get_tuning()
    det = g.dets[-1]
    nb = det["nx"] * det["ny"] * det["nE"]
    last = len(g.dets) - 1
    out = (torch.empty(nb, dtype=torch.int64, device=device), torch.empty(nb, dtype=torch.float64, device=device),
           torch.empty(nb, dtype=torch.float64, device=device))
    flush = torch.empty(FLUSH_BYTES, dtype=torch.uint8, device=device)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    for _ in range(warmup):
        g.trace(n_rays, first=first)
        g.tally(last, out)
    torch.cuda.synchronize(device)
    g.reset()
    launches0 = g.launch_count()
    marks = []
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    for _ in range(steps):
        flush.zero_()                                   # L2 flush, outside the event brackets
        e0, e1, e2 = ev(), ev(), ev()
        e0.record()
        g.trace(n_rays, first=first)
        e1.record()
        g.tally(last, out)
        e2.record()
        marks.append((e0, e1, e2))
    torch.cuda.synchronize(device)
    clocks = sampler.result()
    launches = g.launch_count() - launches0
    t_trace = [a.elapsed_time(b) for a, b, _ in marks]
    t_step = [a.elapsed_time(c) for a, _, c in marks]
    counters = g.counters()
    traced = int(counters["absorbed"].sum()) + counters["detected"] + counters["missed"] + counters["degenerate"]
    assert traced == steps * n_rays, "ray accounting does not add up"
    per_trace = {k: (v / steps if not isinstance(v, np.ndarray) else v / steps) for k, v in counters.items()}
    # the same steps once more with the library's own events around every sort / trace_kernel launch (kept out of the
    # steps timed above: three event records per chunk are visible in a 60 us step)
    g.set_timing(True)
    for _ in range(steps):
        flush.zero_()
        g.trace(n_rays, first=first)
        g.tally(last, out)
    split = g.timing()
    ms_sort, ms_kernel = split["sort_ms"] / steps, split["trace_ms"] / steps
    res = {"n_rays": n_rays, "ms_per_step": float(np.mean(t_step)), "ms_step_min": float(np.min(t_step)),
           "kernel_ms": {"sort_kernels": ms_sort, "trace_kernel": ms_kernel,
                         "tally_read_kernel": float(np.mean(t_step) - np.mean(t_trace)),
                         "trace_kernel_launches_per_step": split["launches"] / steps,
                         "how": "CUDA events on the launching stream: around every sort / trace_kernel launch inside the "
                                "library (mcx_instrument_set_timing), around mcx_tally_read in bench.py"},
           "rays_per_s": n_rays / (np.mean(t_step) * 1e-3), "launches": launches, "clocks": clocks,
           "detected_fraction": counters["detected"] / traced, "tally_bytes": 32 * nb}
    # rooflines of the dominant kernel (trace_kernel): every candidate is algorithmic work per
    # launch / trace_kernel's own device time / a peak measured in this run; the binding one is the largest fraction
    work = oracle_work_per_ray(inst)
    ops = algorithmic_ops(inst, n_rays, per_trace, work)
    byt = algorithmic_bytes(inst, n_rays, per_trace, work)
    sec = ms_kernel * 1e-3
    hbm_peak = (peaks or {}).get("hbm_gbs", 6650.0)
    cand = {"alu": {"achieved": ops / sec / 1e12, "peak": probes["dfma"] / 1e12, "unit": "Tlane-op/s (fp64)",
                    "frac": ops / sec / probes["dfma"], "per_ray": ops / n_rays,
                    "peak_source": "mcx_probe_dfma, measured in this run",
                    "note": "fp64 lane-operations the METHOD needs (work model at the top of bench.py); the voxel walk does "
                            "its 6 per voxel step as integer carries and skips most steps (DESIGN.md 5.3)"},
            "hbm": {"achieved": byt / sec / 1e9, "peak": hbm_peak, "unit": "GB/s", "frac": byt / sec / 1e9 / hbm_peak,
                    "per_ray": byt / n_rays, "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback 6650 GB/s"}}
    n_rec = 1 << (int(nb).bit_length() - 1)
    tally_peak = probes["tally"](n_rec)
    det_rate = res["detected_fraction"] * n_rays / sec
    cand["tally"] = {"achieved": det_rate, "peak": tally_peak, "unit": "records/s", "frac": det_rate / tally_peak,
                     "per_ray": res["detected_fraction"],
                     "peak_source": f"mcx_probe_tally, {n_rec} random 32-byte records, measured in this run"}
    ml2 = mesh_l2(inst, n_rays, per_trace, work)
    if ml2 is not None:
        sectors, footprint = ml2
        table = 1 << int(np.ceil(np.log2(footprint)))
        l2_peak = probes["l2"](table)
        cand["l2"] = {"achieved": sectors / sec * 32 / 1e9, "peak": l2_peak * 32 / 1e9, "unit": "GB/s of 32-byte sectors",
                      "frac": sectors / sec / l2_peak, "per_ray": 32 * sectors / n_rays,
                      "peak_source": f"mcx_probe_l2, random sectors of a {table >> 20} MiB table (BVH + triangles = "
                                     f"{footprint / 2**20:.1f} MiB), measured in this run",
                      "note": "sectors the per-ray walk needs; warps that walk one beam share them (DESIGN.md 5.1)"}
    if tuning["tally_mode"] == "block":
        cand["tally"]["bypassed"] = ("block-private shared-memory tallies (mcx_tally_mode MCX_TALLY_BLOCK): the records in "
                                     "L2 see one flush per block, so this roof does not bind; frac > 1 is the gain over it")
    vox = [c for c in inst["components"] if c["kind"] == "voxels" and c.get("scatter_order", 0) > 0]
    if vox:
        # after its first scattering event a ray walks voxel by voxel in a direction of its own: one 32-byte sector of
        # the volume per voxel visited, at random as far as the memory system is concerned
        sectors = float(n_rays) * work["voxel_steps"]
        footprint = 2 * sum(int(np.prod(c["ids"].shape)) for c in vox)          # cells of {ID, run}
        table = 1 << int(np.ceil(np.log2(footprint)))
        l2_peak = probes["l2"](table)
        cand["l2"] = {"achieved": sectors / sec * 32 / 1e9, "peak": l2_peak * 32 / 1e9, "unit": "GB/s of 32-byte sectors",
                      "frac": sectors / sec / l2_peak, "per_ray": 32 * sectors / n_rays,
                      "peak_source": f"mcx_probe_l2, random sectors of a {table >> 20} MiB table (voxel cells = "
                                     f"{footprint / 2**20:.0f} MiB), measured in this run",
                      "note": "one sector per voxel visited on the legs of scattered rays"}
    for k, c in cand.items():
        # a roof the kernel goes past cannot bind it: the kernel does less of that resource's work than the per-ray model
        # counts (a warp's beam walk reads a BVH sector once for 32 rays; cube-radius skipping does not visit every voxel)
        if c["frac"] > 1.0 and "bypassed" not in c:
            c["bypassed"] = "frac > 1: the kernel needs less of this than the per-ray model counts (DESIGN.md 5.1, 5.4); not binding"
    bound = max((k for k in cand if "bypassed" not in cand[k]), key=lambda k: cand[k]["frac"])
    res["work_per_ray"] = work
    res["tuning"] = tuning
    res["roofline"] = {"bound": bound, "achieved": cand[bound]["achieved"], "peak": cand[bound]["peak"],
                       "unit": cand[bound]["unit"], "frac": cand[bound]["frac"], "traffic": None,
                       "traffic_note": TRAFFIC_NOTE,
                       "kernel": "trace_kernel + scatter_walk_kernel + trace_kernel (staged trace, DESIGN.md 5.4)" if tuning.get("staged_walk") == 1
                       else "trace_kernel", "kernel_ms": ms_kernel,
                       "candidates": cand}
    g.close()
    del flush, out
    torch.cuda.empty_cache()
    if with_e2e:
        res["e2e"] = bench_e2e(M, torch, inst, n_rays, first, 4, device)
    return res


def bench_scan(M, torch, inst, device, steps=1, warmup_lines=None):
    """One projection of the paper's line scanner (550 lines of 1e7 rays): per line the sample is
    moved (mcx_instrument_set_pose), the line's rays are traced, all detectors are read into that line's slice of the
    sinogram stack and the tallies are reset.  CUDA events around the whole projection.  The untimed first pass is a whole
    projection, or its first `warmup_lines` lines."""
    g = M.Instrument(inst, device=device)
    scan, comp, n = inst["scan"], inst["sample_component"], inst["n_rays"]
    nb = [d["nx"] * d["ny"] * d["nE"] for d in g.dets]
    stack = [(torch.empty((len(scan), b), dtype=torch.int64, device=device), torch.empty((len(scan), b), dtype=torch.float64, device=device),
              torch.empty((len(scan), b), dtype=torch.float64, device=device)) for b in nb]
    times = []
    for it in range(steps + 1):
        launches0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for line, T in enumerate(scan if (it > 0 or warmup_lines is None) else scan[:warmup_lines]):
            g.set_pose(comp, T=T)
            g.trace(n, first=line * n)
            for d in range(len(nb)):
                g.tally(d, (stack[d][0][line], stack[d][1][line], stack[d][2][line]))
            g.reset()
        e1.record()
        torch.cuda.synchronize(device)
        if it > 0:                                      # first projection = warm-up
            times.append(e0.elapsed_time(e1))
        launches = g.launch_count() - launches0
    detected = int(sum(int(s_[0].sum()) for s_ in stack))
    g.close()
    ms = float(np.mean(times))
    return {"lines": len(scan), "rays_per_line": n, "ms_per_projection": ms, "rays_per_s": len(scan) * n / (ms * 1e-3),
            "launches_per_projection": launches, "detected_per_projection": detected,
            "paper": "~1500 h single thread, ~50 h on 32 cores, < 4 h on an H100 per projection (PAPER.md:274; other hardware, "
                     "other sample physics: context only)"}


def bench_e2e(M, torch, inst, n_rays, first, steps, device):
    """The same metric through the public API with HOST buffers: every step uploads the instrument description
    (tables from host memory, the voxel volume from pinned memory) with mcx_instrument_create, traces, and reads the
    tallies back into pinned host arrays with mcx_tally_read_host.  Wall-clock around a synchronised step."""
    det = [c for c in inst["components"] if c["kind"] == "detector"][-1]
    nb = det["nx"] * det["ny"] * det["nE"]
    host = (torch.empty(nb, dtype=torch.int64).pin_memory(), torch.empty(nb, dtype=torch.float64).pin_memory(),
            torch.empty(nb, dtype=torch.float64).pin_memory())
    vox = [c for c in inst["components"] if c["kind"] == "voxels"]
    pinned_vox = torch.from_numpy(vox[0]["ids"]).pin_memory() if vox else None
    times, h2d = [], 0
    for it in range(steps + 1):
        torch.cuda.synchronize(device)
        t0 = time.perf_counter()
        g = M.Instrument(inst, device=device, voxels_pinned=pinned_vox, sync=False)
        g.set_exec(EXEC_MODE)
        g.trace(n_rays, first=first)
        g.tally_host(host, len(g.dets) - 1)
        torch.cuda.synchronize(device)
        dt = time.perf_counter() - t0
        h2d = g.upload_bytes()
        g.close()
        if it > 0:                                      # first pass = warm-up (allocator, pinned pages)
            times.append(dt)
    t = float(np.mean(times))
    return {"value": n_rays / t, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(24 * nb),
            "ms_per_step": t * 1e3, "steps": steps, "detected": int(host[0].sum())}


def make_instrument(W, k, n_rays=None):
    kw = {} if n_rays is None else {"n_rays": int(n_rays)}
    return W.config(k, **kw)


def run_reference(args):
    """--impl reference: the oracle (single-threaded C++, as it stands) on host cores, same metric and config; each
    step is a bounded prefix of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import workloads as W
    inst = make_instrument(W, args.config, args.rays)
    rate, n_probe, _ = time_oracle(inst, budget_s=1.0)
    total = args.steps + args.warmup
    n_step = int(max(1000, min(inst["n_rays"], rate * min(8.0, 120.0 / total))))
    from oracle import oracle as O
    oi = O.Instrument(inst)
    has_mesh = any(s["shape"] == "mesh" for c in inst["components"] if c["kind"] == "solids" for s in c["solids"])
    ts = []
    for it in range(total):
        t0 = time.perf_counter()
        O.trace(oi, first=it * n_step, n=n_step, mesh_accel=1 if has_mesh else 0)
        if it >= args.warmup:
            ts.append(time.perf_counter() - t0)
    t = float(np.mean(ts))
    v = n_step / t
    sample = f"{n_step} consecutive ray indices of {inst['name']} per step (of {inst['n_rays']})"
    det_last = [c for c in inst["components"] if c["kind"] == "detector"][-1]
    nb_last = det_last["nx"] * det_last["ny"] * det_last["nE"]
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[{args.config}] {inst['name']}", "n_rays_per_gpu": inst["n_rays"],
                       "detector_bins": int(nb_last), "seed": inst["seed"], "l2": L2_NOTE},
            "sampling": {"rays_per_step": n_step, "what": "each step traces a bounded window of the workload's ray indices"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def make_probes(M, device):
    """Peaks measured in this run (memoised per footprint): FP64 pipe, random L2 sectors, random tally records."""
    dev = str(device)
    memo_l2, memo_tally = {}, {}

    def l2(table_bytes):
        if table_bytes not in memo_l2:
            memo_l2[table_bytes] = max(M.probe_l2(table_bytes, N_SM * 8, 256, device=dev) for _ in range(2))
        return memo_l2[table_bytes]

    def tally(n_rec):
        if n_rec not in memo_tally:
            memo_tally[n_rec] = max(M.probe_tally(n_rec, N_SM * 8, 128, device=dev) for _ in range(2))
        return memo_tally[n_rec]

    # 8 independent DFMA chains per thread, 148 x 8 blocks of 256: the rate the chip holds at its clock under this load
    dfma = max(M.probe_dfma(N_SM * 8, 1 << 15, device=dev) for _ in range(3))
    return {"dfma": dfma, "l2": l2, "tally": tally,
            "latency_ns": {"unloaded_32MiB": M.probe_latency(32 << 20, 1, 32, 4096, device=dev) * 1e9}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs[k] of the headline line")
    ap.add_argument("--rays", type=float, default=None, help="override n_rays of the headline config")
    ap.add_argument("--instruments", default="0,2,3,4,5,6,7,8,9",
                    help="other configs to report under 'instruments' ('' = none); 5-7 are the paper's own three instruments, "
                         "8 and 9 the voxel samples with scattering")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the configs[4] throughput sweep 1e6..1e10 rays")
    ap.add_argument("--exec", default="auto", choices=["auto", "direct", "sorted"], help="lane scheduling (row a13)")
    args = ap.parse_args()
    global EXEC_MODE
    EXEC_MODE = args.exec
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    import workloads as W
    ks = [args.config] + ([int(x) for x in args.instruments.split(",") if x != "" and int(x) != args.config]
                          if (rank == 0 and world == 1) else [])
    insts = {k: make_instrument(W, k, args.rays if k == args.config else None) for k in ks}

    # CPU baselines first: the oracle's worker processes are forked, which must happen before CUDA is initialised
    cpu = {}
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        for k in ks:
            cpu[k] = cpu_baseline(insts[k])

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the mcx hot path has no CPU fallback")
    import paper_2410_08747_b200 as M
    from paper_2410_08747_b200.shard import ray_range, reduce_tallies
    M.lib()
    device = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(device)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    peaks = measured_peaks()
    probes = make_probes(M, device)

    inst = insts[args.config]
    n_rays = inst["n_rays"]
    first, _ = ray_range(rank, world, n_rays, "weak")   # every rank traces n_rays of its own index window
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(device)
    head = bench_instrument(M, torch, inst, n_rays, first, args.steps, args.warmup, device, probes, peaks,
                            with_e2e=True, local_rank=local_rank)
    torch.cuda.synchronize(device)
    ms = head["ms_per_step"]
    e2e_ms = head["e2e"]["ms_per_step"]
    reduce_info = None
    if dist is not None:
        t = torch.tensor([ms, e2e_ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, e2e_ms = float(t[0]), float(t[1])
        dist.barrier()
        # the paper's gather/add of the monitor arrays: one sum-reduce of (N, p, p2) to rank 0 over
        # NCCL, after the timed path and reported on its own
        g = M.Instrument(inst, device=device)
        g.trace(min(n_rays, 1 << 22), first=first)
        tl = list(g.tally(len(g.dets) - 1))
        torch.cuda.synchronize(device)
        dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        reduce_tallies(tl, dst=0)
        e1.record()
        torch.cuda.synchronize(device)
        tr = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=device)
        dist.all_reduce(tr, op=dist.ReduceOp.MAX)
        reduce_info = {"ms": float(tr[0]), "bytes_per_rank": int(sum(x.numel() * x.element_size() for x in tl)),
                       "what": "ncclReduce (sum) of N, p, p2 of the last detector to rank 0; not part of the timed step"}
        g.close()
    value = world * n_rays / (ms * 1e-3)

    instruments = {}
    if rank == 0 and world == 1:
        head_entry = slim(head)
        if args.config in cpu:
            head_entry["cpu_baseline"] = cpu[args.config]
        instruments[f"c{args.config}_{inst['name']}"] = head_entry
        for k in ks[1:]:
            ik = insts[k]
            r = bench_instrument(M, torch, ik, ik["n_rays"], 0, args.steps, args.warmup, device, probes, peaks, with_e2e=True)
            e = slim(r)
            if k in cpu:
                e["cpu_baseline"] = cpu[k]
            instruments[f"c{k}_{ik['name']}"] = e
            if k == 0:                                  # 1e6 rays is launch-latency sized: also the asymptote
                r = bench_instrument(M, torch, ik, 100_000_000, 0, args.steps, args.warmup, device, probes, peaks, with_e2e=True)
                e = slim(r)
                if k in cpu:
                    e["cpu_baseline"] = cpu[k]
                instruments["c0_minimal_1e8_rays"] = e
        if 7 in insts:
            instruments["c7_projection_scan"] = bench_scan(M, torch, insts[7], device)
        if 8 in insts:                                  # the same projection with the scattering sample (~11 s)
            instruments["c8_projection_scan"] = bench_scan(M, torch, insts[8], device, warmup_lines=20)
        if 4 in insts and not args.no_sweep:            # configs[4]: "also run a throughput sweep at 1e6-1e10 rays"
            sweep = {}
            for n in (10**6, 10**7, 10**8, 10**9, 10**10):
                r = bench_instrument(M, torch, insts[4], n, 0, args.steps if n < 10**9 else 1, 3 if n < 10**9 else 1, device,
                                     probes, peaks, with_e2e=False)
                sweep[f"{n:.0e}"] = {"rays_per_s": r["rays_per_s"], "ms_per_step": r["ms_per_step"],
                                     "kernel_ms": {k_: v for k_, v in r["kernel_ms"].items() if k_ != "how"}}
            instruments["c4_sweep"] = sweep

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0
    roof = dict(head["roofline"])
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"configs[{args.config}] {inst['name']}", "n_rays_per_gpu": n_rays,
                       "detector_bins": head["tally_bytes"] // 32, "seed": inst["seed"], "l2": L2_NOTE},
            "timing": {"step": "mcx_trace + mcx_tally_read", "how": "steps timed one by one with CUDA events on the launching stream",
                       "parallelism": f"ray-index shards x{world}, no data-path collective"},
            "e2e": {"value": world * n_rays / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": head["e2e"]["h2d_bytes_per_step"], "d2h_bytes_per_step": head["e2e"]["d2h_bytes_per_step"],
                    "ms_per_step": e2e_ms, "what": "mcx_instrument_create (host tables) + mcx_trace + mcx_tally_read_host (pinned)"},
            "gpu_launches": head["launches"], "clocks": head["clocks"], "roofline": roof,
            "kernel_ms": head["kernel_ms"],
            "peaks_measured_in_this_run": {"fp64_tlaneops": probes["dfma"] / 1e12,
                                           "fp64_nominal_tlaneops": N_SM * NOMINAL_FP64_LANES_PER_SM * 1.965e9 / 1e12,
                                           "dependent_load_latency_ns": probes["latency_ns"]}}
    if args.config in cpu:
        line["cpu_baseline"] = cpu[args.config]
    if reduce_info is not None:
        line["tally_reduce"] = reduce_info
    if instruments:
        line["instruments"] = instruments
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def slim(r):
    keep = ("n_rays", "rays_per_s", "ms_per_step", "kernel_ms", "launches", "detected_fraction", "tally_bytes", "clocks",
            "roofline", "e2e", "tuning")
    out = {k: r[k] for k in keep if k in r}
    out["kernel_ms"] = {k: v for k, v in r["kernel_ms"].items() if k != "how"}
    return out


if __name__ == "__main__":
    sys.exit(main())
