#!/usr/bin/env python
"""bench.py -- rays/s of the mcx hot path on B200 (BASELINE.json: "rays/sec on 1 B200 per instrument; achieved % of
binding roofline").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--instruments 0,1,2,3,4] [--impl reference]

A step = one pass of the whole hot path over one batch of synthetic rays: mcx_trace(n_rays) + mcx_tally_read.
The headline line is BASELINE.json configs[1] (polychromatic energy-dispersive instrument, 1e8 rays); the other four
instruments are measured the same way and reported under "instruments" in the same JSON line (north_star: "all five
configs ... each reported in rays/s with its achieved fraction of the binding roofline").
states the algorithmic work model used for the roofline fractions.
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
FLUSH_BYTES = 256 << 20          # > the 126 MB L2

# ---------------------------------------------------------------------------------------------------------------
# Algorithmic work model: fp64-pipe lane-operations the method itself needs per unit.
# One DFMA / DADD / DMUL / compare = 1; library functions at the length of a correctly rounded-to-1-ulp fp64
# evaluation (sqrt, div ~ 12; exp ~ 25; log, asin ~ 35; sincos ~ 45; tan ~ 50).  Philox is integer work (not counted).
# ---------------------------------------------------------------------------------------------------------------
OPS_SOURCE = {("disk", "target", "mono"): 120, ("gauss", "target", "spectrum"): 250, ("point", "target", "spectrum"): 150,
              ("gauss", "gauss", "uniform"): 330}
OPS_SLIT, OPS_DETECTOR, OPS_MIRROR, OPS_CRYSTAL = 35, 80, 250, 180
OPS_SOLIDS_ENTRY, OPS_PRIMITIVE_TEST, OPS_SEGMENT, OPS_MU, OPS_EXP = 35, 45, 10, 35, 25
OPS_VOXEL_ENTRY, OPS_VOXEL_STEP = 100, 6
OPS_TRI_TEST, OPS_BVH_NODE = 45, 14
NOMINAL_FP64_LANES_PER_SM, N_SM = 64, 148
# DRAM bytes per ray of trace_kernel (dram__bytes_read.sum + dram__bytes_write.sum of one launch of 2^26 rays / 2^26) from
# the ncu --set full captures summarised in profiles/r01d_README.md (c0, c2: whole run / n_rays; their tallies stay in L2).
NCU_DRAM_BYTES_PER_RAY = {"c0_minimal": 0.001, "c1_polychromatic": 10.5, "c2_beamline": 0.01, "c3_mesh": 17.3, "c4_edxct": 28.6}


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


def bench_instrument(M, torch, inst, n_rays, first, steps, warmup, device, dfma_peak, peaks, with_e2e=True, local_rank=0):
    """Times `steps` steps of mcx_trace + mcx_tally_read for one instrument on the current stream.  Returns a dict."""
    g = M.Instrument(inst, device=device)
    g.set_exec(EXEC_MODE)
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
    res = {"n_rays": n_rays, "ms_per_step": float(np.mean(t_step)), "ms_trace_kernel": float(np.mean(t_trace)),
           "ms_tally_read": float(np.mean(t_step) - np.mean(t_trace)), "ms_step_min": float(np.min(t_step)),
           "rays_per_s": n_rays / (np.mean(t_step) * 1e-3), "launches": launches, "clocks": clocks,
           "detected_fraction": counters["detected"] / traced, "tally_bytes": 32 * nb}
    # roofline of the dominant kernel (trace_kernel), DESIGN.md "Measurement"
    work = oracle_work_per_ray(inst)
    ops = algorithmic_ops(inst, n_rays, per_trace, work)
    byt = algorithmic_bytes(inst, n_rays, per_trace, work)
    sec = np.mean(t_trace) * 1e-3
    alu_frac = ops / sec / dfma_peak
    hbm_peak = (peaks or {}).get("hbm_gbs", 6650.0)
    hbm_frac = byt / sec / 1e9 / hbm_peak
    res["work_per_ray"] = work
    bpr = NCU_DRAM_BYTES_PER_RAY.get(inst["name"])
    traffic = None if bpr is None else bpr * n_rays      # bytes per step (all launches of the step)
    traffic_src = None if bpr is None else f"ncu dram bytes {bpr} B/ray (profiles/r01d_README.md) x n_rays"
    res["roofline"] = {"bound": "alu", "achieved": ops / sec / 1e12, "peak": dfma_peak / 1e12, "unit": "Tlane-op/s (fp64)",
                       "frac": alu_frac, "traffic": traffic, "traffic_source": traffic_src, "kernel": "trace_kernel",
                       "ops_per_ray": ops / n_rays, "peak_source": "mcx_probe_dfma, measured in this run",
                       "hbm": {"achieved": byt / sec / 1e9, "peak": hbm_peak, "unit": "GB/s", "frac": hbm_frac,
                               "bytes_per_ray": byt / n_rays,
                               "peak_source": "MEASURED_PEAKS.json" if peaks else "fallback 6650 GB/s"}}
    if with_e2e:
        # the second candidate roofline: random tally-record updates at this detector's footprint
        n_rec = 1 << (int(nb).bit_length() - 1)
        g.close()
        g = None
        torch.cuda.empty_cache()
        tally_peak = max(M.probe_tally(n_rec, N_SM * 8, 128, device=str(device)) for _ in range(2))
        det_rate = res["detected_fraction"] * n_rays / sec
        res["roofline"]["tally"] = {"achieved": det_rate, "peak": tally_peak, "unit": "records/s", "frac": det_rate / tally_peak,
                                    "peak_source": f"mcx_probe_tally, {n_rec} random 32-byte records, measured in this run"}
        res["e2e"] = bench_e2e(M, torch, inst, n_rays, first, max(2, min(steps, 3)), device)
    if g is not None:
        g.close()
    del flush, out
    torch.cuda.empty_cache()
    return res


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
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[{args.config}] {inst['name']}", "n_rays": inst["n_rays"], "rays_per_step": n_step},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json configs[k] of the headline line")
    ap.add_argument("--rays", type=float, default=None, help="override n_rays of the headline config")
    ap.add_argument("--instruments", default="0,2,3,4", help="other configs to report under 'instruments' ('' = none)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs[4] throughput sweep 1e6..1e10 rays")
    ap.add_argument("--exec", default="auto", choices=["auto", "direct", "sorted"], help="lane scheduling (row a13)")
    args = ap.parse_args()
    global EXEC_MODE
    EXEC_MODE = args.exec
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the mcx hot path has no CPU fallback")
    import paper_2410_08747_b200 as M
    from paper_2410_08747_b200.shard import ray_range
    import workloads as W
    M.lib()
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    device = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(device)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)
    peaks = measured_peaks()

    # FP64 pipe peak at the clock the chip holds (8 independent DFMA chains per thread, 148 x 8 blocks of 256)
    dfma_peak = max(M.probe_dfma(N_SM * 8, 1 << 15, device=str(device)) for _ in range(3))

    inst = make_instrument(W, args.config, args.rays)
    n_rays = inst["n_rays"]
    first, _ = ray_range(rank, world, n_rays, "weak")   # every rank traces n_rays of its own index window
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(device)
    head = bench_instrument(M, torch, inst, n_rays, first, args.steps, args.warmup, device, dfma_peak, peaks,
                            with_e2e=True, local_rank=local_rank)
    torch.cuda.synchronize(device)
    ms = head["ms_per_step"]
    e2e_ms = head["e2e"]["ms_per_step"]
    if dist is not None:
        t = torch.tensor([ms, e2e_ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms, e2e_ms = float(t[0]), float(t[1])
        dist.barrier()
    value = world * n_rays / (ms * 1e-3)

    others = {}
    if rank == 0 and world == 1 and args.instruments:
        for k in [int(x) for x in args.instruments.split(",") if x != ""]:
            if k == args.config:
                continue
            ik = make_instrument(W, k)
            r = bench_instrument(M, torch, ik, ik["n_rays"], 0, args.steps, args.warmup, device, dfma_peak, peaks, with_e2e=False)
            others[f"c{k}_{ik['name']}"] = slim(r)
            if k == 0:                                  # 1e6 rays is launch-latency sized: also the asymptote
                r = bench_instrument(M, torch, ik, 100_000_000, 0, args.steps, args.warmup, device, dfma_peak, peaks, with_e2e=False)
                others["c0_minimal_1e8_rays"] = slim(r)
            del ik
    if rank == 0 and world == 1 and args.sweep:
        i4 = make_instrument(W, 4)
        for n in (10**6, 10**7, 10**8, 10**9, 10**10):
            r = bench_instrument(M, torch, i4, n, 0, max(1, args.steps if n < 10**10 else 1), 3 if n < 10**9 else 1, device,
                                 dfma_peak, peaks, with_e2e=False)
            others[f"c4_sweep_{n:.0e}"] = slim(r)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        rate, n_s, dt = time_oracle(inst, budget_s=15.0)
        cpu = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"first {n_s} ray indices of {inst['name']} ({dt:.1f} s, one thread of {os.cpu_count()} host cores)"}
    roof = dict(head["roofline"])
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"configs[{args.config}] {inst['name']}", "n_rays_per_gpu": n_rays,
                       "detector_bins": head["tally_bytes"] // 32, "seed": inst["seed"],
                       "step": "mcx_trace + mcx_tally_read", "l2": "flushed between steps (256 MiB memset, untimed); "
                       "steps timed one by one with CUDA events on the launching stream",
                       "parallelism": f"ray-index shards x{world}, no data-path collective"},
            "e2e": {"value": world * n_rays / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": head["e2e"]["h2d_bytes_per_step"], "d2h_bytes_per_step": head["e2e"]["d2h_bytes_per_step"],
                    "ms_per_step": e2e_ms, "what": "mcx_instrument_create (host tables) + mcx_trace + mcx_tally_read_host (pinned)"},
            "gpu_launches": head["launches"], "clocks": head["clocks"], "roofline": roof,
            "kernel_ms": {"trace_kernel": head["ms_trace_kernel"], "tally_read_kernel": head["ms_tally_read"]},
            "dfma_peak_measured_tlaneops": dfma_peak / 1e12,
            "dfma_peak_nominal_tlaneops": N_SM * NOMINAL_FP64_LANES_PER_SM * 1.965e9 / 1e12}
    if cpu is not None:
        line["cpu_baseline"] = cpu
    if others:
        line["instruments"] = others
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def slim(r):
    keep = ("n_rays", "rays_per_s", "ms_per_step", "ms_trace_kernel", "ms_tally_read", "launches", "detected_fraction",
            "tally_bytes", "clocks")
    out = {k: r[k] for k in keep}
    rf = r["roofline"]
    out["roofline"] = {"bound": rf["bound"], "frac": rf["frac"], "achieved": rf["achieved"], "peak": rf["peak"], "unit": rf["unit"],
                       "ops_per_ray": rf["ops_per_ray"], "hbm_frac": rf["hbm"]["frac"], "hbm_gbs": rf["hbm"]["achieved"],
                       "bytes_per_ray": rf["hbm"]["bytes_per_ray"]}
    return out


if __name__ == "__main__":
    sys.exit(main())
