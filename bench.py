#!/usr/bin/env python
"""bench.py -- throughput of the DEM hot path (arXiv:1607.02427) on B200, one JSON line on stdout.

A "step" is one NVE time step of the whole hot path (neighbour-list upkeep, pair-feature kernel, per-particle
reduction, integrator) over one synthetic configuration of BASELINE.json.  Default workload at N = 1: config 4
(3D rounded octahedra, N = 262,144, fp32, dt = 2e-4), the largest single-GPU 3D NVE configuration.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg3|cfg4|cfg5|cfg2]

metric  = particle-timesteps/s (BASELINE.json); feature-pair evaluations/s are reported beside it.
value   = N_particles * K / (device time of dem_step(nsteps=K)), state resident in HBM, max over ranks.
e2e     = the same metric through dem_step_host (HOST buffers: every step copies the state host->device and back).
roofline= the pair-feature kernel (dominant): algorithmic FP32 flops per launch / its CUDA-event time, against the
          FP32 peak 148 SM x 128 lanes x 2 x clocks.max.sm.
cpu_baseline = the FP64 oracle (oracle/dem_oracle.c, as it stands) timed on this box's host cores on a bounded sample.
`--impl reference` times the oracle as the reference arm (this tier has no reference implementation to install).
With --gpus N > 1 (torchrun) every rank runs an independent replica of the workload (the path does not shard:
DESIGN.md "Multi-GPU"): weak scaling, no data-path collective, one MAX all-reduce of the elapsed time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import dem_inputs as di  # noqa: E402

WORKLOADS = {"cfg2": 2, "cfg3": 3, "cfg4": 4, "cfg5": 5}
SKIN = {2: 0.3, 3: 0.2, 4: 0.3, 5: 0.3}
L2_FLUSH_BYTES = 160 << 20  # larger than the 126 MB L2

# Algorithmic FP32 flop per Eq. 1 / Eq. 2 term of the search formulation in csrc/dem_fast.cuh (FMA = 2, every other
# arithmetic instruction = 1).  The rare candidate terms' scalar evaluation is not counted.
FLOP_VE_2D = 15           # point - segment, 2D: side 4, along 4, over 1, excess 2, r^2 - rc^2 4
FLOP_EE = 49              # segment - segment: r 3, b c f 15, nn num 4, rcp 1, s 1, t 4, s' 3, d 12, r^2 - rc^2 6
FLOP_VF_FACE = 22         # projection on the face frame 18, h^2 - rc^2 2, inside select + add 2
FLOP_VF_EDGE = 16         # per boundary edge of the face: side 4, along 4, over 1, excess 2, d^2 3, two minima 2


def pair_flops(dim, a, b):
    """Algorithmic flop of one unique pair with shapes a (first) and b (second)."""
    if dim == 2:
        return FLOP_VE_2D * (len(a["verts"]) * len(b["edges"]) + len(b["verts"]) * len(a["edges"]))
    fa = sum(FLOP_VF_FACE + FLOP_VF_EDGE * len(f) for f in a["faces"])
    fb = sum(FLOP_VF_FACE + FLOP_VF_EDGE * len(f) for f in b["faces"])
    return FLOP_EE * len(a["edges"]) * len(b["edges"]) + len(a["verts"]) * fb + len(b["verts"]) * fa


def pair_terms(dim, a, b):
    if dim == 2:
        return len(a["verts"]) * len(b["edges"]) + len(b["verts"]) * len(a["edges"])
    return len(a["edges"]) * len(b["edges"]) + len(a["verts"]) * len(b["faces"]) + len(b["verts"]) * len(a["faces"])


def class_pair_counts(st, counts, rows):
    """Unique neighbour pairs per (shape, shape) class from the neighbour list (host-side bookkeeping for the flop
    count only)."""
    sid = st["shape_id"]
    ns = len(st["shapes"])
    out = np.zeros((ns, ns), dtype=np.int64)
    i = np.repeat(np.arange(len(sid)), rows.shape[1])
    j = rows.reshape(-1)
    ok = (j >= 0) & (j > i)
    a, b = sid[i[ok]], sid[j[ok]]
    lo, hi = np.minimum(a, b), np.maximum(a, b)
    np.add.at(out, (lo, hi), 1)
    return out


class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region (B200_PROFILING.md): NVML read directly from
    a thread every millisecond (one nvidia-smi process start alone outlasts a 20-step region); the first sample is taken
    when the region starts, the last when it ends."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, gpu_index):
        self.rows, self.h, self.nv = [], None, None
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = None
            try:  # the device torch uses (CUDA_VISIBLE_DEVICES may renumber it)
                import torch
                uuid = str(torch.cuda.get_device_properties(gpu_index).uuid)
                h = nv.nvmlDeviceGetHandleByUUID(("GPU-" + uuid) if not uuid.startswith("GPU-") else uuid)
            except Exception:
                h = nv.nvmlDeviceGetHandleByIndex(gpu_index)
            self.nv, self.h = nv, h
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
        except Exception:
            self.h = None
        self._stop = threading.Event()
        self.t = None
        if self.h is not None:
            self._sample()
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()

    def _sample(self):
        nv, h = self.nv, self.h
        try:
            mhz = float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
            watts = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
            try:
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(h))
            except Exception:
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))
            self.rows.append((mhz, watts, mask))
        except Exception:
            pass

    def _run(self):
        while not self._stop.wait(0.001):
            self._sample()

    def stop(self):
        if self.h is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["NVML unavailable"]}
        self._stop.set()
        self.t.join(timeout=5)
        self._sample()
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = [r[0] for r in self.rows]
        power = [r[1] for r in self.rows]
        reasons = set()
        for r in self.rows:
            for bit, name in self.REASONS.items():
                if r[2] & bit:
                    reasons.add(name)
        load = [s_ for s_, p_ in zip(sm, power) if p_ >= 0.5 * max(power)] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": self.max_mhz, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power)}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        return json.load(open(path)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


def _oracle_rate(orc, st, rows, cells, threads=None):
    """Rows/s of one oracle force evaluation of `rows` random particles (cells: the cell-grid variant, which is the
    all-pairs sum bit for bit without the O(N) scan per particle)."""
    rng = np.random.default_rng(123)
    sub = np.sort(rng.choice(st["N"], min(rows, st["N"]), replace=False)).astype(np.int32)
    if threads is not None:
        orc.set_num_threads(threads)
    t0 = time.perf_counter()
    orc.compute(st, subset=sub, cells=cells)
    return len(sub) / (time.perf_counter() - t0), len(sub)


def oracle_baseline(st, target_seconds):
    """The oracle (oracle/dem_oracle.c, as it stands) timed on this box's host cores on a bounded sample of the workload.
    value: all cores, neighbours found through the oracle's plain cell grid (the same sums over the same pairs as the
    all-pairs definition, bit for bit) -- the CPU does what the GPU does, a list-limited evaluation of every Eq. 1/2
    term.  Also reported: the same on ONE thread (the paper's CPU column is one core) and the all-pairs
    definition itself (an O(N) scan per particle, which at N = 262,144 costs more than the feature work)."""
    from oracle import dem_oracle as orc

    orc.build()
    st = dict(st, _tab=orc.ShapeTable(st["shapes"]))
    cores = orc.num_threads()
    probe, _ = _oracle_rate(orc, st, 256, True)
    rows = int(max(256, min(st["N"], 0.6 * target_seconds * probe)))
    rate, rows = _oracle_rate(orc, st, rows, True)
    one, rows1 = _oracle_rate(orc, st, int(max(64, min(st["N"], 0.2 * target_seconds * probe / max(cores, 1)))), True, threads=1)
    orc.set_num_threads(cores)
    probe_ap, _ = _oracle_rate(orc, st, 64, False)
    allp, rows_ap = _oracle_rate(orc, st, int(max(64, min(st["N"], 0.2 * target_seconds * probe_ap))), False)
    return {"value": rate, "unit": "particle-timesteps/s", "cores": cores, "kind": "oracle",
            "sample": "%d of %d particles, one full force evaluation each (every Eq. 1/2 term of every neighbour inside "
                      "the reach; neighbours from the oracle's cell grid, same sums as the all-pairs loop), fp64" % (rows, st["N"]),
            "single_thread_value": one, "single_thread_sample": "%d particles, 1 thread" % rows1,
            "all_pairs_value": allp, "all_pairs_sample": "%d particles, %d threads, O(N) minimum-image scan per particle "
                                                         "(the definition the parity tests use)" % (rows_ap, cores)}


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    k = WORKLOADS[args.workload]
    st = di.make_config(k)
    from oracle import dem_oracle as orc

    orc.build()
    st["_tab"] = orc.ShapeTable(st["shapes"])
    n = st["N"]
    rng = np.random.default_rng(7)
    probe, _ = _oracle_rate(orc, st, 256, True)
    budget = 150.0 / (args.steps + args.warmup)       # whole run within a few minutes
    rows = int(max(64, min(n, budget * probe)))
    for _ in range(args.warmup):
        orc.compute(st, subset=np.sort(rng.choice(n, rows, replace=False)).astype(np.int32), cells=True)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        orc.compute(st, subset=np.sort(rng.choice(n, rows, replace=False)).astype(np.int32), cells=True)
    dt = time.perf_counter() - t0
    value = rows * args.steps / dt
    sample = ("each step = one oracle force evaluation of %d of %d particles (every Eq. 1/2 term of every neighbour "
              "inside the reach, neighbours from the oracle's cell grid), fp64" % (rows, n))
    line = {"impl": "reference", "metric": "particle-timesteps/s", "value": value, "unit": "particle-timesteps/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": di.CONFIG_NAMES[k], "N": n, "dt": st["dt"], "skin": SKIN[k]},
            "cpu_baseline": {"value": value, "unit": "particle-timesteps/s", "cores": orc.num_threads(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "particle-timesteps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def max_over_ranks(x, world, device):
    """The slowest rank's figure (replicas only: the one collective of a multi-GPU run)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(n_particles, world, steps, elapsed_ms):
    """Whole-job particle-timesteps/s of `world` replicas that each advanced n_particles by `steps` steps."""
    return n_particles * world * steps / (elapsed_ms * 1e-3)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg4", choices=sorted(WORKLOADS))
    ap.add_argument("--no-l2-flush", action="store_true")
    ap.add_argument("--slices", type=int, default=0, help="lanes per pair in the pair kernel (0 = library heuristic)")
    ap.add_argument("--cull", action="store_true",
                    help="headline arm with exact per-feature culling (default: every Eq. 1 term swept; culling is the second arm)")
    ap.add_argument("--pair-kernel", default="auto", choices=["auto", "search", "generic"],
                    help="search = packed FP32 contact search; generic = fused scalar kernel; auto = library default")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--thermalise", type=int, default=2000,
                    help="NVE steps before the 'thermalised' arm (0 = skip it)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    import paper_1607_02427_b200 as pkg

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    k = WORKLOADS[args.workload]
    st = di.make_config(k, seed=rank)  # independent replica per rank
    n, dt_step, skin = st["N"], st["dt"], SKIN[k]
    dem, t = pkg.from_state(st, "f32")
    if args.slices:
        dem.set_slices(args.slices)
    # headline arm: every Eq. 1 / Eq. 2 term is swept (the paper's method as stated); the
    # library's default, exact per-feature culling, is measured as a second arm ("culled") on the same state
    search3d = st["dim"] == 3 and args.pair_kernel != "generic"
    # (in 2D the one-kernel path is HBM / latency bound either way: its headline is the library default, culling on, and
    # the every-term sweep is the second arm)
    if st["dim"] == 2 and args.pair_kernel == "auto":
        args.cull = True
    dem.set_culling(bool(args.cull))
    if args.pair_kernel != "auto":
        dem.set_pair_kernel({"search": 0, "generic": 1}[args.pair_kernel])
    if not args.no_l2_flush:
        dem.set_l2_flush(L2_FLUSH_BYTES)
    force = torch.empty((n, 4), dtype=torch.float32, device="cuda")
    torque = torch.empty((n, 4), dtype=torch.float32, device="cuda")

    def step(nsteps):
        dem.step(t["pos"], t["quat"], t["vel"], t["angmom"], t["shape_id"], st["box"], dt_step, nsteps, skin, force, torque)

    # ---- device-resident throughput ---------------------------------------------------------------------------
    def timed(nwarm, nsteps, sample_clocks, level=1):
        """nwarm untimed + nsteps timed steps; (ms, clocks, launches, kernel times by kind, swept totals)."""
        step(nwarm)
        dem.set_timing(level)
        dem.kernel_times()
        l0 = dem.launch_count()
        sampler = ClockSampler(local) if (rank == 0 and sample_clocks) else None
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        step(nsteps)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        clk = sampler.stop() if sampler else None
        nl = dem.launch_count() - l0
        kt = dem.kernel_times()
        tot = dem.swept_totals()
        dem.set_timing(0)
        return max_over_ranks(ms, world, "cuda"), clk, nl, kt, tot

    def swept_flops(tot):
        """Algorithmic flop of the terms whose search was executed, summed over the timed evaluations (library counters)."""
        if st["dim"] == 2:
            return FLOP_VE_2D * tot["ee_swept"]
        return FLOP_EE * tot["ee_swept"] + FLOP_VF_FACE * tot["vf_swept"] + FLOP_VF_EDGE * tot["face_edges_swept"]

    def counters_now():
        """Counters of one dem_compute on the current state (dem_step's kernels keep none)."""
        dem.build_neighbors(t["pos"], t["shape_id"], st["box"], st["r_cut"])
        dem.compute(t["pos"], t["quat"], t["shape_id"], virial=False)
        return dem.get_counters()

    elapsed_ms, clocks, gpu_launches, kt, tot = timed(args.warmup, args.steps, True)
    value = aggregate_value(n, world, args.steps, elapsed_ms)
    n_pair_launches, pair_ms, pose_ms = kt["pair"][0], kt["pair"][1], kt["pose"][1]

    # ---- roofline of the dominant kernel ---------------------------------------------------------------------------
    counts, rows = dem.get_neighbors()
    counts_h, rows_h = counts.cpu().numpy(), rows.cpu().numpy()
    cls = class_pair_counts(st, counts_h, rows_h)
    flops = sum(int(cls[a, b]) * pair_flops(st["dim"], st["shapes"][a], st["shapes"][b])
                for a in range(len(st["shapes"])) for b in range(a, len(st["shapes"])))
    terms = sum(int(cls[a, b]) * pair_terms(st["dim"], st["shapes"][a], st["shapes"][b])
                for a in range(len(st["shapes"])) for b in range(a, len(st["shapes"])))
    prims = 0
    if st["dim"] == 3:   # triangle primitives behind the polygon faces: a face with m edges fans into m - 2
        tri = [sum(len(f) - 2 for f in s["faces"]) for s in st["shapes"]]
        prims = sum(int(cls[a, b]) * (len(st["shapes"][a]["edges"]) * len(st["shapes"][b]["edges"])
                                      + len(st["shapes"][a]["verts"]) * tri[b] + len(st["shapes"][b]["verts"]) * tri[a])
                    for a in range(len(st["shapes"])) for b in range(a, len(st["shapes"])))
    n_classes = int((cls > 0).sum())
    peaks, peak_kind = measured_peaks()
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    peak_tf = sm_count * 128 * 2 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    hbm_gbs = float(peaks.get("hbm_gbs", 6650.0))
    particle2d = st["dim"] == 2 and args.pair_kernel == "auto"
    searched = (st["dim"] == 3 and args.pair_kernel != "generic") or args.pair_kernel == "search" or particle2d
    traffic = None
    prof = os.path.join(ROOT, "profiles", "r02_step_%s_ncu.md" % args.workload)
    if os.path.exists(prof):
        for ln in open(prof):
            if ln.startswith("traffic_bytes_per_launch"):
                traffic = int(ln.split(":")[1])
    if particle2d:
        # ONE kernel per step (k_particle2d: neighbour gather, Eq. 2, reduction, integrator): HBM-bound.  Algorithmic
        # bytes per particle and launch: x, q, v, L read and written (8 x 32 B, the FP64 state of R15b), the position of
        # the last list build (32 B), the particle's neighbour row (4 B per listed neighbour + its count)
        evals = max(n_pair_launches, 1)
        kern_ms_per_eval = pair_ms / evals
        bytes_per_launch = n * (8 * 32 + 32 + 4) + 4 * int(counts_h.sum())
        achieved = bytes_per_launch / (kern_ms_per_eval * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "k_particle2d", "achieved": achieved, "peak": hbm_gbs, "unit": "GB/s",
                    "frac": achieved / hbm_gbs, "traffic": traffic,
                    "peak_source": "MEASURED_PEAKS.json hbm_gbs (%s)" % peak_kind, "bytes_per_launch": bytes_per_launch,
                    "kernel_ms": kern_ms_per_eval, "launches_timed": n_pair_launches,
                    "kernel_share_of_step": pair_ms / elapsed_ms,
                    "flops_swept_per_launch": swept_flops(tot) / evals,
                    "note": "the Eq. 2 terms swept after exact per-vertex culling cost %.2f Gflop per launch: not the bound" % (
                        swept_flops(tot) / evals / 1e9)}
    else:
        # force evaluations timed (several classes: one fork-to-join span per evaluation, pose kernels included)
        evals = max(n_pair_launches if n_classes > 1 else n_pair_launches, 1)
        kern_ms_per_eval = pair_ms / evals
        # per evaluation: summed over the timed evaluations by the search kernels themselves; the generic kernel sweeps
        # every term of every listed pair in reach (nominal count)
        flops_swept = swept_flops(tot) / evals if searched else flops
        achieved_tf = flops_swept / (kern_ms_per_eval * 1e-3) / 1e12
        kname = ("k_pair_cull" if args.cull else "k_pair_fast") if searched else "k_pair"
        roofline = {"bound": "alu", "kernel": kname, "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": achieved_tf / peak_tf, "traffic": traffic,
                    "peak_source": "%d SM x 128 FP32 lanes x 2 x %.0f MHz (clocks.max.sm, %s)" % (
                        sm_count, float(peaks.get("sm_max_mhz", 1965.0)), peak_kind),
                    "flops_per_launch": flops_swept, "flops_all_terms": flops, "kernel_ms": kern_ms_per_eval,
                    "pose_kernel_ms": pose_ms / evals, "launches_timed": n_pair_launches,
                    "kernel_share_of_step": pair_ms / elapsed_ms,
                    "fma_chain_measured_tflops": dem.fp32_peak(1 << 15)}

    # ---- second arm: the library default (exact per-feature culling), same state, and the per-kernel breakdown -----------
    def hbm_line(us, nbytes):
        return {"us_per_launch": us, "algorithmic_bytes": nbytes, "GB_per_s": nbytes / (us * 1e-6) / 1e9 if us > 0 else None,
                "frac_of_hbm_peak": nbytes / (us * 1e-6) / 1e9 / hbm_gbs if us > 0 else None}

    def breakdown(kt2, npairs_listed, npairs_eval):
        """Per-kernel microseconds per launch (timing level 2) and, for the HBM-bound kernels, algorithmic bytes and GB/s."""
        us = {k: (1e3 * v[1] / v[0] if v[0] else 0.0) for k, v in kt2.items()}
        out = {"us_per_launch": {k: round(x, 2) for k, x in us.items() if x}, "launches": {k: v[0] for k, v in kt2.items() if v[0]}}
        nsum = int(counts_h.sum())
        if st["dim"] == 3 and us.get("pose"):
            # k_pose: pair list (8 B), positions and orientations of N particles in double (64 B each, gathered), pose
            # records of the pairs inside the reach (48 B R, t + 16 B work-list entry), one flag byte per pair
            out["k_pose"] = hbm_line(us["pose"], npairs_listed * 9 + n * 64 + npairs_eval * 64)
        if us.get("reduce"):
            # k_finish: slots (4 B per listed neighbour), flags (1 B per listed neighbour), x q v L read + written, build positions
            out["k_finish"] = hbm_line(us["reduce"], nsum * 5 + n * (8 * 32 + 32 + 4))
        if us.get("neigh"):
            # k_neigh: cell-ordered positions read once (32 B), rows written (4 B per neighbour + count): the kernel is bound
            # by its FP64 predicate arithmetic over 3^dim cells, not by these bytes
            out["k_neigh"] = hbm_line(us["neigh"], n * 36 + nsum * 4)
        return out

    culled = None
    every_term = None
    if particle2d:
        dem.set_culling(False)
        ems, _, _, ekt, etot = timed(3, args.steps, False)
        dem.set_culling(True)
        every_term = {"value": n * world * args.steps / (ems * 1e-3), "unit": "particle-timesteps/s",
                      "ms_per_step": ems / args.steps, "kernel_ms": ekt["pair"][1] / max(ekt["pair"][0], 1),
                      "flops_swept_per_launch": swept_flops(etot) / max(ekt["pair"][0], 1),
                      "note": "culling off: every Eq. 2 term of every in-reach pair swept (each pair from both sides)"}
    if searched and not args.cull and not particle2d:
        dem.set_culling(True)
        cms, _, _, ckt, ctot = timed(3, args.steps, False)
        cev = max(ckt["pair"][0], 1)
        ckern = ckt["pair"][1] / cev
        ctf = swept_flops(ctot) / cev / (ckern * 1e-3) / 1e12
        culled = {"value": n * world * args.steps / (cms * 1e-3), "unit": "particle-timesteps/s",
                  "ms_per_step": cms / args.steps, "kernel": "k_pair_cull", "kernel_ms": ckern,
                  "pose_kernel_ms": ckt["pose"][1] / cev, "flops_per_launch": swept_flops(ctot) / cev, "achieved": ctf,
                  "frac": ctf / peak_tf,
                  "note": "same results; the library default.  The kernel is not ALU-bound (cull tests, queues, pose traffic)"}
    # per-kernel breakdown of the default path (events around every kernel: its own short pass, not the timed one)
    ccnt = counters_now()
    _, _, _, kt2, _ = timed(3, min(args.steps, 50), False, level=2)
    detail = breakdown(kt2, int(ccnt["pairs_listed"]), int(ccnt["pairs_evaluated"]))
    if culled is not None:
        culled["terms_swept_now"] = ccnt["terms_swept"]
        culled["terms_now"] = ccnt["terms"]
        dem.set_culling(False)

    # ---- third arm: the same workload thermalised (the paper's workloads are thermalised fluids) ----------
    thermal = None
    if args.thermalise > 0:
        step(args.thermalise)
        arms = {}
        for name, cull in (("culled", True), ("every_term", False)) if (searched and not particle2d) else (("default", None),):
            if cull is not None:
                dem.set_culling(cull)
            tms, _, _, tkt, ttot = timed(3, min(args.steps, 100), False)
            tev = max(tkt["pair"][0], 1)
            arms[name] = {"value": n * world * min(args.steps, 100) / (tms * 1e-3), "ms_per_step": tms / min(args.steps, 100),
                          "kernel_ms": tkt["pair"][1] / tev, "pose_kernel_ms": tkt["pose"][1] / tev}
            if st["dim"] == 3 and searched:
                tf = swept_flops(ttot) / tev / (tkt["pair"][1] / tev * 1e-3) / 1e12
                arms[name].update({"achieved": tf, "frac": tf / peak_tf})
        if searched and not particle2d:
            dem.set_culling(bool(args.cull))
        if searched and not particle2d:
            dem.set_culling(True)
        tc = counters_now()
        if searched and not particle2d:
            dem.set_culling(bool(args.cull))
        thermal = {"equilibration_steps": args.thermalise, "arms": arms, "active_terms": tc["active"],
                   "pairs_in_reach": tc["pairs_evaluated"], "pairs_listed": tc["pairs_listed"],
                   "terms_swept_culled": None if particle2d else tc["terms_swept"]}

    # ---- end to end through the host-buffer entry point -------------------------------------------------------------
    h = {kk: t[kk].cpu().pin_memory() for kk in ("pos", "quat", "vel", "angmom")}
    hsid = t["shape_id"].cpu().pin_memory()
    hf = torch.empty((n, 4), dtype=torch.float32).pin_memory()
    dem.set_l2_flush(0)
    for _ in range(3):
        dem.step_host(h["pos"], h["quat"], h["vel"], h["angmom"], hsid, st["box"], dt_step, 1, skin, hf, None)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        dem.step_host(h["pos"], h["quat"], h["vel"], h["angmom"], hsid, st["box"], dt_step, 1, skin, hf, None)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value = aggregate_value(n, world, args.e2e_steps, max_over_ranks(e2e_s, world, "cuda") * 1e3)
    h2d = 4 * n * 16 + n * 4
    d2h = 5 * n * 16
    # the same calls with the library's default pair kernel (exact culling on), when the headline arm switched it off
    e2e_default = None
    if searched and not particle2d and not args.cull:
        dem.set_culling(True)
        for _ in range(3):
            dem.step_host(h["pos"], h["quat"], h["vel"], h["angmom"], hsid, st["box"], dt_step, 1, skin, hf, None)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            dem.step_host(h["pos"], h["quat"], h["vel"], h["angmom"], hsid, st["box"], dt_step, 1, skin, hf, None)
        barrier()
        e2e_default = aggregate_value(n, world, args.e2e_steps,
                                      max_over_ranks(time.perf_counter() - t0, world, "cuda") * 1e3)
        dem.set_culling(False)

    # ---- oracle on the host cores (rank 0, N = 1 only) ---------------------------------------------------------------
    cpu_baseline = None
    if rank == 0 and world == 1:
        cpu_baseline = oracle_baseline(di.make_config(k, seed=rank), args.cpu_seconds)

    if rank == 0:
        step_s = elapsed_ms * 1e-3
        line = {
            "metric": "particle-timesteps/s", "value": value, "unit": "particle-timesteps/s", "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": elapsed_ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": di.CONFIG_NAMES[k], "N": n, "dt": dt_step, "skin": skin,
                       "parallelism": "replicas x%d" % world if world > 1 else "1 GPU",
                       "l2": ("flushed before every step (160 MiB memset inside the timed region)"
                              if not args.no_l2_flush else "not flushed (working set < L2)"),
                       "culling": ("2D per-particle kernel with exact per-vertex culling (library default)" if particle2d else
                                   "on" if args.cull else "off: every Eq. 1/2 term of every in-reach pair is swept; 'culled' = "
                                   "the same steps with the library default (exact per-feature culling)")},
            # feature-pair rates of the timed region (nominal Eq. 1/2 terms over unique listed pairs, each once per
            # evaluation; `evaluated` = the terms whose nearest-point search was executed; triangle primitives = the
            # same with every polygon face fanned into triangles)
            "feature_pair_evals_per_s": terms * world * (args.steps + 1) / step_s,
            "feature_pairs_evaluated_per_s": (tot["ee_swept"] + tot["vf_swept"]) * world / step_s if searched else None,
            "triangle_primitives_per_s": prims * world * (args.steps + 1) / step_s if prims else None,
            "feature_pairs_per_step": terms, "unique_pairs": int(cls.sum()), "active_terms_now": ccnt["active"],
            "roofline": roofline, "culled": culled, "every_term": every_term, "thermalised": thermal, "breakdown": detail,
            "cpu_baseline": cpu_baseline,
            "e2e": {"value": e2e_value, "unit": "particle-timesteps/s", "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "steps": args.e2e_steps,
                    "pair_kernel": "as the headline arm (%s)" % ("culling on" if (args.cull or particle2d) else "every term swept"),
                    "value_library_default": e2e_default},
            "gpu_launches": gpu_launches, "clocks": clocks,
            # the 160 MiB memset that flushes the L2 is inside every timed step above (value, culled, thermalised);
            # its own device time per step, from the breakdown pass, is given here for the reader, never subtracted
            "l2_flush_us_per_step": (detail.get("us_per_launch", {}).get("flush") if detail else None),
        }
        print(json.dumps(line))
    dem.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
