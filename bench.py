#!/usr/bin/env python
"""bench.py -- headline benchmark: the exhaustive MI map of BASELINE.json's configs[4] ("C5":
260x311x260 T1-like fixed @0.7 mm, 182x218x182 T2-like moving @1.0 mm, 256 bins, 41^3 translation
grid over +-10 mm, trilinear) in voxel-transform evaluations per second.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config C1..C5|C5ALL|PAPER51|PAPERROT|PAPERSCALE] [--all] [--shard] [--interp trilinear|nearest|pv]

A "step" is one pass of the whole hot path (a2 transform generation, a3 resample, a4 joint
histogram, a5 entropy reduction, a6 map assembly + arg max) over the full grid: one mi_map call.
`value` is timed with CUDA events with both volumes already resident (pre-binned) in HBM; `e2e`
is the same metric through the C ABI with HOST buffers (mi_create from pinned host memory +
mi_map to host outputs + mi_destroy inside the timed region).

Multi-GPU (one process per GPU; `--gpus N` spawns its own ranks through torch.distributed.run when it
was not launched by it): by default every rank maps the whole grid for its own pair -- independent
problems, no data-path collective, "scaling": "weak".  `--shard` maps ONE grid across the ranks
(contiguous p2 slabs through mi_map_range, one NCCL all-gather of the slabs): "scaling": "strong".

`--all` prints one JSON line per BASELINE.json config (C1..C4 first, the headline C5 last), each with
its roofline fraction, MI evaluations per second (the unit of the paper's Table 1)
and a bounded oracle timing.  `--impl reference` times the CPU oracle (test infrastructure) on a
bounded sample of the same grid.  Prints ONE JSON line per workload on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# DRAM traffic of the dominant kernel from the committed `ncu --set full` captures of this command
# (profiles/r2c_ncu.md): dram__bytes_read.sum + dram__bytes_write.sum of ONE launch and the evaluations
# that launch performed; bench.py scales it to a step (bytes per evaluation x evaluations per step).
# Keyed by (config, grid, interpolation).
NCU_DRAM = {
    # C5, zhist_kernel, launch = 5 of the 41 p0 slabs = 8405 transforms (profiles/r2c_ncu.md section 3:
    # dram__bytes_read.sum 16.282388 GB + dram__bytes_write.sum 553.706496 MB)
    ("C5", (41, 41, 41), 1): {"bytes_per_launch": 16282388000 + 553706496, "evals_per_launch": 8405 * 21023600,
                               "source": "profiles/r2c_ncu.md section 3"},
    # C3, resample_quad_kernel, launch = the whole 15^3 map (profiles/r2c_ncu.md section 6: 9.950978 + 4.473929 GB)
    ("C3", (15, 15, 15), 1): {"bytes_per_launch": 9950978000 + 4473929000, "evals_per_launch": 3375 * 21023600,
                               "source": "profiles/r2c_ncu.md section 6"},
}

METRIC = "voxel-transform evaluations per second (MI map, 260x311x260 fixed, 256 bins)"
UNIT = "evals/s"
PAPER_TABLE1 = {0: 116.21, 1: 86.30, 2: 86.30, 3: 99.46, 4: 99.46}   # MI evaluations/s, GTX 1060, PAPER.md:204-206 (context only)


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), float(p.get("sm_max_mhz", 1965.0)), "measured"
    except Exception:
        return 6650.0, 1965.0, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.FIELDS,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        late = False
        if not self.rows:       # a timed region shorter than nvidia-smi's start-up (C1): wait for its first line
            late = True
            deadline = time.perf_counter() + 2.0
            while not self.rows and time.perf_counter() < deadline:
                time.sleep(0.02)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        busy = [c for c, p in zip(sm, power) if p > 250.0] or sm
        out = {"sm_mhz": float(np.median(busy)) if busy else None,
               "sm_max_mhz": max(smax) if smax else None, "reasons": sorted(reasons),
               "samples": len(sm), "power_w_max": max(power) if power else None}
        if late:
            out["note"] = "timed region shorter than one sampling period: sampled right after it"
        return out


def sample_nodes(cfg, count):
    """Deterministic, spread-out sample of grid nodes (linear indices, p0 fastest)."""
    nt = cfg.n_transforms
    count = max(1, min(count, nt))
    stride = 2654435761 % nt
    while np.gcd(stride, nt) != 1:
        stride += 1
    return [(7 + i * stride) % nt for i in range(count)]


def node_matrices(orc, cfg, nodes):
    n0, n1, _ = cfg.n
    T = []
    for t in nodes:
        k = (t % n0, (t // n0) % n1, t // (n0 * n1))
        p = [cfg.lo[d] if cfg.n[d] == 1 else cfg.lo[d] + k[d] * (cfg.hi[d] - cfg.lo[d]) / (cfg.n[d] - 1)
             for d in range(3)]
        T.append(orc.family_matrix(cfg.family, p))
    T = np.stack(T)
    return T, orc.physical_to_index(T, cfg.fixed.shape[::-1], cfg.fixed_spacing, cfg.moving.shape[::-1],
                                    cfg.moving_spacing)


def time_oracle(cfg, interp, budget_s):
    """Oracle as it stands on the host cores, on a bounded sample of the grid: evals/s."""
    import oracle as orc
    cores = orc.max_threads()
    nodes = sample_nodes(cfg, cores)
    _, M = node_matrices(orc, cfg, nodes)
    t0 = time.perf_counter()
    orc.eval_batch(cfg.fixed, cfg.moving, M, cfg.nbins, *cfg.ranges, interp, q=cfg.q)
    per = time.perf_counter() - t0       # one transform per thread ran concurrently
    count = int(max(cores, min(cfg.n_transforms, round(budget_s / max(per, 1e-6)) * cores)))
    nodes = sample_nodes(cfg, count)
    _, M = node_matrices(orc, cfg, nodes)
    t0 = time.perf_counter()
    r = orc.eval_batch(cfg.fixed, cfg.moving, M, cfg.nbins, *cfg.ranges, interp, q=cfg.q)
    dt = time.perf_counter() - t0
    evals = float(cfg.fixed.size) * len(nodes)
    return {"value": evals / dt, "unit": UNIT, "cores": int(r["threads"]), "kind": "oracle",
            "sample": "%d of %d grid nodes of %s (deterministic stride), all %d fixed voxels each, %.1f s"
                      % (len(nodes), cfg.n_transforms, cfg.name, cfg.fixed.size, dt)}, dt


INTERP_NAMES = {0: "nearest", 1: "trilinear", 2: "partial-volume"}


def workload_config(cfg, interp, extra=None):
    c = {"workload": "%s: fixed %s @%.2f mm, moving %s @%.2f mm, %d bins, %s grid %s over [%g,%g], %s, q=%s"
         % (cfg.name, "x".join(str(d) for d in cfg.fixed.shape[::-1]), cfg.fixed_spacing[0],
            "x".join(str(d) for d in cfg.moving.shape[::-1]), cfg.moving_spacing[0], cfg.nbins,
            {0: "translation", 1: "euler-rotation", 2: "versor-rotation", 3: "scale", 4: "log-scale"}.get(cfg.family, str(cfg.family)),
            "x".join(str(d) for d in cfg.n), cfg.lo[0], cfg.hi[0], INTERP_NAMES[interp], list(cfg.q)),
         "fixed_voxels": int(cfg.fixed.size), "transforms": cfg.n_transforms,
         "evaluations_per_step": int(cfg.evaluations)}
    if extra:
        c.update(extra)
    return c


def run_reference(args, cfg, interp):
    if int(os.environ.get("RANK", "0")) != 0:
        return
    budget = 8.0
    vals, ms = [], []
    for i in range(args.warmup + args.steps):
        r, dt = time_oracle(cfg, interp, budget)
        if i >= args.warmup:
            vals.append(r["value"]); ms.append(dt * 1e3)
        last = r
    value = float(np.mean(vals))
    last["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(ms)),
            "higher_is_better": True, "scaling": "strong" if args.shard else "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(cfg, interp),
            "note": "each step = the oracle on a bounded sample of the grid",
            "cpu_baseline": last,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


class Runtime:
    """Per-process CUDA / torch.distributed state shared by the workloads of one invocation."""

    def __init__(self):
        import torch
        self.torch = torch
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
        torch.cuda.set_device(self.local)
        self.dev = torch.device("cuda", self.local)
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            dist.init_process_group("nccl", device_id=self.dev)
            self.dist = dist
        self.stream = torch.cuda.current_stream().cuda_stream
        self.flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=self.dev)   # > 126 MB L2
        self.num_sms = torch.cuda.get_device_properties(self.local).multi_processor_count

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()
        self.torch.cuda.synchronize()

    def max_over_ranks(self, x):
        if self.dist is None:
            return float(x)
        t = self.torch.tensor([x], dtype=self.torch.float64, device=self.dev)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.dist is not None:
            self.dist.destroy_process_group()


def run_ours(rt, args, cfg, interp, cpu_budget_s):
    """One workload: returns the JSON line (rank 0) or None."""
    torch = rt.torch
    from paper_1909_10690_b200 import binding as mi   # raises if the CUDA library is missing
    from paper_1909_10690_b200 import sharding as sh

    hbm_gbs, sm_max_mhz, peak_src = load_peaks()
    fixed_pin = torch.from_numpy(cfg.fixed).pin_memory()
    moving_pin = torch.from_numpy(cfg.moving).pin_memory()
    fixed_dev, moving_dev = fixed_pin.to(rt.dev), moving_pin.to(rt.dev)
    nch = 1 + len(cfg.q)
    shape = (nch,) + tuple(int(v) for v in cfg.n[::-1])
    shard = bool(args.shard) and rt.world > 1
    map_dev = torch.empty(shape, dtype=torch.float64, device=rt.dev)
    am_dev = torch.empty(nch, dtype=torch.int64, device=rt.dev)
    ctx = mi.mi_create(fixed_dev, moving_dev, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                       device=rt.local, cuda_stream=rt.stream)
    for name, val in args.opt:                           # experiments only: the default run sets none
        mi.mi_set_option(ctx, getattr(mi, "MI_OPT_" + name.upper()), val)
    slab = sh.slab_range(cfg.n, rt.rank, rt.world) if shard else None
    if shard and slab is not None:
        slab_dev = torch.empty((nch, slab[1][2] - slab[0][2]) + shape[2:], dtype=torch.float64, device=rt.dev)
        slab_am = torch.empty(nch, dtype=torch.int64, device=rt.dev)

    def map_slab(begin, end):
        mi.mi_map_range(ctx, cfg.family, cfg.lo, cfg.hi, cfg.n, begin, end, cfg.q, interp, map_out=slab_dev, argmax_out=slab_am)
        return slab_dev

    def step():
        if shard:     # one grid over all ranks: p2 slabs + one NCCL all-gather of doubles
            full, am = sh.map_sharded(map_slab, cfg.n, nch, rt.rank, rt.world, dist=rt.dist, device=rt.dev)
            map_dev.copy_(full); am_dev.copy_(am)
        else:
            mi.mi_map(ctx, cfg.family, cfg.lo, cfg.hi, cfg.n, cfg.q, interp, map_out=map_dev, argmax_out=am_dev)

    for _ in range(args.warmup):
        step()
    # ---- timed region: K steps, CUDA events per step on the launching stream, L2 flushed between ----
    sampler = ClockSampler(rt.local)
    rt.barrier()
    if rt.rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = np.zeros(5)
    launches = hist_launches = 0
    updates_issued = 0
    wall0 = time.perf_counter()
    for k in range(args.steps):
        rt.flush.fill_(k & 0xFF)
        ev[k][0].record()
        step()
        ev[k][1].record()
        ms5, ln5 = mi.mi_last_timing(ctx)
        kern_ms += ms5
        launches += int(ln5[:4].sum())      # class 4 (the dominant kernel alone) is a subset of class 1
        hist_launches += int(ln5[4])
        updates_issued = mi.mi_get_option(ctx, mi.MI_INFO_LAST_UPDATES_ISSUED)
    rt.barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop() if rt.rank == 0 else None
    total_ms = rt.max_over_ranks(sum(a.elapsed_time(b) for a, b in ev))
    path = mi.mi_get_option(ctx, mi.MI_INFO_LAST_PATH)
    evals_step = float(cfg.evaluations)
    jobs = 1 if shard else rt.world                     # grids mapped per step over all ranks
    value = evals_step * args.steps * jobs / (total_ms * 1e-3)

    # ---- e2e: HOST buffers through the C ABI, copies inside the timed region ------------------------
    map_host = np.empty(shape if not shard or slab is None else tuple(slab_dev.shape), dtype=np.float64)
    am_host = np.empty(nch, dtype=np.int64)
    e2e_steps = max(1, min(args.steps, 3))

    e2e_kern = np.zeros(5)

    def e2e_step():
        c2 = mi.mi_create(fixed_pin, moving_pin, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                          device=rt.local, cuda_stream=rt.stream)
        for name, val in args.opt:
            mi.mi_set_option(c2, getattr(mi, "MI_OPT_" + name.upper()), val)
        if shard:
            if slab is not None:
                mi.mi_map_range(c2, cfg.family, cfg.lo, cfg.hi, cfg.n, slab[0], slab[1], cfg.q, interp, map_out=map_host,
                                argmax_out=am_host)
        else:
            mi.mi_map(c2, cfg.family, cfg.lo, cfg.hi, cfg.n, cfg.q, interp, map_out=map_host, argmax_out=am_host)
        e2e_kern[:] = mi.mi_last_timing(c2)[0]
        mi.mi_destroy(c2)

    for _ in range(2):      # untimed: the library's memory pool reaches its steady size
        e2e_step()
    rt.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = rt.max_over_ranks(time.perf_counter() - t0)
    e2e_value = evals_step * e2e_steps * jobs / e2e_s
    # mi_create alone (upload from pinned host memory + pre-binning, ranking, padding): one-off cost, reported apart
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    c3 = mi.mi_create(fixed_pin, moving_pin, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                      device=rt.local, cuda_stream=rt.stream)
    torch.cuda.synchronize()
    create_ms = (time.perf_counter() - t0) * 1e3
    mi.mi_destroy(c3)
    h2d = int(cfg.fixed.nbytes + cfg.moving.nbytes + cfg.n_transforms * 48 // (rt.world if shard else 1) + 8 * len(cfg.q))
    d2h = int(map_host.nbytes + am_host.nbytes)
    if not shard:
        assert np.array_equal(am_host, am_dev.cpu().numpy())

    # ---- capture-range analysis of the finished map, outside the timed region ----------
    torch.cuda.synchronize()
    an_reps = 5
    t0 = time.perf_counter()
    for _ in range(an_reps):
        grad = mi.mi_map_gradient(map_dev[0], cfg.lo, cfg.hi, device=rt.local, cuda_stream=rt.stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    for _ in range(an_reps):
        basins = mi.mi_map_basins(map_dev[0], 1, 26, -1, device=rt.local, cuda_stream=rt.stream)
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    analysis = {"map_nodes": cfg.n_transforms, "gradient_ms": (t1 - t0) / an_reps * 1e3,
                "basins_ms": (t2 - t1) / an_reps * 1e3, "channel": "Shannon", "connectivity": 26,
                "n_extrema": int(basins["n_extrema"]), "capture_fraction_of_global_max": float(basins["capture_fraction"]),
                "max_steps": int(basins["max_steps"]),
                "note": "launch-latency bound at the paper's map sizes: no roofline fraction claimed"}
    del grad

    if rt.rank != 0:
        if cfg.family == 1 and interp == 1:
            pass
        mi.mi_destroy(ctx)
        return None

    # ---- roofline of the dominant kernel (resample + histogram) --------------------------------------
    # north_star: t_roof = max(t_HBM, t_atom); one shared-memory histogram update per evaluation.
    nb_probe = min(cfg.nbins, 256)
    r_rand = mi.mi_probe_shared_atomic_rate(rt.local, nb_probe, 1, 8192)
    r_free = mi.mi_probe_shared_atomic_rate(rt.local, nb_probe, 0, 8192)
    r_lattice = mi.mi_probe_shared_atomic_rate(rt.local, nb_probe, 3, 8192)   # round 1's pattern, for continuity
    r_pre = mi.mi_probe_shared_atomic_rate(rt.local, nb_probe, 6, 8192)       # pattern 1 with the hash out of the timed loop
    # dominant kernel: the z-lerp+histogram kernel (separable maps) or the generic resample+histogram
    # kernel, timed alone with CUDA events on the launching stream (mi_last_timing class 4); one step
    # launches it hist_launches times and together the launches do every evaluation of the step once
    my_evals = evals_step if not shard or slab is None else float(cfg.fixed.size) * np.prod(slab_dev.shape[1:])
    hist_ms = kern_ms[4] / args.steps
    hist_launches = max(1, hist_launches // args.steps)
    achieved = my_evals / (hist_ms * 1e-3)                        # updates/s inside the kernel (this rank)
    pass_bytes = cfg.fixed.size * 1 + cfg.moving.size * 4          # fixed bins + moving floats, read once
    t_hbm_b1 = cfg.n_transforms * pass_bytes / (hbm_gbs * 1e9)
    t_hbm_once = pass_bytes / (hbm_gbs * 1e9)
    sm_hz = (clocks["sm_mhz"] or sm_max_mhz) * 1e6
    # The denominator of every shared-atomic line: the larger of the two probed lane-independent random-bin rates
    # (pattern 1 pays for its hash inside the timed loop, pattern 6 does not) -- never a rate the probe's own
    # arithmetic limits.  peak_nominal is the crossbar model: one warp-wide update = 3.53 wavefronts at 1 per clock.
    r_peak = max(r_rand, r_pre)
    r_nominal = rt.num_sms * 32.0 * sm_hz / 3.53
    t_atom = my_evals / r_peak
    t_lsu = 32.0 * my_evals / (rt.num_sms * 128.0 * sm_hz)
    cap = NCU_DRAM.get((cfg.name, tuple(cfg.n), interp))
    traffic = None if cap is None or shard else cap["bytes_per_launch"] / cap["evals_per_launch"] * evals_step
    kernel_names = {1: "zhist_kernel (separable path: z-lerp + joint histogram + fused entropy epilogue)",
                    0: "resample_hist_kernel (generic affine: two 16-byte quad gathers + 7 lerps + joint histogram)",
                    2: "resample_hist_wide_kernel (nbins > 256: global-memory histograms)",
                    3: "resample_hist_pv_kernel (partial volume: 8 byte gathers + 8 weighted histogram updates)"}
    roofline = {"bound": "shared-atomic", "kernel": kernel_names[path],
                "achieved": achieved / 1e9, "peak": r_peak / 1e9, "unit": "G shared-atomic updates/s",
                "frac": achieved / r_peak,
                "achieved_counts": "evaluations (one histogram update each)",
                "peak_nominal": r_nominal / 1e9, "frac_of_nominal": achieved / r_nominal,
                "peak_nominal_source": "num_sms x 32 lanes x sampled SM clock / 3.53 wavefronts per warp-wide update "
                                       "(expected fullest bank of 32 independent lanes over 32 banks)",
                "peak_probe_hash_in_loop": r_rand / 1e9, "peak_probe_hash_hoisted": r_pre / 1e9,
                "traffic": traffic, "traffic_unit": "DRAM bytes per step of the dominant kernel (ncu capture scaled by evaluations)",
                "traffic_capture": cap,
                "algorithmic_bytes_per_step": pass_bytes,
                "all_a3_a4_kernels_ms_per_step": kern_ms[1] / args.steps,
                "peak_source": "mi_probe_shared_atomic_rate measured in this run: the larger of pattern 1 (uniform random "
                               "bins, independent between the lanes of a warp, hashed inside the timed loop) and pattern 6 "
                               "(the same statistics, bins hashed before the loop)",
                "peak_conflict_free": r_free / 1e9,
                "peak_round1_pattern": r_lattice / 1e9,
                "peak_round1_pattern_note": "round 1 drew the bins from one LCG per thread seeded linearly in the thread "
                                            "index: the lanes of a warp then form an arithmetic progression and spread "
                                            "over the banks more evenly than chance (2.70 wavefronts per update against "
                                            "3.53 for independent lanes, profiles/r2c_ncu.md)",
                "t_atom_ms": t_atom * 1e3, "t_hbm_resident_ms": t_hbm_once * 1e3,
                "t_hbm_if_every_transform_restreams_ms": t_hbm_b1 * 1e3,
                "kernel_ms_per_step": hist_ms, "kernel_launches_per_step": hist_launches,
                "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": peak_src,
                "step_frac_of_t_roof": max(t_atom, t_hbm_once) / (total_ms / args.steps * 1e-3)}
    if path == 1 and updates_issued >= 0:
        # evaluations whose z slice falls outside the moving volume issue no update: the rate by updates issued
        # -- THAT rate is this line's achieved / frac; the rate by evaluations is kept beside it.  Still an upper
        # estimate: the kernel's count credits all 8 columns of a thread that has any valid column.
        issued_rate = updates_issued / (hist_ms * 1e-3)
        roofline.update({"updates_issued_per_step": int(updates_issued),
                         "achieved_by_evaluations": achieved / 1e9, "frac_by_evaluations": achieved / r_peak,
                         "achieved": issued_rate / 1e9, "frac": issued_rate / r_peak, "frac_issued": issued_rate / r_peak,
                         "frac_of_nominal": issued_rate / r_nominal,
                         "achieved_counts": "histogram updates the kernel issued (evaluations whose z slice lies outside "
                                            "the moving volume issue none)"})
    if path == 3:
        roofline["updates_per_evaluation"] = "up to 8 weighted updates (zero weights skipped)"
    if path == 0 and interp == 1:
        # rotations: bound by the rate at which L1TEX delivers the eight neighbours of every sample; its ceiling
        # is the same kernel without the histogram updates on the same transforms (mi_probe_gather_rate)
        import math
        nodes = sample_nodes(cfg, min(cfg.n_transforms, 4 * rt.num_sms))
        T = np.stack([mi.mi_family_matrix(cfg.family, [cfg.lo[d] if cfg.n[d] == 1 else cfg.lo[d] + k * (cfg.hi[d] - cfg.lo[d]) / (cfg.n[d] - 1)
                                                       for d, k in enumerate((t % cfg.n[0], (t // cfg.n[0]) % cfg.n[1], t // (cfg.n[0] * cfg.n[1])))])
                      for t in nodes])
        g_rate = mi.mi_probe_gather_rate(ctx, T, 3)
        # The peak of this line is a hardware floor, valid for ANY kernel that brings eight fp32 neighbours per sample
        # into registers: the load/store unit writes 64 B per clock per SM into the register file
        # (profiles/r2c_ncu.md section 6), a warp-wide sample needs 32 x 32 B of neighbours + 128 B of fixed bins
        # = 18 beats, + 2.41 crossbar wavefronts for its update.  The same kernel without its updates
        # (mi_probe_gather_rate) is a ceiling defined by the kernel's own code: a diagnostic, not a roofline.
        clk_per_warp_sample = (32 * 32 + 128) / 64.0 + 2.41
        floor_rate = rt.num_sms * sm_hz * 32.0 / clk_per_warp_sample
        roofline.update({"bound": "l1tex-writeback", "achieved": achieved / 1e9, "peak": floor_rate / 1e9,
                         "unit": "G trilinear samples/s (8 neighbours each)", "frac": achieved / floor_rate,
                         "achieved_counts": "evaluations (one trilinear sample and one histogram update each)",
                         "peak_source": "64 B/clk/SM register-file writeback of the load/store unit (ncu: "
                                        "l1tex__lsu_writeback_active) x %d SMs at the sampled SM clock, %.2f clocks per "
                                        "warp-wide sample" % (rt.num_sms, clk_per_warp_sample),
                         "clocks_per_warp_sample": clk_per_warp_sample,
                         "frac_of_shared_atomic_rate": achieved / r_peak, "frac_of_nominal": achieved / r_nominal,
                         "same_kernel_without_updates": {"rate": g_rate / 1e9, "ratio": achieved / g_rate,
                                                         "source": "mi_probe_gather_rate on %d nodes of this grid, measured "
                                                                   "in this run; says only how much the updates cost" % len(nodes)},
                         "t_lsu_gather_nominal_ms": t_lsu * 1e3})

    eval_batch = None
    if path == 0 and interp == 1:
        # latency of mi_eval_batch (the engine of mi_multimetric_gradient / mi_register) on the same context:
        # N = 1, 19 (one finite-difference step of a nine-parameter registration) and one transform per SM;
        # Shannon + one Tsallis order, outputs to the host, median host wall-clock of 7 calls after 2 warm-ups
        eval_batch = {}
        allT = np.stack([mi.mi_family_matrix(cfg.family, [cfg.lo[d] + k * (cfg.hi[d] - cfg.lo[d]) / max(cfg.n[d] - 1, 1)
                                                          for d, k in enumerate((t % cfg.n[0], (t // cfg.n[0]) % cfg.n[1], t // (cfg.n[0] * cfg.n[1])))])
                         for t in sample_nodes(cfg, min(cfg.n_transforms, rt.num_sms))])
        for nt in (1, 19, rt.num_sms):
            if nt > len(allT):
                continue
            ts = []
            for i in range(9):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                mi.mi_eval_batch(ctx, allT[:nt], (0.5,), interp)
                ts.append((time.perf_counter() - t0) * 1e3)
            eval_batch["n%d_ms" % nt] = float(np.median(ts[2:]))

    cpu_baseline = None
    if cpu_budget_s > 0:
        cpu_baseline, _ = time_oracle(cfg, interp, cpu_budget_s)
        from oracle import map_analysis as ora
        mh = map_dev[0].cpu().numpy()
        t0 = time.perf_counter()
        ora.map_gradient(mh, cfg.lo, cfg.hi)
        t1 = time.perf_counter()
        ob = ora.map_basins(mh, 1, 26, -1)
        t2 = time.perf_counter()
        analysis["oracle_gradient_ms"] = (t1 - t0) * 1e3
        analysis["oracle_basins_ms"] = (t2 - t1) * 1e3
        analysis["matches_oracle"] = bool(np.array_equal(ob["label"], basins["label"].cpu().numpy())
                                          and ob["captured"] == basins["captured"])

    mi_evals = cfg.n_transforms * args.steps * jobs / (total_ms * 1e-3)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": rt.world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if shard else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(cfg, interp, {
                "l2": "flushed between timed steps (256 MiB write)",
                "parallelism": ("one grid sharded x%d (p2 slabs, NCCL all-gather)" if shard else "replicas x%d") % rt.world,
                "mi_evals_per_s": mi_evals,
                "paper_table1_mi_evals_per_s_gtx1060": PAPER_TABLE1.get(cfg.family),
                **({"options": dict(args.opt)} if args.opt else {})}),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "ms_per_step": e2e_s / e2e_steps * 1e3, "mi_create_ms": create_ms,
                    "kernels_ms_last_step": float(e2e_kern[:4].sum())},
            "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "kernel_ms_per_step": {"setup": kern_ms[0] / args.steps, "resample_hist": kern_ms[1] / args.steps,
                                   "entropy": kern_ms[2] / args.steps, "map": kern_ms[3] / args.steps,
                                   "dominant_hist_kernel": kern_ms[4] / args.steps},
            "path": {0: "generic", 1: "separable", 2: "wide", 3: "partial-volume"}[path],
            "rare_voxels": mi.mi_get_option(ctx, mi.MI_INFO_RARE_VOXELS),
            "capture_analysis": analysis, "wall_s_timed_region": wall}
    if eval_batch:
        line["eval_batch_latency"] = eval_batch
    mi.mi_destroy(ctx)
    return line


def respawn_under_torchrun(args):
    """--gpus N without a launcher: start N ranks of this script through torch.distributed.run."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C5", choices=["C1", "C2", "C3", "C4", "C5", "C5ALL", "PAPER51", "PAPERROT", "PAPERSCALE"])
    ap.add_argument("--all", action="store_true", help="one line per BASELINE.json config, C5 (the headline) last")
    ap.add_argument("--shard", action="store_true", help="N > 1: map ONE grid across the ranks (strong scaling)")
    ap.add_argument("--res", type=float, default=1.0, help="development only: reduced-resolution phantom")
    ap.add_argument("--grid", type=int, default=0, help="development only: grid nodes per axis")
    ap.add_argument("--interp", default="trilinear", choices=["trilinear", "nearest", "pv"])
    ap.add_argument("--nbins", type=int, default=0, help="development only: override the config's bin count (e.g. 4096)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="experiments only: mi_set_option(MI_OPT_<NAME>, VALUE) on the context, e.g. zhist_match_any=1")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3  # timing rule: W >= 3
    args.opt = [(kv.split("=")[0], int(kv.split("=")[1])) for kv in args.opt]
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        respawn_under_torchrun(args)

    from paper_1909_10690_b200 import phantoms as ph
    interp = {"nearest": 0, "trilinear": 1, "pv": 2}[args.interp]
    names = ["C1", "C2", "C3", "C4", "C5"] if args.all else [args.config]

    def get(name):
        kw = {}
        if name not in ("C1", "C2") and args.res != 1.0:
            kw["res"] = args.res
        if args.grid:
            kw["grid_n"] = args.grid
        cfg = ph.get_config(name, **kw)
        if args.nbins:
            import dataclasses
            cfg = dataclasses.replace(cfg, nbins=args.nbins)
        return cfg

    if args.impl == "reference":
        for name in names:
            run_reference(args, get(name), interp)
        return

    rt = Runtime()
    for name in names:
        budget = 0.0 if args.no_cpu_baseline else (15.0 if not args.all or name == "C5" else 5.0)
        line = run_ours(rt, args, get(name), interp, budget)
        if line is not None:
            print(json.dumps(line), flush=True)
    rt.close()


if __name__ == "__main__":
    main()
