#!/usr/bin/env python
"""bench.py -- headline benchmark: the exhaustive MI map of BASELINE.json's configs[4] ("C5":
260x311x260 T1-like fixed @0.7 mm, 182x218x182 T2-like moving @1.0 mm, 256 bins, 41^3 translation
grid over +-10 mm, trilinear) in voxel-transform evaluations per second.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path (a2 transform generation, a3 resample, a4 joint
histogram, a5 entropy reduction, a6 map assembly + arg max) over the full grid: one mi_map call.
`value` is timed with CUDA events with both volumes already resident (pre-binned) in HBM; `e2e`
is the same metric through the C ABI with HOST buffers (mi_create from pinned host memory +
mi_map to host outputs + mi_destroy inside the timed region).  At N > 1 every rank maps the whole
grid on its own GPU (independent problems, no data-path collective): weak scaling.
`--impl reference` times the CPU oracle (test infrastructure) on a bounded sample of the same grid.
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel (4 of the 41 p0
# slabs = 6724 transforms = 1.414e11 evaluations), from the committed ncu --set full capture of the
# default command (profiles/r1k_ncu_zhist_final.md); keyed by (config, grid, interpolation)
NCU_DRAM_BYTES_PER_LAUNCH = {("C5", (41, 41, 41), 1): 16264608000 + 553361408}

METRIC = "voxel-transform evaluations per second (MI map, 260x311x260 fixed, 256 bins)"
UNIT = "evals/s"


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
        return {"sm_mhz": float(np.median(busy)) if busy else None,
                "sm_max_mhz": max(smax) if smax else None, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power) if power else None}


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
    dt = time.perf_counter() - t0
    per = dt / 1.0  # one transform per thread ran concurrently -> dt per `cores` transforms
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


def workload_config(cfg, interp, extra=None):
    c = {"workload": "%s: fixed %s @%.2f mm, moving %s @%.2f mm, %d bins, %s grid %s over [%g,%g], %s, q=%s"
         % (cfg.name, "x".join(str(d) for d in cfg.fixed.shape[::-1]), cfg.fixed_spacing[0],
            "x".join(str(d) for d in cfg.moving.shape[::-1]), cfg.moving_spacing[0], cfg.nbins,
            {0: "translation", 1: "euler-rotation", 3: "scale"}.get(cfg.family, str(cfg.family)),
            "x".join(str(d) for d in cfg.n), cfg.lo[0], cfg.hi[0],
            "trilinear" if interp == 1 else "nearest", list(cfg.q)),
         "fixed_voxels": int(cfg.fixed.size), "transforms": cfg.n_transforms,
         "evaluations_per_step": int(cfg.evaluations)}
    if extra:
        c.update(extra)
    return c


def run_reference(args, cfg, interp):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
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
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(cfg, interp, {"note": "each step = bounded sample of the grid"}),
            "cpu_baseline": last,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C5", choices=["C2", "C3", "C4", "C5", "PAPER51"])
    ap.add_argument("--res", type=float, default=1.0, help="development only: reduced-resolution phantom")
    ap.add_argument("--grid", type=int, default=0, help="development only: grid nodes per axis")
    ap.add_argument("--interp", default="trilinear", choices=["trilinear", "nearest"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3  # timing rule: W >= 3

    from paper_1909_10690_b200 import phantoms as ph
    kw = {}
    if args.config != "C2" and args.res != 1.0:
        kw["res"] = args.res
    if args.grid:
        kw["grid_n"] = args.grid
    cfg = ph.get_config(args.config, **kw)
    interp = 1 if args.interp == "trilinear" else 0

    if args.impl == "reference":
        return run_reference(args, cfg, interp)

    import torch
    from paper_1909_10690_b200 import binding as mi   # raises if the CUDA library is missing

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    hbm_gbs, sm_max_mhz, peak_src = load_peaks()
    stream = torch.cuda.current_stream().cuda_stream
    fixed_pin = torch.from_numpy(cfg.fixed).pin_memory()
    moving_pin = torch.from_numpy(cfg.moving).pin_memory()
    fixed_dev, moving_dev = fixed_pin.to(dev), moving_pin.to(dev)
    nch = 1 + len(cfg.q)
    map_dev = torch.empty((nch,) + tuple(int(v) for v in cfg.n[::-1]), dtype=torch.float64, device=dev)
    am_dev = torch.empty(nch, dtype=torch.int64, device=dev)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2

    ctx = mi.mi_create(fixed_dev, moving_dev, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                       device=local, cuda_stream=stream)

    def step():
        mi.mi_map(ctx, cfg.family, cfg.lo, cfg.hi, cfg.n, cfg.q, interp, map_out=map_dev, argmax_out=am_dev)

    for _ in range(args.warmup):
        step()
    # ---- timed region: K steps, CUDA events per step on the launching stream, L2 flushed between ----
    sampler = ClockSampler(local)
    barrier()
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = np.zeros(5)
    launches = 0
    hist_launches = 0
    wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k & 0xFF)
        ev[k][0].record()
        step()
        ev[k][1].record()
        ms5, ln5 = mi.mi_last_timing(ctx)
        kern_ms += ms5
        launches += int(ln5[:4].sum())      # class 4 (the dominant kernel alone) is a subset of class 1
        hist_launches += int(ln5[4])
    barrier()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    if dist is not None:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    evals_step = float(cfg.evaluations)
    value = evals_step * args.steps * world / (total_ms * 1e-3)

    # ---- e2e: HOST buffers through the C ABI, copies inside the timed region ------------------------
    map_host = np.empty(map_dev.shape, dtype=np.float64)
    am_host = np.empty(nch, dtype=np.int64)
    e2e_steps = max(1, min(args.steps, 3))

    def e2e_step():
        c2 = mi.mi_create(fixed_pin, moving_pin, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                          device=local, cuda_stream=stream)
        mi.mi_map(c2, cfg.family, cfg.lo, cfg.hi, cfg.n, cfg.q, interp, map_out=map_host, argmax_out=am_host)
        mi.mi_destroy(c2)

    for _ in range(2):      # untimed: the library's memory pool reaches its steady size
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    if dist is not None:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    e2e_value = evals_step * e2e_steps * world / e2e_s
    # mi_create alone (upload from pinned host memory + pre-binning, ranking, padding): one-off cost, reported apart
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    c3 = mi.mi_create(fixed_pin, moving_pin, cfg.fixed_spacing, cfg.moving_spacing, cfg.nbins, *cfg.ranges,
                      device=local, cuda_stream=stream)
    torch.cuda.synchronize()
    create_ms = (time.perf_counter() - t0) * 1e3
    mi.mi_destroy(c3)
    h2d = int(cfg.fixed.nbytes + cfg.moving.nbytes + cfg.n_transforms * 48 + 8 * len(cfg.q))
    d2h = int(map_host.nbytes + am_host.nbytes)
    assert np.array_equal(am_host, am_dev.cpu().numpy())

    # ---- capture-range analysis of the finished map, outside the timed region ----------
    torch.cuda.synchronize()
    an_reps = 5
    t0 = time.perf_counter()
    for _ in range(an_reps):
        grad = mi.mi_map_gradient(map_dev[0], cfg.lo, cfg.hi, device=local, cuda_stream=stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    for _ in range(an_reps):
        basins = mi.mi_map_basins(map_dev[0], 1, 26, -1, device=local, cuda_stream=stream)
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    analysis = {"map_nodes": cfg.n_transforms, "gradient_ms": (t1 - t0) / an_reps * 1e3,
                "basins_ms": (t2 - t1) / an_reps * 1e3, "channel": "Shannon", "connectivity": 26,
                "n_extrema": int(basins["n_extrema"]), "capture_fraction_of_global_max": float(basins["capture_fraction"]),
                "max_steps": int(basins["max_steps"]),
                "note": "launch-latency bound at the paper's map sizes: no roofline fraction claimed"}
    del grad

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (resample + histogram) --------------------------------------
    # north_star: t_roof = max(t_HBM, t_atom); one shared-memory histogram update per evaluation.
    r_rand = mi.mi_probe_shared_atomic_rate(local, cfg.nbins, 1, 8192)
    r_free = mi.mi_probe_shared_atomic_rate(local, cfg.nbins, 0, 8192)
    # dominant kernel: the z-lerp+histogram kernel (separable maps) or the generic resample+histogram
    # kernel, timed alone with CUDA events on the launching stream (mi_last_timing class 4); one step
    # launches it hist_launches times and together the launches do every evaluation of the step once
    separable = cfg.family in (0, 3, 4)
    hist_ms = kern_ms[4] / args.steps
    hist_launches = max(1, hist_launches // args.steps)
    achieved = evals_step / (hist_ms * 1e-3)                        # updates/s inside the kernel
    pass_bytes = cfg.fixed.size * 1 + cfg.moving.size * 4          # fixed bins + moving floats, read once
    t_hbm_b1 = cfg.n_transforms * pass_bytes / (hbm_gbs * 1e9)
    t_hbm_once = pass_bytes / (hbm_gbs * 1e9)
    t_atom = evals_step / r_rand
    sm_hz = (clocks["sm_mhz"] or sm_max_mhz) * 1e6
    t_lsu = 32.0 * evals_step / (148 * 128.0 * sm_hz)
    # measured DRAM bytes of one launch of the dominant kernel in this exact command; null for the
    # workloads that have no committed capture
    traffic = NCU_DRAM_BYTES_PER_LAUNCH.get((cfg.name, tuple(cfg.n), interp))
    roofline = {"bound": "alu",
                "kernel": ("zhist_kernel (separable path: z-lerp + joint histogram + fused entropy epilogue)" if separable
                           else "resample_hist_kernel (generic affine: 8 gathers + 7 lerps + joint histogram)"),
                "achieved": achieved / 1e9, "peak": r_rand / 1e9, "unit": "G shared-atomic updates/s",
                "frac": achieved / r_rand, "traffic": traffic,
                "all_a3_a4_kernels_ms_per_step": kern_ms[1] / args.steps,
                "peak_source": "mi_probe_shared_atomic_rate(pattern=uniform random bins) measured in this run",
                "peak_conflict_free": r_free / 1e9,
                "t_atom_ms": t_atom * 1e3, "t_hbm_resident_ms": t_hbm_once * 1e3,
                "t_hbm_if_every_transform_restreams_ms": t_hbm_b1 * 1e3,
                "t_lsu_gather_nominal_ms": None if separable else t_lsu * 1e3,
                "kernel_ms_per_step": hist_ms, "kernel_launches_per_step": hist_launches,
                "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": peak_src,
                "step_frac_of_t_roof": max(t_atom, t_hbm_once) / (total_ms / args.steps * 1e-3)}

    cpu_baseline = None
    if not args.no_cpu_baseline:
        cpu_baseline, _ = time_oracle(cfg, interp, 15.0)
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

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": workload_config(cfg, interp, {
                "l2": "flushed between timed steps (256 MiB write)", "parallelism": "replicas x%d" % world,
                "mi_evals_per_s": cfg.n_transforms * args.steps * world / (total_ms * 1e-3)}),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": e2e_steps, "ms_per_step": e2e_s / e2e_steps * 1e3, "mi_create_ms": create_ms},
            "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu_baseline,
            "kernel_ms_per_step": {"setup": kern_ms[0] / args.steps, "resample_hist": kern_ms[1] / args.steps,
                                   "entropy": kern_ms[2] / args.steps, "map": kern_ms[3] / args.steps,
                                   "dominant_hist_kernel": kern_ms[4] / args.steps},
            "capture_analysis": analysis, "wall_s_timed_region": wall}
    print(json.dumps(line))
    mi.mi_destroy(ctx)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
