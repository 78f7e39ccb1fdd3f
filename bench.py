#!/usr/bin/env python
"""bench.py — the driver's measurement contract for the DOCTORS hot path on B200.

One "step" = one whole `doctors_solve` of the workload: ray trace (a1) -> per group fixed source
(a2) -> source iteration {sweep of all 8 octants (a3-a5), convergence (a6)} for every source and
group, to the 1e-5 tolerance.  Default workload = BASELINE.json configs[4] (256x256x128, 47 groups,
P3, S8, 8 cone-beam sources batched in 2 chunks of 4) — the config the >= 50 % HBM-roofline target
is judged on.  Metric: cell*direction*group updates per second over the whole solve.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--impl reference]

N > 1 (torchrun): replicas only — the path does not shard; every rank solves the
same workload, the time is the max over ranks, value = N * updates / time.
`--impl reference` times the fp64 CPU oracle (as it stands) on a bounded sample of the workload.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

CONFIG_LABEL = {0: "cfg0_8c_S2P0", 1: "cfg1_32c_sphere_S8P3", 2: "cfg2_64c_cyl_S8P3", 3: "cfg3_128x128x64_S16P3",
                4: "cfg4_256x256x128_S8P3_8src"}
METRIC = "cell_direction_group_updates_per_s"
UNIT = "updates/s"
TRAFFIC_CSV = "r02_sweep_traffic.csv"
NOMINAL_HBM_GBS = 8000.0      # the ~8 TB/s BASELINE.json north_star quotes


def rank_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def measured_peak():
    """HBM GB/s denominator: MEASURED_PEAKS.json (driver-written), else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic_per_problem_sweep(idx):
    """DRAM bytes (read + write) one problem's share of a sweep launch moved under `ncu --set full`, from the committed
    summary profiles/r02_sweep_traffic.csv (columns: config, problems_in_launch, dram_read_bytes, dram_write_bytes, commit)."""
    try:
        with open(os.path.join(ROOT, "profiles", TRAFFIC_CSV)) as f:
            for ln in f:
                c = ln.strip().split(",")
                if len(c) >= 4 and c[0].strip() == str(idx):
                    return (float(c[2]) + float(c[3])) / float(c[1])
    except Exception:
        pass
    return None


def workload_for(idx, slice_=False):
    from workloads import make_config, single_sweep_case
    if slice_:
        # ncu slice (profiles/): full mesh and quadrature of the config, 2 sources, one mid-spectrum group,
        # 2 sweeps -> 2 launches of the sweep kernel with a workspace small enough for ncu's replay
        g = {0: 0, 1: 9, 2: 9, 3: 9, 4: 20}.get(idx, 45)
        return single_sweep_case(idx, groups=(g,), n_sources=2 if idx == 4 else 1, fixed_iters=2)
    if idx >= 5:
        # the paper's own workload shapes (Table 2) on synthetic cross sections:
        # 5 coarse single projection, 6 coarse CT (16 cone beams summed), 7 fine single, 8 fine CT
        from workloads import paper_shaped
        return paper_shaped(fine=idx >= 7, ct=idx in (6, 8))
    return make_config(idx)


def algorithmic_bytes_per_cell_octant(nm, batch):
    """per (cell, octant, problem) the sweep must read Q_lm (nm*4), read-modify-write
    phi_lm (2*nm*4) and read sigma_t (4 B shared by the `batch` problems swept together)."""
    return nm * 4 + 2 * nm * 4 + 4.0 / batch


# ---- clocks sampling during the timed region -----------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.tmp.flush()
        self.tmp.seek(0)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.tmp.read().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        try:
            os.unlink(self.tmp.name)
        except OSError:
            pass
        if sm:
            out["sm_mhz"] = float(np.median(sm))
            out["sm_max_mhz"] = float(max(mx))
            out["power_w_max"] = float(max(pw))
            out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


# ---- the oracle legs (cpu_baseline and --impl reference) -----------------------------------------
def oracle_sample(idx):
    """Bounded sample of config idx the oracle finishes in ~10-30 s: full mesh and quadrature,
    first source, highest-energy group, ray trace + a fixed number of sweeps."""
    from workloads import single_sweep_case, make_config
    if idx >= 5:
        from workloads import paper_shaped
        import copy
        wl = paper_shaped(fine=idx >= 7, ct=idx in (6, 8), G=90 if idx < 7 else 2)
        if idx >= 7:
            wl.fixed_iters = 2
        return wl, "%s: %s" % (wl.name, "all 90 groups to tolerance" if idx < 7 else "2 of 90 groups, 2 sweeps each")
    if idx <= 1:
        wl = make_config(idx)
        return wl, "%s: whole config (all groups, to tolerance)" % wl.name
    sweeps = {2: 8, 3: 2, 4: 1}[idx]
    wl = single_sweep_case(idx, groups=(0,), n_sources=1, fixed_iters=sweeps)
    return wl, "%s mesh/quadrature, source 0, group 0 only: ray trace + %d sweep(s) of all %d directions" % (
        wl.name, sweeps, wl.n_dir)


def time_oracle(wl, closure, one_thread=True):
    """The fp64 oracle as it stands on the host cores: sweeps timed apart from the ray trace and the fixed-source
    assembly (oracle.solve reports the split), all cores and — BASELINE.md §2, the paper's CPU configuration
     — one thread.  Returns the cpu_baseline object."""
    from oracle import oracle
    oracle.build()
    cores = oracle.default_threads()
    t0 = time.perf_counter()
    res = oracle.solve(wl, closure=closure, threads=cores)
    dt = time.perf_counter() - t0
    updates = int(res["iters"].sum()) * wl.cells * wl.n_dir
    sec = {k: float(v) for k, v in res["seconds"].items()}
    out = {"value": updates / sec["sweep"], "unit": UNIT, "cores": cores, "kind": "oracle",
           "what": "untuned fp64 oracle (test infrastructure), sweeps only; not a tuned CPU solver",
           "updates": updates, "seconds": dict(sec, total=dt), "value_incl_raytrace_and_source": updates / dt}
    if one_thread and cores > 1:
        import copy
        w1 = copy.copy(wl)
        w1.fixed_iters = 1                                   # one sweep per group of the same sample, on one thread
        r1 = oracle.solve(w1, closure=closure, threads=1, raytrace_threads=cores)
        u1 = int(r1["iters"].sum()) * wl.cells * wl.n_dir
        out["value_1thread"] = u1 / r1["seconds"]["sweep"]
        out["seconds_1thread_sweep"] = float(r1["seconds"]["sweep"])
    return out


def run_reference(args):
    rank, world, _ = rank_world()
    if rank != 0:
        return 0
    wl, sample = oracle_sample(args.config)
    steps = []
    for i in range(args.warmup + args.steps):
        c = time_oracle(wl, args.closure, one_thread=False)
        if i >= args.warmup:
            steps.append(c)
    updates = sum(c["updates"] for c in steps)
    sweep_s = sum(c["seconds"]["sweep"] for c in steps)
    total_s = sum(c["seconds"]["total"] for c in steps)
    v = updates / sweep_s
    cfg = bench_config(wl, args, None)                       # the workload that RAN: the bounded sample, named as such
    cfg["sample_of"] = CONFIG_LABEL.get(args.config, "config %d" % args.config)
    cfg["sample"] = sample
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total_s / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
            "ms_per_step_split": {k: 1e3 * sum(c["seconds"][k] for c in steps) / max(1, args.steps)
                                  for k in ("raytrace", "fixed_source", "sweep")},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": steps[-1]["cores"], "kind": "oracle", "sample": sample,
                             "what": steps[-1]["what"]},
            "e2e": {"value": updates / total_s, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def bench_config(wl, args, info):
    c = {"workload": wl.name, "mesh": [wl.nx, wl.ny, wl.nz], "groups": wl.G, "pl_order": wl.L, "sn": wl.sn,
         "n_dir": wl.n_dir, "sources": len(wl.sources), "tol": wl.tol, "closure": args.closure,
         "l2": "inputs larger than L2 (per-group working set > 126 MB)" if wl.cells * 33 * 4 * min(4, len(wl.sources)) > 126e6
               else "working set fits L2; an L2 flush (256 MiB write) runs between steps",
         "parallelism": "replicas only" if args.gpus > 1 else "1 GPU"}
    if info is not None:
        c.update({"source_chunks": info["n_chunks"], "brick": list(info["brick"]), "ctas_per_sm": info["ctas_per_sm"]})
    return c


# ---- N > 1: max over ranks ------------------------------------------------------------------------
def aggregate_over_ranks(ms_local, updates_local, dist=None):
    """Replicas only: time = max over ranks, updates = sum over ranks.  Works on any backend
    (tested with gloo, world_size 2)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return ms_local, updates_local
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([ms_local], dtype=torch.float64, device=dev)
    u = torch.tensor([float(updates_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), int(u.item())


def run_gpu_arm(args):
    import torch
    rank, world, local = rank_world()
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = local if world > 1 else 0
    torch.cuda.set_device(dev)
    from paper_1910_11335_b200 import build
    if rank == 0:
        build.build()
    if dist is not None:
        dist.barrier()
    import paper_1910_11335_b200 as pkg
    pkg.load_library()                       # raises if the CUDA library is missing: no fallback

    wl = workload_for(args.config, args.slice)
    nm = (wl.L + 1) ** 2
    p = pkg.problem_from_workload(wl, device=dev)
    kw = dict(tol=wl.tol, max_iters=wl.max_iters, closure=args.closure,
              fixed_iters=(wl.fixed_iters if wl.fixed_iters else None))
    if args.config == 4 and not args.slice:
        kw["source_chunk"] = 4               # 2 chunks of 4: all-group moments of 8 sources exceed HBM
    if args.projection:
        kw["projection"] = args.projection
    if args.brick:
        kw["brick"] = tuple(int(v) for v in args.brick.split(","))
    if args.ctas:
        kw["ctas_per_sm"] = args.ctas
    flush = None
    if wl.cells * 33 * 4 * min(4, len(wl.sources)) <= 126e6:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def step():
        if flush is not None:
            flush.fill_(1)
        return p.solve(**kw)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(dev) if rank == 0 else None
    ms_dev = ms_sweep = 0.0
    updates = launches = sweep_launches = timed_sweeps = 0
    t0 = time.perf_counter()
    info = None
    for _ in range(args.steps):
        info = step()
        ms_dev += info["ms_total"]; ms_sweep += info["ms_sweep"]
        updates += info["updates"]; launches += info["kernel_launches"]; sweep_launches += info["sweep_launches"]
        timed_sweeps += info["timed_sweeps"]
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    wall_ms = 1e3 * (time.perf_counter() - t0)
    clocks = sampler.stop() if sampler else None
    sweeps_local = int(info["iters"].sum())
    ms_all, upd_all = aggregate_over_ranks(ms_dev, updates, dist)

    # ---- e2e: host buffers in, host buffers out, through the public API, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = torch.empty(wl.cells, dtype=torch.float32).pin_memory()
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        p.set_mesh_materials(wl.material, wl.density, (wl.dx, wl.dy, wl.dz), wl.n_materials)
        p.set_xs(wl.sigma_t, wl.sigma_s)
        p.set_quadrature(wl.sn)
        p.set_source(wl.sources, wl.mode)
        inf2 = p.solve(**kw)
        nprob = p.n_problems()
        for q in range(nprob):
            for g in range(wl.G):
                p.get_flux_moments_into(q, g, 0, pin.data_ptr())
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        e2e_ms, e2e_upd = aggregate_over_ranks(1e3 * e2e_s, inf2["updates"], dist)
        h2d = wl.material.nbytes + wl.density.nbytes + wl.sigma_t.nbytes + wl.sigma_s.nbytes // 2 + 4096
        h2d += sum(s.volume.nbytes for s in wl.sources if s.volume is not None)
        e2e = {"value": e2e_upd / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(nprob * wl.G * wl.cells * 4), "steps": 1,
               "what": "set_* from host arrays + doctors_solve + every (problem, group) scalar flux read to pinned host memory"}
    if rank != 0:
        p.close()
        if dist is not None:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (k_sweep_brick) ----
    peak, peak_src = measured_peak()
    batch = min(4, len(wl.sources)) if wl.mode == 0 else 1
    if args.slice:
        args.no_cpu = True
    bytes_per = algorithmic_bytes_per_cell_octant(nm, batch)
    problem_sweeps = updates / (wl.cells * wl.n_dir)               # sum of K[s][g] over the timed steps
    alg_bytes = problem_sweeps * wl.cells * 8 * bytes_per
    achieved = alg_bytes / (ms_sweep * 1e-3) / 1e9
    traffic = args.traffic
    if traffic is None:
        per = ncu_traffic_per_problem_sweep(args.config)          # one ncu capture, scaled to this run's problems per launch
        if per is not None:
            traffic = per * problem_sweeps / max(1, sweep_launches)
    roofline = {"bound": "hbm", "kernel": "k_sweep_brick", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "peak_source": peak_src, "frac_of_nominal_8tbs": achieved / NOMINAL_HBM_GBS,
                "traffic": traffic, "traffic_unit": "DRAM bytes per launch (one ncu --set full capture of this kernel on the config's "
                "2-problem slice, profiles/%s, scaled to this run's problems per launch)" % TRAFFIC_CSV,
                "timed_sweeps": int(timed_sweeps),
                "launches": int(sweep_launches), "avg_launch_ms": ms_sweep / max(1, sweep_launches),
                "algorithmic_bytes_per_launch": alg_bytes / max(1, sweep_launches),
                "share_of_step": ms_sweep / ms_dev,
                "bytes_per_update": 8 * bytes_per * wl.cells / (wl.cells * wl.n_dir)}

    # ---- oracle beside it (bounded sample), rank 0, N = 1 only ----
    cpu = None
    if world == 1 and not args.no_cpu:
        swl, sample = oracle_sample(args.config)
        cpu = time_oracle(swl, args.closure)
        cpu["sample"] = sample

    value = upd_all / (ms_all * 1e-3)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_all / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": bench_config(wl, args, info),
            "solve_ms": {"total": ms_dev / args.steps, "sweep": ms_sweep / args.steps,
                         "raytrace": info["ms_raytrace"], "fixed_source": info["ms_fixed_source"],
                         "iterate": info["ms_iterate"], "wall_incl_upload": wall_ms / args.steps},
            "sweeps_per_step": sweeps_local, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": int(launches), "clocks": clocks}
    print(json.dumps(line), flush=True)
    p.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs index 0..4 (default 4, the largest); 5..8 = the paper's own workload shapes (coarse/fine x single/CT)")
    ap.add_argument("--closure", type=int, default=1, help="0 pure diamond difference, 1 + set-to-zero fix-up (R2)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--slice", action="store_true", help="profiling slice of the config (see workload_for); not a bench number")
    ap.add_argument("--projection", type=int, default=0, help="doctors_solve_opts.projection (experiments; 0 = the library's default)")
    ap.add_argument("--brick", default="", help="bx,by,bz brick extents (experiments; default automatic)")
    ap.add_argument("--ctas", type=int, default=0, help="persistent CTAs per SM (experiments; default occupancy maximum)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--traffic", type=float, default=None,
                    help="ncu dram bytes per sweep launch (from profiles/), echoed into roofline.traffic")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu_arm(args)


if __name__ == "__main__":
    sys.exit(main())
