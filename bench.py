#!/usr/bin/env python
"""bench.py -- zone-updates/s per RK substep of the GRMHD hot path on B200 (contract: see
DESIGN.md "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--n SIZE]
                  [--impl reference] [--no-cpu-baseline]

A "step" is one full RK step (all stages: every A1-A8 row of the hot path) of one block.
N > 1 (torchrun): independent replicas, one block per rank, no data-path collective
("replicas only"); value = zone-substeps of all ranks / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 GRMHD zone-updates/s per RK substep"
UNIT = "zone-updates/s"
# algorithmic bytes per cell and direction of the flux kernel:
# reads P(5)+B_c(3)+B~^d(1)+alpha,beta,gamma(10) = 19 doubles, writes 7
FLUX_BYTES_PER_CELL_DIR = 26 * 8


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2,
                    help="index into BASELINE.json configs (0..4); default 2 = 256^3 Kerr-Schild")
    ap.add_argument("--n", type=int, default=None, help="override the linear size")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-n", type=int, default=48)
    ap.add_argument("--set", action="append", default=[], metavar="KEY=VALUE",
                    help="grmhd_set_option before the run, e.g. --set emf=1 (upwind CT), "
                         "--set gauge=1 (Lorenz gauge), --set c2p_backup=1")
    ap.add_argument("--no-point-kernels", action="store_true",
                    help="skip the FP64 peak and config-4b con2prim measurements")
    ap.add_argument("--point-kernels-only", action="store_true",
                    help="run only the FP64 peak and config-4b con2prim kernels (SURVEY 8(d): the "
                         "target of the ncu FP64-pipe capture) and print their JSON")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def kernel_source_hash():
    """sha256 over the CUDA sources the library was built from (sorted by name): ties a committed
    ncu capture to the kernels this run executes (the GPU box has no .git to ask)."""
    import hashlib
    d = os.path.join(ROOT, "paper_2406_11669_b200", "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def traffic_for(workload_name, options):
    """DRAM bytes per flux launch (dram__bytes_read.sum + dram__bytes_write.sum of one
    `ncu --set full` capture, profiles/traffic.json) -- only if that capture was taken on THESE
    kernel sources, this workload and these options; otherwise null: a stale number is not
    printed beside live ones."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(p):
        return None, {"traffic_source": None}
    t = json.load(open(p))
    meta = {"traffic_source": t.get("_source"), "traffic_source_commit": t.get("_commit"),
            "traffic_source_kernel_hash": t.get("_kernel_hash")}
    same = (t.get("_kernel_hash") == kernel_source_hash() and not options
            and workload_name in t)
    if not same:
        meta["traffic_note"] = "capture does not match this run (kernel sources, workload or options): not reported"
        return None, meta
    meta["fp64_pipe_active_pct_ncu"] = t.get("_fp64_pipe_active_pct")
    return t[workload_name], meta


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.p = None
        try:
            self.p = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def make_workload(args):
    from paper_2406_11669_b200 import workloads as wl
    return wl.make(args.config, args.n)


def oracle_throughput(w_small, steps, threads):
    """zone-substeps/s of the oracle, as it stands, on `threads` host cores."""
    from oracle import ref
    ref.set_num_threads(threads)
    r = ref.RefSolver(w_small.nx, w_small.ny, w_small.nz, w_small.dx,
                      ref.make_opts(**w_small.opts))
    r.set_metric(w_small.metric)
    r.set_prims(w_small.prims)
    if w_small.vecpot is not None:
        r.set_vecpot(w_small.vecpot)
    if w_small.mask is not None:
        r.set_mask(w_small.mask)
    t0 = time.perf_counter()
    r.step(steps, w_small.cfl)
    dt = time.perf_counter() - t0
    return w_small.ncells * w_small.stages * steps / dt, dt


def sample_workload(args):
    """The bounded CPU sample: the same generator at a reduced linear size."""
    from paper_2406_11669_b200 import workloads as wl
    if args.config == 0:
        return wl.make(0, None), "full config (256x4x4)"
    n = args.cpu_sample_n
    return wl.make(args.config, n), f"same generator at {n}^3"


def cpu_baseline(args, target_s=10.0, target_1core_s=8.0):
    """The oracle as it stands on all host cores and, beside it, on ONE core."""
    ws, what = sample_workload(args)
    cores = os.cpu_count() or 1
    v1, t1 = oracle_throughput(ws, 1, cores)
    steps = int(max(1, min(200, target_s / max(t1, 1e-3))))
    v, t = oracle_throughput(ws, steps, cores)
    _, s1 = oracle_throughput(ws, 1, 1)
    steps1 = int(max(1, min(50, target_1core_s / max(s1, 1e-3))))
    vs, ts = oracle_throughput(ws, steps1, 1)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{what}, {steps} RK{ws.stages} steps, {t:.1f} s wall, OpenMP {cores} threads",
            "one_core": {"value": vs, "unit": UNIT, "cores": 1,
                         "sample": f"{what}, {steps1} RK{ws.stages} steps, {ts:.1f} s wall"}}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    ws, what = sample_workload(args)
    wfull = None
    cores = os.cpu_count() or 1
    for _ in range(max(args.warmup, 0)):
        oracle_throughput(ws, 1, cores)
    t0 = time.perf_counter()
    tot = 0.0
    for _ in range(args.steps):
        _, dt = oracle_throughput(ws, 1, cores)
        tot += dt
    wall = time.perf_counter() - t0
    value = ws.ncells * ws.stages * args.steps / tot
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": config_name(args), "sample": what, "stages": ws.stages,
                       "cells_per_step": ws.ncells},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"{what}; each step = one RK{ws.stages} step of the "
                                       f"oracle, OpenMP {cores} threads; wall {wall:.1f} s"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def config_name(args):
    names = ["config1_balsara1_256x4x4", "config2_blast_128", "config3_kerrschild_256",
             "config4_c2p_stress_256", "config5_bns_512"]
    if args.n is None:
        return names[args.config]
    return names[args.config].rsplit("_", 1)[0] + "_%d" % args.n


ALG_BYTES = {  # algorithmic bytes per interior cell and launch
    "flux_x": FLUX_BYTES_PER_CELL_DIR, "flux_y": FLUX_BYTES_PER_CELL_DIR,
    "flux_z": FLUX_BYTES_PER_CELL_DIR,
    # update: fluxes 15 + 6, sources 4, Y 8, Y0 8 read; Y 8 written
    "update": (21 + 4 + 8 + 8 + 8) * 8,
    # fused post-update kernel (curl A, con2prim, max speed): A 3, B~0 3, alpha/beta/gamma 10,
    # U~ 5 read; B~ 3, B_c 3, P 5 written
    "con2prim": (3 + 3 + 10 + 5 + 3 + 3 + 5) * 8,
    # sources: P 5, B_c 3, metric 16 read; 4 written
    "sources": (5 + 3 + 16 + 4) * 8,
}


def max_over_ranks(ms, world, device):
    """Device time of the job = max over the ranks' own times (one block per rank, no data-path
    collective: "replicas only").  Works on any backend (nccl on the GPUs, gloo in the CPU test)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(ncells, stages, steps, world, ms):
    """zone-updates/s per RK substep of all replicas together."""
    return world * ncells * stages * steps / (ms * 1e-3)


def point_kernels(binding, torch, n=1 << 22):
    """FP64 pipe peak (dependent-free DFMA loop) and 'config 4b': the two con2prim
    schemes alone on n iid states with the config-4 marginals, device resident."""
    from paper_2406_11669_b200 import workloads as wl
    out = {"fp64_peak_tflops_measured": binding.dfma_peak()}
    prim, met = wl.c2p_states(n)
    o = binding.make_opts(gamma_ad=5.0 / 3.0, rho_atm=1e-10, p_floor=1e-10, w_max=100.0)
    P, M = torch.from_numpy(prim).cuda(), torch.from_numpy(met).cuda()
    U = binding.prim2con_batch(P, M, o)
    for name, fn in (("con2prim_2d", binding.con2prim_batch), ("con2prim_1d", binding.con2prim1d_batch)):
        for _ in range(3):   # warm-up (first calls also grow torch's allocator pool)
            fn(U, M, o)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(5):
            _, st, it = fn(U, M, o)
        e1.record()
        e1.synchronize()
        ms = e0.elapsed_time(e1) / 5
        out[name] = {"states": n, "ms": ms, "states_per_s": n / (ms * 1e-3),
                     "mean_iterations": float(it.double().mean()), "failed": int((st & 2).ne(0).sum())}
    return out


def run_b200(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2406_11669_b200 import binding

    w = make_workload(args)
    opts = binding.make_opts(**w.opts)
    dev = f"cuda:{local}"
    s = binding.Solver(w.nx, w.ny, w.nz, w.dx, opts, device=dev)
    pin = lambda a: None if a is None else torch.from_numpy(a).pin_memory()
    h_prims = [pin(a) for a in w.prims]
    h_vec = None if w.vecpot is None else [pin(a) for a in w.vecpot]
    s.set_metric(w.metric)
    if w.mask is not None:
        s.set_mask(w.mask)
    options = {}
    for kv in args.set:
        key, val = kv.split("=", 1)
        s.set_option(key, float(val))
        options[key] = float(val)

    def reset():
        s.set_prims(h_prims)
        if h_vec is not None:
            s.set_vecpot(h_vec)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput -------------------------------------------------
    reset()
    for _ in range(args.warmup):
        s.step(1, w.cfl)
    s.set_option("kernel_timing", 1)
    stream = s.stream
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = s.launch_count()
    e0.record(stream)
    s.step(args.steps, w.cfl)
    e1.record(stream)
    barrier()
    clocks = sampler.stop() if sampler else None
    ms = e0.elapsed_time(e1)
    launches = s.launch_count() - l0
    kt = s.kernel_times()
    s.set_option("kernel_timing", 0)
    # the same K steps without the per-kernel event brackets: one cudaGraphLaunch per step
    # (the library captures the step once; the brackets above force the eager path)
    s.step(2, w.cfl)   # eager step + capture
    barrier()
    e0.record(stream)
    s.step(args.steps, w.cfl)
    e1.record(stream)
    barrier()
    ms_graph = max_over_ranks(e0.elapsed_time(e1), world, dev)
    st = s.stats()
    ms = max_over_ranks(ms, world, dev)
    zone_sub = w.ncells * w.stages * args.steps
    value = whole_job_value(w.ncells, w.stages, args.steps, world, ms)

    # ---- end to end through the C ABI with host buffers --------------------------------
    k_e2e = max(1, min(args.steps, 5))
    out_host = [torch.empty(s.cc_shape, dtype=torch.float64).pin_memory() for _ in range(8)]
    reset(); s.step(1, w.cfl); s.get_cons(out=out_host)   # warm-up of the e2e path
    barrier()
    t0 = time.perf_counter()
    e0.record(stream)
    for _ in range(k_e2e):
        reset()
        s.step(1, w.cfl)
        s.get_cons(out=out_host)
    e1.record(stream)
    barrier()
    wall_e2e = time.perf_counter() - t0
    ms_e2e = max(e0.elapsed_time(e1), 0.0)
    ms_e2e = max_over_ranks(ms_e2e, world, dev)
    h2d = sum(a.numel() * 8 for a in h_prims if a is not None) + \
        (sum(a.numel() * 8 for a in h_vec) if h_vec else 0)
    d2h = sum(a.numel() * 8 for a in out_host)
    e2e = {"value": world * w.ncells * w.stages * k_e2e / (ms_e2e * 1e-3), "unit": UNIT,
           "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": k_e2e,
           "ms_per_step": ms_e2e / k_e2e,
           "call": "set_prims[+set_vecpot](pinned host) -> step(1) -> get_cons(pinned host)"}
    s.close()
    point = None
    if rank == 0 and not args.no_point_kernels:
        point = point_kernels(binding, torch)
    if world > 1:
        dist.destroy_process_group()
    if rank != 0:
        return

    # ---- roofline of the dominant kernel --------------------------------------------------
    peak, peak_src = peaks()
    kernels = {}
    tot_k = sum(v[0] for v in kt.values()) or 1.0
    for k, (kms, cnt) in kt.items():
        if cnt == 0:
            continue
        avg = kms / cnt
        ent = {"ms_avg": avg, "launches": cnt, "share": kms / tot_k}
        if k in ALG_BYTES:
            nd = 3 if (k == "flux_x" and kt["flux_y"][1] == 0) else 1
            ent["alg_GBps"] = nd * ALG_BYTES[k] * w.ncells / (avg * 1e-3) / 1e9
        kernels[k] = ent
    flux_ms = sum(kt[k][0] for k in ("flux_x", "flux_y", "flux_z"))
    flux_n = sum(kt[k][1] for k in ("flux_x", "flux_y", "flux_z")) or 1
    flux_avg = flux_ms / flux_n
    # launch-bound small blocks run x, y and z in one launch (k_flux_all), booked under flux_x
    dirs_per_launch = 3 if kt["flux_y"][1] == 0 and kt["flux_x"][1] > 0 else 1
    achieved = dirs_per_launch * FLUX_BYTES_PER_CELL_DIR * w.ncells / (flux_avg * 1e-3) / 1e9
    traffic, traffic_meta = traffic_for(w.name, options)
    roofline = {"kernel": "flux (reconstruct + Riemann, average of x/y/z launches)",
                "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic,
                "alg_bytes_per_launch": dirs_per_launch * FLUX_BYTES_PER_CELL_DIR * w.ncells,
                "directions_per_launch": dirs_per_launch,
                "alg_bytes_note": "208 B per cell-direction = the method's own bytes (SURVEY 8(d): "
                                  "19 doubles read, 7 written); the kernel reads one more double, "
                                  "the precomputed sqrt(gamma) of the face (216 B)",
                "ms_per_launch": flux_avg, "share_of_step": flux_ms / tot_k,
                "peak_source": peak_src,
                "step_decomposed_frac": (1400.0 * zone_sub / (ms * 1e-3) / 1e9) / peak,
                "step_floor_frac": (344.0 * zone_sub / (ms * 1e-3) / 1e9) / peak}
    roofline.update(traffic_meta)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "cells": [w.nx, w.ny, w.nz], "ghosts": 3,
                       "stages_per_step": w.stages, "recon": "ppm" if w.opts["recon"] else "minmod",
                       "riemann": "lxf" if w.opts.get("riemann") else "hlle", "cfl": w.cfl, "parallelism": "replicas" if world > 1 else "1gpu",
                       "l2": "inputs larger than L2 (every kernel streams > 126 MB)"
                             if w.ncells >= 128 ** 3 else "working set fits L2 (latency-bound config)",
                       "us_per_substep": 1e3 * ms / (args.steps * w.stages)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "options": options,
            "cuda_graph": {"ms_per_step": ms_graph / args.steps,
                           "value": whole_job_value(w.ncells, w.stages, args.steps, world, ms_graph),
                           "unit": UNIT,
                           "note": "same K steps, kernel_timing off: one cudaGraphLaunch per step"},
            "point_kernels": point,
            "roofline": roofline, "kernels": kernels,
            "stats": {k: st[k] for k in ("t", "dt", "c2p_fail", "p_fix", "atmo", "w_cap",
                                         "c2p_maxiter")}}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args)
    print(json.dumps(line))


def main():
    args = parse()
    if args.point_kernels_only:
        import torch
        from paper_2406_11669_b200 import binding
        assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
        print(json.dumps({"point_kernels": point_kernels(binding, torch)}))
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
