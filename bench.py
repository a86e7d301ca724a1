#!/usr/bin/env python
"""bench.py -- throughput of the full coupled step (MLUPS, fp64) on B200, with roofline and CPU-oracle baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload config4] [--precision 64] [--impl ours|reference]

A "step" is one pass of the whole hot path (K_phi + K_main: H1..H7 of DESIGN.md) over the whole grid.  The default
workload is BASELINE.json configs[3], the 3D film-boiling grid 256x256x512 (D3Q19 + D3Q7 + D3Q7, fp64) on which
north_star states the roofline target.  Prints ONE JSON line (rank 0).  N > 1: N independent replicas, one process
per GPU (launched by torchrun), no data-path collective ("replicas only").
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
sys.path.insert(0, ROOT)

from paper_2003_06342_b200 import replicas, workloads as wl  # noqa: E402

METRIC = "MLUPS (full coupled step, fp64)"
FALLBACK_HBM_GBS = 6650.0   # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def make_workload(name: str, seed_offset: int = 0):
    if name == "config4":
        return wl.config4_film3d(seed=4 + seed_offset)
    if name == "config4_q15":        # same grid and recipe with the paper's D3Q15 Navier-Stokes lattice
        return wl.config4_film3d(seed=4 + seed_offset, lat_f="D3Q15")
    if name == "config4_sample":     # bounded sample of config 4 for the CPU oracle: same recipe, a 256x256x128 slab
        return wl.config4_film3d(nx=256, ny=256, nz=128, seed=4 + seed_offset)
    if name == "config4_small":      # the reference arm's per-step sample (128^3)
        return wl.config4_film3d(nx=128, ny=128, nz=128, seed=4 + seed_offset)
    if name == "config3":
        return wl.config3_film2d(seed=3 + seed_offset)
    if name.startswith("config3_"):   # e.g. config3_1024x1024, config3_4096x3072: the paper's film-boiling grids
        nx, ny = (int(v) for v in name.split("_")[1].split("x"))
        over = {"lat_s": "D2Q9"} if "_q9" in name else {}   # _q9: three D2Q9 lattices as in the paper
        if name.endswith("_mm"):                             # _mm: 16-mode interface of the paper's 8-GPU run, Eq.(44)
            over.update(modes=16, amp=1.0)
        return wl.config3_film2d(nx=nx, ny=ny, seed=3 + seed_offset, **over)
    if name.startswith("config5_"):
        return wl.config5_droplets(n=int(name.split("_")[1]), seed=5 + seed_offset)
    if name == "paper_film_1024":     # the paper's own film-boiling run, Table 2 in physical units
        return wl.paper_film_boiling()
    if name == "paper_film_4096x3072":   # its 8-GPU run
        return wl.paper_film_boiling(nx=4096, ny=3072, modes=16, y1=0.004)
    if name == "config1":
        return wl.config1_droplet(seed=1 + seed_offset)
    raise SystemExit("unknown workload %r" % name)


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], [], set()
        for t, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                clk, mx = float(f[1]), float(f[2])
            except ValueError:
                continue
            smax.append(mx)
            if t0 - 0.05 <= t <= t1 + 0.05:
                sm.append(clk)
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        if not sm:   # region shorter than one sample: take the nearest samples
            sm = [float(x[1].split(",")[1]) for x in self.rows[-3:] if len(x[1].split(",")) > 2]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload: str, precision: int):
    """DRAM bytes per K_main launch from the committed ncu --set full capture, if there is one for this workload."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as fh:
            return json.load(fh).get("%s_fp%d" % (workload, precision))
    except Exception:
        return None


def oracle_throughput(name: str, steps: int, warmup: int):
    """Time the CPU oracle, as it stands, on the host cores (bounded sample).  Returns (MLUPS, cores, description)."""
    import oracle
    P, I = make_workload(name)
    o = oracle.Oracle(P)
    o.init(I["phi"], I["T"])
    o.step(warmup)
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    n = P["nx"] * P["ny"] * P["nz"]
    o.close()
    return n * steps / dt / 1e6, oracle.num_threads(), "%s: %d steps of %dx%dx%d" % (I["name"], steps, P["nx"], P["ny"], P["nz"]), dt / steps * 1e3


def run_reference(args):
    """--impl reference: the oracle (unmodified) on the host cores, on a bounded sample of the same workload."""
    rank, _, world = replicas.env_rank()
    if rank != 0:
        return 0
    sample = "config4_small" if args.workload == "config4" else args.workload
    mlups, cores, desc, ms = oracle_throughput(sample, args.steps, args.warmup)
    P, _ = (wl.config4_film3d(nx=8, ny=8, nz=8) if args.workload == "config4" else make_workload(args.workload))
    line = {
        "impl": "reference", "metric": METRIC, "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "sample": desc, "lattices": [P["lat_f"], P["lat_g"], P["lat_s"]]},
        "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    from paper_2003_06342_b200 import binding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path (use --impl reference for the oracle)")
    rank, local_rank, world = replicas.init_process_group("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    prec = args.precision
    np_dt = np.float64 if prec == 64 else np.float32
    t_dt = torch.float64 if prec == 64 else torch.float32

    P, I = make_workload(args.workload, seed_offset=1000 * rank)
    nz, ny, nx = P["nz"], P["ny"], P["nx"]
    N = nx * ny * nz
    K, W = args.steps, args.warmup

    # host buffers in pinned memory (e2e leg) -- inputs phi, T; outputs phi, u, p, T
    h_phi = torch.empty((nz, ny, nx), dtype=t_dt).pin_memory()
    h_T = torch.empty((nz, ny, nx), dtype=t_dt).pin_memory()
    h_phi.numpy()[...] = I["phi"].astype(np_dt)
    h_T.numpy()[...] = I["T"].astype(np_dt)
    outs = (torch.empty((nz, ny, nx), dtype=t_dt).pin_memory(), torch.empty((3, nz, ny, nx), dtype=t_dt).pin_memory(),
            torch.empty((nz, ny, nx), dtype=t_dt).pin_memory(), torch.empty((nz, ny, nx), dtype=t_dt).pin_memory())
    del I

    sim = binding.LBM(P, prec)
    sim.init(h_phi, h_T)                      # inputs resident in HBM from here on
    sim.step(W)
    sim.sync()

    # ---- device-resident leg: K steps, CUDA events on the launching stream, clocks sampled during the region
    sampler = ClockSampler(local_rank) if rank == 0 else None
    time.sleep(0.25 if sampler else 0.0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = sim.launch_count
    # per-kernel CUDA events inside lbm_step: on large grids they ride in the timed region itself; small (launch-bound) grids
    # replay their steps from a CUDA graph, which per-kernel events would switch off, so those get a second pass for them
    events_inside = N > (1 << 21)
    sim.set_timing(events_inside)
    replicas.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e0.record(sim.stream)
    sim.step(K)
    e1.record(sim.stream)
    torch.cuda.synchronize()
    replicas.barrier()
    t1 = time.perf_counter()
    ms_local = e0.elapsed_time(e1)
    launches = sim.launch_count - launches0
    if not events_inside:
        sim.set_timing(True)
        sim.step(K)
    ms_phi, ms_main, nsteps_timed = sim.kernel_times()
    sim.set_timing(False)
    clocks = sampler.stop(t0, t1) if sampler else None
    ms_job, lu_job = replicas.reduce_job(ms_local, float(N) * K, dev)
    value = replicas.job_throughput_mlups(ms_job, lu_job)

    # ---- end-to-end leg through the public API with HOST buffers: init (H2D) + K steps + read_macro (D2H)
    es = 8 if prec == 64 else 4
    h2d, d2h = 2 * N * es, 6 * N * es
    replicas.barrier()
    torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(sim.stream)
    sim.init(h_phi, h_T)
    sim.step(K)
    sim.read_macro(out=outs)
    f1.record(sim.stream)
    torch.cuda.synchronize()
    ms_e2e, lu_e2e = replicas.reduce_job(f0.elapsed_time(f1), float(N) * K, dev)
    e2e_value = replicas.job_throughput_mlups(ms_e2e, lu_e2e)
    # the same with the host copies around EVERY step (what a per-step host round trip would cost): 3 iterations
    s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    s0.record(sim.stream)
    for _ in range(3):
        sim.init(h_phi, h_T)
        sim.step(1)
        sim.read_macro(out=outs)
    s1.record(sim.stream)
    torch.cuda.synchronize()
    ms_strict, lu_strict = replicas.reduce_job(s0.elapsed_time(s1), float(N) * 3, dev)
    e2e_strict = replicas.job_throughput_mlups(ms_strict, lu_strict)
    finite = bool(torch.isfinite(outs[0]).all() and torch.isfinite(outs[3]).all())

    if rank != 0:
        return 0

    # ---- roofline of the dominant kernel (K_main), algorithmic bytes / live CUDA-event duration
    q = {"D2Q5": 5, "D2Q9": 9, "D3Q7": 7, "D3Q19": 19, "D3Q15": 15}
    Q = q[P["lat_f"]] + q[P["lat_g"]] + q[P["lat_s"]]
    main_vals = (Q + 3) + (Q + 1)                    # reads: pops, phi^{n+1}, phi^n, Pdot; writes: pops, Pdot
    phi_vals = q[P["lat_g"]] + 1                    # reads: g; write: phi (dt/2 Pdot rides in the stored rest population)
    main_bytes = (main_vals * es + 2 * (8 - es)) * N    # the two phi values are doubles in both precisions
    main_ms = ms_main / max(nsteps_timed, 1)
    phi_ms = ms_phi / max(nsteps_timed, 1)
    peak, peak_src = measured_peak()
    achieved = main_bytes / (main_ms * 1e-3) / 1e9
    step_bytes = wl.bytes_per_lu(P, es) * N
    roofline = {
        "bound": "hbm", "kernel": "k_main", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
        "peak_source": peak_src, "traffic": ncu_traffic(args.workload, prec),
        "algorithmic_bytes_per_launch": main_bytes, "ms_per_launch": main_ms,
        "k_phi": {"ms_per_launch": phi_ms, "achieved": (phi_vals * es + (8 - es)) * N / (phi_ms * 1e-3) / 1e9 if phi_ms > 0 else None},
        "step": {"bytes_per_lu": wl.bytes_per_lu(P, es), "achieved": step_bytes / (ms_job / K * 1e-3) / 1e9,
                 "frac_of_peak": step_bytes / (ms_job / K * 1e-3) / 1e9 / peak,
                 "frac_of_8TBs": step_bytes / (ms_job / K * 1e-3) / 1e9 / 8000.0},
        "k_main_share_of_step": ms_main / max(ms_main + ms_phi, 1e-30),
    }

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        sample = "config4_sample" if args.workload == "config4" else ("config5_128" if args.workload.startswith("config5") else args.workload)
        steps_cpu = 16 if sample == "config4_sample" else (6 if sample != "config3" else 20)   # about 10-30 s of CPU work
        mlups, cores, desc, _ = oracle_throughput(sample, steps_cpu, 1)
        cpu = {"value": mlups, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": desc}

    line = {
        "metric": METRIC if prec == 64 else "MLUPS (full coupled step, fp32)", "value": value, "unit": "MLUPS",
        "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_job / K, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if prec == 64 else "f32", "data": "synthetic",
        "config": {"workload": args.workload, "grid": [nx, ny, nz], "lattices": [P["lat_f"], P["lat_g"], P["lat_s"]],
                   "parallelism": "replicas x%d" % world, "variant": sim.variant,
                   "l2": "state (%.2f GB) is larger than the 126 MB L2; no flush needed" % (sim.workspace_bytes / 1e9)
                   if sim.workspace_bytes > 4 * 126e6 else
                   ("state (%.0f MB) is not far above the 126 MB L2: partly L2-resident, no flush" % (sim.workspace_bytes / 1e6)
                    if sim.workspace_bytes > 126e6 else "state fits L2: numbers are L2-resident"),
                   "finite": finite},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "MLUPS", "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
                "region": "lbm_init(host phi,T) + lbm_step(%d) + lbm_read_macro(host phi,u,p,T), pinned host buffers" % K,
                "ms": ms_e2e,
                "per_step_io": {"value": e2e_strict, "unit": "MLUPS", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                                "region": "3 x [lbm_init(host) + lbm_step(1) + lbm_read_macro(host)]"}},
        "gpu_launches": launches,
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    return 0


def run_slabs(args):
    """Slab decomposition of the workload along its slowest axis (paper's multi-GPU mode).

    --slabs N (one process, one GPU): the N slabs run one after the other on one stream -- measures what the
    decomposition costs (ghost layers, pack/unpack launches, shorter launches), not a speed-up.
    --parallelism slabs under torchrun: one slab per rank, WEAK scaling (config 4 stacked N times along z), ghost layers
    exchanged with NCCL point-to-point calls between the two phases of every step."""
    import torch
    from paper_2003_06342_b200 import slabs

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path")
    rank, local_rank, world = replicas.init_process_group("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    K, W, prec = args.steps, args.warmup, args.precision
    if args.parallelism == "slabs":
        if not args.workload.startswith("config4"):
            raise SystemExit("bench.py: --parallelism slabs is defined for config4 (stacked along z)")
        P, _ = wl.config4_film3d(16, 16, 16)                      # parameters only
        P.update(nx=256, ny=256, nz=512 * world)
        sim = slabs.DistSlab(P, rank, world, prec, overlap=not args.no_overlap, transport=args.transport)
        z0, z1 = sim.slab.layer_range()
        _, I = wl.config4_film3d(256, 256, 512 * world, zrange=(z0, z1))
        sim.init(I["phi"], I["T"], local=True)
        n_slabs, mode = world, "slabs x%d (one per rank, %s ghost exchange)" % (world, "NCCL p2p" if args.transport == "p2p" else "peer-memory push")
        owned = sim.slab.P["slab"]["count"] * 256 * 256
        scaling = "weak"
    elif args.parallelism == "slabs-strong":
        # the paper's decomposed runs: ONE domain cut into one slab per rank along its slowest axis,
        # e.g. --workload config3_1024x1024_q9 on 4 ranks (4 x 1024x256), config3_4096x3072_q9_mm on 8
        P, I = make_workload(args.workload)
        sim = slabs.DistSlab(P, rank, world, prec, overlap=not args.no_overlap, transport=args.transport)
        sim.init(I["phi"], I["T"])
        n_slabs, mode = world, "one domain cut into %d slabs (one per rank, %s ghost exchange)" % (world, "NCCL p2p" if args.transport == "p2p" else "peer-memory push")
        owned = sim.slab.P["slab"]["count"] * (P["nx"] * P["ny"] if P["nz"] > 1 else P["nx"])
        scaling = "strong"
    else:
        P, I = make_workload(args.workload)
        sim = slabs.SlabGroup(P, args.slabs, prec, overlap=not args.no_overlap)
        sim.init(I["phi"], I["T"])
        n_slabs, mode = args.slabs, "slabs x%d in one process on one GPU" % args.slabs
        owned = P["nx"] * P["ny"] * P["nz"]
        scaling = "weak"
    del I
    sim.step(W)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    replicas.barrier()
    torch.cuda.synchronize()
    e0.record(sim.stream)
    sim.step(K)
    e1.record(sim.stream)          # the compute stream: every step ends there, after the last exchange has been waited for
    torch.cuda.synchronize()
    replicas.barrier()
    ms_job, lu_job = replicas.reduce_job(e0.elapsed_time(e1), float(owned) * K, dev)
    phi = sim.read_macro()[0]
    finite = bool(np.isfinite(phi).all())
    if rank == 0:
        print(json.dumps({
            "metric": METRIC if prec == 64 else "MLUPS (full coupled step, fp32)",
            "value": replicas.job_throughput_mlups(ms_job, lu_job), "unit": "MLUPS", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_job / K, "higher_is_better": True, "scaling": scaling, "vs_baseline": None,
            "dtype": "f64" if prec == 64 else "f32", "data": "synthetic",
            "config": {"workload": args.workload, "grid": [P["nx"], P["ny"], P["nz"]], "parallelism": mode,
                       "slabs": n_slabs, "finite": finite,
                       "schedule": "plain (one stream)" if args.no_overlap else "boundary layers first, exchange on a second stream"}}))
    sim.destroy()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="config4")
    ap.add_argument("--precision", type=int, default=64, choices=(32, 64))
    ap.add_argument("--impl", default="ours", choices=("ours", "reference"))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--parallelism", default="replicas", choices=("replicas", "slabs", "slabs-strong"),
                    help="N > 1: independent replicas (default, the bench contract), one slab of a stacked domain per rank (weak), "
                         "or ONE domain cut into one slab per rank (strong; the paper's decomposed runs)")
    ap.add_argument("--transport", default="p2p", choices=("p2p", "peer"),
                    help="slabs under torchrun: ghost layers by torch.distributed point-to-point calls (NCCL) or pushed into the "
                         "neighbours' CUDA-IPC-mapped workspaces (same node)")
    ap.add_argument("--no-overlap", action="store_true", help="slabs: the plain one-stream schedule instead of boundary layers first")
    ap.add_argument("--slabs", type=int, default=0, help="cut the workload into this many slabs on ONE GPU (overhead measurement)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        if args.steps > 20:
            args.steps = 20          # bounded: the oracle runs at a few MLUPS
        args.warmup = min(args.warmup, 2)
        return run_reference(args)
    if args.slabs > 0 or args.parallelism in ("slabs", "slabs-strong"):
        return run_slabs(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
