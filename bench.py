#!/usr/bin/env python
"""bench.py - throughput of the micromagnetic hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--size 4096] [--impl ours|reference]

A "step" is one Dormand-Prince RK45 step (6 torque evaluations: demag FFT convolution + exchange +
Zeeman, torque, stage combinations, error norm, controller) of the C4 workload of BASELINE.json: a
size x size x 1 Permalloy film, 4x4x2 nm cells, seeded random m, B_ext = 10 mT, fixed dt = 1e-13 s
(deterministic count, no rejections).  metric: cell-updates/s = cells * steps / time, whole job.
N > 1 runs N independent replicas (the path does not shard): weak scaling.
Prints ONE JSON line on rank 0.
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
sys.path.insert(0, ROOT)

METRIC = "LLG cell-updates/s per RK45 step (demag+exchange)"
UNIT = "cell-updates/s"
STEP_BYTES_PER_CELL = 1272.0      # algorithmic bytes per cell per RK45 step, 2D open


def measured_peak_gbs():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"       # B200_PROFILING.md fallback


def kernel_bytes(kind, n, P):
    """Algorithmic bytes of ONE launch of a kernel class of the 2D path.
    n = cells per side, P = padded FFT length; Cx = P/2+1 stored kx, Hy = P/2+1 kernel rows."""
    N, Cx, Hy = n * n, P // 2 + 1, P // 2 + 1
    spec = n * Cx * 8               # one component of the half spectrum, rows y < n
    table = {
        "x_fwd": 12 * N + N + 3 * spec,
        "last_xy": 2 * spec + 3 * Hy * Cx * 4 + 2 * spec,
        "last_z": spec + Hy * Cx * 4 + spec,
        "x_inv": 3 * spec + 12 * N,
        # fused local kernels (Nx % 4 == 0): per step 6 x (y, B_demag, regions in; k out) + 5 x (m0 in, next y out)
        # + 19 slope reads of the non-zero tableau / error weights = 570 N bytes over 6 launches
        "local": 95 * N,
        "rk_stage": 36 * N,                                   # only y_2 = m0 + h a21 k1 is left to the stage kernel
        "rk_error": 12 * N * 6,
        # register-FFT kernels of the fast 2D path (transposed spectrum, Cx = n + 1 stored kx)
        "f2_xfwd": 12 * N + N + 3 * spec,
        "f2_ycol": 6 * spec + 4 * Hy * Cx * 4,
        "f2_xinv": 3 * spec + 12 * N,
    }
    return float(table.get(kind, 0.0))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm)}
        return out


def _oracle_threads():
    import oracle.field as of
    return int(of.FFT_WORKERS)


def _time_oracle(n, steps, budget_s):
    """Time `steps` RK45 steps of the oracle (as it stands: numpy fp64, library FFT threaded over the host cores)
    on the C4 recipe at n x n x 1; stops early when the time budget is spent. Returns (cell-updates/s, steps done, s)."""
    from oracle import RefSim
    from synth import config_c4
    cfg = config_c4(n)
    ref = RefSim(cfg["grid"], cfg["cell"], cfg["pbc"], demag_method="fft")
    ref.set_params(cfg["params"]); ref.set_m(cfg["m0"]); ref.set_solver(fix_dt=cfg["fix_dt"])
    ref.step()                                   # warm-up: kernel spectrum, FSAL slope
    done, t0 = 0, time.perf_counter()
    while done < steps:
        ref.step(); done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return n * n * done / dt, done, dt


def cpu_baseline(args):
    """The oracle on the box's host cores: a bounded sample of the C4 workload at the largest size that fits the
    time budget (args.cpu_size, default 1024^2) and at 256^2; cell-updates/s is not size-invariant, both are given."""
    big, nbig, sbig = _time_oracle(args.cpu_size, args.cpu_steps, args.cpu_budget)
    small, nsmall, ssmall = _time_oracle(256, 20, 0.3 * args.cpu_budget) if args.cpu_size != 256 else (big, nbig, sbig)
    thr = _oracle_threads()
    return {"value": big, "unit": UNIT, "cores": thr, "host_cores": os.cpu_count(), "kind": "oracle",
            "sample": "C4 recipe at %dx%dx1, %d RK45 steps in %.1f s (numpy fp64 oracle, FFT demag, library FFT on %d threads, "
                      "the rest of the step on one)" % (args.cpu_size, args.cpu_size, nbig, sbig, thr),
            "also": {"size": 256, "value": small, "steps": nsmall, "seconds": ssmall}}


def run_reference(args, rank):
    """--impl reference: the oracle as it stands, on the host cores, each step a bounded sample of the workload."""
    if rank != 0:
        return
    n = args.cpu_size
    steps = max(1, min(args.steps, args.cpu_steps))
    value, done, dt = _time_oracle(n, steps, args.cpu_budget)
    thr = _oracle_threads()
    sample = "C4 recipe at %dx%dx1, %d RK45 steps (numpy fp64, FFT demag, library FFT on %d threads)" % (n, n, done, thr)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": done,
            "warmup": 1, "ms_per_step": 1e3 * dt / done, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "C4 film %dx%dx1 (bounded sample of the %d^2 workload)" % (n, n, args.size),
                       "cells": n * n, "fix_dt": 1e-13},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": thr, "host_cores": os.cpu_count(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (the driver's torchrun line)."""
    import socket
    with socket.socket() as so:
        so.bind(("127.0.0.1", 0))
        port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def run_batch(args, mm, torch, replicas, rank, world, local_rank):
    """B independent C4 boxes per GPU stepping concurrently: aggregate cell-updates/s and time per box and step."""
    from synth import config_c4
    n, B = args.size, args.batch
    sims = []
    for b in range(B):
        cfg = config_c4(n, seed_offset=replicas.replica_seed(b, rank))
        sim = mm.from_config(cfg)
        sim.set_solver(fix_dt=cfg["fix_dt"])
        sims.append(sim)
    mm.batch_steps(sims, args.warmup)
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = sum(s_.launch_count() for s_ in sims)
    streams = [s_.stream for s_ in sims]
    e0 = [torch.cuda.Event(enable_timing=True) for _ in sims]
    e1 = [torch.cuda.Event(enable_timing=True) for _ in sims]
    for a_, st in zip(e0, streams):
        a_.record(st)
    mm.batch_steps(sims, args.steps)
    for b_, st in zip(e1, streams):
        b_.record(st)
    torch.cuda.synchronize()
    ms = max(a_.elapsed_time(b_) for a_ in e0 for b_ in e1)          # first start to last end, on the device
    launches = sum(s_.launch_count() for s_ in sims) - l0
    clocks = sampler.stop() if sampler else None
    cells = n * n * B
    value, ms = replicas.aggregate_throughput(cells * args.steps, ms, device="cuda")
    if rank == 0:
        working = sum(s_.stats()["peak_device_bytes"] for s_ in sims)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms / args.steps, "ms_per_box_step": ms / args.steps / B, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "%d independent C4 films %dx%dx1 advancing together (mm_batch_steps), fix_dt 1e-13 s" % (B, n, n),
                           "cells": cells, "batch": B, "parallelism": "replicas x%d" % world,
                           "l2": "working set %.2f GB (all boxes)" % (working / 1e9), "evals_per_step": 6},
                "clocks": clocks, "gpu_launches": launches,
                "step_roofline": {"achieved": STEP_BYTES_PER_CELL * value / 1e9, "peak": measured_peak_gbs()[0], "unit": "GB/s",
                                  "frac": STEP_BYTES_PER_CELL * value / 1e9 / measured_peak_gbs()[0]}}
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--size", type=int, default=4096)
    ap.add_argument("--workload", default="c4", choices=["c4", "c4regions", "c5", "c5pbc", "c3"],
                    help="c4: size x size x 1 film (default, the metric's workload); c4regions: the same film cut into 64 "
                         "Voronoi regions with an inter-region exchange table; c5 / c5pbc: size^3 cube, open / "
                         "PBC(4,4,0); c3: 128 x 128 x 32 multi-region block, adaptive steps (--size is ignored)")
    ap.add_argument("--batch", type=int, default=0,
                    help="c4 only: this many independent boxes of --size advance together (mm_batch_steps, one stream "
                         "per handle): the paper's batch use of small simulations (L426, L800-L803)")
    ap.add_argument("--adaptive", action="store_true",
                    help="c4: adaptive RK45 (MaxErr 1e-5) instead of the fixed step; attempts (accepted or not) count as steps")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-size", type=int, default=1024, help="film edge of the timed oracle sample")
    ap.add_argument("--cpu-steps", type=int, default=8)
    ap.add_argument("--cpu-budget", type=float, default=25.0, help="seconds of oracle time per sample")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the mm_b200 path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    from paper_1406_7635_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    import paper_1406_7635_b200 as mm
    from paper_1406_7635_b200 import replicas
    from synth import config_c4

    n = args.size
    if args.batch > 0:
        run_batch(args, mm, torch, replicas, rank, world, local_rank)
        if world > 1:
            dist.destroy_process_group()
        return
    if args.workload == "c4":
        cfg = config_c4(n, seed_offset=replicas.replica_seed(0, rank))     # one independent replica per rank
        cells, step_bytes = n * n, STEP_BYTES_PER_CELL
        wname = "C4 film %dx%dx1, 4x4x2 nm, Permalloy, random m, B_ext 10 mT, fix_dt 1e-13 s" % (n, n)
    elif args.workload == "c4regions":
        from synth import config_c4_regions
        cfg = config_c4_regions(n)
        cells, step_bytes = n * n, STEP_BYTES_PER_CELL
        wname = "C4 film %dx%dx1 in 64 Voronoi regions (Msat +-10 %%, inter-region exchange 0.5-1), fix_dt 1e-13 s" % (n, n)
    elif args.workload == "c3":
        from synth import config_c3
        cfg = config_c3()
        cfg["fix_dt"] = 0.0                                   # adaptive RK45, MaxErr 1e-5; attempts are counted as steps
        nx, ny, nz = cfg["grid"]
        cells, step_bytes = nx * ny * nz, 2472.0
        wname = "C3 block %dx%dx%d, 2 nm, 64 Voronoi regions, Ku1 + inter-region exchange, random m, adaptive RK45" % (nx, ny, nz)
    else:
        from synth import config_c5
        cfg = config_c5(n, pbc=args.workload == "c5pbc")
        cells = n ** 3
        step_bytes = 6 * 140.0 + 372.0 if args.workload == "c5pbc" else 2472.0
        wname = "C5 cube %d^3, 2 nm, Kc1 -5e3, random m, %s, fix_dt 1e-13 s" % (n, "PBC (4,4,0)" if args.workload == "c5pbc" else "open")
    if args.adaptive and args.workload in ("c4", "c4regions"):
        cfg["fix_dt"] = 0.0
        wname = wname.replace("fix_dt 1e-13 s", "adaptive RK45 (MaxErr 1e-5, attempts counted)")
    sim = mm.from_config(cfg)
    sim.set_solver(fix_dt=cfg["fix_dt"])
    P = sim.fft_size()[0]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between two events
    sim.steps(args.warmup)
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    l0 = sim.launch_count()
    # L2: a step streams its whole working set several times, so nothing of one step survives to the next when
    # the set is much larger than the cache; a set that fits is flushed (a 256 MB memset) before every timed step
    l2_bytes = torch.cuda.get_device_properties(local_rank).L2_cache_size
    working = sim.stats()["peak_device_bytes"]
    flush = torch.empty(2 * l2_bytes, dtype=torch.uint8, device="cuda") if working < 4 * l2_bytes else None
    hstream = sim.stream                      # the handle's own stream: events must be recorded where its kernels run
    if flush is None:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(hstream)
        for _ in range(args.steps):
            sim.step(want_info=False)
        e1.record(hstream)
        barrier()
        ms = e0.elapsed_time(e1)
    else:
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a_, b_ in ev:
            with torch.cuda.stream(hstream):
                flush.zero_()
            a_.record(hstream)
            sim.step(want_info=False)
            b_.record(hstream)
        barrier()
        ms = sum(a_.elapsed_time(b_) for a_, b_ in ev)
    launches = sim.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    value, ms = replicas.aggregate_throughput(cells * args.steps, ms, device="cuda")   # all ranks' units / max time

    # ---- per-kernel CUDA-event timing of the same K steps (separate pass: events bracket every launch)
    sim.profile(True)
    for _ in range(args.steps):
        sim.step(want_info=False)
    prof = sim.profile_read()
    sim.profile(False)
    peak, peak_src = measured_peak_gbs()
    roofline, kernels = None, {}
    tot_ms = sum(v[0] for v in prof.values()) or 1.0
    for name, (kms, cnt) in prof.items():
        b = kernel_bytes(name, n, P) if args.workload in ("c4", "c4regions") else 0.0     # byte table is for the 2D path
        kernels[name] = {"ms_per_launch": kms / cnt, "launches_per_step": cnt / args.steps, "share": kms / tot_ms,
                         "GBps": (b / (kms / cnt * 1e-3) / 1e9) if b else None}
    if prof and args.workload in ("c4", "c4regions"):
        top = max(prof, key=lambda k: prof[k][0])
        b = kernel_bytes(top, n, P)
        ach = b / (prof[top][0] / prof[top][1] * 1e-3) / 1e9
        traffic, traffic_src = None, None
        try:
            with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
                tj = json.load(f)
            traffic = tj.get("%s@%d" % (top, n))
            traffic_src = tj.get("_captured")       # which ncu capture the figure is from (not measured in this run)
        except Exception:
            pass
        roofline = {"bound": "hbm", "kernel": top, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic, "traffic_source": traffic_src if traffic else None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": b, "share_of_step": prof[top][0] / tot_ms}
    step_gbs = step_bytes * cells * args.steps / (ms * 1e-3) / 1e9
    step_roofline = {"achieved": step_gbs, "peak": peak, "unit": "GB/s", "frac": step_gbs / peak,
                     "frac_of_8TBps": step_gbs / 8000.0, "bytes_per_cell_step": step_bytes}

    # ---- end to end through the C ABI with HOST buffers: per step H2D of m, one RK45 step, D2H of m
    host_in = torch.from_numpy(cfg["m0"].copy()).pin_memory()
    host_out = torch.empty_like(host_in).pin_memory()
    ke = max(1, min(args.e2e_steps, args.steps))
    sim.set_m(host_in); sim.step(want_info=False); sim.get_m(host_out)       # warm the path
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        sim.set_m(host_in)                  # host -> device, normalise
        sim.step(want_info=False)           # FSAL slope is stale after set_m: 7 evaluations
        sim.get_m(host_out)                 # device -> host (synchronises)
        host_in, host_out = host_out, host_in
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_value, e2e_ms = replicas.aggregate_throughput(cells * ke, 1e3 * e2e_s, device="cuda")
    e2e_s = 1e-3 * e2e_ms
    nbytes = int(host_in.numel() * 4)
    e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
           "steps": ke, "ms_per_step": 1e3 * e2e_s / ke}

    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": wname,
                           "cells": cells, "fft": list(sim.fft_size()), "parallelism": "replicas x%d" % world,
                           "l2": ("working set %.2f GB vs %d MB L2: " % (working / 1e9, l2_bytes >> 20)) +
                                 ("streams through, no flush" if flush is None else "L2 flushed before every timed step"),
                           "evals_per_step": 6},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "step_roofline": step_roofline, "kernels": kernels,
                "peak_device_bytes": sim.stats()["peak_device_bytes"], "resident_device_bytes": sim.memory()[0]}
        line["cpu_baseline"] = None if (args.no_cpu_baseline or world > 1) else cpu_baseline(args)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
