#!/usr/bin/env python
"""bench.py -- MLUPS of the full LB+FD step and achieved HBM bandwidth of the LB kernel.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--config 3] [--precision fp32s|fp64|fp32u] [--size NX NY NZ]

Workload (default): BASELINE.json configs[3] -- two skyrmion tubes in Poiseuille flow on
256x256x64, FD/LB ratio r = 10, shifted FP32 (the configuration north_star's target is quoted on).
One bench "step" is one pass over every row of the hot path: r LB steps (collide+stream+force),
then the velocity store, predictor, corrector and force update.  MLUPS = fluid cells x LB steps /
seconds / 1e6 (reading G21).

Prints ONE JSON line (rank 0).  Beyond the contract's keys: `roofline` (dominant LB kernel: `bound` "hbm" for the one-step
kernels, "latency" for the two-step kernel with `own_dram_floor_frac`, its time against one pass over HBM per pair of steps),
`sustained` (the same loop for >= 3 s: clocks, power, `mlups_per_watt`), `fp64` and `one_step` sub-records, `e2e` through
the C ABI with pinned host buffers, `cpu_baseline` (the oracle on the host cores).  Both arms take `config` from config_of().  Multi-GPU (--gpus N, under torchrun or started by bench.py itself): ONE lattice of N
times the config's rows, cut into N y-slabs, one per rank, halo rows exchanged over NCCL (weak scaling; DESIGN.md
section 8); --replicas runs N independent lattices instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PRECISIONS = {"fp64": 0, "fp32s": 1, "fp32u": 2, "fp64u": 3}
DTYPE = {0: "f64", 1: "f32", 2: "f32", 3: "f64"}
METRIC = "MLUPS (LB+FD step)"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs index; 5 = the paper's 320x320x16 "
                    "many-skyrmion demonstration (PAPER.md:284) on its test-case material, Delta t_FD = 250")
    ap.add_argument("--precision", default="fp32s", choices=sorted(PRECISIONS))
    ap.add_argument("--size", type=int, nargs=3, default=None, help="configs[4] grid (nx ny nz)")
    ap.add_argument("--options", type=lambda v: int(v, 0), default=0, help="nh_set_options bits (kernel variants)")
    ap.add_argument("--two-step", action="store_true", help="NH_OPT_LB_TWOSTEP: force two LB steps per launch through the L2")
    ap.add_argument("--one-step", action="store_true", help="NH_OPT_LB_ONESTEP: one LB step per launch")
    ap.add_argument("--graph", action="store_true", help="NH_OPT_GRAPH: replay nh_step through CUDA graphs (pays where the LB "
                    "launches are short and the two-step kernel does not apply, e.g. --config 5)")
    ap.add_argument("--tune", action="append", default=[], metavar="KEY=VALUE",
                    help="nh_debug_tune knob (include/nh_debug.h), e.g. --tune lb2_lead=3 --tune lb2_ring=6")
    ap.add_argument("--leslie", type=float, default=0.0,
                    help="scale of the paper's Table-1 Leslie viscosities in the force (row f1; 0 = elastic stress only)")
    ap.add_argument("--fd-ratio", type=int, default=None, help="override the config's Delta t_FD / Delta t_LB")
    ap.add_argument("--frank3", action="store_true",
                    help="three-constant Frank energy (row f2): K11 = K, K22 : K33 in the ratios of the paper's Table 1")
    ap.add_argument("--slabs", type=int, default=0,
                    help="ONE lattice cut into y-slabs with halo exchange (paper_2503_06610_b200/slabs.py).  With more than one "
                         "GPU this is the default: one slab per rank over NCCL, the config's ny rows PER RANK (weak scaling; the "
                         "value is ignored).  On one GPU: the config's lattice cut into this many slabs held by one process "
                         "(measures the decomposition's overhead)")
    ap.add_argument("--replicas", action="store_true",
                    help="with more than one GPU: N independent lattices, one per rank, no communication, instead of slabs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the sustained (>= 3 s) loop and the fp64 / one_step sub-records")
    return ap.parse_args()


def workload(args):
    import nh_inputs as I
    over = {}
    if args.config == 4 and args.size:
        over["size"] = tuple(args.size)
    if args.fd_ratio is not None:
        over["fd_ratio"] = args.fd_ratio
    p = I.many_skyrmions(**over) if args.config == 5 else I.config(args.config, **over)
    if args.leslie:
        # alpha1..alpha6 of MBBA in simulation units as printed in the paper's Table 1
        table1 = (0.0373, -0.4496, -0.0203, 0.9318, 0.3084, -0.1617)
        p["alpha"] = tuple(args.leslie * a for a in table1)
    if args.frank3:
        # K11 : K22 : K33 = 1.67 : 0.788 : 2.62
        p["K3"] = (p["K"], p["K"] * 0.788 / 1.67, p["K"] * 2.62 / 1.67)
    if args.leslie and args.config == 5:
        p["alpha"] = tuple(args.leslie * a for a in I.MBBA_ALPHA)
    d = p.pop("director")
    p.pop("steps")
    name = {0: "configs[0] tiny channel", 1: "configs[1] single skyrmion tube", 2: "configs[2] precision sweep domain",
            3: "configs[3] two skyrmion tubes in Poiseuille flow", 4: "configs[4] skyrmion lattice",
            5: "many-skyrmion demonstration (PAPER.md:284), 20 tubes, free plates, W0"}[args.config]
    desc = {"workload": "%s %dx%dx%d" % (name, p["nx"], p["ny"], p["nz"]), "grid": [p["nx"], p["ny"], p["nz"]],
            "fd_ratio": p["fd_ratio"], "tau": p["tau"], "K": p.get("K", 0.0), "pitch": p["pitch"], "xi": p["xi"],
            "g_x": p["g"][0], "precision": args.precision}
    if args.leslie:
        desc["leslie_viscous_stress"] = "Table 1 x %g" % args.leslie
    if args.frank3 or args.config == 5:
        desc["frank_constants"] = list(p["K3"])
    return p, d, desc


B200_L2_MB = 126.0          # nominal L2 of a B200: the config line's L2 statement depends on the workload only, so
                            # that both arms (--impl ours / reference) print the same `config`


def base_options(args):
    # NH_OPT_LB_TWOSTEP, NH_OPT_LB_ONESTEP, NH_OPT_GRAPH of include/nh.h (literal: the reference arm prints the same
    # config and must not import the CUDA package)
    return args.options | (64 if args.two_step else 0) | (128 if args.one_step else 0) | (1 if args.graph else 0)


def tune_knobs(args):
    return {kv.split("=")[0]: int(kv.split("=")[1]) for kv in args.tune}


def config_of(args, p, desc, world):
    """The `config` of the JSON line: the workload and how a step is counted.  The same for both arms."""
    r = max(1, p["fd_ratio"])
    N = p["nx"] * p["ny"] * p["nz"]
    word = 8 if PRECISIONS[args.precision] in (0, 3) else 4
    pop_mb = 19 * N * word / 1e6
    fits = 2 * pop_mb <= B200_L2_MB * 1.048576
    l2 = (("populations (2 x %.0f MB) exceed the %.0f MB L2; no flush needed" if not fits else
           "populations (2 x %.1f MB) FIT the %.0f MB L2 and nothing is flushed between steps: this grid is "
           "L2-resident by nature (a time step follows a time step); MLUPS is the figure, GB/s is not") % (pop_mb, B200_L2_MB))
    return dict(desc, lb_steps_per_step=r, fluid_cells=p["nx"] * p["ny"] * (p["nz"] - 2),
                step="one step = %d LB steps + 1 director update + 1 force update" % r,
                parallelism="replicas x%d" % world, l2=l2, options=base_options(args), tune=tune_knobs(args))


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


LB_SOURCES = ("paper_2503_06610_b200/csrc/nh_lb.cuh", "paper_2503_06610_b200/csrc/nh_lb2.cuh")


def lb_source_sha():
    """First 16 hex digits of the SHA-256 of the LB kernel sources: profiles/lb_traffic.csv records the value a
    capture was taken at, so that a capture of an older kernel is never quoted for a newer one."""
    import hashlib
    h = hashlib.sha256()
    for rel in LB_SOURCES:
        with open(os.path.join(ROOT, rel), "rb") as f:
            h.update(f.read())
    return h.hexdigest()[:16]


def ncu_traffic(precision_name, grid):
    """(DRAM bytes per launch, warp instructions per launch, where it comes from) of the dominant LB kernel, from
    the committed `ncu --set full` capture (profiles/lb_traffic.csv: a STORED capture, not measured in this run).
    Only a row taken from the kernel source as it stands now counts: otherwise (None, None, why)."""
    path = os.path.join(ROOT, "profiles", "lb_traffic.csv")
    if not os.path.exists(path):
        return None, None, "no capture (profiles/lb_traffic.csv missing)"
    try:
        want = "%dx%dx%d" % tuple(grid)
        now = lb_source_sha()
        row = stale = None
        for line in open(path).read().splitlines()[1:]:
            c = line.split(",")
            if len(c) >= 5 and c[0] == precision_name and c[1] == want:
                if len(c) >= 7 and c[6] == now:
                    row = c                  # the last matching row is the newest capture
                else:
                    stale = c
        if row is not None:
            return float(row[3]), (float(row[5]) if row[5] else None), "stored capture %s (kernel source sha %s)" % (row[4], now)
        if stale is not None:
            return None, None, ("stale: the newest capture of this kernel and grid (%s) was taken from another version "
                                "of the kernel source (now %s)" % (stale[4], now))
        return None, None, "no capture for %s on %s" % (precision_name, want)
    except Exception as e:  # noqa: BLE001
        return None, None, "unreadable capture table: %s" % e


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)          # nvidia-smi -lms needs a moment to print its first line on short runs
        self.proc.terminate()
        try:
            out = self.proc.communicate(timeout=5)[0]
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); power.append(float(c[3]))
            except ValueError:
                continue
            for nme, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power), "power_w_mean": sum(power) / len(power)}


def run_reference(args):
    """The oracle, as it stands, on the host cores (tier contract: the reference arm)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import Oracle, num_threads
    p, d, desc = workload(args)
    o = Oracle(**dict(p, precision=PRECISIONS[args.precision]))
    o.set_director(d)
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    r = max(1, p["fd_ratio"])
    # a step is what the GPU arm calls a step: r LB steps, then the director and force update (one FD period)
    for _ in range(args.warmup):
        o.step(r)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.step(r)
    dt = time.perf_counter() - t0
    mlups = nf * r * args.steps / dt / 1e6
    sample = ("each step = %d LB steps + 1 FD update of the full %dx%dx%d grid (%d steps timed, %.1f s)"
              % (r, p["nx"], p["ny"], p["nz"], args.steps, dt))
    line = {"impl": "reference", "metric": METRIC, "value": mlups, "unit": "MLUPS", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": config_of(args, p, desc, 1),
            "cpu_baseline": {"value": mlups, "unit": "MLUPS", "cores": num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": mlups, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def cpu_baseline(p, d, precision):
    from oracle import Oracle, num_threads
    o = Oracle(**dict(p, precision=precision))
    o.set_director(d)
    r = max(1, p["fd_ratio"])
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    # bounded sample: whole FD periods of the same workload, about 10-30 s of CPU work; the first
    # period sizes the sample, the rest is what is timed
    t0 = time.perf_counter()
    o.step(r)
    first = time.perf_counter() - t0
    periods = max(1, min(200, int(12.0 / max(first, 1e-3))))
    t0 = time.perf_counter()
    o.step(periods * r)
    dt = time.perf_counter() - t0
    return {"value": nf * periods * r / dt / 1e6, "unit": "MLUPS", "cores": num_threads(), "kind": "oracle",
            "sample": "%d FD period(s) = %d LB steps + %d FD update(s) of the same %dx%dx%d workload, %.1f s"
                      % (periods, periods * r, periods, p["nx"], p["ny"], p["nz"], dt)}


def max_over_ranks(ms, world, device="cuda"):
    """Step time of the job = the slowest rank's device time (replicas only: no data-path collective)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_mlups(world, fluid_cells, lb_steps, ms):
    """Whole-job throughput: every rank advanced its own replica by lb_steps LB steps in ms."""
    return world * fluid_cells * lb_steps / (ms * 1e-3) / 1e6


def run_slabs(args, world, rank, local):
    """One lattice cut along y.  N > 1: the global lattice has world x ny rows, rank s holds slab s;
    N = 1: the config's own lattice in args.slabs slabs on this device.  Same timing rules as the main line."""
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200.slabs import SlabLattice

    p, d, desc = workload(args)
    prec = PRECISIONS[args.precision]
    r = max(1, p["fd_ratio"])
    if world > 1:
        d = np.concatenate([d] * world, axis=2)          # the config's director tiled along y: still periodic
        p = dict(p, ny=p["ny"] * world)
    nslabs = world if world > 1 else args.slabs
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    lat = SlabLattice(slabs=nslabs, group=dist.group.WORLD if world > 1 else None, device="cuda:%d" % local,
                      **dict(p, precision=prec))
    lat.set_director(d)
    # the kernel-variant flags act on every slab's lattice, as they do on the undivided one
    base_opt, knobs = base_options(args), tune_knobs(args)
    for L in lat.local.values():
        L.debug_tune(**knobs)
        L.set_options(base_opt)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        lat.step(r)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = sum(x.launch_count for x in lat.local.values())
    x0, b0 = lat.exchanges, lat.bytes_sent
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        lat.step(r)
    ev1.record()
    barrier()
    ms = max_over_ranks(ev0.elapsed_time(ev1), world)
    launches = sum(x.launch_count for x in lat.local.values()) - l0
    clocks = sampler.stop() if rank == 0 else None
    # second pass of the same steps with an event pair around every launch: where each slab's time goes
    for L in lat.local.values():
        L.set_options((base_opt & ~nh.OPT_GRAPH) | nh.OPT_TIMING)
    barrier()
    for _ in range(args.steps):
        lat.step(r)
    kernel_ms = {str(sl): {k: round(L.kernel_time(k)[0], 4) for k in nh.KERNEL_CLASSES} for sl, L in sorted(lat.local.items())}
    for L in lat.local.values():
        L.set_options(base_opt)
    if rank == 0:
        line = {"metric": METRIC, "value": nf * r * args.steps / (ms * 1e-3) / 1e6, "unit": "MLUPS", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": DTYPE[prec], "data": "synthetic",
                "config": dict(desc, grid=[p["nx"], p["ny"], p["nz"]], lb_steps_per_step=r, fluid_cells=nf,
                               parallelism="y-slabs x%d, halo %d rows%s" % (nslabs, lat.H, "" if world > 1 else " (one device)"),
                               exchanges_per_step=(lat.exchanges - x0) / args.steps,
                               halo_bytes_sent_per_step_per_process=(lat.bytes_sent - b0) / args.steps,
                               options=base_opt, tune=knobs),
                "clocks": clocks, "gpu_launches": launches, "roofline": None,
                "kernel_ms_per_slab": {"slabs_of_rank_0": kernel_ms,
                                       "timed": "second pass of the same K steps with per-launch CUDA events"}}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not launched by torchrun: start the N ranks ourselves (one process per GPU, NCCL over NVLink)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)

    import torch
    import torch.distributed as dist
    import paper_2503_06610_b200 as nh
    from paper_2503_06610_b200 import build as nh_build

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    # test hooks (tests/test_gpu_slabs.py runs the N = 2 path on a one-GPU box): all ranks on one device, gloo instead of NCCL
    backend = os.environ.get("NH_BENCH_BACKEND", "nccl")
    if "NH_BENCH_DEVICE" in os.environ:
        local = int(os.environ["NH_BENCH_DEVICE"])
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl ours needs a CUDA device (there is no CPU path)")
    torch.cuda.set_device(local)
    # a stream of its own: the lattice, the copies and the timing events all go to torch's current stream, and
    # graph replay (--graph) cannot capture the legacy default stream
    torch.cuda.set_stream(torch.cuda.Stream())
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(backend)
        if rank == 0:
            sys.stderr.write("bench.py: communicator backend=%s nranks=%d (NCCL_DEBUG=INFO shows its rings and NVLS)\n"
                             % (dist.get_backend(), dist.get_world_size()))
    if rank == 0:
        nh_build.build()
    if world > 1:
        dist.barrier()

    # more than one GPU: the path shards as y-slabs with a halo exchange; --replicas opts out
    if args.slabs or (world > 1 and not args.replicas):
        return run_slabs(args, world, rank, local)

    p, d, desc = workload(args)
    prec = PRECISIONS[args.precision]
    r = max(1, p["fd_ratio"])
    nf = p["nx"] * p["ny"] * (p["nz"] - 2)
    N = p["nx"] * p["ny"] * p["nz"]
    word = 8 if prec in (0, 3) else 4
    lat = nh.Lattice(device="cuda:%d" % local, **dict(p, precision=prec))
    d_pinned = torch.from_numpy(d).pin_memory()
    lat.set_director(d_pinned)
    base_opt = base_options(args)
    knobs = tune_knobs(args)
    lat.debug_tune(**knobs)
    l2_bytes = int(getattr(torch.cuda.get_device_properties(local), "L2_cache_size", 0)) or 126 * 1024 * 1024
    peak, peak_src = peaks()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn):
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        ev0.record()
        fn()
        ev1.record()
        barrier()
        return max_over_ranks(ev0.elapsed_time(ev1), world)

    def measure(L, opt, precision_name, w, steps, warmup, sample_clocks=True):
        """W warm-up steps, exactly K steps between barriers (CUDA events, max over ranks), then a second pass of the
        same K steps with a CUDA-event pair around every launch for the dominant kernel's roofline."""
        L.set_options(opt)
        for _ in range(warmup):
            L.step(r)
        sampler = ClockSampler(local)
        if rank == 0 and sample_clocks:
            sampler.start()
        l0 = L.launch_count
        ms = timed(lambda: [L.step(r) for _ in range(steps)])
        launches = L.launch_count - l0
        clocks = sampler.stop() if rank == 0 and sample_clocks else None
        L.set_options((opt & ~nh.OPT_GRAPH) | nh.OPT_TIMING)      # per-launch events need plain launches: same kernels
        barrier()
        for _ in range(steps):
            L.step(r)
        kt = {k: L.kernel_time(k) for k in nh.KERNEL_CLASSES}
        L.set_options(opt)
        # dominant kernel: the one-step LB launch, or the two-step launch (2 LB steps each) when it is on
        two = kt["lb2"][0] > kt["lb"][0]
        lb_ms, lb_n = kt["lb2"] if two else kt["lb"]
        # (small lattices take all the LB steps between two director updates in one cooperative launch)
        steps_per_launch = 2 if two else max(1, int(round(r * steps / max(lb_n, 1))))
        lb_avg = lb_ms / max(lb_n, 1)
        total_k = sum(v[0] for v in kt.values())
        # 19 read + 19 write + 3 (F^LC) words per fluid cell and LB step
        alg_bytes = 41 * w * nf * steps_per_launch
        achieved = alg_bytes / (lb_avg * 1e-3) / 1e9 if lb_avg > 0 else 0.0
        kname = ("lb_wave (2 x collide+stream+force per launch)" if two else
                 "lb_step (collide+stream+force)" if steps_per_launch == 1 else
                 "lb_resident (%d x collide+stream+force per cooperative launch)" % steps_per_launch)
        traffic, inst, tsrc = ncu_traffic(precision_name + ("+2step" if two else ""), desc["grid"])
        pop_bytes = 2 * 19 * N * w
        in_l2 = pop_bytes <= l2_bytes
        # The one-step kernels move their algorithmic bytes through the DRAM at the copy rate: HBM-bound.  The two-step
        # kernel halves the DRAM traffic through the L2 and is then held by latency (barrier and scoreboard stalls,
        # DRAM and L2 each about half busy: profiles/r02_lbwave_full.txt), so `frac` against the section-8(d) byte model
        # exceeds 1 and the fraction that says how far it is from ITS limit is own_dram_floor_frac below.
        roof = {"bound": "latency" if two else "hbm", "kernel": kname, "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": tsrc,
                "peak_source": peak_src, "frac_of_nominal_8000_gbs": achieved / 8000.0,
                "algorithmic_bytes_per_launch": alg_bytes,
                "lb_steps_per_launch": steps_per_launch,
                "avg_launch_ms": lb_avg, "launches_timed": lb_n, "share_of_step": lb_ms / total_k if total_k else None,
                "kernel_ms": {k: round(v[0], 4) for k, v in kt.items()},
                "full_step_bytes_per_cell": (41 + 30.0 / r) * w,
                "full_step_achieved_gbs": (41 + 30.0 / r) * w * nf * r * steps / (ms * 1e-3) / 1e9,
                "timed": "second pass of the same K steps with per-launch CUDA events on the launch stream"}
        if in_l2:
            roof["resident_in_l2"] = True
            roof["note"] = ("both population buffers (%.1f MB) fit the %.0f MB L2: the gathers are served by the L2, "
                            "`achieved` is algorithmic bytes over time and says nothing about HBM; SURVEY 8(d): report "
                            "MLUPS for such grids, not GB/s" % (pop_bytes / 1e6, l2_bytes / 1e6))
        if traffic and lb_avg > 0:
            # what the DRAM moved in the STORED ncu capture of this same kernel source, over the live launch time
            roof["dram_gbs"] = traffic / (lb_avg * 1e-3) / 1e9
            roof["dram_frac"] = roof["dram_gbs"] / peak
            roof["dram_gbs_is"] = "derived: stored capture's bytes / this run's launch time"
        if inst and lb_avg > 0 and clocks and clocks.get("sm_mhz"):
            # second ceiling: warp instructions issued against SMs x 4 issue slots per clock
            sms = torch.cuda.get_device_properties(local).multi_processor_count
            roof["issue_frac"] = inst / (lb_avg * 1e-3) / (sms * 4 * clocks["sm_mhz"] * 1e6)
            roof["warp_instructions_per_launch"] = inst
        if two and lb_avg > 0:
            # the kernel's own DRAM floor: 19 read + 19 written + 3 (F^LC) words per cell for the PAIR of steps
            roof["own_dram_floor_bytes_per_launch"] = 41 * w * nf
            roof["own_dram_floor_frac"] = 41 * w * nf / (lb_avg * 1e-3) / 1e9 / peak
            roof["bound_is"] = ("latency: two LB steps per pass over HBM through an L2-resident plane ring; neither DRAM "
                                "nor L2 nor the issue slots are saturated (profiles/): own_dram_floor_frac = time at the "
                                "measured copy rate for the kernel's own 41 words per cell and launch / measured time")
        if two:
            roof["note"] = ("two LB steps share one pass over HBM (the intermediate step lives in an L2-resident "
                            "plane ring), so the algorithmic bytes of two steps move in about the DRAM traffic of "
                            "one: frac > 1 is expected; dram_frac is the DRAM's own utilisation")
        return {"ms": ms, "mlups": job_mlups(world, nf, r * steps, ms), "launches": launches, "clocks": clocks,
                "roofline": roof, "pop_bytes": pop_bytes, "in_l2": in_l2}

    # ---- the headline: device-resident timing, W warm-up steps, then exactly K steps ---------------
    m = measure(lat, base_opt, args.precision, word, args.steps, args.warmup)
    ms, mlups, launches, clocks, roofline = m["ms"], m["mlups"], m["launches"], m["clocks"], m["roofline"]

    # ---- the same loop kept up for >= 3 s: does the number hold once power management has had time to act? ----
    sustained = None
    if not args.no_extras:
        reps = max(args.steps, int(3000.0 / max(ms / args.steps, 1e-3)) + 1)
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        ms_long = timed(lambda: [lat.step(r) for _ in range(reps)])
        cl = sampler.stop() if rank == 0 else None
        sustained = {"value": job_mlups(world, nf, r * reps, ms_long), "unit": "MLUPS", "steps": reps,
                     "seconds": ms_long * 1e-3, "ms_per_step": ms_long / reps, "clocks": cl,
                     "what": "the headline loop (same lattice, same options) repeated back to back for at least 3 s, "
                             "clocks and throttle reasons sampled over that window"}
        if cl and cl.get("power_w_mean"):
            sustained["mlups_per_watt"] = sustained["value"] / cl["power_w_mean"]
        # the issue-slot ceiling at the clock the SMs run at under load (the headline's few samples are mostly idle ones)
        inst = roofline.get("warp_instructions_per_launch")
        if inst and cl and cl.get("sm_mhz") and roofline["avg_launch_ms"] > 0:
            sms = torch.cuda.get_device_properties(local).multi_processor_count
            roofline["issue_frac"] = inst / (roofline["avg_launch_ms"] * 1e-3) / (sms * 4 * cl["sm_mhz"] * 1e6)
            roofline["issue_frac_clock_mhz"] = cl["sm_mhz"]
            roofline["issue_frac_clock_from"] = "sustained window"

    # ---- what `metric` also names: FP64, and the one-step FP32 kernel, each timed like the headline ----
    extras = {}
    if not args.no_extras and world == 1:
        def sub(precision_name, opt):
            pr = PRECISIONS[precision_name]
            w2 = 8 if pr in (0, 3) else 4
            L2 = nh.Lattice(device="cuda:%d" % local, **dict(p, precision=pr))
            L2.debug_tune(**knobs)
            L2.set_director(d_pinned)
            mm = measure(L2, opt, precision_name, w2, args.steps, args.warmup)
            L2.close()
            rf = mm["roofline"]
            return {"value": mm["mlups"], "unit": "MLUPS", "ms_per_step": mm["ms"] / args.steps, "dtype": DTYPE[pr],
                    "options": opt, "gpu_launches": mm["launches"], "clocks": mm["clocks"],
                    "roofline": {k: rf.get(k) for k in ("bound", "kernel", "achieved", "peak", "unit", "frac", "traffic",
                                                        "traffic_source", "avg_launch_ms", "launches_timed",
                                                        "share_of_step", "lb_steps_per_launch", "kernel_ms",
                                                        "full_step_achieved_gbs", "resident_in_l2")}}
        if args.precision != "fp64":
            extras["fp64"] = sub("fp64", base_opt)
        if not (base_opt & nh.OPT_LB_ONESTEP) and roofline["lb_steps_per_launch"] != 1:
            extras["one_step"] = sub(args.precision, (base_opt & ~nh.OPT_LB_TWOSTEP) | nh.OPT_LB_ONESTEP)

    # ---- end to end through the C ABI with host buffers --------------------------------------------
    e2e = None
    if not args.no_e2e:
        out = {"u": torch.empty((3, p["nz"], p["ny"], p["nx"]), dtype=torch.float64).pin_memory(),
               "n": torch.empty((3, p["nz"], p["ny"], p["nx"]), dtype=torch.float64).pin_memory()}

        def job():
            lat.set_director(d_pinned)                      # H2D 3N doubles
            for _ in range(args.steps):
                lat.step(r)
            lat.get_fields(out=out, which=("u", "n"))       # D2H 6N doubles

        job()
        ms_job = timed(job)
        # where the job's time goes (each part timed on its own, same buffers): PCIe copies of FP64 host arrays
        # (the contract's choice) against the device-resident steps
        ms_h2d = timed(lambda: lat.set_director(d_pinned))
        ms_steps = timed(lambda: [lat.step(r) for _ in range(args.steps)])
        ms_d2h = timed(lambda: lat.get_fields(out=out, which=("u", "n")))

        def every():
            for _ in range(3):
                lat.set_director(d_pinned)
                lat.step(r)
                lat.get_fields(out=out, which=("u", "n"))

        ms_every = timed(every)
        e2e = {"value": job_mlups(world, nf, r * args.steps, ms_job), "unit": "MLUPS",
               "h2d_bytes_per_step": 24 * N / args.steps, "d2h_bytes_per_step": 48 * N / args.steps,
               "what": "one job = nh_set_director(pinned host n) + K steps + nh_get_fields(u, n -> pinned host), "
                       "all inside the timed region; bytes are the job's copies divided by K",
               "split_ms": {"set_director_h2d": ms_h2d, "steps": ms_steps, "get_fields_d2h": ms_d2h, "job": ms_job,
                            "h2d_gbs": 24 * N / (ms_h2d * 1e-3) / 1e9, "d2h_gbs": 48 * N / (ms_d2h * 1e-3) / 1e9},
               "copies_every_step": {"value": job_mlups(world, nf, r * 3, ms_every), "unit": "MLUPS",
                                     "h2d_bytes_per_step": 24 * N, "d2h_bytes_per_step": 48 * N}}

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return 0

    line = {"metric": METRIC, "value": mlups, "unit": "MLUPS", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": DTYPE[prec], "data": "synthetic",
            "config": config_of(args, p, desc, world),
            "clocks": clocks, "gpu_launches": launches, "roofline": roofline}
    if sustained is not None:
        line["sustained"] = sustained
    line.update(extras)
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(p, d, prec)
    print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
