#!/usr/bin/env python
"""bench.py -- the per-level time step (ghost fill + x-sweep + y-sweep + CFL reduction) on config 5 of BASELINE.json:
one spherical level of NxN cells (default 8192 x 8192, 0.5 arcmin) tiled into square patches, all resident in one pool.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--side S] [--n NCELLS] [--impl reference]

A "step" = gc_fill_ghost + gc_level_step_auto (dt chain on the device, no host sync) over the whole level.
metric  = fp64 cell updates/s (interior cells x steps / device time, CUDA events, max over ranks).
N > 1   = replicas only (the contract fixes one GPU per problem; no collective is invented): every rank
          advances its own copy of the workload; value = units all ranks processed / max time.
--impl reference = the oracle (plain C, one thread) timed on a bounded sample of the same recipe on the host cores.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

# Algorithmic work per cell per sweep, counted per kernel from the ncu source page of the default marching
# kernels k_marchp<0> (x-sweep) / k_marchp<1> (y-sweep), profiles/r01_marchp.md: thread instructions / cells of one launch.
#   x-sweep: 140.7 DMUL + 103.7 DADD + 81.2 DFMA (x 2 flops) = 407 flops, + 60.5 DSETP = 386 fp64-pipe instructions
#   y-sweep: 143.9 DMUL + 104.8 DADD + 81.2 DFMA (x 2 flops) = 411 flops, + 64.6 DSETP = 394 fp64-pipe instructions
# (divides and square roots expanded into their correctly rounded Newton sequences; no FMA contraction elsewhere)
FLOP_PER_SWEEP = {"xsweep": 407.0, "ysweep": 411.0}
FP64_SLOTS_PER_SWEEP = {"xsweep": 386.0, "ysweep": 394.0}
BYTES_PER_UPDATE = 56.0   # read h, hu, hv, b + write h, hu, hv once; the two-pass design moves 112
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of each sweep kernel at the bench size 8192^2 / side 256, from the
# ncu --set full capture summarised in profiles/r01_marchp.md (k_marchp; not valid for GC_MARCH=regs or GC_SWEEP=edge)
NCU_TRAFFIC_BYTES = {"xsweep": 4.385e9, "ysweep": 3.906e9}
METRIC = "fp64 cell updates/sec per level step (device-timed)"
UNIT = "cell updates/s"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)).get("hbm_gbs", 6650.0), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    def __init__(self, index):
        self.rows = []
        q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
            "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + q, "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 6:
                continue
            try:
                mx = float(f[1])
                if t0 - 0.05 <= ts <= t1 + 0.15:
                    sm.append(float(f[0]))
                    for n, v in zip(names, f[2:6]):
                        if v.lower().startswith("active"):
                            reasons.add(n)
            except ValueError:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


# ---- N > 1: replicas only.  One process per GPU, each advancing its own copy of the level; no data-path collective.
# The only exchanges are a barrier on both sides of a timed region and the max over ranks of its duration.
def init_ranks(backend="nccl", device=None):
    """-> (rank, world, local_rank, dist or None) from torchrun's environment; joins the process group when world > 1."""
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1:
        return rank, world, local, None
    import torch.distributed as dist
    if device is not None:
        dist.init_process_group(backend, device_id=device)
    else:
        dist.init_process_group(backend)
    return rank, world, local, dist


def max_over_ranks(x, dist, device="cpu"):
    """the slowest rank's value of a duration (every rank gets it); x itself without a process group"""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.item()


def job_rate(units_per_rank, world, seconds):
    """whole-job throughput of `world` replicas that each processed units_per_rank in `seconds` (the max over ranks)"""
    return world * units_per_rank / seconds


def oracle_rate(n, steps, warmup=0):
    """The oracle as it stands, one thread: config-5 recipe at n x n, one patch.  -> (updates/s, seconds)"""
    import workloads
    from oracle import gco
    from harness import driver
    wl = workloads.cfg5(n)
    L = driver.setup_level(gco.Context(**wl.params), wl)
    dt = driver.probe_dt(L, wl.cfl)
    for _ in range(warmup):
        L.fill_ghost(None, 1.0); st = L.step(dt); dt = wl.cfl / st["s_over_dx_max"]
    t0 = time.time()
    for _ in range(steps):
        L.fill_ghost(None, 1.0); st = L.step(dt); dt = wl.cfl / st["s_over_dx_max"]
    el = time.time() - t0
    return n * n * steps / el, el


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = 1024
    rate, el = oracle_rate(n, args.steps, args.warmup)
    sample = "config-5 recipe at %dx%d (one patch), %d steps, single thread" % (n, n, args.steps)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / max(args.steps, 1), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5 spherical single level, oracle sample", "sample": sample},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--n", type=int, default=8192, help="level is n x n cells")
    ap.add_argument("--side", type=int, default=256, help="patch side")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--sweep", action="store_true", help="also report every tiling 16..256 in config.tilings")
    ap.add_argument("--gauges", type=int, default=0,
                    help="bind this many seeded gauges and record them into a device-resident series every step (DESIGN.md 3.10)")
    ap.add_argument("--manning", type=float, default=0.0,
                    help="Manning n of the friction step (DESIGN.md 3.9); 0 = off, as BASELINE.json's configs state no n")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import workloads
    from paper_1901_06798_b200 import binding
    from harness import driver

    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    rank, world, local, dist = init_ranks("nccl", torch.device("cuda", local))
    dev = "cuda:%d" % local
    W = max(args.warmup, 3)
    n = args.n
    wl = workloads.cfg5(n)
    if args.manning > 0.0:
        wl.params = dict(wl.params, manning_n=args.manning)
    ctx = binding.Context(device=dev, **wl.params)

    def make(side):
        L = ctx.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, workloads.tile(n, n, side))
        # inputs generated on the host in row blocks (bounded memory), handed over through the C ABI
        rows = max(1, (1 << 24) // n)
        for j0 in range(0, n, rows):
            nr = min(rows, n - j0)
            b, h, hu, hv = wl.fields(i0=0, j0=j0, nx=n, ny=nr)
            L.set_global("b", b, 0, j0); L.set_global("h", h, 0, j0); L.set_global("hu", hu, 0, j0); L.set_global("hv", hv, 0, j0)
        L.fill_ghost_b()
        return L

    def timed(L, K, warm):
        dt0 = driver.probe_dt(L, wl.cfl)
        dt_dev = torch.tensor([dt0], dtype=torch.float64, device=dev)
        series = None
        if args.gauges > 0:      # seeded points, each bound to the patch that holds it; one record per step, kept on the device
            rng = np.random.default_rng(1901067985)
            pts = np.stack([wl.xlo + rng.uniform(0.0, 1.0, args.gauges) * n * wl.dx * (1 - 1e-12),
                            wl.ylo + rng.uniform(0.0, 1.0, args.gauges) * n * wl.dy * (1 - 1e-12)], axis=1)
            L.gauges_bind([driver.GaugeRecorder.patch_of(L, x, y) for x, y in pts], pts)
            series = torch.empty((max(K, warm), args.gauges, 4), dtype=torch.float64, device=dev)
            torch.cuda.synchronize()
        def one_step(k):
            L.fill_ghost(None, 1.0)
            if series is not None:
                L.gauges_sample_into(series[k])      # one record per step, straight into the device-resident series
            L.step_auto(dt_dev, wl.cfl)
        for k in range(warm):
            one_step(k)
        torch.cuda.synchronize()
        if dist: dist.barrier()
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        lc0 = ctx.launch_count()
        e0.record()
        for k in range(K):
            one_step(k)
        e1.record()
        torch.cuda.synchronize()
        if dist: dist.barrier()
        ms = e0.elapsed_time(e1)
        launches = ctx.launch_count() - lc0
        # same K steps again with the library's per-kernel event brackets (separate pass: brackets perturb a little)
        ctx.profile(True)
        for k in range(K):
            one_step(k)
        prof = ctx.profile_read()
        ctx.profile(False)
        st = L.stats()
        assert st["nan_seen"] == 0 and np.isfinite(dt_dev.item())
        return ms, launches, prof

    L = make(args.side)
    sampler = ClockSampler(local)
    time.sleep(0.3)
    t0 = time.time()
    ms, launches, prof = timed(L, args.steps, W)
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = max_over_ranks(ms, dist, dev)
    cells = n * n
    value = job_rate(cells * args.steps, world, ms * 1e-3)

    # end to end through the C ABI with HOST buffers: every step copies the state host -> device and back (the paper's own
    # pipeline) around fill + step; pinned host memory
    Ke = args.e2e_steps
    host = [torch.empty((n, n), dtype=torch.float64).pin_memory() for _ in range(3)]
    for k, f in enumerate(("h", "hu", "hv")):
        host[k].copy_(torch.from_numpy(L.get_global(f)))
    hnp = [t.numpy() for t in host]
    dt = driver.probe_dt(L, wl.cfl)
    torch.cuda.synchronize()
    if dist: dist.barrier()
    w0 = time.time()
    for _ in range(Ke):
        for k, f in enumerate(("h", "hu", "hv")):
            L.set_global(f, hnp[k])
        L.fill_ghost(None, 1.0)
        st = L.step(dt)
        dt = wl.cfl / st["s_over_dx_max"]
        for k, f in enumerate(("h", "hu", "hv")):
            ctx._chk(binding.lib().gc_level_get_global(L.h, k, 0, hnp[k].ctypes.data, 0, n, 0, 0, n, n), "get")
    torch.cuda.synchronize()
    e2e_s = time.time() - w0
    e2e_s = max_over_ranks(e2e_s, dist, dev)
    e2e = job_rate(cells * Ke, world, e2e_s)

    tilings = None
    if args.sweep and rank == 0:
        tilings = {}
        L.destroy(); L = None
        for side in (16, 32, 64, 128, 256):
            Ls = make(side)
            m, _, pr = timed(Ls, args.steps, W)
            tilings[str(side)] = {"updates_per_s": cells * args.steps / (m * 1e-3), "ms_per_step": m / args.steps,
                                  "kernel_ms_per_step": {k: v[0] / args.steps for k, v in pr.items() if v[1]}}
            Ls.destroy()

    if rank != 0:
        return
    hbm_peak, which = peaks()
    fp64_peak = ctx.fp64_peak()
    # dominant kernel = the largest slot of the per-kernel brackets
    dom = max(prof, key=lambda k: prof[k][0])
    dom_ms = prof[dom][0] / max(prof[dom][1], 1)
    share = {k: v[0] / max(sum(x[0] for x in prof.values()), 1e-12) for k, v in prof.items() if v[1]}
    # cells one launch of the dominant kernel updates: the x-sweep also covers the 4 ghost rows of every patch (S-5)
    per_launch = {"xsweep": cells * (1.0 + 4.0 / args.side), "ysweep": float(cells)}.get(dom, float(cells))
    flop_sweep = FLOP_PER_SWEEP.get(dom, 411.0)
    alu_achieved = flop_sweep * per_launch / (dom_ms * 1e-3) / 1e12
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    slot_peak = nsm * 64.0 * (clocks.get("sm_mhz") or 1965.0) * 1e6      # fp64 pipe: 64 lanes per SM per clock
    slot_frac = FP64_SLOTS_PER_SWEEP.get(dom, 394.0) * per_launch / (dom_ms * 1e-3) / slot_peak
    default_kernels = True
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5: spherical single level %dx%d at 0.5 arcmin, %dx%d patches of side %d, ghost fill + level step"
                               % (n, n, n // args.side, n // args.side, args.side),
                   "l2": "inputs (%.1f GB pool) larger than L2, no flush" % (L.ncells * 8 * 10 * (1 + 4 / args.side) ** 2 / 1e9 if L else 0),
                   "parallelism": "replicas only" if world > 1 else "single GPU", "cfl": wl.cfl, "fmad": False,
                   "manning_n": args.manning, "gauges": args.gauges},
        "clocks": clocks,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 3 * cells * 8, "d2h_bytes_per_step": 3 * cells * 8 + 40,
                "steps": Ke, "note": "state copied host->device and back every step through the C ABI (P:166 pipeline)"},
        "gpu_launches": int(launches),
        "roofline": {"bound": "alu", "kernel": dom, "achieved": alu_achieved, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                     "frac": alu_achieved / (fp64_peak / 1e12), "traffic": NCU_TRAFFIC_BYTES.get(dom) if default_kernels else None,
                     "peak_source": "DFMA micro-benchmark in this run (gc_probe_fp64_peak = 2 flop x 64 lanes x SMs x clock); "
                                    "the scheme is compiled without FMA contraction, so add/mul code tops out at 0.5",
                     "flop_per_cell_per_sweep": flop_sweep, "cells_per_launch": per_launch, "kernel_ms": dom_ms,
                     "fp64_pipe_slot_frac": slot_frac, "kernel_share_of_step": share},
        "hbm": {"achieved_gbs": BYTES_PER_UPDATE * (cells * args.steps / (ms * 1e-3)) / 1e9, "peak_gbs": hbm_peak,
                "frac": BYTES_PER_UPDATE * (cells * args.steps / (ms * 1e-3)) / 1e9 / hbm_peak, "of": which,
                "bytes_per_update": BYTES_PER_UPDATE},
    }
    if tilings:
        out["config"]["tilings"] = tilings
    if not args.no_cpu:
        rate, el = oracle_rate(1024, 60)
        out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": "config-5 recipe at 1024x1024 (one patch), 60 steps, %.1f s" % el}
    print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
