#!/usr/bin/env python
"""bench.py -- the per-level time step (ghost fill + x-sweep + y-sweep + CFL reduction) on config 5 of BASELINE.json:
one spherical level of NxN cells (default 8192 x 8192, 0.5 arcmin) tiled into square patches, all resident in one pool.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--side S] [--n NCELLS] [--impl reference]

A "step" = gc_fill_ghost_step + gc_level_step_auto (dt chain on the device, no host sync) over the whole level
(gc_fill_ghost_step = gc_fill_ghost without the same-level copies the step does not read; --full-fill: gc_fill_ghost).
metric  = fp64 cell updates/s (interior cells x steps / device time, CUDA events, max over ranks).
config.tilings = the same step on the five tilings BASELINE.json's configs[4] names (sides 16 ... 256), each with its updates/s,
          HBM GB/s at 56 B per update and fp64-pipe slot fraction (N = 1 only).
roofline = the dominant sweep kernel against the DFMA rate measured in this run ("alu": the scheme is bound by the fp64 pipe,
          DESIGN.md 6).  Its per-cell instruction counts and its DRAM traffic come from profiles/r02_counts.json, which
          paper_1901_06798_b200/counts.py writes from an ncu capture together with a hash of the kernel sources; when the
          sources have changed since, the counts are NOT printed (null) and the roofline falls back to the algorithmic bytes.
e2e     = the same metric through the C ABI with HOST buffers: every step uploads its state from pinned host memory and reads the
          result back.  "value": copies overlapped with the kernels (gc_level_upload_state_async / download, three streams, two
          level pools used alternately, the pattern of P:174-186); "serial": copy, step, copy in sequence.
cpu_baseline = the oracle (oracle/, plain C) on the SAME workload (8192 x 8192 in patches of 256), its loop over patches on all
          host cores, core count stated, and on one core.
N > 1   = replicas only (the contract fixes one GPU per problem; no collective is invented): every rank advances its
          own copy of the workload; value = units all ranks processed / max time.  Launch with torch.distributed.run; --gpus must
          equal WORLD_SIZE.
--impl reference = the oracle alone, timed on the host cores on the same workload (rank 0 only).
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

BYTES_PER_UPDATE = 56.0   # read h, hu, hv, b + write h, hu, hv once; the two-pass design moves 112
METRIC = "fp64 cell updates/sec per level step (device-timed)"
UNIT = "cell updates/s"
COUNTS = os.path.join(ROOT, "profiles", "r02_counts.json")


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)).get("hbm_gbs", 6650.0), "measured"
    return 6650.0, "fallback"


def load_counts():
    """per-kernel counts of the committed ncu capture, or None when the sources have changed since it was taken"""
    if not os.path.exists(COUNTS):
        return None, "profiles/r02_counts.json missing"
    c = json.load(open(COUNTS))
    from paper_1901_06798_b200.counts import source_hash
    if c.get("source_sha256") != source_hash():
        return None, "kernel sources changed since the capture (hash differs): counts withheld"
    return c, "profiles/r02_counts.json (written by paper_1901_06798_b200/counts.py from %s)" % c.get("capture", "?")


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


def host_fields(wl, n):
    """the seeded analytic inputs of config 5 at every cell centre, generated on the host in row blocks -> dict of (n, n) arrays"""
    import numpy as np
    out = {f: np.empty((n, n)) for f in ("b", "h", "hu", "hv")}
    rows = max(1, (1 << 24) // n)
    for j0 in range(0, n, rows):
        nr = min(rows, n - j0)
        for f, v in zip(("b", "h", "hu", "hv"), wl.fields(i0=0, j0=j0, nx=n, ny=nr)):
            out[f][j0:j0 + nr] = v
    return out


def oracle_leg(wl, n, side, fields, steps, warmup, threads, budget_s=None, unsplit=False):
    """The oracle as it stands on the bench workload (n x n in patches of `side`), its loop over patches on `threads` host
    cores (0 = all).  steps = None: as many steps as fit budget_s after the first.  -> (updates/s, seconds, steps, threads)"""
    import workloads
    from oracle import gco
    nt = gco.set_threads(threads)
    L = gco.Context(**wl.params).level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, workloads.tile(n, n, side))
    for f in ("b", "h", "hu", "hv"):
        L.set_global(f, fields[f])
    L.fill_ghost_b(); L.fill_ghost(None, 1.0)
    dt = wl.cfl / L.step(0.0)["s_over_dx_max"]

    def one(dt):
        L.fill_ghost(None, 1.0)
        return wl.cfl / (L.step_unsplit(dt) if unsplit else L.step(dt))["s_over_dx_max"]
    for _ in range(warmup):
        dt = one(dt)
    t0 = time.time()
    dt = one(dt)
    first = time.time() - t0
    k = 1
    if steps is None:
        steps = max(1, min(50, int(budget_s / max(first, 1e-3))))
    while k < steps:
        dt = one(dt); k += 1
    el = time.time() - t0
    L.destroy(); gco.set_threads(1)
    return n * n * k / el, el, k, nt


def run_reference(args):
    """--impl reference: there is no reference implementation to install (/root/reference holds the paper only); the oracle, as it
    stands, is timed on the host cores on the same workload.  Rank 0 alone runs and prints; the other ranks exit 0 without work."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import workloads
    n, side = args.n, args.side
    wl = workloads.cfg5(n)
    fields = host_fields(wl, n)
    rate, el, k, nt = oracle_leg(wl, n, side, fields, max(args.steps, 1), args.warmup, 0, unsplit=args.scheme == "unsplit")
    sample = "cfg5 spherical %dx%d in patches of side %d (the whole workload), %d steps after %d warm-up, loop over patches on %d threads" \
             % (n, n, side, k, args.warmup, nt)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": k,
        "warmup": args.warmup, "ms_per_step": 1e3 * el / k, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5: spherical single level %dx%d at 0.5 arcmin, patches of side %d, ghost fill + level step (oracle)" % (n, n, side),
                   "sample": sample},
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": nt, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--n", type=int, default=8192, help="level is n x n cells")
    ap.add_argument("--side", type=int, default=256, help="patch side of the headline line")
    ap.add_argument("--e2e-steps", type=int, default=4)
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--no-tilings", action="store_true", help="skip config.tilings (sides 16 ... 256)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the end-to-end legs")
    ap.add_argument("--full-fill", action="store_true", help="gc_fill_ghost (every ghost cell) instead of gc_fill_ghost_step before each step")
    ap.add_argument("--no-chains", action="store_true", help="marching lines stop at every patch boundary (GC_OPT_CHAINS = 1): same bits")
    ap.add_argument("--seg", type=int, default=0, help="GC_OPT_MARCH_SEG: cells per marching segment (0: the library's choice)")
    ap.add_argument("--chain-max", type=int, default=0, help="GC_OPT_CHAINS = k: patches of k cells or more are not chained")
    ap.add_argument("--scheme", default="split", choices=("split", "unsplit"),
                    help="split: the paper's dimensionally split step (the headline); unsplit: the step with transverse Riemann solves "
                         "(DESIGN.md 3.13; fixed dt, no tilings / e2e legs)")
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
    unsplit = args.scheme == "unsplit"
    if unsplit:
        args.no_tilings = args.no_e2e = True
    assert args.gpus == world, "--gpus %d but WORLD_SIZE %d: launch N > 1 with torch.distributed.run (one rank per GPU)" % (args.gpus, world)
    dev = "cuda:%d" % local
    W = args.warmup
    n = args.n
    wl = workloads.cfg5(n)
    if args.manning > 0.0:
        wl.params = dict(wl.params, manning_n=args.manning)
    if args.seg:
        binding.DEFAULT_OPTIONS[binding.OPT_MARCH_SEG] = args.seg
    if args.no_chains:
        binding.DEFAULT_OPTIONS[binding.OPT_CHAINS] = 1
    elif args.chain_max >= 8:
        binding.DEFAULT_OPTIONS[binding.OPT_CHAINS] = args.chain_max
    ctx = binding.Context(device=dev, **wl.params)
    fields = host_fields(wl, n)

    def make(side):
        L = ctx.level_create(1, wl.xlo, wl.ylo, wl.dx, wl.dy, n, n, 1, workloads.tile(n, n, side))
        rows = max(1, (1 << 24) // n)          # handed over through the C ABI in row blocks (bounded staging)
        for j0 in range(0, n, rows):
            for f in ("b", "h", "hu", "hv"):
                L.set_global(f, fields[f][j0:j0 + rows], 0, j0)
        L.fill_ghost_b()
        return L

    def timed(L, K, warm, use_dist=True, full_fill=False):
        d = dist if use_dist else None
        dt0 = driver.probe_dt(L, wl.cfl)
        dt_dev = torch.tensor([dt0], dtype=torch.float64, device=dev)
        series = None
        if args.gauges > 0:      # seeded points, each bound to the patch that holds it; one record per step, kept on the device
            rng = np.random.default_rng(1901067985)
            pts = np.stack([wl.xlo + rng.uniform(0.0, 1.0, args.gauges) * n * wl.dx * (1 - 1e-12),
                            wl.ylo + rng.uniform(0.0, 1.0, args.gauges) * n * wl.dy * (1 - 1e-12)], axis=1)
            L.gauges_bind([driver.GaugeRecorder.patch_of(L, x, y) for x, y in pts], pts)
            series = torch.empty((max(K, warm, 1), args.gauges, 4), dtype=torch.float64, device=dev)
            torch.cuda.synchronize()

        # gc_fill_ghost_step: the ghost cells the split step reads (where marching lines run through chained patches the copy
        # between them is dead work; same bits); gauges and the unsplit step read other ghost cells: gc_fill_ghost
        step_fill = not (full_fill or args.full_fill or unsplit or series is not None)

        def one_step(k):
            if step_fill:
                L.fill_ghost_step(None, 1.0)
            else:
                L.fill_ghost(None, 1.0)
            if series is not None:
                L.gauges_sample_into(series[k])      # one record per step, straight into the device-resident series
            if unsplit:
                L.step_unsplit(dt0)                  # fixed dt (gc_level_step_unsplit returns its statistics to the host)
            else:
                L.step_auto(dt_dev, wl.cfl)
        for k in range(warm):
            one_step(k)
        torch.cuda.synchronize()
        if d: d.barrier()
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        lc0 = ctx.launch_count()
        # the library brackets each of its kernels with CUDA events on the launching stream during the timed steps themselves
        # (they cost nothing measurable: plain against bracketed passes alternating, profiles/r02_marchp.md), so that the
        # per-kernel times of the roofline object come from the same steps, at the same clock, as ms_per_step
        ctx.profile(True)
        e0.record()
        for k in range(K):
            one_step(k)
        e1.record()
        torch.cuda.synchronize()
        prof = ctx.profile_read()
        ctx.profile(False)
        if d: d.barrier()
        ms = e0.elapsed_time(e1)
        launches = ctx.launch_count() - lc0
        st = L.stats()
        assert st["nan_seen"] == 0 and np.isfinite(dt_dev.item())
        return ms, launches, prof

    cells = n * n
    L = make(args.side)
    xcells_full, xcells_step, ycells = L.sweep_cells()          # cells one launch of each marching sweep updates on this tiling
    sampler = ClockSampler(local)
    time.sleep(0.3)
    t0 = time.time()
    ms, launches, prof = timed(L, args.steps, W)
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = max_over_ranks(ms, dist, dev)
    value = job_rate(cells * args.steps, world, ms * 1e-3)

    hbm_peak, which = peaks()
    fp64_peak = ctx.fp64_peak()
    nsm = torch.cuda.get_device_properties(dev).multi_processor_count
    slot_peak = nsm * 64.0 * (clocks.get("sm_mhz") or 1965.0) * 1e6      # fp64 pipe: 64 lanes per SM per clock
    counts, counts_src = load_counts()

    def slot_fraction(xc, rate):
        """fp64-pipe issue slots per interior cell update (the x-sweep also covers the ghost rows a y line reads: xc cells per
        launch for n * n interior cells) x rate / peak"""
        if counts is None:
            return None
        kx, ky = counts["kernels"]["xsweep"], counts["kernels"]["ysweep"]
        return (kx["fp64_slots_per_cell"] * (xc / float(cells)) + ky["fp64_slots_per_cell"]) * rate / slot_peak

    # ---- end to end through the C ABI with HOST buffers (pinned): serial, then copies overlapped with the kernels
    e2e = None
    if not args.no_e2e:
        Ke = max(args.e2e_steps, 2)
        hin = [torch.from_numpy(fields[f]).clone().pin_memory() for f in ("h", "hu", "hv")]
        hout = [torch.empty((n, n), dtype=torch.float64).pin_memory() for _ in range(3)]
        hnp_in, hnp_out = [t.numpy() for t in hin], [t.numpy() for t in hout]
        dt = driver.probe_dt(L, wl.cfl)
        torch.cuda.synchronize()
        if dist: dist.barrier()
        w0 = time.time()
        for _ in range(Ke):
            for k, f in enumerate(("h", "hu", "hv")):
                L.set_global(f, hnp_in[k])
            L.fill_ghost_step(None, 1.0)
            st = L.step(dt)
            for k, f in enumerate(("h", "hu", "hv")):
                ctx._chk(binding.lib().gc_level_get_global(L.h, k, 0, hnp_out[k].ctypes.data, 0, n, 0, 0, n, n), "get")
        torch.cuda.synchronize()
        serial_s = max_over_ranks(time.time() - w0, dist, dev)
        # overlapped: two level pools used alternately, uploads and downloads on their own streams
        L2 = make(args.side)
        pools = [L, L2]
        dts = [torch.tensor([dt], dtype=torch.float64, device=dev) for _ in range(2)]
        s_up, s_dn = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)

        def pipelined(K):
            for s in range(K):
                P = pools[s % 2]
                P.upload_state_async(hin, s_up)
                P.fill_ghost_step(None, 1.0)
                P.step_auto(dts[s % 2], wl.cfl)
                P.download_state_async(hout, s_dn)
            s_dn.synchronize(); torch.cuda.synchronize()
        pipelined(2)                                   # first use allocates the staging planes
        if dist: dist.barrier()
        w0 = time.time()
        pipelined(Ke)
        over_s = max_over_ranks(time.time() - w0, dist, dev)
        assert np.isfinite(hnp_out[0]).all() and abs(float(hnp_out[0].mean()) - float(fields["h"].mean())) < 1.0
        L2.destroy()
        nbytes = 3 * cells * 8
        e2e = {"value": job_rate(cells * Ke, world, over_s), "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
               "steps": Ke, "serial": job_rate(cells * Ke, world, serial_s),
               "h2d_gbs": nbytes * Ke / over_s / 1e9,
               "note": "every step uploads h, hu, hv from pinned host memory and reads the new state back, through the C ABI. value: "
                       "gc_level_upload_state_async / gc_level_download_state_async on their own streams, two level pools used "
                       "alternately, so one step's copies overlap the neighbouring steps' kernels (P:174-186); serial: "
                       "gc_level_set_global, fill + step, gc_level_get_global in sequence (P:166)"}
        del hin, hout

    # ---- the five tilings of BASELINE.json configs[4] (N = 1 only: no barrier inside, nothing for other ranks to wait on)
    tilings = None
    if not args.no_tilings and world == 1:
        tilings = {}
        if L is not None:
            L.destroy(); L = None
        both_fills = not (args.full_fill or args.no_chains or unsplit or args.gauges > 0)
        for side in (16, 32, 64, 128, 256):
            Ls = make(side)
            xc = Ls.sweep_cells()[0 if (args.full_fill or unsplit) else 1]
            if side == args.side:
                m, pr = ms, prof                                # the headline run above
            else:
                m, _, pr = timed(Ls, args.steps, W, use_dist=False)
            mf = timed(Ls, args.steps, W, use_dist=False, full_fill=True)[0] if both_fills else m   # every ghost cell filled
            Ls.destroy()
            rate = cells * args.steps / (m * 1e-3)
            tilings[str(side)] = {"updates_per_s": rate, "ms_per_step": m / args.steps,
                                  "ms_per_step_full_fill": mf / args.steps,
                                  "hbm_gbs_at_56B": BYTES_PER_UPDATE * rate / 1e9, "hbm_frac": BYTES_PER_UPDATE * rate / 1e9 / hbm_peak,
                                  "fp64_pipe_slot_frac": slot_fraction(xc, rate), "xsweep_cells_per_launch": xc,
                                  "kernel_ms_per_step": {k: v[0] / args.steps for k, v in pr.items() if v[1]}}

    if rank != 0:
        if dist: dist.destroy_process_group()
        return
    # dominant kernel = the largest slot of the per-kernel brackets
    dom = max(prof, key=lambda k: prof[k][0])
    dom_ms = prof[dom][0] / max(prof[dom][1], 1)
    share = {k: v[0] / max(sum(x[0] for x in prof.values()), 1e-12) for k, v in prof.items() if v[1]}
    # cells one launch of the dominant kernel updates: the x-sweep also covers the ghost rows a y line reads (S-5; gc_level_sweep_cells)
    per_launch = {"xsweep": float(xcells_full if (args.full_fill or unsplit) else xcells_step), "ysweep": float(ycells)}.get(dom, float(cells))
    kc = counts["kernels"].get(dom) if counts and not unsplit else None
    if unsplit:
        # planes of 8 bytes per cell the kernels of DESIGN.md 3.13 must move: the edge kernels read h, hu, hv, b and write
        # (A-dQ, A+dQ, F~); the update reads those 18 and h, hu, hv and writes the new state
        ub = {"xsweep": 104.0, "ysweep": 104.0, "fused": 192.0}.get(dom, 56.0)
        gbs = ub * cells / (dom_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": {"xsweep": "k_uns_xedges", "ysweep": "k_uns_yedges", "fused": "k_uns_update"}.get(dom, dom),
                    "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak, "traffic": None,
                    "peak_source": "MEASURED_PEAKS.json" if which == "measured" else "fallback 6650 GB/s",
                    "bytes_per_cell": ub, "cells_per_launch": float(cells), "kernel_ms": dom_ms, "kernel_share_of_step": share}
    elif kc:
        achieved = kc["flop_per_cell"] * per_launch / (dom_ms * 1e-3) / 1e12
        traffic = kc["dram_bytes_per_launch"] if (n, args.side) == (counts.get("n"), counts.get("side")) else None
        roofline = {"bound": "alu", "kernel": dom, "achieved": achieved, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                    "frac": achieved / (fp64_peak / 1e12), "traffic": traffic,
                    "peak_source": "DFMA micro-benchmark in this run (gc_probe_fp64_peak = 2 flop x 64 lanes x SMs x clock)",
                    "flop_per_cell": kc["flop_per_cell"], "fp64_slots_per_cell": kc["fp64_slots_per_cell"],
                    "thread_inst_per_cell": kc["thread_inst_per_cell"], "cells_per_launch": per_launch, "kernel_ms": dom_ms,
                    "fp64_pipe_slot_frac": kc["fp64_slots_per_cell"] * per_launch / (dom_ms * 1e-3) / slot_peak,
                    "counts_source": counts_src, "kernel_share_of_step": share}
    else:
        gbs = BYTES_PER_UPDATE * per_launch / (dom_ms * 1e-3) / 1e9       # one sweep reads 4 planes and writes 3: 56 B per cell
        roofline = {"bound": "hbm", "kernel": dom, "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                    "traffic": None, "peak_source": "MEASURED_PEAKS.json" if which == "measured" else "fallback 6650 GB/s",
                    "cells_per_launch": per_launch, "kernel_ms": dom_ms, "counts_source": counts_src,
                    "note": "the kernel is bound by the fp64 pipe (DESIGN.md 6); its instruction counts are withheld because the "
                            "committed capture does not match the sources, so only the algorithmic-bytes figure is given",
                    "kernel_share_of_step": share}
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "cfg5: spherical single level %dx%d at 0.5 arcmin, %dx%d patches of side %d, ghost fill + level step"
                               % (n, n, n // args.side, n // args.side, args.side),
                   "l2": "inputs (%.1f GB pool) larger than L2, no flush" % (cells * 8 * 10 * (1 + 4 / args.side) ** 2 / 1e9),
                   "parallelism": "replicas only" if world > 1 else "single GPU", "cfl": wl.cfl,
                   "fma": "explicit, where DESIGN.md 3 writes it (both sides)", "manning_n": args.manning, "gauges": args.gauges,
                   "scheme": args.scheme,
                   "ghost_fill": "gc_fill_ghost (every ghost cell)" if (args.full_fill or unsplit or args.gauges > 0) else
                                 "gc_fill_ghost_step (the ghost cells the step reads: chained patches are read through, DESIGN.md 5); "
                                 "tilings[side].ms_per_step_full_fill is the same step after gc_fill_ghost"},
        "clocks": clocks, "gpu_launches": launches, "roofline": roofline,
        "hbm": {"achieved_gbs": BYTES_PER_UPDATE * value / world / 1e9, "peak_gbs": hbm_peak,
                "frac": BYTES_PER_UPDATE * value / world / 1e9 / hbm_peak, "of": which, "bytes_per_update": BYTES_PER_UPDATE},
    }
    if e2e:
        out["e2e"] = e2e
    if tilings:
        out["config"]["tilings"] = tilings
    if not args.no_cpu and world == 1:
        if L is not None:
            L.destroy()
        rate, el, k, nt = oracle_leg(wl, n, args.side, fields, None, 0, 0, budget_s=12.0, unsplit=unsplit)
        rate1, el1, k1, _ = oracle_leg(wl, n, args.side, fields, 1, 0, 1, unsplit=unsplit)
        out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": nt, "kind": "oracle",
                               "sample": "the bench workload itself (%dx%d in patches of side %d): %d steps in %.1f s, loop over patches on "
                                         "%d threads" % (n, n, args.side, k, el, nt),
                               "one_core": {"value": rate1, "steps": k1, "seconds": el1}}
    print(json.dumps(out))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
