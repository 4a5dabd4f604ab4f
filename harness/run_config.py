"""Run one of the five BASELINE.json configurations on the GPU and report its end-to-end rate.

    python -m harness.run_config --config N [--scale S] [--max-steps M] [--max-wall SECONDS] [--graph K]

Prints ONE JSON line: total interior-cell updates over all levels / wall time of the whole run (ghost fills, level
steps, regrids incl. flag download and host clustering, average-down, fix-up), the kernel launches, and how far the run
got (steps, simulated time) when a cap stopped it.  Single-level configs (1, 2, 5) keep dt on the device
(gc_level_step_auto: no host synchronisation inside the run) and can replay the step as a CUDA graph of K steps.
The AMR configs (3, 4) go through driver.Hierarchy (host dt control, one synchronisation per level step).
Inputs: the seeded synthetic recipes of workloads/ (DESIGN.md 4).  GPU only: there is no CPU fallback.
"""
import argparse
import json
import time

import numpy as np


def fallback_of(L):
    """P:345 accounting of a level still alive at the end of the run: the share of the marching kernels' warp iterations in which
    some lane left the guarded open-ocean code, and the share of lane-level edges redone with the general code (0 / None for a
    level swept by the edge-parallel kernels)"""
    c = L.fallback_counts()
    if c["warp_iters"] == 0:
        return dict(level=int(L.level), cells=int(L.ncells), marching=False)
    return dict(level=int(L.level), cells=int(L.ncells), marching=True, warp_iters=int(c["warp_iters"]),
                warp_iter_fraction=c["fb_warp_iters"] / c["warp_iters"],
                edge_fraction=0.5 * (c["fb_solves"] + c["fb_fluxes"]) / (32.0 * c["warp_iters"]))


def run_single(cfg, wl, patches, max_steps, graph_k, device):
    import torch
    from paper_1901_06798_b200 import binding
    from harness import driver
    s = torch.cuda.Stream(device=device)
    with torch.cuda.stream(s):
        ctx = binding.Context(device=device, stream=s, **wl.params)
        L = driver.setup_level(ctx, wl, patches=patches)
        nsteps = wl.nsteps if max_steps is None else min(wl.nsteps, max_steps)
        dt0 = driver.probe_dt(L, wl.cfl)
        dt_dev = torch.tensor([dt0], dtype=torch.float64, device=device)
        t_dev = torch.zeros(1, dtype=torch.float64, device=device)

        def one():
            L.fill_ghost_step(None, 1.0)           # the ghost cells the step reads (every one of them unless patches are chained)
            t_dev.add_(dt_dev)                     # simulated time, accumulated on the device
            L.step_auto(dt_dev, wl.cfl)

        lcw = ctx.launch_count()
        for _ in range(3):                         # warm-up, then restore the initial state
            one()
        per_step = (ctx.launch_count() - lcw) // 3
        driver.set_initial(L, wl, state=True)
        dt_dev.fill_(dt0); t_dev.zero_()
        g = None
        if graph_k and graph_k > 1 and nsteps >= graph_k:
            # an even number of steps per graph: the NEW/OLD buffer roles are back where the capture started
            graph_k -= graph_k % 2
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=s):
                for _ in range(graph_k):
                    one()
            driver.set_initial(L, wl, state=True)
            dt_dev.fill_(dt0); t_dev.zero_()
        s.synchronize()
        lc0 = ctx.launch_count()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        w0 = time.time()
        e0.record(s)
        done = 0
        if g is not None:
            while done + graph_k <= nsteps:
                g.replay(); done += graph_k
        launched_by_graph = done * per_step        # kernels replayed from the graph are not counted by the library
        while done < nsteps:
            one(); done += 1
        e1.record(s)
        s.synchronize()
        wall = time.time() - w0
        st = L.stats()
        assert st["nan_seen"] == 0
        out = dict(levels=1, patches=int(len(L.patches)), steps=done, sim_time=float(t_dev.item()), updates=int(L.ncells) * done,
                   wall_s=wall, device_ms=e0.elapsed_time(e1), launches=int(ctx.launch_count() - lc0) + launched_by_graph,
                   graph_steps=int(graph_k or 0) if g is not None else 0, wet_cells=int(L.wet_mask().sum()), mass=L.mass(),
                   fallback=[fallback_of(L)])
        L.destroy()
    return out


def run_amr(cfg, wl, max_steps, max_wall, device, max_levels=None):
    import torch
    from paper_1901_06798_b200 import binding
    from harness import driver
    ctx = binding.Context(device=device, **wl.params)
    t_setup = time.time()
    H = driver.Hierarchy(ctx, wl, max_levels=max_levels)
    torch.cuda.synchronize()
    t_setup = time.time() - t_setup
    lc0 = ctx.launch_count()
    w0 = time.time()
    dt = H.probe()
    n = 0
    while H.t < wl.t_end and (max_steps is None or n < max_steps) and (max_wall is None or time.time() - w0 < max_wall):
        if H.t + dt > wl.t_end:
            dt = wl.t_end - H.t
        dt = H.step(dt)
        n += 1
    torch.cuda.synchronize()
    wall = time.time() - w0
    out = dict(levels=len(H.levels), patches=[int(len(L.patches)) for L in H.levels], cells=[int(L.ncells) for L in H.levels],
               steps=n, sim_time=H.t, t_end=wl.t_end, finished=bool(H.t >= wl.t_end), updates=int(H.updates), regrids=int(H.regrids),
               wall_s=wall, setup_s=t_setup, launches=int(ctx.launch_count() - lc0),
               fallback=[fallback_of(L) for L in H.levels])
    H.destroy()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, required=True, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--scale", type=int, default=None, help="coarse cells per side (config 4: in x); default = BASELINE.json's")
    ap.add_argument("--side", type=int, default=256, help="config 5: patch side")
    ap.add_argument("--max-steps", type=int, default=None)
    ap.add_argument("--max-wall", type=float, default=None)
    ap.add_argument("--max-levels", type=int, default=None)
    ap.add_argument("--boxes-from-start", action="store_true",
                    help="config 4: switch the forced coastal boxes on at t = 0 instead of 6 h / 6.5 h, so that all four levels exist at once")
    ap.add_argument("--graph", type=int, default=0, help="single-level configs: replay the step as a CUDA graph of this many steps")
    ap.add_argument("--device", default="cuda:0")
    ap.add_argument("--family", choices=["auto", "edge", "march"], default="auto", help="sweep kernel family (gc_ctx_set_option)")
    ap.add_argument("--seg", type=int, default=0, help="marching segment length in cells (0 = by level size)")
    a = ap.parse_args()
    import workloads
    from paper_1901_06798_b200 import binding
    binding.DEFAULT_OPTIONS[binding.OPT_SWEEP_FAMILY] = {"auto": 0, "edge": 1, "march": 2}[a.family]
    binding.DEFAULT_OPTIONS[binding.OPT_MARCH_SEG] = a.seg
    if a.config == 1:
        wl = workloads.cfg1(a.scale or 64); res = run_single(1, wl, None, a.max_steps, a.graph, a.device)
    elif a.config == 2:
        wl = workloads.cfg2(a.scale or 512); res = run_single(2, wl, None, a.max_steps, a.graph, a.device)
    elif a.config == 5:
        n = a.scale or 8192
        wl = workloads.cfg5(n); res = run_single(5, wl, workloads.tile(n, n, a.side), a.max_steps, a.graph, a.device)
    elif a.config == 3:
        wl = workloads.cfg3(a.scale or 256); res = run_amr(3, wl, a.max_steps, a.max_wall, a.device, a.max_levels)
    else:
        nx = a.scale or 1800
        wl = workloads.cfg4(nx, nx // 2)
        if a.boxes_from_start:
            wl.forced_boxes = tuple((lv, x0, x1, y0, y1, 0.0, t1) for lv, x0, x1, y0, y1, t0, t1 in wl.forced_boxes)
        res = run_amr(4, wl, a.max_steps, a.max_wall, a.device, a.max_levels)
    res.update(config=a.config, workload=wl.name, e2e_updates_per_s=res["updates"] / res["wall_s"], unit="cell updates/s")
    if "device_ms" in res:
        res["device_updates_per_s"] = res["updates"] / (res["device_ms"] * 1e-3)
    print(json.dumps(res))


if __name__ == "__main__":
    main()
