"""Per-kernel instruction counts and DRAM traffic of the sweep kernels, from an ncu capture, for bench.py's roofline.

    python -m paper_1901_06798_b200.counts gpurun_out/<capture>.ncu-rep --n 8192 --side 256 [--out profiles/r02_counts.json]

The capture is the one the profiling recipe prescribes (`ncu --set full --clock-control none --import-source on
-k regex:k_marchp ... python bench.py --steps 2 --warmup 3 --no-cpu --no-tilings --no-e2e`); this script reads its raw and
SASS-source pages through `ncu -i`, divides by the cells one launch updates, and stores the result together with a hash of the
kernel sources.  bench.py prints the counts only while that hash still matches the tree (a stale count is worse than none).
"""
import argparse
import collections
import csv
import hashlib
import io
import json
import os
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def source_hash():
    """sha256 over what the sweep kernels are compiled from: gc_sweep.cu and the internal headers beside it (gc_internal.h, *.cuh);
    the public headers only declare the ABI and are left out, so that a new entry point does not make the counts stale"""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_1901_06798_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f == "gc_sweep.cu" or f.endswith((".cuh", ".h")):
            h.update(f.encode()); h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()


def _ncu(rep, *page):
    return subprocess.run(["ncu", "-i", rep] + list(page), capture_output=True, text=True, check=True).stdout


def _sweep_of(kernel_name):
    if "k_marchp<(int)0" in kernel_name or "k_marchp<0" in kernel_name:
        return "xsweep"
    if "k_marchp<(int)1" in kernel_name or "k_marchp<1" in kernel_name:
        return "ysweep"
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("rep")
    ap.add_argument("--n", type=int, default=8192)
    ap.add_argument("--side", type=int, default=256)
    ap.add_argument("--out", default=os.path.join(ROOT, "profiles", "r02_counts.json"))
    ap.add_argument("--x-cells", type=float, default=0.0,
                    help="cells one x-sweep launch updates (bench.py prints it as roofline.cells_per_launch / config.tilings[side]."
                         "xsweep_cells_per_launch); default: n * (n + 4), the regular tiling with chains (only the level's own 4 ghost rows)")
    a = ap.parse_args()
    cells = {"xsweep": a.x_cells if a.x_cells > 0 else float(a.n) * (a.n + 4), "ysweep": float(a.n * a.n)}

    raw = list(csv.reader(io.StringIO(_ncu(a.rep, "--page", "raw", "--csv"))))
    hdr = raw[0]
    per = {}
    for r in raw[2:]:
        d = dict(zip(hdr, r))
        k = _sweep_of(d.get("Kernel Name", ""))
        if k is None or k in per:
            continue                                     # first captured launch of each sweep
        f = lambda name: float(d[name].replace(",", ""))
        tunit = raw[1][hdr.index("gpu__time_duration.sum")]
        per[k] = {"duration_ms": f("gpu__time_duration.sum") * {"second": 1e3, "msecond": 1.0, "usecond": 1e-3, "nsecond": 1e-6}.get(tunit, 1.0),
                  "dram_bytes_per_launch": None, "registers": int(f("launch__registers_per_thread")),
                  "warp_inst": f("smsp__inst_executed.sum"),
                  "fp64_pipe_pct": f("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"),
                  "issue_active_pct": f("smsp__issue_active.avg.pct_of_peak_sustained_active")}
        rd, wr = f("dram__bytes_read.sum"), f("dram__bytes_write.sum")
        units = raw[1][hdr.index("dram__bytes_read.sum")]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(units, 1.0)
        per[k]["dram_bytes_per_launch"] = (rd + wr) * scale

    src = _ncu(a.rep, "--page", "source", "--csv", "--print-source", "sass")
    kern, hdr2, seen = None, None, set()
    ops = collections.defaultdict(collections.Counter)
    for r in csv.reader(io.StringIO(src)):
        if len(r) >= 2 and r[0] == "Kernel Name":
            k = _sweep_of(r[1])
            kern = k if (k and k not in seen) else None
            if kern:
                seen.add(kern)
            hdr2 = None
            continue
        if r and r[0] == "Address":
            hdr2 = r
            continue
        if kern and hdr2 and len(r) > 6:
            d = dict(zip(hdr2, r))
            t = d["Source"].split()
            op = (t[1] if t[0].startswith("@") else t[0]).split(".")[0]
            ops[kern][op] += int(d["Thread Instructions Executed"])
            ops[kern]["_all"] += int(d["Thread Instructions Executed"])
    kernels = {}
    for k in ("xsweep", "ysweep"):
        c = cells[k]
        o = ops[k]
        dmul, dadd, dfma, dsetp = (o[x] / c for x in ("DMUL", "DADD", "DFMA", "DSETP"))
        kernels[k] = dict(per[k], cells_per_launch=c, thread_inst_per_cell=o["_all"] / c,
                          dmul_per_cell=dmul, dadd_per_cell=dadd, dfma_per_cell=dfma, dsetp_per_cell=dsetp,
                          flop_per_cell=dmul + dadd + 2.0 * dfma, fp64_slots_per_cell=dmul + dadd + dfma + dsetp,
                          top_opcodes={x: round(v / c, 2) for x, v in o.most_common(16) if x != "_all"})
    out = {"source_sha256": source_hash(), "capture": os.path.basename(a.rep), "n": a.n, "side": a.side, "kernels": kernels}
    with open(a.out, "w") as f:
        json.dump(out, f, indent=1, sort_keys=True)
    print(json.dumps(out, indent=1, sort_keys=True))


if __name__ == "__main__":
    main()
