"""Writes tests/golden/oracle_anchors.txt from the oracle alone (imports only oracle/, the seeded input recipes and the
host driver; nothing from the CUDA path):

    python tests/golden/make_golden.py

The paper (arXiv 1901.06798) prints no numeric worked example of the method -- its tables are run times on its own
hardware -- so there is no paper value to store.  These are regression anchors of the oracle's own
arithmetic, as C99 hex floats (exact): a later change to the oracle that moves one of them has to name, in its commit
message, the passage of the paper or the DESIGN.md reading that justifies it.  What the oracle must satisfy mathematically
is pinned elsewhere (tests/test_oracle_*.py: closed forms, invariants, brute force)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_anchors.txt")


def anchors():
    import workloads
    from oracle import gco
    from harness import driver                    # neutral AMR harness (host control code); nothing under paper_1901_06798_b200 is imported
    rows = []

    def put(key, values, cite):
        rows.append((key, [float(v).hex() for v in np.atleast_1d(values)], cite))

    # Riemann solver: f-waves and speeds of four canonical problems
    for name, args in (("dam_break_wet", (9.81, 1e-3, 2.0, 0.0, 0.0, -2.0, 1.0, 0.0, 0.0, -2.0)),
                       ("step_at_rest", (9.81, 1e-3, 3.0, 0.0, 0.0, -3.0, 2.5, 0.0, 0.0, -2.5)),
                       ("wall_dry_right", (9.81, 1e-3, 0.5, 0.3, 0.1, -0.5, 0.0, 0.0, 0.0, 0.8)),
                       ("oblique_flow", (9.81, 1e-3, 4000.0, 800.0, -300.0, -4000.0, 3999.5, 790.0, -310.0, -3999.0))):
        Z, s = gco.riemann(*args)
        put("riemann.%s.Z" % name, Z.ravel(), "P:122, DESIGN.md 3.3 R0-R8")
        put("riemann.%s.s" % name, s, "P:122, DESIGN.md 3.3 R4-R6")
    # config 1 (BASELINE.json configs[0]): 64 x 64, 100 steps -- dt sequence head, final mass, a row of cells
    wl = workloads.cfg1(64)
    L = driver.setup_level(gco.Context(**wl.params), wl)
    hist = driver.run_single_level(L, wl.nsteps, wl.cfl)
    put("cfg1.dt[0:3]", [d for d, _ in hist[:3]], "P:124-128 eq. 15, DESIGN.md 3.4")
    put("cfg1.dt[99]", hist[99][0], "P:124-128 eq. 15")
    put("cfg1.mass", L.mass(), "eq. 1a (conservation), closed basin")
    H, U = L.get_global("h"), L.get_global("hu")
    put("cfg1.h[32,0:64:9]", H[32, 0:64:9], "P:65-120 eqs. 4-14")
    put("cfg1.hu[20,0:64:9]", U[20, 0:64:9], "P:65-120 eqs. 4-14")
    # config 2 recipe at 64 x 64 (wet/dry shoreline), 60 steps
    wl = workloads.cfg2(64)
    L = driver.setup_level(gco.Context(**wl.params), wl)
    hist = driver.run_single_level(L, 60, wl.cfl)
    put("cfg2_64.wet_cells", float(L.wet_mask().sum()), "P:122 dry states, DESIGN.md 3.4 S-9")
    put("cfg2_64.clipped_cells", float(sum(s["n_clipped"] for _, s in hist)), "DESIGN.md 3.4 S-9")
    H, V = L.get_global("h"), L.get_global("hv")
    put("cfg2_64.h[10,40:64:3]", H[10, 40:64:3], "P:65-120, wetting and drying")
    put("cfg2_64.hv[33,30:64:5]", V[33, 30:64:5], "P:65-120, wetting and drying")
    # config 5 recipe at 96 x 96 on the sphere, 12 steps
    wl = workloads.cfg5(96)
    L = driver.setup_level(gco.Context(**wl.params), wl)
    hist = driver.run_single_level(L, 12, wl.cfl)
    put("cfg5_96.dt[11]", hist[11][0], "eq. 15 with the capacity function, DESIGN.md 3.5")
    put("cfg5_96.h[50,0:96:13]", L.get_global("h")[50, 0:96:13], "DESIGN.md 3.5 (lon/lat capacity form)")
    # friction (eq. 2): the cube-root sequence and one cell's step
    put("cbrt(2),cbrt(0.025),cbrt(4500)", [gco.cbrt(2.0), gco.cbrt(0.025), gco.cbrt(4500.0)], "DESIGN.md 3.9")
    put("friction(dt=1,h=2,hu=3,hv=4,n=0.025)", gco.friction(1.0, 2.0, 3.0, 4.0, manning_n=0.025), "P:52-57 eq. 1b-1c, 2; DESIGN.md 3.9")
    return rows


def main():
    with open(OUT, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ alone; key | C99 hex floats | passage that defines the quantity\n")
        for key, vals, cite in anchors():
            f.write("%s | %s | %s\n" % (key, " ".join(vals), cite))
    print(OUT)


if __name__ == "__main__":
    main()
