/* gco_bathy.c -- ORACLE (test infrastructure).  Time-dependent bathymetry: the seafloor-deformation source.
 *
 * P:52 has B = B(x, y, t); both of the paper's benchmarks start from "earthquake source deformation files ... converted to
 * deformation information on uniform grids" ("ground deformation file").  The paper gives no more than that; the
 * reading is DESIGN.md 3.12 (S-20): a deformation field dz on a uniform node grid, bilinear between nodes and zero outside the
 * grid, added to the bathymetry with a weight w that the driver takes from a linear ramp over [t0, t1]:
 *     b <- fma(w, dz(x_c, y_c), b)      for every storage cell of the level (ghost cells too) whose centre lies in the domain;
 * the water column h is left as it is -- the water rides on the seafloor, so the surface eta = h + b moves with it (that is
 * what makes a tsunami) -- and cells outside the domain are left to gco_fill_ghost_b.
 */
#include <math.h>
#include "gco_int.h"

/* dz at (x, y): node (m, n) of the grid sits at (x0 + m ddx, y0 + n ddy), m = 0..mx-1, n = 0..my-1, values row-major (n, m) */
double gco_deform_at(const gco_deform *D, double x, double y)
{
    double s = (x - D->x0) / D->ddx, t = (y - D->y0) / D->ddy;
    if (!(s >= 0.0) || !(t >= 0.0) || !(s <= (double)(D->mx - 1)) || !(t <= (double)(D->my - 1))) return 0.0;
    int64_t m = (int64_t)floor(s), n = (int64_t)floor(t);
    if (m > D->mx - 2) m = D->mx - 2;      /* the last node belongs to the last interval */
    if (n > D->my - 2) n = D->my - 2;
    double a = s - (double)m, c = t - (double)n;
    const double *z = D->dz + n * D->mx + m;
    double lo = (1.0 - a) * z[0] + a * z[1];
    double hi = (1.0 - a) * z[D->mx] + a * z[D->mx + 1];
    return (1.0 - c) * lo + c * hi;
}

int gco_bathy_update(gco_level *L, const gco_deform *D, double w)
{
    int p, i, j;
    if (!L || !D || !D->dz || D->mx < 2 || D->my < 2 || !(D->ddx > 0.0) || !(D->ddy > 0.0)) return GCO_ERR_BADARG;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 0; j < Pp->ny + 4; j++) for (i = 0; i < pitch; i++) {
            int64_t gi = (int64_t)Pp->i0 + i - 2, gj = (int64_t)Pp->j0 + j - 2;
            if (gi < 0 || gi >= L->nxl || gj < 0 || gj >= L->nyl) continue;
            double x = L->xlo + ((double)gi + 0.5) * L->dx, y = L->ylo + ((double)gj + 0.5) * L->dy;
            int64_t c = L->off[p] + (int64_t)j * pitch + i;
            L->b[c] = fma(w, gco_deform_at(D, x, y), L->b[c]);
        }
    }
    return GCO_OK;
}
