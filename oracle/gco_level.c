/* gco_level.c -- ORACLE (test infrastructure).  Level storage, metric tables, ghost fill,
 * the level step (x-sweep then y-sweep, eqs. 13-14), wet mask and mass.
 * Readings: DESIGN.md 3.2 (storage), 3.5 (sphere), 3.6 (ghost fill), 3.4 (ranges, clean-up).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "gco_int.h"

static double max2(double a, double b) { return a > b ? a : b; }

int gco_ctx_create(const gco_params *P, gco_ctx **out)
{
    if (!P || !out) return GCO_ERR_BADARG;
    gco_ctx *c = calloc(1, sizeof *c);
    if (!c) return GCO_ERR_NOMEM;
    c->P = *P;
    *out = c;
    return GCO_OK;
}
int gco_ctx_destroy(gco_ctx *c) { free(c); return GCO_OK; }

/* per global row j (index j+2 in the tables, j = -2..ny+1):
 * kappa_j = (pi/180) R^2 (sin(phi_{j+1/2}) - sin(phi_{j-1/2})) / dy   [m^2 per deg^2]
 * e_x = R pi/180, e_y(edge j) = R cos(phi_{j-1/2}) pi/180  (edge j = lower edge of row j).
 * Ghost rows outside a wall are mirrored together with the state; Cartesian: all 1. */
static void build_metric(gco_level *L)
{
    const gco_params *P = &L->ctx->P;
    int64_t ny = L->nyl, j;
    int64_t nr = ny + 4, ne = ny + 5;
    L->kappa = malloc(sizeof(double) * nr);
    L->rdx = malloc(sizeof(double) * nr);
    L->rdy = malloc(sizeof(double) * nr);
    L->ey = malloc(sizeof(double) * ne);
    const double PI = 3.14159265358979323846;
    const double d2r = PI / 180.0;
    if (P->coord == 0) {
        for (j = 0; j < nr; j++) L->kappa[j] = 1.0;
        for (j = 0; j < ne; j++) L->ey[j] = 1.0;
        L->ex = 1.0;
    } else {
        double R = P->earth_radius;
        L->ex = R * d2r;
        for (j = -2; j <= ny + 2; j++) { /* edges */
            double lat = (L->ylo + (double)j * L->dy) * d2r;
            L->ey[j + 2] = R * cos(lat) * d2r;
        }
        for (j = -2; j <= ny + 1; j++) { /* rows */
            double lat0 = (L->ylo + (double)j * L->dy) * d2r;
            double lat1 = (L->ylo + (double)(j + 1) * L->dy) * d2r;
            L->kappa[j + 2] = d2r * (R * R) * (sin(lat1) - sin(lat0)) / L->dy;
        }
        if (P->bc[2] == 1) { /* wall at ylo: mirror rows -1,-2 and edges -1,-2 */
            L->kappa[1] = L->kappa[2]; L->kappa[0] = L->kappa[3];
            L->ey[1] = L->ey[3]; L->ey[0] = L->ey[4];
        }
        if (P->bc[3] == 1) { /* wall at yhi: rows ny, ny+1 mirror ny-1, ny-2; edges ny+1, ny+2 mirror ny-1, ny-2 */
            L->kappa[ny + 2] = L->kappa[ny + 1]; L->kappa[ny + 3] = L->kappa[ny];
            L->ey[ny + 3] = L->ey[ny + 1]; L->ey[ny + 4] = L->ey[ny];
        }
    }
    for (j = 0; j < nr; j++) {
        L->rdx[j] = 1.0 / (L->kappa[j] * L->dx);
        L->rdy[j] = 1.0 / (L->kappa[j] * L->dy);
    }
}

int gco_level_metric(const gco_level *L, double *kappa, double *rdx, double *rdy, double *ey)
{
    int64_t nr = L->nyl + 4, ne = L->nyl + 5;
    if (kappa) memcpy(kappa, L->kappa, sizeof(double) * nr);
    if (rdx) memcpy(rdx, L->rdx, sizeof(double) * nr);
    if (rdy) memcpy(rdy, L->rdy, sizeof(double) * nr);
    if (ey) memcpy(ey, L->ey, sizeof(double) * ne);
    return GCO_OK;
}

/* which patch's interior holds global cell (gi,gj)?  -1 if none.  Linear search. */
int gco_find_patch(const gco_level *L, int64_t gi, int64_t gj)
{
    int q;
    for (q = 0; q < L->np; q++) {
        const gco_patch *Q = &L->pat[q];
        if (gi >= Q->i0 && gi < (int64_t)Q->i0 + Q->nx && gj >= Q->j0 && gj < (int64_t)Q->j0 + Q->ny) return q;
    }
    return -1;
}

int gco_level_create(gco_ctx *ctx, int level, double xlo, double ylo, double dx, double dy,
                     int64_t nxl, int64_t nyl, int ratio, int np, const gco_patch *pat, gco_level **out)
{
    int p, f, w;
    if (!ctx || !out || np < 0 || nxl < 1 || nyl < 1 || !(dx > 0.0) || !(dy > 0.0) || ratio < 1) return GCO_ERR_BADARG;
    for (p = 0; p < np; p++) {
        if (pat[p].nx < 2 || pat[p].ny < 2 || pat[p].i0 < 0 || pat[p].j0 < 0 ||
            (int64_t)pat[p].i0 + pat[p].nx > nxl || (int64_t)pat[p].j0 + pat[p].ny > nyl) return GCO_ERR_BADARG;
        if (level > 1 && (pat[p].i0 % ratio || pat[p].j0 % ratio || pat[p].nx % ratio || pat[p].ny % ratio))
            return GCO_ERR_BADARG; /* fine patches are aligned with coarse cells */
    }
    gco_level *L = calloc(1, sizeof *L);
    if (!L) return GCO_ERR_NOMEM;
    L->ctx = ctx; L->level = level; L->xlo = xlo; L->ylo = ylo; L->dx = dx; L->dy = dy;
    L->nxl = nxl; L->nyl = nyl; L->ratio = ratio; L->np = np;
    L->pat = malloc(sizeof(gco_patch) * (np > 0 ? np : 1));
    L->off = malloc(sizeof(int64_t) * (np + 1));
    memcpy(L->pat, pat, sizeof(gco_patch) * np);
    L->off[0] = 0; L->ncells = 0;
    for (p = 0; p < np; p++) {
        L->off[p + 1] = L->off[p] + (int64_t)(pat[p].nx + 4) * (pat[p].ny + 4);
        L->ncells += (int64_t)pat[p].nx * pat[p].ny;
    }
    int64_t tot = L->off[np] > 0 ? L->off[np] : 1;
    for (w = 0; w < 2; w++) for (f = 0; f < 3; f++) L->q[w][f] = calloc(tot, sizeof(double));
    L->b = calloc(tot, sizeof(double));
    L->cur = 0;
    build_metric(L);
    /* ghost source map: for every ghost cell, >=0 same-level source patch, -1 coarse, -2 outside domain */
    L->gsrc = malloc(sizeof(int32_t) * tot);
    for (p = 0; p < np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4, i, j;
        for (j = 0; j < Pp->ny + 4; j++) for (i = 0; i < pitch; i++) {
            int64_t gi = (int64_t)Pp->i0 + i - 2, gj = (int64_t)Pp->j0 + j - 2;
            int32_t v;
            if (i >= 2 && i < Pp->nx + 2 && j >= 2 && j < Pp->ny + 2) v = p;
            else if (gi < 0 || gi >= nxl || gj < 0 || gj >= nyl) v = -2;
            else v = gco_find_patch(L, gi, gj);
            L->gsrc[L->off[p] + (int64_t)j * pitch + i] = v;
        }
    }
    *out = L;
    return GCO_OK;
}

int gco_level_destroy(gco_level *L)
{
    int w, f;
    if (!L) return GCO_OK;
    for (w = 0; w < 2; w++) for (f = 0; f < 3; f++) free(L->q[w][f]);
    free(L->b); free(L->pat); free(L->off); free(L->gsrc);
    free(L->kappa); free(L->rdx); free(L->rdy); free(L->ey);
    gco_flux_free(L);
    free(L);
    return GCO_OK;
}

double *gco_field(const gco_level *L, int field, int which)
{
    if (field == GCO_B) return L->b;
    return L->q[which == 0 ? L->cur : 1 - L->cur][field];
}

int gco_level_set_field(gco_level *L, int p, int field, const double *src, int64_t ld)
{
    if (!L || p < 0 || p >= L->np || field < 0 || field > 3 || !src) return GCO_ERR_BADARG;
    int pitch = L->pat[p].nx + 4, j;
    double *d = gco_field(L, field, 0) + L->off[p];
    for (j = 0; j < L->pat[p].ny + 4; j++) memcpy(d + (int64_t)j * pitch, src + j * ld, sizeof(double) * pitch);
    return GCO_OK;
}

int gco_level_get_field(const gco_level *L, int p, int field, int which, double *dst, int64_t ld)
{
    if (!L || p < 0 || p >= L->np || field < 0 || field > 3 || !dst) return GCO_ERR_BADARG;
    int pitch = L->pat[p].nx + 4, j;
    const double *s = gco_field(L, field, which) + L->off[p];
    for (j = 0; j < L->pat[p].ny + 4; j++) memcpy(dst + j * ld, s + (int64_t)j * pitch, sizeof(double) * pitch);
    return GCO_OK;
}

int gco_level_set_global(gco_level *L, int field, const double *src, int64_t ld,
                         int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    if (!L || field < 0 || field > 3 || !src) return GCO_ERR_BADARG;
    double *d = gco_field(L, field, 0);
    int p, i, j;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 0; j < Pp->ny + 4; j++) for (i = 0; i < pitch; i++) {
            int64_t gi = (int64_t)Pp->i0 + i - 2 - gi0, gj = (int64_t)Pp->j0 + j - 2 - gj0;
            if (gi < 0 || gi >= gnx || gj < 0 || gj >= gny) continue;
            d[L->off[p] + (int64_t)j * pitch + i] = src[gj * ld + gi];
        }
    }
    return GCO_OK;
}

int gco_level_get_global(const gco_level *L, int field, int which, double *dst, int64_t ld,
                         int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    if (!L || field < 0 || field > 3 || !dst) return GCO_ERR_BADARG;
    const double *s = gco_field(L, field, which);
    int p, i, j;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 2; j < Pp->ny + 2; j++) for (i = 2; i < Pp->nx + 2; i++) {
            int64_t gi = (int64_t)Pp->i0 + i - 2 - gi0, gj = (int64_t)Pp->j0 + j - 2 - gj0;
            if (gi < 0 || gi >= gnx || gj < 0 || gj >= gny) continue;
            dst[gj * ld + gi] = s[L->off[p] + (int64_t)j * pitch + i];
        }
    }
    return GCO_OK;
}

/* DESIGN.md 3.6 step (3): physical boundary.  x-faces over rows inside the domain, then y-faces
 * over all columns (corners = BC of BC).  Wall: mirror cell, normal momentum negated;
 * extrapolation: nearest interior cell.  fields[f] selects what is filled; sign[f][0/1] is the
 * factor under a wall for x-faces / y-faces. */
static void fill_physical(gco_level *L, double *const fld[], int nf, const double sgn[][2])
{
    const gco_params *P = &L->ctx->P;
    int p, i, j, f;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        int64_t o = L->off[p];
        /* x-faces */
        for (j = 0; j < Pp->ny + 4; j++) {
            int64_t gj = (int64_t)Pp->j0 + j - 2;
            if (gj < 0 || gj >= L->nyl) continue;
            for (i = 0; i < pitch; i++) {
                int64_t gi = (int64_t)Pp->i0 + i - 2;
                int64_t gs; int wall;
                if (gi < 0) { wall = P->bc[0]; gs = wall ? -1 - gi : 0; }
                else if (gi >= L->nxl) { wall = P->bc[1]; gs = wall ? 2 * L->nxl - 1 - gi : L->nxl - 1; }
                else continue;
                int is = (int)(gs - Pp->i0 + 2);
                for (f = 0; f < nf; f++) {
                    double v = fld[f][o + (int64_t)j * pitch + is];
                    fld[f][o + (int64_t)j * pitch + i] = wall ? sgn[f][0] * v : v;
                }
            }
        }
        /* y-faces */
        for (j = 0; j < Pp->ny + 4; j++) {
            int64_t gj = (int64_t)Pp->j0 + j - 2;
            int64_t gs; int wall;
            if (gj < 0) { wall = P->bc[2]; gs = wall ? -1 - gj : 0; }
            else if (gj >= L->nyl) { wall = P->bc[3]; gs = wall ? 2 * L->nyl - 1 - gj : L->nyl - 1; }
            else continue;
            int js = (int)(gs - Pp->j0 + 2);
            for (i = 0; i < pitch; i++)
                for (f = 0; f < nf; f++) {
                    double v = fld[f][o + (int64_t)js * pitch + i];
                    fld[f][o + (int64_t)j * pitch + i] = wall ? sgn[f][1] * v : v;
                }
        }
    }
}

/* same-level copy, DESIGN.md 3.6 step (1) ("copying cell values from adjacent level l+1 patches") */
static void fill_same(gco_level *L, double *const fld[], int nf)
{
    int p, i, j, f;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 0; j < Pp->ny + 4; j++) for (i = 0; i < pitch; i++) {
            int64_t c = L->off[p] + (int64_t)j * pitch + i;
            int32_t q = L->gsrc[c];
            if (q < 0 || q == p) continue;
            const gco_patch *Q = &L->pat[q];
            int64_t gi = (int64_t)Pp->i0 + i - 2, gj = (int64_t)Pp->j0 + j - 2;
            int64_t s = L->off[q] + (gj - Q->j0 + 2) * (int64_t)(Q->nx + 4) + (gi - Q->i0 + 2);
            for (f = 0; f < nf; f++) fld[f][c] = fld[f][s];
        }
    }
}

int gco_fill_ghost_b(gco_level *L)
{
    if (!L) return GCO_ERR_BADARG;
    double *const fld[1] = { L->b };
    const double sgn[1][2] = { {1.0, 1.0} };
    fill_same(L, fld, 1);
    fill_physical(L, fld, 1, sgn);
    return GCO_OK;
}

int gco_fill_ghost(gco_level *L, const gco_level *coarser, double alpha)
{
    if (!L) return GCO_ERR_BADARG;
    double *const fld[3] = { L->q[L->cur][0], L->q[L->cur][1], L->q[L->cur][2] };
    const double sgn[3][2] = { {1.0, 1.0}, {-1.0, 1.0}, {1.0, -1.0} };
    fill_same(L, fld, 3);
    if (coarser) {
        int rc = gco_fill_coarse(L, coarser, alpha, 0 /* ghosts only */);
        if (rc) return rc;
    } else {
        int64_t c;
        for (c = 0; c < L->off[L->np]; c++) if (L->gsrc[c] == -1) return GCO_ERR_STATE; /* uncovered ghost, no coarser level */
    }
    fill_physical(L, fld, 3, sgn);
    return GCO_OK;
}

/* P:52-57 eq. 2 needs h^(7/3) = h^2 * h^(1/3).  A library cbrt differs between compilers, so the cube root is the fixed
 * sequence of DESIGN.md 3.9: bit pattern / 3 + K as the seed (K minimises the seed's worst relative error, 3.2 %), then
 * three Halley steps y <- y (y^3 + 2x) / (2 y^3 + x); x positive and normal. */
double gco_cbrt(double x)
{
    uint64_t i;
    double y, y3;
    int k;
    memcpy(&i, &x, 8);
    i = i / 3u + 0x2A9F762500000000ull;
    memcpy(&y, &i, 8);
    for (k = 0; k < 3; k++) {
        y3 = (y * y) * y;
        y = y * ((y3 + 2.0 * x) / (2.0 * y3 + x));
    }
    return y;
}

/* P:52-57 eq. 1b-1c: (hu)_t = ... - D hu, (hv)_t = ... - D hv with D = g n^2 sqrt(hu^2 + hv^2) / h^(7/3) (eq. 2 read over the
 * momenta), as a fractional step that is implicit in hu, hv and explicit in D. */
void gco_friction(const gco_params *P, double dt, double h, double *hu, double *hv)
{
    double m, c, gam, d;
    if (!(P->manning_n > 0.0) || !(h > P->dry_tol) || !(h <= P->friction_depth)) return;
    m = sqrt(fma(*hu, *hu, (*hv) * (*hv)));
    c = gco_cbrt(h);
    gam = ((P->g * (P->manning_n * P->manning_n)) * m) / ((h * h) * c);
    d = fma(dt, gam, 1.0);
    *hu = *hu / d;
    *hv = *hv / d;
}

/* One patch of the level step: x-sweep on all rows, y-sweep on interior columns, dry clean-up.  Patches are independent inside a
 * level step (their ghost cells are filled beforehand); what they contribute to the level's statistics comes back per patch. */
static void step_patch(gco_level *L, int p, double dt, double *sdx_out, double *clipped_out, int64_t *nclip_out, int *nan_out)
{
    const gco_params *P = &L->ctx->P;
    double eps = P->dry_tol;
    double sdx = 0.0, clipped = 0.0;
    int64_t nclip = 0; int nan_seen = 0;
    int cur = L->cur, nxt = 1 - cur, i, j, k;
    {
        const gco_patch *Pp = &L->pat[p];
        int nx = Pp->nx, ny = Pp->ny, pitch = nx + 4, rows = ny + 4;
        int64_t o = L->off[p];
        const double *h = L->q[cur][0] + o, *hu = L->q[cur][1] + o, *hv = L->q[cur][2] + o, *b = L->b + o;
        double *hn = L->q[nxt][0] + o, *hun = L->q[nxt][1] + o, *hvn = L->q[nxt][2] + o;
        size_t sz = (size_t)pitch * rows;
        double *hs = calloc(sz, sizeof(double)), *hus = calloc(sz, sizeof(double)), *hvs = calloc(sz, sizeof(double));
        int nmax = (nx > ny ? nx : ny) + 5;
        double *rd = malloc(sizeof(double) * nmax), *ef = malloc(sizeof(double) * nmax);
        double *lin[4], *lout[3];
        for (k = 0; k < 4; k++) lin[k] = malloc(sizeof(double) * nmax);
        for (k = 0; k < 3; k++) lout[k] = malloc(sizeof(double) * nmax);
        double *fmx = NULL, *fpx = NULL, *fmy = NULL, *fpy = NULL;
        if (L->save_flux) { /* flux-like quantities for the registers */
            fmx = L->fmx + o * 3; fpx = L->fpx + o * 3; fmy = L->fmy + o * 3; fpy = L->fpy + o * 3;
        }
        double *lfm = malloc(sizeof(double) * 3 * nmax), *lfp = malloc(sizeof(double) * 3 * nmax);

        /* x-sweep: every row (ghost rows too, S-5); normal = hu, transverse = hv */
        for (j = 0; j < rows; j++) {
            int64_t gr = (int64_t)Pp->j0 + j; /* table index = global row + 2 */
            for (i = 0; i < pitch; i++) rd[i] = L->rdx[gr];
            for (i = 0; i < pitch + 1; i++) ef[i] = L->ex;
            int interior_row = (j >= 2 && j < ny + 2);
            gco_sweep_line(P, nx, h + (size_t)j * pitch, hu + (size_t)j * pitch, hv + (size_t)j * pitch,
                           b + (size_t)j * pitch, rd, ef, dt, lout[0], lout[1], lout[2], lfm, lfp,
                           interior_row, &sdx);
            for (i = 2; i < nx + 2; i++) {
                hs[(size_t)j * pitch + i] = lout[0][i];
                hus[(size_t)j * pitch + i] = lout[1][i];
                hvs[(size_t)j * pitch + i] = lout[2][i];
            }
            if (fmx) for (i = 2; i <= nx + 2; i++) for (k = 0; k < 3; k++) {
                fmx[((size_t)j * pitch + i) * 3 + k] = lfm[i * 3 + k];
                fpx[((size_t)j * pitch + i) * 3 + k] = lfp[i * 3 + k];
            }
        }
        if (L->save_flux) {
            memcpy(L->qs[0] + o, hs, sz * sizeof(double));
            memcpy(L->qs[1] + o, hus, sz * sizeof(double));
            memcpy(L->qs[2] + o, hvs, sz * sizeof(double));
        }
        /* y-sweep: interior columns; normal = hv, transverse = hu */
        for (i = 2; i < nx + 2; i++) {
            for (j = 0; j < rows; j++) {
                int64_t gr = (int64_t)Pp->j0 + j;
                lin[0][j] = hs[(size_t)j * pitch + i];
                lin[1][j] = hvs[(size_t)j * pitch + i];
                lin[2][j] = hus[(size_t)j * pitch + i];
                lin[3][j] = b[(size_t)j * pitch + i];
                rd[j] = L->rdy[gr];
                ef[j] = L->ey[gr];
            }
            ef[rows] = L->ey[(int64_t)Pp->j0 + rows];
            gco_sweep_line(P, ny, lin[0], lin[1], lin[2], lin[3], rd, ef, dt, lout[0], lout[1], lout[2],
                           lfm, lfp, 1, &sdx);
            for (j = 2; j < ny + 2; j++) {
                double hh = lout[0][j], uu = lout[2][j], vv = lout[1][j];
                /* dry clean-up, DESIGN.md 3.4 (S-9) */
                if (hh < eps && dt > 0.0) {
                    if (hh < 0.0) { nclip++; clipped += (-hh) * gco_cell_area(L, (int64_t)Pp->j0 + j - 2); }
                    hh = max2(hh, 0.0); uu = 0.0; vv = 0.0;
                }
                if (dt > 0.0) gco_friction(P, dt, hh, &uu, &vv);   /* DESIGN.md 3.9 (S-16) */
                if (hh != hh || uu != uu || vv != vv) nan_seen = 1;
                if (dt > 0.0) { /* dt = 0 probe leaves both buffers untouched */
                    hn[(size_t)j * pitch + i] = hh; hun[(size_t)j * pitch + i] = uu; hvn[(size_t)j * pitch + i] = vv;
                }
            }
            if (fmy) for (j = 2; j <= ny + 2; j++) for (k = 0; k < 3; k++) {
                fmy[((size_t)j * pitch + i) * 3 + k] = lfm[j * 3 + k];
                fpy[((size_t)j * pitch + i) * 3 + k] = lfp[j * 3 + k];
            }
        }
        free(hs); free(hus); free(hvs); free(rd); free(ef); free(lfm); free(lfp);
        for (k = 0; k < 4; k++) free(lin[k]);
        for (k = 0; k < 3; k++) free(lout[k]);
    }
    *sdx_out = sdx; *clipped_out = clipped; *nclip_out = nclip; *nan_out = nan_seen;
}

/* Threads for the level step's loop over patches (the N-core baseline SURVEY 8(d) asks for; default 1: the oracle is a
 * single-thread program unless a caller says otherwise).  Patches are independent inside a step and the statistics are
 * combined per patch in patch order afterwards, so no result bit depends on the thread count. */
static int g_threads = 1;
int gco_set_threads(int n) { if (n < 1) return GCO_ERR_BADARG; g_threads = n; return GCO_OK; }
int gco_get_threads(void) { return g_threads; }

/* One level step (P:140-142 step 1; eqs. 13-14): x-sweep on all rows, y-sweep on interior columns,
 * dry clean-up, swap buffers.  dt = 0 is a legal probe: state unchanged, speeds returned. */
int gco_level_step(gco_level *L, double dt, gco_step_stats *out)
{
    if (!L || !(dt >= 0.0)) return GCO_ERR_BADARG;
    double sdx = 0.0, clipped = 0.0;
    int64_t nclip = 0; int nan_seen = 0;
    int p, np = L->np;
    double *psdx = malloc(sizeof(double) * (np + 1)), *pclip = malloc(sizeof(double) * (np + 1));
    int64_t *pn = malloc(sizeof(int64_t) * (np + 1));
    int *pnan = malloc(sizeof(int) * (np + 1));
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(g_threads) if (g_threads > 1)
#endif
    for (p = 0; p < np; p++) step_patch(L, p, dt, &psdx[p], &pclip[p], &pn[p], &pnan[p]);
    for (p = 0; p < np; p++) {         /* patch order, whatever the thread count */
        sdx = max2(sdx, psdx[p]); clipped = clipped + pclip[p]; nclip += pn[p]; nan_seen |= pnan[p];
    }
    free(psdx); free(pclip); free(pn); free(pnan);
    if (dt > 0.0) {
        L->cur = 1 - L->cur;
        if (L->save_flux) gco_flux_accumulate_own(L, dt);
    }
    L->last.cfl_max = dt * sdx; L->last.s_over_dx_max = sdx; L->last.clipped_mass = clipped;
    L->last.n_clipped = nclip; L->last.nan_seen = nan_seen;
    if (out) *out = L->last;
    return GCO_OK;
}

double gco_cell_area(const gco_level *L, int64_t grow)
{
    return L->kappa[grow + 2] * L->dx * L->dy;
}

int gco_wet_mask(const gco_level *L, uint8_t *mask)
{
    if (!L || !mask) return GCO_ERR_BADARG;
    double eps = L->ctx->P.dry_tol;
    const double *h = L->q[L->cur][0];
    int64_t n = 0; int p, i, j;
    for (p = 0; p < L->np; p++) {
        int pitch = L->pat[p].nx + 4;
        for (j = 2; j < L->pat[p].ny + 2; j++) for (i = 2; i < L->pat[p].nx + 2; i++)
            mask[n++] = h[L->off[p] + (int64_t)j * pitch + i] > eps ? 1 : 0;
    }
    return GCO_OK;
}

/* sum of h*area over interior cells, patch order then row-major (fixed order) */
double gco_level_mass(const gco_level *L)
{
    const double *h = L->q[L->cur][0];
    double m = 0.0; int p, i, j;
    for (p = 0; p < L->np; p++) {
        int pitch = L->pat[p].nx + 4;
        for (j = 2; j < L->pat[p].ny + 2; j++) {
            double a = gco_cell_area(L, (int64_t)L->pat[p].j0 + j - 2);
            for (i = 2; i < L->pat[p].nx + 2; i++) m += h[L->off[p] + (int64_t)j * pitch + i] * a;
        }
    }
    return m;
}

int64_t gco_level_ncells(const gco_level *L) { return L->ncells; }
