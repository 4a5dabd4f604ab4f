/* gco_amr.c -- ORACLE (test infrastructure).  Level-transfer operations of the AMR algorithm:
 * coarse-to-fine interpolation in space and time (P:143 step 2), fine-to-coarse averaging
 * ("updating", P:145 step 4), refinement flags and new-patch
 * initialisation at regrid.  Formulas the paper defers to LeVeque et al. (2011) are the
 * readings of DESIGN.md 3.6-3.7.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "gco_int.h"

static double max2(double a, double b) { return a > b ? a : b; }

/* minmod of two one-sided differences */
static double minmod(double a, double b)
{
    if (a * b <= 0.0) return 0.0;
    return (fabs(a) < fabs(b)) ? a : b;
}

/* DESIGN.md 3.6 step (2): value of one fine cell (global fine index gi,gj; fine bathymetry bf)
 * from the coarser level at time fraction alpha.  Coarse state in time: Q = Q_old + alpha (Q_new - Q_old)
 * (P:143).  In space: eta = h+b and the velocities are reconstructed linearly in the coarse cell
 * containing the fine cell centre, minmod slopes; any dry cell in the 5-point stencil -> slopes 0.
 * Interpolating eta (not h) keeps the flat ocean flat. */
static int interp_cell(const gco_level *C, int r, double alpha, int use_old, int64_t gi, int64_t gj,
                       double bf, double eps, double out[3])
{
    int64_t I = gi / r, J = gj / r; /* gi,gj >= 0 inside the domain */
    int cp = gco_find_patch(C, I, J);
    if (cp < 0) return GCO_ERR_STATE; /* not properly nested */
    const gco_patch *Q = &C->pat[cp];
    int pitch = Q->nx + 4;
    int64_t c0 = C->off[cp] + (int64_t)(J - Q->j0 + 2) * pitch + (I - Q->i0 + 2);
    const int64_t nb[5] = { c0, c0 - 1, c0 + 1, c0 - pitch, c0 + pitch }; /* C, W, E, S, N */
    double eta[5], u[5], v[5], hh[5];
    int k, anydry = 0;
    for (k = 0; k < 5; k++) {
        double q[3]; int f;
        for (f = 0; f < 3; f++) {
            double qn = C->q[C->cur][f][nb[k]];
            if (use_old) { double qo = C->q[1 - C->cur][f][nb[k]]; q[f] = qo + alpha * (qn - qo); }
            else q[f] = qn;
        }
        hh[k] = q[0];
        eta[k] = q[0] + C->b[nb[k]];
        if (q[0] > eps) { double rh = 1.0 / q[0]; u[k] = q[1] * rh; v[k] = q[2] * rh; }
        else { u[k] = 0.0; v[k] = 0.0; anydry = 1; }
    }
    if (!(hh[0] > eps)) { out[0] = 0.0; out[1] = 0.0; out[2] = 0.0; return GCO_OK; }
    double xi = ((double)(gi - I * r) + 0.5) / (double)r - 0.5;
    double ze = ((double)(gj - J * r) + 0.5) / (double)r - 0.5;
    double sx[3] = {0, 0, 0}, sy[3] = {0, 0, 0};
    if (!anydry) {
        sx[0] = minmod(eta[0] - eta[1], eta[2] - eta[0]); sy[0] = minmod(eta[0] - eta[3], eta[4] - eta[0]);
        sx[1] = minmod(u[0] - u[1], u[2] - u[0]);         sy[1] = minmod(u[0] - u[3], u[4] - u[0]);
        sx[2] = minmod(v[0] - v[1], v[2] - v[0]);         sy[2] = minmod(v[0] - v[3], v[4] - v[0]);
    }
    double ef = (eta[0] + xi * sx[0]) + ze * sy[0];
    double uf = (u[0] + xi * sx[1]) + ze * sy[1];
    double vf = (v[0] + xi * sx[2]) + ze * sy[2];
    double hf = max2(0.0, ef - bf);
    double huf = hf * uf, hvf = hf * vf;
    if (hf < eps) { huf = 0.0; hvf = 0.0; } /* clean-up rule */
    out[0] = hf; out[1] = huf; out[2] = hvf;
    return GCO_OK;
}

/* fills ghost cells whose source is the coarser level (all_cells = 0), or every interior cell not
 * marked in `keep` (regrid transfer: all_cells = 1, handled by gco_level_init_from). */
int gco_fill_coarse(gco_level *L, const gco_level *C, double alpha, int all_cells)
{
    double eps = L->ctx->P.dry_tol;
    int r = L->ratio, p, i, j, f;
    (void)all_cells;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 0; j < Pp->ny + 4; j++) for (i = 0; i < pitch; i++) {
            int64_t c = L->off[p] + (int64_t)j * pitch + i;
            if (L->gsrc[c] != -1) continue;
            double out[3];
            int rc = interp_cell(C, r, alpha, 1, (int64_t)Pp->i0 + i - 2, (int64_t)Pp->j0 + j - 2, L->b[c], eps, out);
            if (rc) return rc;
            for (f = 0; f < 3; f++) L->q[L->cur][f][c] = out[f];
        }
    }
    return GCO_OK;
}

/* P:136 "newly generated level l+1 grid patches get their initial solution from either copying data
 * from existing old level l+1 grid patches or, if no such grid patch exists, interpolating from
 * level l".  b of the new level must have been set already.  Interior cells only. */
int gco_level_init_from(gco_level *N, const gco_level *O, const gco_level *C)
{
    if (!N || !C) return GCO_ERR_BADARG;
    double eps = N->ctx->P.dry_tol;
    int r = N->ratio, p, i, j, f;
    for (p = 0; p < N->np; p++) {
        const gco_patch *Pp = &N->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 2; j < Pp->ny + 2; j++) for (i = 2; i < Pp->nx + 2; i++) {
            int64_t c = N->off[p] + (int64_t)j * pitch + i;
            int64_t gi = (int64_t)Pp->i0 + i - 2, gj = (int64_t)Pp->j0 + j - 2;
            int q = O ? gco_find_patch(O, gi, gj) : -1;
            if (q >= 0) {
                const gco_patch *Q = &O->pat[q];
                int64_t s = O->off[q] + (gj - Q->j0 + 2) * (int64_t)(Q->nx + 4) + (gi - Q->i0 + 2);
                for (f = 0; f < 3; f++) N->q[N->cur][f][c] = O->q[O->cur][f][s];
            } else {
                double out[3];
                int rc = interp_cell(C, r, 1.0, 0, gi, gj, N->b[c], eps, out);
                if (rc) return rc;
                for (f = 0; f < 3; f++) N->q[N->cur][f][c] = out[f];
            }
        }
    }
    return GCO_OK;
}

/* P:145 step 4 / P:162: covered coarse cell <- average of the r*r fine cells on top.  All fine cells
 * wet: average eta, h_c = max(0, eta_bar - b_c) (keeps the ocean at rest); else average h.  Momenta
 * are averaged.  Weights kappa_f (cell area) on the sphere.  Then the clean-up rule. */
int gco_average_down(gco_level *C, const gco_level *F)
{
    if (!C || !F) return GCO_ERR_BADARG;
    double eps = C->ctx->P.dry_tol;
    int r = F->ratio, p, ii, jj;
    int64_t I, J;
    for (p = 0; p < F->np; p++) {
        const gco_patch *Pp = &F->pat[p];
        int pitch = Pp->nx + 4;
        for (J = Pp->j0 / r; J < (Pp->j0 + Pp->ny) / r; J++) for (I = Pp->i0 / r; I < (Pp->i0 + Pp->nx) / r; I++) {
            int cp = gco_find_patch(C, I, J);
            if (cp < 0) return GCO_ERR_STATE;
            const gco_patch *Q = &C->pat[cp];
            int64_t cc = C->off[cp] + (int64_t)(J - Q->j0 + 2) * (Q->nx + 4) + (I - Q->i0 + 2);
            double sw = 0.0, se = 0.0, sh = 0.0, su = 0.0, sv = 0.0;
            int allwet = 1;
            for (jj = 0; jj < r; jj++) {
                int64_t gj = J * r + jj;
                double w = F->kappa[gj + 2];
                for (ii = 0; ii < r; ii++) {
                    int64_t gi = I * r + ii;
                    int64_t c = F->off[p] + (gj - Pp->j0 + 2) * (int64_t)pitch + (gi - Pp->i0 + 2);
                    double h = F->q[F->cur][0][c];
                    if (!(h > eps)) allwet = 0;
                    sw = sw + w;
                    se = se + w * (h + F->b[c]);
                    sh = sh + w * h;
                    su = su + w * F->q[F->cur][1][c];
                    sv = sv + w * F->q[F->cur][2][c];
                }
            }
            double hc = allwet ? max2(0.0, se / sw - C->b[cc]) : sh / sw;
            double huc = su / sw, hvc = sv / sw;
            if (hc < eps) { hc = max2(hc, 0.0); huc = 0.0; hvc = 0.0; }
            C->q[C->cur][0][cc] = hc; C->q[C->cur][1][cc] = huc; C->q[C->cur][2][cc] = hvc;
        }
    }
    return GCO_OK;
}

/* flag = wet and (|eta - eta_sea| > tol_eta or slope > tol_slope), optionally only
 * where b < 0; or the cell centre lies in an active forced box; then dilation by `buffer` cells
 * (Chebyshev distance) over the cells of this level.  Needs ghost cells filled (slope criterion).
 * Output: uint8 per interior cell, packed patch after patch, row-major. */
int gco_flag_cells(const gco_level *L, const gco_flag_params *fp, double t, uint8_t *flags, int64_t *nflag)
{
    if (!L || !fp || !flags) return GCO_ERR_BADARG;
    const gco_params *P = &L->ctx->P;
    double eps = P->dry_tol;
    const double *h = L->q[L->cur][0], *b = L->b;
    int p, q, i, j, k;
    int64_t *poff = malloc(sizeof(int64_t) * (L->np + 1));
    poff[0] = 0;
    for (p = 0; p < L->np; p++) poff[p + 1] = poff[p] + (int64_t)L->pat[p].nx * L->pat[p].ny;
    uint8_t *raw = calloc(poff[L->np] > 0 ? poff[L->np] : 1, 1);
    memset(flags, 0, poff[L->np]);
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        int pitch = Pp->nx + 4;
        for (j = 2; j < Pp->ny + 2; j++) for (i = 2; i < Pp->nx + 2; i++) {
            int64_t c = L->off[p] + (int64_t)j * pitch + i;
            int fl = 0;
            int wet = h[c] > eps;
            int wave_ok = wet && (!fp->offshore_only || b[c] < 0.0);
            if (wave_ok && fp->tol_eta > 0.0 && fabs((h[c] + b[c]) - P->sea_level) > fp->tol_eta) fl = 1;
            if (wave_ok && fp->tol_slope > 0.0) {
                /* central differences of eta over wet neighbours, per unit cell */
                const int64_t lo[2] = { c - 1, c - pitch }, hi[2] = { c + 1, c + pitch };
                for (k = 0; k < 2; k++)
                    if (h[lo[k]] > eps && h[hi[k]] > eps) {
                        double sl = 0.5 * fabs((h[hi[k]] + b[hi[k]]) - (h[lo[k]] + b[lo[k]]));
                        if (sl > fp->tol_slope) fl = 1;
                    }
            }
            if (!fl) {
                double xc = L->xlo + ((double)((int64_t)Pp->i0 + i - 2) + 0.5) * L->dx;
                double yc = L->ylo + ((double)((int64_t)Pp->j0 + j - 2) + 0.5) * L->dy;
                for (k = 0; k < fp->nboxes; k++) {
                    const double *B = fp->boxes + 6 * k;
                    if (xc >= B[0] && xc <= B[1] && yc >= B[2] && yc <= B[3] && t >= B[4] && t <= B[5]) fl = 1;
                }
            }
            raw[poff[p] + (int64_t)(j - 2) * Pp->nx + (i - 2)] = (uint8_t)fl;
        }
    }
    /* dilation */
    int bw = fp->buffer > 0 ? fp->buffer : 0;
    for (p = 0; p < L->np; p++) {
        const gco_patch *Pp = &L->pat[p];
        for (j = 0; j < Pp->ny; j++) for (i = 0; i < Pp->nx; i++) {
            if (!raw[poff[p] + (int64_t)j * Pp->nx + i]) continue;
            int64_t gi = (int64_t)Pp->i0 + i, gj = (int64_t)Pp->j0 + j;
            for (q = 0; q < L->np; q++) {
                const gco_patch *Q = &L->pat[q];
                int64_t a0 = gi - bw > Q->i0 ? gi - bw : Q->i0;
                int64_t a1 = gi + bw < (int64_t)Q->i0 + Q->nx - 1 ? gi + bw : (int64_t)Q->i0 + Q->nx - 1;
                int64_t b0 = gj - bw > Q->j0 ? gj - bw : Q->j0;
                int64_t b1 = gj + bw < (int64_t)Q->j0 + Q->ny - 1 ? gj + bw : (int64_t)Q->j0 + Q->ny - 1;
                int64_t a, bb;
                for (bb = b0; bb <= b1; bb++) for (a = a0; a <= a1; a++)
                    flags[poff[q] + (bb - Q->j0) * Q->nx + (a - Q->i0)] = 1;
            }
        }
    }
    int64_t n = 0, c;
    for (c = 0; c < poff[L->np]; c++) n += flags[c];
    if (nflag) *nflag = n;
    free(raw); free(poff);
    return GCO_OK;
}

/* P:166 "finding the best grid patch ..., interpolating from cell values": DESIGN.md 3.10 (S-19).  The best patch is found by the
 * caller (host bookkeeping); this is the interpolation, in the order DESIGN.md states. */
int gco_gauges_sample(const gco_level *L, int n, const int32_t *patch, const double *xy, double *out)
{
    int k, f;
    if (!L || n < 0 || (n > 0 && (!patch || !xy || !out))) return GCO_ERR_BADARG;
    for (k = 0; k < n; k++) {
        const gco_patch *Pp;
        const double *fld[3];
        const double *bb;
        double eps = L->ctx->P.dry_tol;
        double gx, gy, xi, et, a, b, v[4][4];
        int64_t ic, jc, i, j, pitch, c00;
        int dry = 0, m;
        if (patch[k] < 0 || patch[k] >= L->np) return GCO_ERR_BADARG;
        Pp = &L->pat[patch[k]];
        pitch = (int64_t)Pp->nx + 4;
        gx = (xy[2 * k] - L->xlo) / L->dx;  gy = (xy[2 * k + 1] - L->ylo) / L->dy;
        ic = (int64_t)floor(gx); jc = (int64_t)floor(gy);                 /* the cell that contains the point */
        if (ic < Pp->i0 || ic >= (int64_t)Pp->i0 + Pp->nx || jc < Pp->j0 || jc >= (int64_t)Pp->j0 + Pp->ny) return GCO_ERR_BADARG;
        xi = gx - 0.5; et = gy - 0.5;
        i = (int64_t)floor(xi); j = (int64_t)floor(et);
        a = xi - (double)i; b = et - (double)j;
        for (f = 0; f < 3; f++) fld[f] = L->q[L->cur][f] + L->off[patch[k]];
        bb = L->b + L->off[patch[k]];
        c00 = (j - Pp->j0 + 2) * pitch + (i - Pp->i0 + 2);
        for (m = 0; m < 4; m++) {                                          /* m = 0: (i, j), 1: (i+1, j), 2: (i, j+1), 3: (i+1, j+1) */
            int64_t c = c00 + (m & 1) + (m >> 1) * pitch;
            v[0][m] = fld[0][c]; v[1][m] = fld[1][c]; v[2][m] = fld[2][c]; v[3][m] = fld[0][c] + bb[c];
            if (!(fld[0][c] > eps)) dry = 1;
        }
        if (dry) {
            int64_t c = (jc - Pp->j0 + 2) * pitch + (ic - Pp->i0 + 2);
            out[4 * k] = fld[0][c]; out[4 * k + 1] = fld[1][c]; out[4 * k + 2] = fld[2][c]; out[4 * k + 3] = fld[0][c] + bb[c];
        } else {
            for (f = 0; f < 4; f++)
                out[4 * k + f] = (1.0 - b) * ((1.0 - a) * v[f][0] + a * v[f][1]) + b * ((1.0 - a) * v[f][2] + a * v[f][3]);
        }
    }
    return GCO_OK;
}
