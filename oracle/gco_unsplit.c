/* gco_unsplit.c -- ORACLE (test infrastructure).  The unsplit wave-propagation step with transverse Riemann solves.
 *
 * P:309 and P:371 name it: "the original GeoClaw ... with the unsplit algorithm", which the paper's GPU code simplifies to
 * dimensional splitting and validates against.  The paper gives no formula; the reading is DESIGN.md 3.13 (S-21),
 * LeVeque's unsplit wave-propagation method with second-order corrections split transversely:
 *   1. from Q^n (ghost cells filled) every x-edge and every y-edge gets its fluctuations A-dQ, A+dQ (B-dQ, B+dQ) and its limited
 *      correction flux F~ (G~), exactly as in the 1-D sweep (gco_line_terms: steps (1)-(5) of DESIGN.md 3.4);
 *   2. at every x-edge the vectors  a- = A-dQ + F~  (it enters the cell on the left) and  a+ = A+dQ - F~  (the cell on the right)
 *      are split by the y-direction Jacobian of that cell into a down-going part and an up-going part (gco_transverse), which
 *      change the correction fluxes of that cell's lower and upper y-edge:  G~ <- fma(-(1/2 dt rdx_row), part, G~);  every y-edge
 *      vector is split in x likewise and changes F~ of the cell's left and right x-edge;
 *   3. Q <- fma(-dt rdy, gm_{j+1} - gp_j, fma(-dt rdx, fm_{i+1} - fp_i, Q)), fm = F~' + A-dQ, fp = F~' - A+dQ (gm, gp likewise),
 *      then the dry clean-up, friction and statistics of the split step.
 * Storage indices below: cell (i, j), i = 0..nx+3, j = 0..ny+3; x-edge (e, j) between cells (e-1, j) and (e, j).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "gco_int.h"

static double max2(double a, double b) { return a > b ? a : b; }

/* Transverse split of a vector a = (a0, a1, a2) given in the frame of the TARGET direction -- a0: depth component, a1: momentum
 * along the target direction, a2: momentum across it -- by the Jacobian of that direction at the cell state (h, pn, pt):
 * eigenvalues w - c, w, w + c (w = pn / h, c = sqrt(g h)), eigenvectors (1, w - c, z), (0, 0, 1), (1, w + c, z), z = pt / h.
 * bm = sum over negative eigenvalues of lambda beta r, bp = over positive ones (zero eigenvalue: dropped); a dry cell: both zero. */
void gco_transverse(double g, double eps, double h, double pn, double pt, const double a[3], double bm[3], double bp[3])
{
    int k, p;
    for (k = 0; k < 3; k++) { bm[k] = 0.0; bp[k] = 0.0; }
    if (!(h > eps)) return;
    double rh = 1.0 / h;
    double w = pn * rh, z = pt * rh, c = sqrt(g * h);
    double l1 = w - c, l2 = w, l3 = w + c;
    double rho = 1.0 / (l3 - l1);
    double b1 = fma(l3, a[0], -a[1]) * rho;
    double b3 = fma(-l1, a[0], a[1]) * rho;
    double b2 = fma(-z, a[0], a[2]);
    double lam[3] = { l1, l2, l3 };
    double V[3][3];
    V[0][0] = l1 * b1; V[0][1] = V[0][0] * l1; V[0][2] = V[0][0] * z;
    V[1][0] = 0.0;     V[1][1] = 0.0;          V[1][2] = l2 * b2;
    V[2][0] = l3 * b3; V[2][1] = V[2][0] * l3; V[2][2] = V[2][0] * z;
    for (p = 0; p < 3; p++)
        for (k = 0; k < 3; k++) {
            if (lam[p] < 0.0) bm[k] = bm[k] + V[p][k];
            else if (lam[p] > 0.0) bp[k] = bp[k] + V[p][k];
        }
}

/* one patch of the unsplit step; statistics come back per patch (see gco_level.c: step_patch) */
static void unsplit_patch(gco_level *L, int p, double dt, double *sdx_out, double *clipped_out, int64_t *nclip_out, int *nan_out)
{
    const gco_params *P = &L->ctx->P;
    const gco_patch *Pp = &L->pat[p];
    double eps = P->dry_tol, sdx = 0.0, clipped = 0.0;
    int64_t nclip = 0; int nan_seen = 0;
    int nx = Pp->nx, ny = Pp->ny, pitch = nx + 4, rows = ny + 4, i, j, e, k;
    int cur = L->cur, nxt = 1 - cur;
    int64_t o = L->off[p];
    const double *h = L->q[cur][0] + o, *hu = L->q[cur][1] + o, *hv = L->q[cur][2] + o, *b = L->b + o;
    double *hn = L->q[nxt][0] + o, *hun = L->q[nxt][1] + o, *hvn = L->q[nxt][2] + o;
    size_t sz = (size_t)pitch * rows * 3;
    /* per storage cell (j, i), 3 components: terms of the x-edge at its left side / of the y-edge at its lower side */
    double *amx = calloc(sz, sizeof(double)), *apx = calloc(sz, sizeof(double)), *Fx = calloc(sz, sizeof(double));
    double *bmy = calloc(sz, sizeof(double)), *bpy = calloc(sz, sizeof(double)), *Gy = calloc(sz, sizeof(double));
    int nmax = (nx > ny ? nx : ny) + 5;
    double *rd = malloc(sizeof(double) * nmax), *ef = malloc(sizeof(double) * nmax);
    double *lin[4], *lam = malloc(sizeof(double) * 3 * nmax), *lap = malloc(sizeof(double) * 3 * nmax);
    double *lF = malloc(sizeof(double) * 3 * nmax), *ls = malloc(sizeof(double) * 3 * nmax);
    for (k = 0; k < 4; k++) lin[k] = malloc(sizeof(double) * nmax);
#define AT(j, i) (((size_t)(j) * pitch + (i)) * 3)

    /* 1a. x-edges of rows 1..ny+2 (one ghost row each side feeds the transverse terms), normal = hu, transverse = hv */
    for (j = 1; j <= ny + 2; j++) {
        int64_t gr = (int64_t)Pp->j0 + j; /* table index = global row + 2 */
        for (i = 0; i < pitch; i++) rd[i] = L->rdx[gr];
        for (i = 0; i < pitch + 1; i++) ef[i] = L->ex;
        gco_line_terms(P, nx, h + (size_t)j * pitch, hu + (size_t)j * pitch, hv + (size_t)j * pitch, b + (size_t)j * pitch,
                       rd, ef, dt, lam, lap, lF, ls);
        for (e = 2; e <= nx + 2; e++) for (k = 0; k < 3; k++) {
            amx[AT(j, e) + k] = lam[e * 3 + k]; apx[AT(j, e) + k] = lap[e * 3 + k]; Fx[AT(j, e) + k] = lF[e * 3 + k];
        }
        if (j >= 2 && j < ny + 2) /* eq. 15 over interior lines */
            for (e = 2; e <= nx + 2; e++) for (k = 0; k < 3; k++) {
                sdx = max2(sdx, max2(ls[e * 3 + k], 0.0) * rd[e]);
                sdx = max2(sdx, max2(-ls[e * 3 + k], 0.0) * rd[e - 1]);
            }
    }
    /* 1b. y-edges of columns 1..nx+2, normal = hv, transverse = hu */
    for (i = 1; i <= nx + 2; i++) {
        for (j = 0; j < rows; j++) {
            int64_t gr = (int64_t)Pp->j0 + j;
            lin[0][j] = h[(size_t)j * pitch + i]; lin[1][j] = hv[(size_t)j * pitch + i];
            lin[2][j] = hu[(size_t)j * pitch + i]; lin[3][j] = b[(size_t)j * pitch + i];
            rd[j] = L->rdy[gr]; ef[j] = L->ey[gr];
        }
        ef[rows] = L->ey[(int64_t)Pp->j0 + rows];
        gco_line_terms(P, ny, lin[0], lin[1], lin[2], lin[3], rd, ef, dt, lam, lap, lF, ls);
        for (e = 2; e <= ny + 2; e++) for (k = 0; k < 3; k++) {
            bmy[AT(e, i) + k] = lam[e * 3 + k]; bpy[AT(e, i) + k] = lap[e * 3 + k]; Gy[AT(e, i) + k] = lF[e * 3 + k];
        }
        if (i >= 2 && i < nx + 2)
            for (e = 2; e <= ny + 2; e++) for (k = 0; k < 3; k++) {
                sdx = max2(sdx, max2(ls[e * 3 + k], 0.0) * rd[e]);
                sdx = max2(sdx, max2(-ls[e * 3 + k], 0.0) * rd[e - 1]);
            }
    }

    /* 2. transverse splits.  F2, G2: the correction fluxes as the update will see them */
    double *F2 = malloc(sz * sizeof(double)), *G2 = malloc(sz * sizeof(double));
    memcpy(F2, Fx, sz * sizeof(double)); memcpy(G2, Gy, sz * sizeof(double));
    /* 2a. x-edge vectors, split in y; they change G2 of interior columns */
    for (j = 1; j <= ny + 2; j++) {
        int64_t gr = (int64_t)Pp->j0 + j;
        double half = 0.5 * (dt * L->rdx[gr]);
        for (e = 2; e <= nx + 2; e++) {
            int part;
            for (part = 0; part < 2; part++) {           /* a- = A-dQ + F~ enters cell e-1, a+ = A+dQ - F~ enters cell e */
                int ic = part == 0 ? e - 1 : e;
                if (ic < 2 || ic > nx + 1) continue;
                double a[3], at[3], bm[3], bp[3];
                for (k = 0; k < 3; k++)
                    a[k] = part == 0 ? amx[AT(j, e) + k] + Fx[AT(j, e) + k] : apx[AT(j, e) + k] - Fx[AT(j, e) + k];
                at[0] = a[0]; at[1] = a[2]; at[2] = a[1];              /* target frame: (h, hv, hu) */
                size_t c = (size_t)j * pitch + ic;
                gco_transverse(P->g, eps, h[c], hv[c], hu[c], at, bm, bp);
                if (P->coord == 1) for (k = 0; k < 3; k++) { bm[k] = bm[k] * L->ey[gr]; bp[k] = bp[k] * L->ey[gr + 1]; }
                if (j >= 2) for (k = 0; k < 3; k++) G2[AT(j, ic) + k] = fma(-half, bm[k], G2[AT(j, ic) + k]);            /* lower y-edge of the cell */
                if (j <= ny + 1) for (k = 0; k < 3; k++) G2[AT(j + 1, ic) + k] = fma(-half, bp[k], G2[AT(j + 1, ic) + k]); /* upper y-edge */
            }
        }
    }
    /* 2b. y-edge vectors, split in x; they change F2 of interior rows */
    for (i = 1; i <= nx + 2; i++) {
        for (e = 2; e <= ny + 2; e++) {
            int part;
            for (part = 0; part < 2; part++) {
                int jc = part == 0 ? e - 1 : e;
                if (jc < 2 || jc > ny + 1) continue;
                int64_t gr = (int64_t)Pp->j0 + jc;
                double half = 0.5 * (dt * L->rdy[gr]);
                double a[3], at[3], cm[3], cp[3];
                for (k = 0; k < 3; k++)
                    a[k] = part == 0 ? bmy[AT(e, i) + k] + Gy[AT(e, i) + k] : bpy[AT(e, i) + k] - Gy[AT(e, i) + k];
                at[0] = a[0]; at[1] = a[2]; at[2] = a[1];              /* target frame: (h, hu, hv) */
                size_t c = (size_t)jc * pitch + i;
                gco_transverse(P->g, eps, h[c], hu[c], hv[c], at, cm, cp);
                if (P->coord == 1) for (k = 0; k < 3; k++) { cm[k] = cm[k] * L->ex; cp[k] = cp[k] * L->ex; }
                if (i >= 2) for (k = 0; k < 3; k++) F2[AT(jc, i) + k] = fma(-half, cm[k], F2[AT(jc, i) + k]);            /* left x-edge of the cell */
                if (i <= nx + 1) for (k = 0; k < 3; k++) F2[AT(jc, i + 1) + k] = fma(-half, cp[k], F2[AT(jc, i + 1) + k]); /* right x-edge */
            }
        }
    }

    /* 3. update of the interior, clean-up (S-9), friction (S-16) */
    for (j = 2; j <= ny + 1; j++) {
        int64_t gr = (int64_t)Pp->j0 + j;
        double dtdx = dt * L->rdx[gr], dtdy = dt * L->rdy[gr];
        for (i = 2; i <= nx + 1; i++) {
            size_t c = (size_t)j * pitch + i;
            double dfx[3], dgy[3];
            for (k = 0; k < 3; k++) {
                double fm = F2[AT(j, i + 1) + k] + amx[AT(j, i + 1) + k], fp = F2[AT(j, i) + k] - apx[AT(j, i) + k];
                double gm = G2[AT(j + 1, i) + k] + bmy[AT(j + 1, i) + k], gp = G2[AT(j, i) + k] - bpy[AT(j, i) + k];
                dfx[k] = fm - fp; dgy[k] = gm - gp;
            }
            double hh = fma(-dtdy, dgy[0], fma(-dtdx, dfx[0], h[c]));
            double uu = fma(-dtdy, dgy[2], fma(-dtdx, dfx[1], hu[c]));
            double vv = fma(-dtdy, dgy[1], fma(-dtdx, dfx[2], hv[c]));
            if (hh < eps && dt > 0.0) {
                if (hh < 0.0) { nclip++; clipped += (-hh) * gco_cell_area(L, (int64_t)Pp->j0 + j - 2); }
                hh = max2(hh, 0.0); uu = 0.0; vv = 0.0;
            }
            if (dt > 0.0) gco_friction(P, dt, hh, &uu, &vv);
            if (hh != hh || uu != uu || vv != vv) nan_seen = 1;
            if (dt > 0.0) { hn[c] = hh; hun[c] = uu; hvn[c] = vv; }
        }
    }
#undef AT
    free(amx); free(apx); free(Fx); free(bmy); free(bpy); free(Gy); free(F2); free(G2);
    free(rd); free(ef); free(lam); free(lap); free(lF); free(ls);
    for (k = 0; k < 4; k++) free(lin[k]);
    *sdx_out = sdx; *clipped_out = clipped; *nclip_out = nclip; *nan_out = nan_seen;
}

/* One unsplit level step.  dt = 0 is a legal probe.  Flux registers are defined for the split step only. */
int gco_level_step_unsplit(gco_level *L, double dt, gco_step_stats *out)
{
    if (!L || !(dt >= 0.0)) return GCO_ERR_BADARG;
    if (L->save_flux) return GCO_ERR_STATE;
    double sdx = 0.0, clipped = 0.0;
    int64_t nclip = 0; int nan_seen = 0;
    int p, np = L->np, nt = gco_get_threads();
    double *psdx = malloc(sizeof(double) * (np + 1)), *pclip = malloc(sizeof(double) * (np + 1));
    int64_t *pn = malloc(sizeof(int64_t) * (np + 1));
    int *pnan = malloc(sizeof(int) * (np + 1));
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt) if (nt > 1)
#endif
    for (p = 0; p < np; p++) unsplit_patch(L, p, dt, &psdx[p], &pclip[p], &pn[p], &pnan[p]);
    for (p = 0; p < np; p++) { sdx = max2(sdx, psdx[p]); clipped = clipped + pclip[p]; nclip += pn[p]; nan_seen |= pnan[p]; }
    free(psdx); free(pclip); free(pn); free(pnan);
    if (dt > 0.0) L->cur = 1 - L->cur;
    L->last.cfl_max = dt * sdx; L->last.s_over_dx_max = sdx; L->last.clipped_mass = clipped;
    L->last.n_clipped = nclip; L->last.nan_seen = nan_seen;
    if (out) *out = L->last;
    return GCO_OK;
}
