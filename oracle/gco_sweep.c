/* gco_sweep.c -- ORACLE (test infrastructure).  One 1-D sweep of the wave-propagation scheme.
 *
 * Follows P:65-105 (section 2.2, eqs. 4-11) in f-wave form (Z^p = lambda^p W^p, so that
 * A-dQ = sum_{s<0} Z, A+dQ = sum_{s>0} Z, eq. 5-6) and the capacity form of DESIGN.md 3.4-3.5.
 * Order of operations: (1) solve every edge 1..n+3; (2) scale by the edge factor; (3) fluctuations;
 * (4) limiter (eq. 10-11 with the reading S-1 theta = (Z_I . Z_e)/(Z_e . Z_e), MC limiter P:292);
 * (5) correction flux (eq. 9); (6) fm = F~ + A-dQ, fp = F~ - A+dQ; (7) update (eq. 8 / 13 / 14)
 *     Q_c <- fma(-dt*rdx_c, fm_{c+1} - fp_c, Q_c); (8) CFL (eq. 15).
 * fma(a, b, c) = a*b + c rounded once, at exactly the places DESIGN.md 3.4 writes it (C99 fma; -ffp-contract=off elsewhere).
 */
#include <math.h>
#include <stdlib.h>
#include "gco.h"

static double max2(double a, double b) { return a > b ? a : b; }
static double min2(double a, double b) { return a < b ? a : b; }

/* steps (1)-(5) on one line: fluctuations am = A-dQ, ap = A+dQ and limited correction flux F at edges 2..n+2 (3 doubles each,
 * index [e*3+k]), speeds s at edges 1..n+3.  Shared by the dimensionally split sweep below and the unsplit step (gco_unsplit.c). */
void gco_line_terms(const gco_params *P, int n, const double *h, const double *p, const double *t,
                    const double *b, const double *rdx, const double *efac, double dt,
                    double *am_out, double *ap_out, double *F_out, double *s_out)
{
    int ne = n + 4; /* edge index e = 1..n+3 used */
    double (*Z)[3][3] = malloc(sizeof(double[3][3]) * ne);
    double (*s)[3] = malloc(sizeof(double[3]) * ne);
    double (*am)[3] = malloc(sizeof(double[3]) * ne);
    double (*ap)[3] = malloc(sizeof(double[3]) * ne);
    int e, w, k;

    /* (1)-(3): Riemann problems, edge scaling, fluctuations (eq. 5-6; tie S-4) */
    for (e = 1; e <= n + 3; e++) {
        gco_riemann(P->g, P->dry_tol, h[e - 1], p[e - 1], t[e - 1], b[e - 1],
                    h[e], p[e], t[e], b[e], Z[e], s[e]);
        if (P->coord == 1) {
            for (w = 0; w < 3; w++) {
                s[e][w] = s[e][w] * efac[e];
                for (k = 0; k < 3; k++) Z[e][w][k] = Z[e][w][k] * efac[e];
            }
        }
        for (k = 0; k < 3; k++) { am[e][k] = 0.0; ap[e][k] = 0.0; }
        for (w = 0; w < 3; w++) {
            for (k = 0; k < 3; k++) {
                if (s[e][w] < 0.0) am[e][k] = am[e][k] + Z[e][w][k];
                else if (s[e][w] > 0.0) ap[e][k] = ap[e][k] + Z[e][w][k];
                else { am[e][k] = am[e][k] + 0.5 * Z[e][w][k]; ap[e][k] = ap[e][k] + 0.5 * Z[e][w][k]; }
            }
        }
    }

    /* (4)-(5): limited second-order correction at edges 2..n+2 */
    for (e = 2; e <= n + 2; e++) {
        double F[3] = {0.0, 0.0, 0.0};
        double T[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
        if (P->limiter != 0) {
            double dtdx_ave = 0.5 * fma(dt, rdx[e - 1], dt * rdx[e]);
            for (w = 0; w < 3; w++) {
                double sw = s[e][w];
                if (sw == 0.0) continue; /* sgn(0) = 0, S-4 */
                double zz = fma(Z[e][w][2], Z[e][w][2], fma(Z[e][w][1], Z[e][w][1], Z[e][w][0] * Z[e][w][0]));
                double phi = 1.0;
                if (zz != 0.0) {
                    int I = (sw > 0.0) ? e - 1 : e + 1; /* eq. 11 */
                    double zi = fma(Z[I][w][2], Z[e][w][2], fma(Z[I][w][1], Z[e][w][1], Z[I][w][0] * Z[e][w][0]));
                    double theta = zi / zz; /* eq. 10, reading S-1 */
                    /* MC: max(0, min((1+theta)/2, 2, 2 theta)) */
                    phi = max2(0.0, min2(min2(0.5 * (1.0 + theta), 2.0), 2.0 * theta));
                }
                double coef = ((sw > 0.0) ? 0.5 : -0.5) * fma(-fabs(sw), dtdx_ave, 1.0);
                double cphi = coef * phi;
                for (k = 0; k < 3; k++) T[w][k] = cphi * Z[e][w][k];
            }
            for (k = 0; k < 3; k++) F[k] = (T[0][k] + T[2][k]) + T[1][k];
        }
        for (k = 0; k < 3; k++) { am_out[e * 3 + k] = am[e][k]; ap_out[e * 3 + k] = ap[e][k]; F_out[e * 3 + k] = F[k]; }
    }
    for (e = 1; e <= n + 3; e++) for (w = 0; w < 3; w++) s_out[e * 3 + w] = s[e][w];
    free(Z); free(s); free(am); free(ap);
}

void gco_sweep_line(const gco_params *P, int n, const double *h, const double *p, const double *t,
                    const double *b, const double *rdx, const double *efac, double dt,
                    double *ho, double *po, double *to, double *fm_out, double *fp_out,
                    int count_cfl, double *sdx)
{
    int ne = n + 4; /* edge index e = 1..n+3 used */
    double *am = malloc(sizeof(double) * 3 * ne), *ap = malloc(sizeof(double) * 3 * ne), *F = malloc(sizeof(double) * 3 * ne);
    double *s = malloc(sizeof(double) * 3 * ne);
    double (*fm)[3] = malloc(sizeof(double[3]) * ne);
    double (*fp)[3] = malloc(sizeof(double[3]) * ne);
    int e, c, w, k;

    gco_line_terms(P, n, h, p, t, b, rdx, efac, dt, am, ap, F, s);          /* (1)-(5) */
    for (e = 2; e <= n + 2; e++)                                              /* (6) */
        for (k = 0; k < 3; k++) {
            fm[e][k] = F[e * 3 + k] + am[e * 3 + k];
            fp[e][k] = F[e * 3 + k] - ap[e * 3 + k];
        }

    /* (7) update of cells 2..n+1 */
    for (c = 2; c <= n + 1; c++) {
        double dtdx = dt * rdx[c];
        ho[c] = fma(-dtdx, fm[c + 1][0] - fp[c][0], h[c]);
        po[c] = fma(-dtdx, fm[c + 1][1] - fp[c][1], p[c]);
        to[c] = fma(-dtdx, fm[c + 1][2] - fp[c][2], t[c]);
    }

    /* (8) CFL: right-going waves enter cell e, left-going waves enter cell e-1 */
    if (count_cfl) {
        double m = *sdx;
        for (e = 2; e <= n + 2; e++)
            for (w = 0; w < 3; w++) {
                m = max2(m, max2(s[e * 3 + w], 0.0) * rdx[e]);
                m = max2(m, max2(-s[e * 3 + w], 0.0) * rdx[e - 1]);
            }
        *sdx = m;
    }
    if (fm_out) for (e = 2; e <= n + 2; e++) for (k = 0; k < 3; k++) fm_out[e * 3 + k] = fm[e][k];
    if (fp_out) for (e = 2; e <= n + 2; e++) for (k = 0; k < 3; k++) fp_out[e * 3 + k] = fp[e][k];
    free(am); free(ap); free(F); free(s); free(fm); free(fp);
}
