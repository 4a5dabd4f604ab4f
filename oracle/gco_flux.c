/* gco_flux.c -- ORACLE (test infrastructure).  Flux registers and the conservative fix-up
 * (refluxing), P:146 step 5 as the paper DESCRIBES it (the paper's GPU code drops it).
 * Form: DESIGN.md 3.8.  With fm = F~ + A-dQ and fp = F~ - A+dQ the true numerical flux at an edge is
 * fm + f(Q_left) = fp + f(Q_right); a register holds, for a coarse edge E on the boundary of the
 * fine region with uncovered coarse neighbour C,
 *   delta_E = dt_c l_E (fm_E or fp_E, whichever C used)
 *             - sum_substeps sum_k dt_f l_k [ (fp_k or fm_k used by fine cell f_k) + J_k ],
 *   J_k = f(Q_fk) - f(Q_C^n) minus the source jump: mass component p(f_k) - p(C^n) in closed form,
 *   momentum components from sum_p Z^p of the Riemann problem between the two states in geometric
 *   order.  Fix-up: Q_C += side * delta_E / area_C, then the clean-up rule.
 */
#include <stdlib.h>
#include <string.h>
#include "gco_int.h"

static double max2(double a, double b) { return a > b ? a : b; }

void gco_flux_free(gco_level *L)
{
    int f;
    free(L->fmx); free(L->fpx); free(L->fmy); free(L->fpy);
    for (f = 0; f < 3; f++) free(L->qs[f]);
    free(L->reg);
    L->fmx = L->fpx = L->fmy = L->fpy = NULL; L->reg = NULL; L->nreg = 0;
    for (f = 0; f < 3; f++) L->qs[f] = NULL;
}

static void enable_save(gco_level *L)
{
    int f;
    if (L->save_flux) return;
    int64_t tot = L->off[L->np] > 0 ? L->off[L->np] : 1;
    L->fmx = calloc(tot * 3, sizeof(double)); L->fpx = calloc(tot * 3, sizeof(double));
    L->fmy = calloc(tot * 3, sizeof(double)); L->fpy = calloc(tot * 3, sizeof(double));
    for (f = 0; f < 3; f++) L->qs[f] = calloc(tot, sizeof(double));
    L->save_flux = 1;
}

static void add_reg(gco_level *C, const gco_freg *r)
{
    C->reg = realloc(C->reg, sizeof(gco_freg) * (C->nreg + 1));
    C->reg[C->nreg++] = *r;
}

int gco_flux_attach(gco_level *C, gco_level *F)
{
    if (!C || !F) return GCO_ERR_BADARG;
    int r = F->ratio, p, side;
    free(C->reg); C->reg = NULL; C->nreg = 0;
    enable_save(C); enable_save(F);
    C->reg_fine = F; F->reg_coarse = C;
    for (p = 0; p < F->np; p++) {
        const gco_patch *Pp = &F->pat[p];
        int64_t I0 = Pp->i0 / r, I1 = (Pp->i0 + Pp->nx) / r, J0 = Pp->j0 / r, J1 = (Pp->j0 + Pp->ny) / r;
        for (side = 0; side < 4; side++) { /* xlo, xhi, ylo, yhi side of the fine patch */
            int dir = side / 2;
            int64_t n = dir == 0 ? J1 - J0 : I1 - I0, m;
            for (m = 0; m < n; m++) {
                int64_t I, J;
                if (side == 0) { I = I0 - 1; J = J0 + m; } else if (side == 1) { I = I1; J = J0 + m; }
                else if (side == 2) { I = I0 + m; J = J0 - 1; } else { I = I0 + m; J = J1; }
                if (I < 0 || J < 0 || I >= C->nxl || J >= C->nyl) continue;       /* physical boundary */
                if (gco_find_patch(F, I * r, J * r) >= 0) continue;              /* fine-fine boundary */
                int cp = gco_find_patch(C, I, J);
                if (cp < 0) return GCO_ERR_STATE;
                gco_freg R; memset(&R, 0, sizeof R);
                R.cp = cp; R.ci = (int32_t)(I - C->pat[cp].i0 + 2); R.cj = (int32_t)(J - C->pat[cp].j0 + 2);
                R.dir = dir;
                R.side = (side == 0 || side == 2) ? +1 : -1; /* fine region on the high side of C for lo sides */
                R.fpat = p;
                if (side == 0) { R.fi = 2; R.fj = (int32_t)(2 + m * r); }
                else if (side == 1) { R.fi = Pp->nx + 1; R.fj = (int32_t)(2 + m * r); }
                else if (side == 2) { R.fi = (int32_t)(2 + m * r); R.fj = 2; }
                else { R.fi = (int32_t)(2 + m * r); R.fj = Pp->ny + 1; }
                add_reg(C, &R);
            }
        }
    }
    return GCO_OK;
}

static double p_used(double h, double p, double eps) { return (h <= eps) ? 0.0 : p; }

/* called at the end of every step of L (after the buffer swap): q[1-cur] = Q^n, qs = Q* */
void gco_flux_accumulate_own(gco_level *L, double dt)
{
    const gco_params *P = &L->ctx->P;
    int n, k, m;
    /* (a) L is the coarse side */
    for (n = 0; n < L->nreg; n++) {
        gco_freg *R = &L->reg[n];
        int pitch = L->pat[R->cp].nx + 4;
        int64_t o = L->off[R->cp], c = o + (int64_t)R->cj * pitch + R->ci;
        const double *F; double len;
        if (R->dir == 0) {
            len = L->dy;
            F = (R->side > 0) ? L->fmx + (c + 1) * 3 : L->fpx + c * 3;
            R->base[0] = L->q[1 - L->cur][0][c]; R->base[1] = L->q[1 - L->cur][1][c]; R->base[2] = L->q[1 - L->cur][2][c];
        } else {
            len = L->dx;
            F = (R->side > 0) ? L->fmy + (c + pitch) * 3 : L->fpy + c * 3;
            R->base[0] = L->qs[0][c]; R->base[1] = L->qs[2][c]; R->base[2] = L->qs[1][c];
        }
        R->base[3] = L->b[c];
        for (k = 0; k < 3; k++) R->delta[k] = R->delta[k] + dt * len * F[k];
    }
    /* (b) L is the fine side of its coarser level's registers */
    gco_level *C = L->reg_coarse;
    if (!C || C->reg_fine != L) return;
    int r = L->ratio;
    for (n = 0; n < C->nreg; n++) {
        gco_freg *R = &C->reg[n];
        const gco_patch *Pp = &L->pat[R->fpat];
        int pitch = Pp->nx + 4;
        int64_t o = L->off[R->fpat];
        for (m = 0; m < r; m++) {
            int fi = R->fi + (R->dir == 1 ? m : 0), fj = R->fj + (R->dir == 0 ? m : 0);
            int64_t c = o + (int64_t)fj * pitch + fi;
            double st[4]; const double *F; double len, ef;
            if (R->dir == 0) {
                len = L->dy; ef = (P->coord == 1) ? L->ex : 1.0;
                st[0] = L->q[1 - L->cur][0][c]; st[1] = L->q[1 - L->cur][1][c]; st[2] = L->q[1 - L->cur][2][c];
                F = (R->side > 0) ? L->fpx + c * 3 : L->fmx + (c + 1) * 3;
            } else {
                len = L->dx;
                /* edge row of the fine table: the shared edge */
                int64_t ge = (int64_t)Pp->j0 + fj - 2 + (R->side > 0 ? 0 : 1);
                ef = (P->coord == 1) ? L->ey[ge + 2] : 1.0;
                st[0] = L->qs[0][c]; st[1] = L->qs[2][c]; st[2] = L->qs[1][c];
                F = (R->side > 0) ? L->fpy + c * 3 : L->fmy + (c + pitch) * 3;
            }
            st[3] = L->b[c];
            double Z[3][3], s[3], J[3];
            if (R->side > 0) /* C is the left/lower state */
                gco_riemann(P->g, P->dry_tol, R->base[0], R->base[1], R->base[2], R->base[3],
                            st[0], st[1], st[2], st[3], Z, s);
            else
                gco_riemann(P->g, P->dry_tol, st[0], st[1], st[2], st[3],
                            R->base[0], R->base[1], R->base[2], R->base[3], Z, s);
            double sg = (R->side > 0) ? 1.0 : -1.0;
            J[0] = p_used(st[0], st[1], P->dry_tol) - p_used(R->base[0], R->base[1], P->dry_tol);
            J[1] = sg * ((Z[0][1] + Z[1][1]) + Z[2][1]);
            J[2] = sg * ((Z[0][2] + Z[1][2]) + Z[2][2]);
            for (k = 0; k < 3; k++) R->delta[k] = R->delta[k] - dt * len * (F[k] + ef * J[k]);
        }
    }
}

int gco_flux_fixup(gco_level *C, gco_level *F)
{
    if (!C || !F || C->reg_fine != F) return GCO_ERR_BADARG;
    double eps = C->ctx->P.dry_tol;
    int n, k;
    for (n = 0; n < C->nreg; n++) {
        gco_freg *R = &C->reg[n];
        int pitch = C->pat[R->cp].nx + 4;
        int64_t c = C->off[R->cp] + (int64_t)R->cj * pitch + R->ci;
        double area = gco_cell_area(C, (int64_t)C->pat[R->cp].j0 + R->cj - 2);
        double sg = (double)R->side;
        int fn = (R->dir == 0) ? 1 : 2, ft = (R->dir == 0) ? 2 : 1;
        C->q[C->cur][0][c] = C->q[C->cur][0][c] + sg * R->delta[0] / area;
        C->q[C->cur][fn][c] = C->q[C->cur][fn][c] + sg * R->delta[1] / area;
        C->q[C->cur][ft][c] = C->q[C->cur][ft][c] + sg * R->delta[2] / area;
        for (k = 0; k < 3; k++) R->delta[k] = 0.0;
    }
    for (n = 0; n < C->nreg; n++) { /* clean-up rule on the corrected cells */
        gco_freg *R = &C->reg[n];
        int pitch = C->pat[R->cp].nx + 4;
        int64_t c = C->off[R->cp] + (int64_t)R->cj * pitch + R->ci;
        double h = C->q[C->cur][0][c];
        if (h < eps) { C->q[C->cur][0][c] = max2(h, 0.0); C->q[C->cur][1][c] = 0.0; C->q[C->cur][2][c] = 0.0; }
    }
    return GCO_OK;
}
