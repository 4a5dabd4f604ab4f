/* gco_riemann.c -- ORACLE (test infrastructure).  Augmented shallow-water Riemann solver.
 *
 * The paper gives one sentence (section 2.2): "An approximate Riemann solver has been
 * implemented by George (2008) ... for this augmented system ... preserving steady state of the
 * ocean, handling dry states in the Riemann problem, and maintaining non-negative depth".  The
 * steps R0..R9 below are the reading of that sentence fixed in DESIGN.md section 3.3: an
 * f-wave decomposition of the jump in (h, hu, phi = hu*u + g h^2/2) onto the eigenvectors
 * (1, lambda, lambda^2) for the two outer Einfeldt speeds plus the (0,0,1) corrector, after the
 * steady-state (bathymetry) jump has been removed.  Every step is written in the order of
 * DESIGN.md; there is no blocking, fusion or reordering.
 */
#include <math.h>
#include "gco.h"

static double max2(double a, double b) { return a > b ? a : b; }
static double min2(double a, double b) { return a < b ? a : b; }
/* fma(a, b, c) = a*b + c with ONE rounding (C99 fma, correctly rounded by libm with or without hardware
 * support), used at exactly the places DESIGN.md 3.3-3.4 write it; every other operation rounds on its own
 * (-ffp-contract=off).  north_star: "both sides fp64, FMA contraction stated". */

#define TAU 1.0e-6      /* critical-flow tolerance */
#define SQRT_TAU 1.0e-3

/* R5 -- flat-bottom two-wave middle state M(hL,hR,uL,uR) -> (hm, sigma1, sigma2).
 * Depth function F(h) = fL(h) + fR(h) + (uR-uL); fK = 2(sqrt(g h) - cK) for h <= hK (rarefaction),
 * (h - hK) sqrt(g/2 (1/h + 1/hK)) for h > hK (shock).  Exactly one Newton step (two shocks) or one
 * secant step (mixed), DESIGN.md 3.3 R5. cL, cR = sqrt(g hL), sqrt(g hR). */
void gco_middle_state(double g, double eps, double hL, double hR, double uL, double uR,
                      double cL, double cR, double *hm, double *s1m, double *s2m)
{
    double hmin = min2(hL, hR), hmax = max2(hL, hR);
    double du = uR - uL;
    if (hmin <= eps) { /* a side dry: dry-front speed */
        double s = ((uR + uL) - 2.0 * cR) + 2.0 * cL;
        *hm = 0.0; *s1m = s; *s2m = s;
        return;
    }
    double cmin = (hL < hR) ? cL : cR; /* = sqrt(g hmin) */
    double cmax = (hL > hR) ? cL : cR; /* = sqrt(g hmax) */
    if (hL == hR) { cmin = cL; cmax = cL; }
    double Fmin = du + 2.0 * (cmin - cmax);
    double Fmax = fma(hmax - hmin, sqrt(0.5 * g * (hmax + hmin) / (hmax * hmin)), du);
    if (Fmin > 0.0) { /* two rarefactions: closed form */
        double cm = 0.25 * max2(0.0, 2.0 * (cL + cR) - du);
        *hm = cm * cm / g;
        *s1m = fma(-3.0, cm, uL + 2.0 * cL);
        *s2m = fma(3.0, cm, uR - 2.0 * cR);
    } else if (Fmax <= 0.0) { /* two shocks: one Newton step in sqrt(h) from hmax */
        double h0 = hmax;
        double gL = sqrt(0.5 * g * (1.0 / h0 + 1.0 / hL));
        double gR = sqrt(0.5 * g * (1.0 / h0 + 1.0 / hR));
        double F0 = fma(h0 - hR, gR, fma(h0 - hL, gL, du));
        double dfdh = (gL - g * (h0 - hL) / (4.0 * (h0 * h0) * gL))
                    + (gR - g * (h0 - hR) / (4.0 * (h0 * h0) * gR));
        double sq0 = sqrt(h0);
        double slope = 2.0 * sq0 * dfdh;
        double sq = sq0 - F0 / slope;
        double h1 = sq * sq;
        double u1m = fma(-(h1 - hL), sqrt(0.5 * g * (1.0 / h1 + 1.0 / hL)), uL);
        double u2m = fma(h1 - hR, sqrt(0.5 * g * (1.0 / h1 + 1.0 / hR)), uR);
        double cm = sqrt(g * h1);
        *hm = h1;
        *s1m = u1m - cm;
        *s2m = u2m + cm;
    } else { /* one shock, one rarefaction: one secant step from hmin on [hmin, hmax] */
        double h1 = hmin - Fmin * (hmax - hmin) / (Fmax - Fmin);
        double cm = sqrt(g * h1);
        *hm = h1;
        if (hL > hR) { /* 1-rarefaction on the deeper (left) side */
            *s1m = fma(-3.0, cm, uL + 2.0 * cL);
            *s2m = (uL + 2.0 * cL) - cm;
        } else {
            *s2m = fma(3.0, cm, uR - 2.0 * cR);
            *s1m = (uR - 2.0 * cR) + cm;
        }
    }
}

void gco_riemann(double g, double eps, double hL, double pL, double tL, double bL,
                 double hR, double pR, double tR, double bR, double Z[3][3], double s[3])
{
    int p, k;
    for (p = 0; p < 3; p++) { s[p] = 0.0; for (k = 0; k < 3; k++) Z[p][k] = 0.0; }

    /* R0 sanitise negative depth */
    if (hL < 0.0) { hL = 0.0; pL = 0.0; tL = 0.0; }
    if (hR < 0.0) { hR = 0.0; pR = 0.0; tR = 0.0; }
    /* R1 both dry */
    if (hL <= eps && hR <= eps) return;

    /* R2 primitive variables per side */
    double uL, vL, phiL, cL, uR, vR, phiR, cR;
    if (hL <= eps) { hL = 0.0; pL = 0.0; tL = 0.0; uL = 0.0; vL = 0.0; phiL = 0.0; }
    else { double rh = 1.0 / hL; uL = pL * rh; vL = tL * rh; phiL = fma(pL, uL, 0.5 * g * (hL * hL)); }
    if (hR <= eps) { hR = 0.0; pR = 0.0; tR = 0.0; uR = 0.0; vR = 0.0; phiR = 0.0; }
    else { double rh = 1.0 / hR; uR = pR * rh; vR = tR * rh; phiR = fma(pR, uR, 0.5 * g * (hR * hR)); }
    cL = sqrt(g * hL);
    cR = sqrt(g * hR);

    /* R3 dry-side wall test */
    double w0 = 1.0, w1 = 1.0, w2 = 1.0;
    if (hR <= eps) {
        double hw, a1, a2;
        gco_middle_state(g, eps, hL, hL, uL, -uL, cL, cL, &hw, &a1, &a2);
        double htest = max2(hL, hw);
        if (htest + bL < bR) { /* right cell is a wall: mirror state, keep only family 1 */
            w1 = 0.0; w2 = 0.0;
            hR = hL; pR = -pL; tR = tL; bR = bL; phiR = phiL; uR = -uL; vR = vL; cR = cL;
        } else if (hL + bL < bR) {
            bR = hL + bL;
        }
    } else if (hL <= eps) {
        double hw, a1, a2;
        gco_middle_state(g, eps, hR, hR, -uR, uR, cR, cR, &hw, &a1, &a2);
        double htest = max2(hR, hw);
        if (htest + bR < bL) {
            w0 = 0.0; w1 = 0.0;
            hL = hR; pL = -pR; tL = tR; bL = bR; phiL = phiR; uL = -uR; vL = vR; cL = cR;
        } else if (hR + bR < bL) {
            bL = hR + bR;
        }
    }

    /* R4 Einfeldt speeds */
    double sL = uL - cL, sR = uR + cR;
    double uhat = (cL * uL + cR * uR) / (cL + cR);
    double chat = sqrt(g * (0.5 * (hL + hR)));
    double sE1 = min2(sL, uhat - chat);
    double sE2 = max2(sR, uhat + chat);

    /* R5 middle state of the flat-bottom problem */
    double hm, s1m, s2m;
    gco_middle_state(g, eps, hL, hR, uL, uR, cL, cR, &hm, &s1m, &s2m);
    (void)hm;

    /* R6 widen the outer speeds; corrector speed */
    double l1 = min2(sE1, s2m);
    double l3 = max2(sE2, s1m);
    double l2 = 0.5 * (l1 + l3);

    /* R7 steady-state jump */
    double delb = bR - bL;
    double hbar = max2(0.5 * (hL + hR), 0.0);
    double ghbar = g * hbar;
    double su = uL + uR;
    double pbar = fma(0.25 * su, su, -ghbar);          /* \bar P */
    double ptil = max2(0.0, uL * uR) - ghbar;         /* \tilde P */
    double hsd = max2(0.0, fma(-l1, hL, fma(l3, hR, pL - pR))); /* h*_HLL (l3 - l1) */
    int sonic = 0;
    if (fabs(pbar) <= TAU) sonic = 1;
    if (pbar * ptil <= TAU) sonic = 1;
    if (pbar * l1 * l3 <= TAU) sonic = 1;
    if (min2(fabs(l1), fabs(l3)) < SQRT_TAU) sonic = 1;
    if (l1 < SQRT_TAU && s1m > -SQRT_TAU) sonic = 1;
    if (l3 > -SQRT_TAU && s2m < SQRT_TAU) sonic = 1;
    if ((uL + cL) * (uR + cR) < 0.0) sonic = 1;
    if ((uL - cL) * (uR - cR) < 0.0) sonic = 1;

    double dh, dphi;
    if (sonic) {
        dh = -delb;
        dphi = -ghbar * delb;
    } else {
        double q = ghbar / pbar;
        dh = delb * q;
        dphi = -delb * (q * ptil);
    }
    if (l1 < -TAU && l3 > TAU) {
        dh = min2(dh, hsd / l3);
        dh = max2(dh, hsd / l1);
    } else if (l1 >= TAU) {
        dh = min2(dh, hsd / l1);
        dh = max2(dh, -hL);
    } else if (l3 <= -TAU) {
        dh = min2(dh, hR);
        dh = max2(dh, hsd / l3);
    }
    {
        double a = -hL * delb, c = -hR * delb;
        dphi = min2(dphi, g * max2(a, c));
        dphi = max2(dphi, g * min2(a, c));
    }

    /* R8 decomposition */
    double d1 = (hR - hL) - dh;
    double d2 = pR - pL;
    double d3 = (phiR - phiL) - dphi;
    double rdl = 1.0 / (l3 - l1);
    double l1sq = l1 * l1, l3sq = l3 * l3;
    double b1 = fma(l3, d1, -d2) * rdl;
    double b3 = fma(-l1, d1, d2) * rdl;
    double b2 = fma(-l3sq, b3, fma(-l1sq, b1, d3));

    Z[0][0] = b1 * l1;  Z[0][1] = b1 * l1sq;  Z[0][2] = vL * Z[0][0];
    Z[2][0] = b3 * l3;  Z[2][1] = b3 * l3sq;  Z[2][2] = vR * Z[2][0];
    Z[1][0] = 0.0;      Z[1][1] = b2;         Z[1][2] = ((pR * vR - pL * vL) - Z[0][2]) - Z[2][2];
    s[0] = l1; s[1] = l2; s[2] = l3;

    /* wall mask */
    if (w0 == 0.0) { s[0] = 0.0; Z[0][0] = 0.0; Z[0][1] = 0.0; Z[0][2] = 0.0; }
    if (w1 == 0.0) { s[1] = 0.0; Z[1][0] = 0.0; Z[1][1] = 0.0; Z[1][2] = 0.0; }
    if (w2 == 0.0) { s[2] = 0.0; Z[2][0] = 0.0; Z[2][1] = 0.0; Z[2][2] = 0.0; }
}
