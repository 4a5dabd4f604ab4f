// gc_riemann.cuh -- device Riemann solver of the sweep kernels (A5/A6).
//
// P:122 names the solver (George 2008, augmented system with topography and momentum flux) and its
// properties; the steps R0-R8 implemented here are DESIGN.md section 3.3.  Every expression is
// evaluated in the order DESIGN.md states: fused multiply-adds exactly where it writes fma(a, b, c) (__fma_rn here, C99
// fma in the oracle), no contraction anywhere else (the library is built with -fmad=false), '/' and sqrt IEEE, so the
// result is bit-identical to a plain C evaluation.  Divides, reciprocals and
// square roots go through a math policy M (gc_math.cuh): MathIeee = the operators, MathFast = the same
// correctly rounded results without a branch per operation (valid inside an exponent window, else M.failed()).
#pragma once
#include <cuda_runtime.h>
#include "gc_math.cuh"

#define GC_TAU 1.0e-6
#define GC_SQRT_TAU 1.0e-3

__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }

struct RState { double h, p, t, b, u, v, phi, c; };   // depth, normal/transverse momentum, bathymetry, velocities, momentum flux, celerity

// R2: primitive variables of one side (h <= eps: dry, everything zero)
template <class M>
__device__ __forceinline__ void gc_prim(M &m, RState &S, double g, double eps)
{
    if (S.h < 0.0) { S.h = 0.0; S.p = 0.0; S.t = 0.0; }      // R0
    if (S.h <= eps) {
        S.h = 0.0; S.p = 0.0; S.t = 0.0; S.u = 0.0; S.v = 0.0; S.phi = 0.0;
        S.c = g * S.h;                                        // sqrt(g * 0) = sqrt(+-0) = +-0 = g * 0 itself: no call of the root, whose
    } else {                                                  // zero operand takes the IEEE sequence's out-of-line path (land cells)
        double rh = m.rcp(S.h);
        S.u = S.p * rh; S.v = S.t * rh;
        S.phi = __fma_rn(S.p, S.u, 0.5 * g * (S.h * S.h));
        S.c = m.sqrt_(g * S.h);
    }
}

// R5: flat-bottom two-wave middle state M(hL, hR, uL, uR) -> (hm, sigma1, sigma2)
template <class M>
__device__ __forceinline__ void gc_middle(M &m, double g, double eps, double hL, double hR, double uL, double uR,
                                          double cL, double cR, double &hm, double &s1m, double &s2m)
{
    double hmin = dmin(hL, hR), hmax = dmax(hL, hR);
    double du = uR - uL;
    if (hmin <= eps) {
        double s = ((uR + uL) - 2.0 * cR) + 2.0 * cL;
        hm = 0.0; s1m = s; s2m = s;
        return;
    }
    double cmin = (hL < hR) ? cL : cR;
    double cmax = (hL < hR) ? cR : cL;
    double Fmin = du + 2.0 * (cmin - cmax);
    double Fmax = __fma_rn(hmax - hmin, m.sqrt_(m.div(0.5 * g * (hmax + hmin), hmax * hmin)), du);
    if (Fmin > 0.0) {                       // two rarefactions
        double cm = 0.25 * dmax(0.0, 2.0 * (cL + cR) - du);
        hm = m.div(cm * cm, g);
        s1m = __fma_rn(-3.0, cm, uL + 2.0 * cL);
        s2m = __fma_rn(3.0, cm, uR - 2.0 * cR);
    } else if (Fmax <= 0.0) {               // two shocks: one Newton step in sqrt(h) from hmax
        double h0 = hmax;
        double gL = m.sqrt_(0.5 * g * (m.rcp(h0) + m.rcp(hL)));
        double gR = m.sqrt_(0.5 * g * (m.rcp(h0) + m.rcp(hR)));
        double F0 = __fma_rn(h0 - hR, gR, __fma_rn(h0 - hL, gL, du));
        double dfdh = (gL - m.div(g * (h0 - hL), 4.0 * (h0 * h0) * gL))
                    + (gR - m.div(g * (h0 - hR), 4.0 * (h0 * h0) * gR));
        double sq0 = m.sqrt_(h0);
        double slope = 2.0 * sq0 * dfdh;
        double sq = sq0 - m.div(F0, slope);
        double h1 = sq * sq;
        double u1m = __fma_rn(-(h1 - hL), m.sqrt_(0.5 * g * (m.rcp(h1) + m.rcp(hL))), uL);
        double u2m = __fma_rn(h1 - hR, m.sqrt_(0.5 * g * (m.rcp(h1) + m.rcp(hR))), uR);
        double cm = m.sqrt_(g * h1);
        hm = h1; s1m = u1m - cm; s2m = u2m + cm;
    } else {                                // shock + rarefaction: one secant step from hmin
        double h1 = hmin - m.div(Fmin * (hmax - hmin), Fmax - Fmin);
        double cm = m.sqrt_(g * h1);
        hm = h1;
        if (hL > hR) { s1m = __fma_rn(-3.0, cm, uL + 2.0 * cL); s2m = (uL + 2.0 * cL) - cm; }
        else         { s2m = __fma_rn(3.0, cm, uR - 2.0 * cR); s1m = (uR - 2.0 * cR) + cm; }
    }
}

// Full solve.  L and R must have gone through gc_prim.  Z[p][k]: f-wave of family p, component k
// (0: h, 1: normal momentum, 2: transverse momentum); s[p]: speeds.
template <class M>
__device__ __forceinline__ void gc_riemann(M &m, double g, double eps, RState L, RState R, double (&Z)[3][3], double (&s)[3])
{
#pragma unroll
    for (int p = 0; p < 3; p++) { s[p] = 0.0; Z[p][0] = 0.0; Z[p][1] = 0.0; Z[p][2] = 0.0; }
    if (L.h <= eps && R.h <= eps) return;                       // R1

    bool m0 = true, m1 = true, m2 = true;                      // R3 wall mask
    if (R.h <= eps) {
        double hw, a1, a2;
        gc_middle(m, g, eps, L.h, L.h, L.u, -L.u, L.c, L.c, hw, a1, a2);
        double htest = dmax(L.h, hw);
        if (htest + L.b < R.b) {
            m1 = false; m2 = false;
            R.h = L.h; R.p = -L.p; R.t = L.t; R.b = L.b; R.phi = L.phi; R.u = -L.u; R.v = L.v; R.c = L.c;
        } else if (L.h + L.b < R.b) {
            R.b = L.h + L.b;
        }
    } else if (L.h <= eps) {
        double hw, a1, a2;
        gc_middle(m, g, eps, R.h, R.h, -R.u, R.u, R.c, R.c, hw, a1, a2);
        double htest = dmax(R.h, hw);
        if (htest + R.b < L.b) {
            m0 = false; m1 = false;
            L.h = R.h; L.p = -R.p; L.t = R.t; L.b = R.b; L.phi = R.phi; L.u = -R.u; L.v = R.v; L.c = R.c;
        } else if (R.h + R.b < L.b) {
            L.b = R.h + R.b;
        }
    }

    // R4 Einfeldt speeds
    double sL = L.u - L.c, sR = R.u + R.c;
    double uhat = m.div(L.c * L.u + R.c * R.u, L.c + R.c);
    double chat = m.sqrt_(g * (0.5 * (L.h + R.h)));
    double sE1 = dmin(sL, uhat - chat);
    double sE2 = dmax(sR, uhat + chat);

    // R5, R6
    double hm, s1m, s2m;
    gc_middle(m, g, eps, L.h, R.h, L.u, R.u, L.c, R.c, hm, s1m, s2m);
    double l1 = dmin(sE1, s2m);
    double l3 = dmax(sE2, s1m);
    double l2 = 0.5 * (l1 + l3);

    // R7 steady-state jump
    double delb = R.b - L.b;
    double hbar = dmax(0.5 * (L.h + R.h), 0.0);
    double ghbar = g * hbar;
    double su = L.u + R.u;
    double pbar = __fma_rn(0.25 * su, su, -ghbar);
    double ptil = dmax(0.0, L.u * R.u) - ghbar;
    double hsd = dmax(0.0, __fma_rn(-l1, L.h, __fma_rn(l3, R.h, L.p - R.p)));
    bool sonic = false;
    if (fabs(pbar) <= GC_TAU) sonic = true;
    if (pbar * ptil <= GC_TAU) sonic = true;
    if (pbar * l1 * l3 <= GC_TAU) sonic = true;
    if (dmin(fabs(l1), fabs(l3)) < GC_SQRT_TAU) sonic = true;
    if (l1 < GC_SQRT_TAU && s1m > -GC_SQRT_TAU) sonic = true;
    if (l3 > -GC_SQRT_TAU && s2m < GC_SQRT_TAU) sonic = true;
    if ((L.u + L.c) * (R.u + R.c) < 0.0) sonic = true;
    if ((L.u - L.c) * (R.u - R.c) < 0.0) sonic = true;

    double dh, dphi;
    if (sonic) {
        dh = -delb;
        dphi = -ghbar * delb;
    } else {
        double q = m.div(ghbar, pbar);
        dh = delb * q;
        dphi = -delb * (q * ptil);
    }
    if (l1 < -GC_TAU && l3 > GC_TAU) {
        dh = dmin(dh, m.div(hsd, l3));
        dh = dmax(dh, m.div(hsd, l1));
    } else if (l1 >= GC_TAU) {
        dh = dmin(dh, m.div(hsd, l1));
        dh = dmax(dh, -L.h);
    } else if (l3 <= -GC_TAU) {
        dh = dmin(dh, R.h);
        dh = dmax(dh, m.div(hsd, l3));
    }
    {
        double a = -L.h * delb, c = -R.h * delb;
        dphi = dmin(dphi, g * dmax(a, c));
        dphi = dmax(dphi, g * dmin(a, c));
    }

    // R8 decomposition onto (1, l1, l1^2), (0, 0, 1), (1, l3, l3^2)
    double d1 = (R.h - L.h) - dh;
    double d2 = R.p - L.p;
    double d3 = (R.phi - L.phi) - dphi;
    double rdl = m.rcp(l3 - l1);
    double l1sq = l1 * l1, l3sq = l3 * l3;
    double b1 = __fma_rn(l3, d1, -d2) * rdl;
    double b3 = __fma_rn(-l1, d1, d2) * rdl;
    double b2 = __fma_rn(-l3sq, b3, __fma_rn(-l1sq, b1, d3));

    Z[0][0] = b1 * l1; Z[0][1] = b1 * l1sq; Z[0][2] = L.v * Z[0][0];
    Z[2][0] = b3 * l3; Z[2][1] = b3 * l3sq; Z[2][2] = R.v * Z[2][0];
    Z[1][0] = 0.0;     Z[1][1] = b2;        Z[1][2] = ((R.p * R.v - L.p * L.v) - Z[0][2]) - Z[2][2];
    s[0] = l1; s[1] = l2; s[2] = l3;
    if (!m0) { s[0] = 0.0; Z[0][0] = 0.0; Z[0][1] = 0.0; Z[0][2] = 0.0; }
    if (!m1) { s[1] = 0.0; Z[1][0] = 0.0; Z[1][1] = 0.0; Z[1][2] = 0.0; }
    if (!m2) { s[2] = 0.0; Z[2][0] = 0.0; Z[2][1] = 0.0; Z[2][2] = 0.0; }
}

// ---- guarded open-ocean path -------------------------------------------------------------------------------------
// The same R0-R8 result, for the edges a tsunami model meets almost everywhere (both cells wet, small Froude number,
// similar depths), written without control flow and WITHOUT step R5.  DESIGN.md 5 ("guard") gives the argument; in short:
// with c- = min(cL, cR) and the guard
//     G:  |cL - cR| <= c-/4,   |uL| <= c-/4,   |uR| <= c-/4,   c- >= 0.1,
// every branch of R5 (two rarefactions, two shocks after its one Newton step, shock + rarefaction after its one secant step)
// returns sigma1 <= -c-/4 and sigma2 >= c-/4, while sE1 <= uL - cL < 0 < uR + cR <= sE2.  Hence R6 gives lambda1 = sE1 and
// lambda3 = sE2 whatever R5 returned, none of the eight near-critical tests of R7 can fire (each quantity they compare with
// tau = 1e-6 or sqrt(tau) is bounded away from it by more than a factor 50), and the clamp case is lambda1 < -tau < tau <
// lambda3.  R5 only ever decides these comparisons, so it is not evaluated at all.  The slack in every inequality is >= 0.02
// absolute against rounding errors of 1e-16 c.  tests/test_oracle_guard.py checks the claim on the oracle's own R5.
// Both functions return false when the cell / edge is not of that kind; the caller then runs the general code above.
// Where they return true they produce its bits.  Division and roots use the unchecked sequences of gc_math.cuh; their
// operands are inside the window by the same bounds: h in (hlo, 2^100], c in [0.1, 2^54], |p-bar| >= (15/16) c-^2,
// lambda3 - lambda1 >= 1.5 c-; the numerator of u-hat may be zero or tiny, and is then absorbed by -+ c-hat.

// R0 + R2 of a cell.  hlo = max(dry tolerance, 2^-100); hg = 0.5 * g.  false: dry, or h outside (hlo, 2^100].
__device__ __forceinline__ bool gc_prim_fast(RState &S, double g, double hg, double hlo)
{
    const double rh = gc_frcp(S.h);
    S.u = S.p * rh; S.v = S.t * rh;
    S.phi = __fma_rn(S.p, S.u, hg * (S.h * S.h));
    S.c = gc_fsqrt(g * S.h);
    return (S.h > hlo) & (S.h <= 0x1p100);
}

// R3-R8 of an edge whose two cells passed gc_prim_fast.  Writes all of Z and s (garbage when it returns false).
__device__ __forceinline__ bool gc_riemann_fast(double g, const RState &L, const RState &R, double (&Z)[3][3], double (&s)[3])
{
    const double hL = L.h, hR = R.h, cL = L.c, cR = R.c;
    // guard G
    const double cmn = dmin(cL, cR);
    const double c4 = 0.25 * cmn;
    bool ok = (fabs(cL - cR) <= c4) & (fabs(L.u) <= c4) & (fabs(R.u) <= c4) & (cmn >= 0.1);      // bitwise: no short-circuit branches
    // R4 (= R6 under G)
    const double hsum = hL + hR;
    const double ghbar = g * (0.5 * hsum);                               // max(0.5 (hL + hR), 0) = 0.5 (hL + hR): both wet
    const double uhat = gc_fdiv(cL * L.u + cR * R.u, cL + cR);
    const double chat = gc_fsqrt(ghbar);
    const double l1 = dmin(L.u - cL, uhat - chat);
    const double l3 = dmax(R.u + cR, uhat + chat);
    const double l2 = 0.5 * (l1 + l3);
    // R7, not near-critical, subcritical clamp
    const double delb = R.b - L.b;
    const double su = L.u + R.u;
    const double pbar = __fma_rn(0.25 * su, su, -ghbar);
    const double ptil = dmax(0.0, L.u * R.u) - ghbar;
    const double hsd = dmax(0.0, __fma_rn(-l1, hL, __fma_rn(l3, hR, L.p - R.p)));
    const double q = gc_fdiv(ghbar, pbar);
    const double dh = delb * q;
    double dphi = -delb * (q * ptil);
    // The clamp dh <- max(min(dh, hsd / l3), hsd / l1) is the identity when dh lies inside the bounds.  That is decided
    // without the two divides, with a margin far above the rounding of the products and of the quotients:
    //   dh * l3 < hsd (1 - 1e-7)  =>  dh < fl(hsd / l3);   dh * l1 < hsd (1 - 1e-7)  =>  dh > fl(hsd / l1)   (l1 < 0 < l3).
    // hsd > 1e-100 and |dh| < 1e100 keep every product away from underflow / overflow.  Otherwise: general code.
    {
        const double hs = hsd * 0.9999999;
        ok = ok & (hsd > 1.0e-100) & (fabs(dh) < 1.0e100) & (dh * l3 < hs) & (dh * l1 < hs);
    }
    {
        const double a = -hL * delb, c = -hR * delb;
        dphi = dmin(dphi, g * dmax(a, c));
        dphi = dmax(dphi, g * dmin(a, c));
    }
    // R8
    const double d1 = (hR - hL) - dh;
    const double d2 = R.p - L.p;
    const double d3 = (R.phi - L.phi) - dphi;
    const double rdl = gc_frcp(l3 - l1);
    const double l1sq = l1 * l1, l3sq = l3 * l3;
    const double b1 = __fma_rn(l3, d1, -d2) * rdl;
    const double b3 = __fma_rn(-l1, d1, d2) * rdl;
    const double b2 = __fma_rn(-l3sq, b3, __fma_rn(-l1sq, b1, d3));
    Z[0][0] = b1 * l1; Z[0][1] = b1 * l1sq; Z[0][2] = L.v * Z[0][0];
    Z[2][0] = b3 * l3; Z[2][1] = b3 * l3sq; Z[2][2] = R.v * Z[2][0];
    Z[1][0] = 0.0;     Z[1][1] = b2;        Z[1][2] = ((R.p * R.v - L.p * L.v) - Z[0][2]) - Z[2][2];
    s[0] = l1; s[1] = l2; s[2] = l3;
    return ok;
}
