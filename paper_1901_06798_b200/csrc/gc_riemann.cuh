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
    } else {
        double rh = m.rcp(S.h);
        S.u = S.p * rh; S.v = S.t * rh;
        S.phi = __fma_rn(S.p, S.u, 0.5 * g * (S.h * S.h));
    }
    S.c = m.sqrt_(g * S.h);
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

// ---- straight-line variants for the common case --------------------------------------------------------------
// The same expressions in the same order as gc_prim / gc_riemann, specialised to the branch an open-ocean edge takes
// (both sides wet, one shock + one rarefaction in R5, not near-critical in R7, subcritical clamp l1 < -tau < tau < l3)
// and written without control flow, so that the independent divide / square-root chains can overlap.  They return
// false when the edge is not of that kind (or a fast-math operand left its window); the caller then runs the
// general code above.  Where both apply they produce identical bits.

// R0 + R2 without branches (the reciprocal of a dry cell's depth is taken of 1 and discarded)
__device__ __forceinline__ void gc_prim_fast(MathFast &m, RState &S, double g, double eps)
{
    const bool wet = S.h > eps;                       // h < 0 and h <= eps both end as the zero state
    const double hs = wet ? S.h : 1.0;
    const double rh = m.rcp(hs);
    const double u = S.p * rh, v = S.t * rh;
    const double phi = __fma_rn(S.p, u, 0.5 * g * (S.h * S.h));
    S.h = wet ? S.h : 0.0; S.p = wet ? S.p : 0.0; S.t = wet ? S.t : 0.0;
    S.u = wet ? u : 0.0; S.v = wet ? v : 0.0; S.phi = wet ? phi : 0.0;
    S.c = m.sqrt_(g * S.h);
}

// Lanes whose edge is not of that kind compute garbage (possibly Inf / NaN: harmless, nothing traps) that the caller
// discards; only the returned flag decides.
__device__ __forceinline__ bool gc_riemann_fast(MathFast &m, double g, double eps, const RState &L, const RState &R,
                                                double (&Z)[3][3], double (&s)[3])
{
    bool ok = (L.h > eps) && (R.h > eps);
    const double hL = L.h, hR = R.h, cL = L.c, cR = R.c;
    // R4
    const double sL = L.u - cL, sR = R.u + cR;
    const double uhat = m.div(cL * L.u + cR * R.u, cL + cR);
    const double chat = m.sqrt_(g * (0.5 * (hL + hR)));
    const double sE1 = dmin(sL, uhat - chat);
    const double sE2 = dmax(sR, uhat + chat);
    // R5, shock + rarefaction branch
    const bool deepL = hL > hR, shalL = hL < hR;
    const double hmin = shalL ? hL : hR, hmax = hL > hR ? hL : hR;
    const double du = R.u - L.u;
    const double cmin = shalL ? cL : cR;
    const double cmax = shalL ? cR : cL;
    const double Fmin = __fma_rn(2.0, cmin - cmax, du);                 // = du + 2 (cmin - cmax) bit for bit (x 2 is exact)
    const double Fmax = __fma_rn(hmax - hmin, m.sqrt_(m.div(0.5 * g * (hmax + hmin), hmax * hmin)), du);
    ok = ok && !(Fmin > 0.0) && !(Fmax <= 0.0);
    const double h1 = hmin - m.div(Fmin * (hmax - hmin), Fmax - Fmin);
    const double cm = m.sqrt_(g * h1);
    const double aL = __fma_rn(2.0, cL, L.u), aR = __fma_rn(-2.0, cR, R.u);   // = u + 2c, u - 2c bit for bit
    const double s1m = deepL ? __fma_rn(-3.0, cm, aL) : (aR + cm);
    const double s2m = deepL ? (aL - cm) : __fma_rn(3.0, cm, aR);
    // R6
    const double l1 = dmin(sE1, s2m);
    const double l3 = dmax(sE2, s1m);
    const double l2 = 0.5 * (l1 + l3);
    // R7, not near-critical, subcritical clamp
    const double delb = R.b - L.b;
    const double hbar = dmax(0.5 * (hL + hR), 0.0);
    const double ghbar = g * hbar;
    const double su = L.u + R.u;
    const double pbar = __fma_rn(0.25 * su, su, -ghbar);
    const double ptil = dmax(0.0, L.u * R.u) - ghbar;
    const double hsd = dmax(0.0, __fma_rn(-l1, hL, __fma_rn(l3, hR, L.p - R.p)));
    bool sonic = fabs(pbar) <= GC_TAU;
    sonic = sonic || (pbar * ptil <= GC_TAU);
    sonic = sonic || (pbar * l1 * l3 <= GC_TAU);
    sonic = sonic || (dmin(fabs(l1), fabs(l3)) < GC_SQRT_TAU);
    sonic = sonic || (l1 < GC_SQRT_TAU && s1m > -GC_SQRT_TAU);
    sonic = sonic || (l3 > -GC_SQRT_TAU && s2m < GC_SQRT_TAU);
    sonic = sonic || ((L.u + cL) * (R.u + cR) < 0.0);
    sonic = sonic || ((L.u - cL) * (R.u - cR) < 0.0);
    ok = ok && !sonic && (l1 < -GC_TAU) && (l3 > GC_TAU);
    const double q = m.div(ghbar, pbar);
    const double dh = delb * q;
    double dphi = -delb * (q * ptil);
    // The clamp dh <- max(min(dh, hsd / l3), hsd / l1) is the identity when dh lies inside the bounds.  That is decided
    // without the two divides, with a margin far above the rounding of the products and of the quotients:
    //   dh * l3 < hsd (1 - 1e-7)  =>  dh < fl(hsd / l3);   dh * l1 < hsd (1 - 1e-7)  =>  dh > fl(hsd / l1)   (l1 < 0 < l3).
    // hsd > 1e-100 and |dh| < 1e100 keep every product away from underflow / overflow (|l| >= tau).  Otherwise: general code.
    {
        const double hs = hsd * 0.9999999;
        ok = ok && (hsd > 1.0e-100) && (fabs(dh) < 1.0e100) && (dh * l3 < hs) && (dh * l1 < hs);
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
    const double rdl = m.rcp(l3 - l1);
    const double l1sq = l1 * l1, l3sq = l3 * l3;
    const double b1 = __fma_rn(l3, d1, -d2) * rdl;
    const double b3 = __fma_rn(-l1, d1, d2) * rdl;
    const double b2 = __fma_rn(-l3sq, b3, __fma_rn(-l1sq, b1, d3));
    Z[0][0] = b1 * l1; Z[0][1] = b1 * l1sq; Z[0][2] = L.v * Z[0][0];
    Z[2][0] = b3 * l3; Z[2][1] = b3 * l3sq; Z[2][2] = R.v * Z[2][0];
    Z[1][0] = 0.0;     Z[1][1] = b2;        Z[1][2] = ((R.p * R.v - L.p * L.v) - Z[0][2]) - Z[2][2];
    s[0] = l1; s[1] = l2; s[2] = l3;
    return ok && !m.failed();
}
