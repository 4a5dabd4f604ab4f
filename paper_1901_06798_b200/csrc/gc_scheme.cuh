// gc_scheme.cuh -- the per-edge arithmetic of the wave-propagation scheme shared by every kernel that needs
// a flux-like quantity at an edge (sweep kernels A5/A6, flux registers A8).
//
// P:65-105 (eqs. 4-11) in f-wave form; (1) Riemann solve (gc_riemann.cuh), (2) edge scaling
// on the sphere, (3) fluctuations A-dQ / A+dQ (eq. 5-6, tie S-4), (4) MC-limited waves
// (eq. 10-11, S-1), (5) correction flux (eq. 9), (6) fm = F~ + A-dQ, fp = F~ - A+dQ.
// Every expression is written in the order of DESIGN.md -- fused multiply-adds exactly where it writes fma (__fma_rn), no
// contraction elsewhere (-fmad=false) -- so that all users get the same bits.
#pragma once
#include "gc_riemann.cuh"

struct Waves { double Z[3][3]; double s[3]; };

__device__ __forceinline__ void gc_waves_zero(Waves &W)
{
#pragma unroll
    for (int w = 0; w < 3; w++) { W.s[w] = 0.0; W.Z[w][0] = 0.0; W.Z[w][1] = 0.0; W.Z[w][2] = 0.0; }
}

// (1)+(2) with the primitive variables of both sides already computed (gc_prim applied by the caller)
template <class M>
__device__ __forceinline__ void gc_solve_edge_prim(M &m, double g, double eps, const RState &L, const RState &R, int coord, double ef, Waves &W)
{
    gc_riemann(m, g, eps, L, R, W.Z, W.s);
    if (coord == 1) {
#pragma unroll
        for (int w = 0; w < 3; w++) { W.s[w] = W.s[w] * ef; W.Z[w][0] = W.Z[w][0] * ef; W.Z[w][1] = W.Z[w][1] * ef; W.Z[w][2] = W.Z[w][2] * ef; }
    }
}

// (1)+(2): solve the edge between two cells given as raw (h, p, t, b) and scale by the edge factor ef
template <class M>
__device__ __forceinline__ void gc_solve_edge(M &m, double g, double eps, RState L, RState R, int coord, double ef, Waves &W)
{
    gc_prim(m, L, g, eps);
    gc_prim(m, R, g, eps);
    gc_solve_edge_prim(m, g, eps, L, R, coord, ef, W);
}

// Z_a^w . Z_b^w per family.  The product is commutative term by term, so the same three numbers serve the
// limiter of edge a (upwind neighbour b) and of edge b (upwind neighbour a) -- eq. 10 with reading S-1.
__device__ __forceinline__ void gc_wave_dots(const Waves &A, const Waves &B, double (&d)[3])
{
#pragma unroll
    for (int w = 0; w < 3; w++) d[w] = __fma_rn(A.Z[w][2], B.Z[w][2], __fma_rn(A.Z[w][1], B.Z[w][1], A.Z[w][0] * B.Z[w][0]));
}

// MC limiter value for one family: zi = Z_I . Z_e, zz = Z_e . Z_e (zz != 0)
template <class M>
__device__ __forceinline__ double gc_mc(M &m, double zi, double zz)
{
    double theta = m.div(zi, zz);                                                    // eq. 10 (S-1)
    return dmax(0.0, dmin(dmin(__fma_rn(0.5, theta, 0.5), 2.0), 2.0 * theta));  // MC; fma(.5, t, .5) = .5 (1 + t) bit for bit
}

// (3)-(5) for edge e: fluctuations am = A-dQ, ap = A+dQ and limited correction flux F.  dlo[w] = Z_{e-1}^w . Z_e^w, dhi[w] = Z_{e+1}^w . Z_e^w (eq. 11: I = e-1 if s > 0, e+1 if s < 0).
// rdL, rdR = 1/(kappa dx) of the left / right cell.
template <class M>
__device__ __forceinline__ void gc_edge_terms(M &m, const Waves &W, const double (&dlo)[3], const double (&dhi)[3], int limiter,
                                              double dt, double rdL, double rdR, double (&am)[3], double (&ap)[3], double (&F)[3])
{
#pragma unroll
    for (int c = 0; c < 3; c++) { am[c] = 0.0; ap[c] = 0.0; F[c] = 0.0; }
    double T[3][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};
#pragma unroll
    for (int w = 0; w < 3; w++) {
#pragma unroll
        for (int c = 0; c < 3; c++) {
            if (W.s[w] < 0.0) am[c] = am[c] + W.Z[w][c];
            else if (W.s[w] > 0.0) ap[c] = ap[c] + W.Z[w][c];
            else { am[c] = am[c] + 0.5 * W.Z[w][c]; ap[c] = ap[c] + 0.5 * W.Z[w][c]; }
        }
    }
    if (limiter != 0) {
        double dtdx_ave = 0.5 * __fma_rn(dt, rdL, dt * rdR);
#pragma unroll
        for (int w = 0; w < 3; w++) {
            double sw = W.s[w];
            if (sw != 0.0) {
                double zz = __fma_rn(W.Z[w][2], W.Z[w][2], __fma_rn(W.Z[w][1], W.Z[w][1], W.Z[w][0] * W.Z[w][0]));
                double phi = 1.0;
                if (zz != 0.0) phi = gc_mc(m, (sw > 0.0) ? dlo[w] : dhi[w], zz);
                double cphi = (((sw > 0.0) ? 0.5 : -0.5) * __fma_rn(-fabs(sw), dtdx_ave, 1.0)) * phi;
#pragma unroll
                for (int c = 0; c < 3; c++) T[w][c] = cphi * W.Z[w][c];               // eq. 9, one family
            }
        }
#pragma unroll
        for (int c = 0; c < 3; c++) F[c] = (T[0][c] + T[2][c]) + T[1][c];             // outer families first: mirror-symmetric
    }
}
// (3)-(6): fm = F~ + A-dQ, fp = F~ - A+dQ
template <class M>
__device__ __forceinline__ void gc_edge_flux(M &m, const Waves &W, const double (&dlo)[3], const double (&dhi)[3], int limiter,
                                             double dt, double rdL, double rdR, double (&fm)[3], double (&fp)[3])
{
    double am[3], ap[3], F[3];
    gc_edge_terms(m, W, dlo, dhi, limiter, dt, rdL, rdR, am, ap, F);
#pragma unroll
    for (int c = 0; c < 3; c++) { fm[c] = F[c] + am[c]; fp[c] = F[c] - ap[c]; }
}

// eq. 15: right-going waves enter the right cell, left-going waves the left cell
__device__ __forceinline__ double gc_edge_cfl(const Waves &W, double rdL, double rdR)
{
    double m = 0.0;
#pragma unroll
    for (int w = 0; w < 3; w++) {
        m = dmax(m, dmax(W.s[w], 0.0) * rdR);
        m = dmax(m, dmax(-W.s[w], 0.0) * rdL);
    }
    return m;
}

// (3)-(6) for a "standard" edge, without control flow: the edge was solved by gc_riemann_fast, so s[0] < 0 < s[2] (the edge
// factor is positive) and families 1 and 3 need no sign tests; only the corrector family 2 keeps them.  Requires limiter = MC.
// Same values as gc_edge_flux: the fluctuation sums are formed in the same order, a skipped term is added as +0.0 (no bit
// changes: the partial sums start at +0.0 and are therefore never -0.0), -|s0| = s0 exactly, Z[1][0] is +0.0 by construction
// (so its square drops out of zz: fma(x, x, +0) = fl(x x) for every x).  The three limiter divides use the unchecked
// sequence: the function returns false -- and the caller redoes the edge with gc_edge_flux -- unless, for every family, the
// wave is exactly zero (then Phi = 1) or it is inside the window and the upwind product is zero (Phi = that signed zero) or inside
// the window too.  dtdx_ave = 0.5 fma(dt, rdL, dt rdR).
__device__ __forceinline__ double gc_mc_fast(double theta)
{
    return dmax(0.0, dmin(dmin(__fma_rn(0.5, theta, 0.5), 2.0), 2.0 * theta));                      // MC
}
__device__ __forceinline__ bool gc_edge_terms_std(const Waves &W, const double (&dlo)[3], const double (&dhi)[3],
                                                  double dtdx_ave, double (&am)[3], double (&ap)[3], double (&F)[3])
{
    const double s0 = W.s[0], s1 = W.s[1], s2 = W.s[2];
    const bool neg1 = s1 < 0.0, pos1 = s1 > 0.0;
    am[0] = 0.0 + W.Z[0][0];
    ap[0] = 0.0 + W.Z[2][0];
#pragma unroll
    for (int c = 1; c < 3; c++) {                       // s1 = 0 (still water over a flat bed): half of the wave each way (S-4)
        const double z = W.Z[1][c], hz = 0.5 * z;
        am[c] = (0.0 + W.Z[0][c]) + (neg1 ? z : (pos1 ? 0.0 : hz));
        ap[c] = (0.0 + (pos1 ? z : (neg1 ? 0.0 : hz))) + W.Z[2][c];
    }
    // eq. 10 (S-1), eq. 11: upwind neighbour e+1 for family 1 (s < 0), e-1 for family 3 (s > 0), by sign for family 2
    const double zz0 = __fma_rn(W.Z[0][2], W.Z[0][2], __fma_rn(W.Z[0][1], W.Z[0][1], W.Z[0][0] * W.Z[0][0]));
    const double zz1 = __fma_rn(W.Z[1][2], W.Z[1][2], W.Z[1][1] * W.Z[1][1]);
    const double zz2 = __fma_rn(W.Z[2][2], W.Z[2][2], __fma_rn(W.Z[2][1], W.Z[2][1], W.Z[2][0] * W.Z[2][0]));
    const double zi0 = dhi[0], zi1 = pos1 ? dlo[1] : dhi[1], zi2 = dlo[2];
    // a family whose wave is exactly zero (an ocean at rest: most of the domain before the tsunami arrives) takes Phi = 1, as in
    // gc_edge_flux; its quotient is garbage and discarded.  A non-zero wave needs both operands inside the divide's window.
    // A zero upwind product (the neighbour's wave vanishes: common in still water, where the corrector wave is rounding noise and
    // now and then exactly 0) gives theta = zi / zz = zi, a signed zero, and Phi(+-0) = +-0 with that sign: Phi = zi itself.
    const bool z0 = gc_is_zero(zz0), z1 = gc_is_zero(zz1), z2 = gc_is_zero(zz2);
    const bool y0 = gc_is_zero(zi0), y1 = gc_is_zero(zi1), y2 = gc_is_zero(zi2);
    const bool on1 = neg1 | pos1;                                                 // sgn(0) = 0: no correction from a steady wave
    const bool ok = (z0 | (gc_in_window(zz0) & (y0 | gc_in_window(zi0)))) & (!on1 | z1 | (gc_in_window(zz1) & (y1 | gc_in_window(zi1))))
                    & (z2 | (gc_in_window(zz2) & (y2 | gc_in_window(zi2))));    // bitwise on purpose: no short-circuit branches
    const double p0 = gc_mc_fast(gc_fdiv(zi0, zz0)), p1 = gc_mc_fast(gc_fdiv(zi1, zz1)), p2 = gc_mc_fast(gc_fdiv(zi2, zz2));
    const double c0 = (-0.5 * __fma_rn(s0, dtdx_ave, 1.0)) * (z0 ? 1.0 : (y0 ? zi0 : p0));
    const double c1 = ((pos1 ? 0.5 : -0.5) * __fma_rn(-fabs(s1), dtdx_ave, 1.0)) * (z1 ? 1.0 : (y1 ? zi1 : p1));
    const double c2 = (0.5 * __fma_rn(-s2, dtdx_ave, 1.0)) * (z2 ? 1.0 : (y2 ? zi2 : p2));
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const double t1 = c1 * W.Z[1][c];
        F[c] = (c0 * W.Z[0][c] + c2 * W.Z[2][c]) + (on1 ? t1 : 0.0);                                 // eq. 9, outer families first
    }
    return ok;
}
// (6) on top of it: fm = F~ + A-dQ, fp = F~ - A+dQ
__device__ __forceinline__ bool gc_edge_flux_std(const Waves &W, const double (&dlo)[3], const double (&dhi)[3],
                                                 double dtdx_ave, double (&fm)[3], double (&fp)[3])
{
    double am[3], ap[3], F[3];
    const bool ok = gc_edge_terms_std(W, dlo, dhi, dtdx_ave, am, ap, F);
#pragma unroll
    for (int c = 0; c < 3; c++) { fm[c] = F[c] + am[c]; fp[c] = F[c] - ap[c]; }
    return ok;
}

// eq. 15 for a standard edge (s[0] < 0 < s[2]): max(s0, 0) and max(-s2, 0) are +0, and the corrector speed
// s1 = 0.5 (s0 + s2) lies between the outer two, so its terms are never the largest (rounding is monotone):
// the edge's value is max(-s0 rdL, s2 rdR), the same number gc_edge_cfl returns.
__device__ __forceinline__ double gc_edge_cfl_std(const Waves &W, double rdL, double rdR)
{
    return dmax((-W.s[0]) * rdL, W.s[2] * rdR);
}

// ---- Manning friction (eq. 1b-1c, 2, reading S-16) -----------------------------------------
// Cube root of a positive normal double by a fixed sequence (no library call, so that every compiler produces the same
// bits): bit pattern / 3 + K as the seed (worst relative error 3.2 %), then three Halley steps -- gc_cbrt_m below.

// Semi-implicit fractional step of one cell over dt: hu, hv <- hu / d, hv / d with d = 1 + dt g n^2 |(hu, hv)| / h^(7/3)
// (D of eq. 2 read over the momenta), for dry_tol < h <= friction_depth; gn2 = g * (n * n) formed by the host in that order.
// Returns the new (hu, hv) by value (references would give the calling kernel a stack frame); out of line, so that the default
// (friction off) path of the marching kernels keeps its registers.  M = MathFast: the six divides and the square root as the
// branch-free correctly rounded sequences of gc_math.cuh (the two final divides share their reciprocal); operands outside
// its window fall back to M = MathIeee.  Both give the oracle's bits.
template <class M>
__device__ __forceinline__ double gc_cbrt_m(M &m, double x)
{
    unsigned long long i = (unsigned long long)__double_as_longlong(x);
    i = i / 3ull + 0x2A9F762500000000ull;
    double y = __longlong_as_double((long long)i);
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const double y3 = (y * y) * y;
        y = y * m.div(y3 + 2.0 * x, 2.0 * y3 + x);
    }
    return y;
}
template <class M>
__device__ __forceinline__ double2 gc_friction_m(M &m, double gn2, double dt, double h, double hu, double hv)
{
    const double mag = m.sqrt_(__fma_rn(hu, hu, hv * hv));
    const double c = gc_cbrt_m(m, h);
    const double gam = m.div(gn2 * mag, (h * h) * c);
    const double d = __fma_rn(dt, gam, 1.0);
    return make_double2(m.div(hu, d), m.div(hv, d));
}
static __device__ __noinline__ double2 gc_friction_apply(double gn2, double eps, double fdepth, double dt, double h, double hu, double hv)
{
    if (!(h > eps) || !(h <= fdepth)) return make_double2(hu, hv);
    MathFast mf;
    const double2 q = gc_friction_m(mf, gn2, dt, h, hu, hv);
    if (!mf.failed()) return q;
    MathIeee mi;
    return gc_friction_m(mi, gn2, dt, h, hu, hv);
}
