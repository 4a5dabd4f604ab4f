// gc_unsplit.cu -- the unsplit wave-propagation step with transverse Riemann solves.
//
// P:309 and P:371 name it ("the original GeoClaw ... with the unsplit algorithm"); the paper's GPU code simplifies it to
// dimensional splitting.  DESIGN.md 3.13 (reading S-21) fixes the formulas.  Three kernels per step, all reading Q^n only:
//   k_uns_xedges  thread <-> x-edge: fluctuations A-dQ, A+dQ and limited correction flux F~ of the edges e = 2..nx+2 of rows
//                 1..ny+2.  The solved edges of a patch (e = 1..nx+3 of every row) form one flat sequence; a block takes windows of
//                 128 consecutive ones, 126 apart, hands the waves to the neighbours through shared memory (double-buffered: one
//                 barrier per window) and finishes the 126 in the middle.  Coalesced; 1.03 Riemann problems per edge.
//   k_uns_yedges  thread <-> column segment (32 y-edges of one of the columns 1..nx+2), lanes <-> consecutive columns, marching
//                 upwards with the last two wave sets in registers: coalesced, no barrier, 1.06 Riemann problems per edge.
//                 Both store (A-dQ, A+dQ, F~) per edge: 18 doubles per cell; eq. 15 over the edges of interior lines.
//   k_uns_update  thread <-> column segment of interior cells, lanes <-> consecutive columns (30 updating + 1 halo lane each
//                 side), marching upwards.  Row r: the four transverse splits of cell r (a+ of its left and a- of
//                 its right x-edge by the y-Jacobian, b+ of its lower and b- of its upper y-edge by the x-Jacobian, each computed
//                 ONCE -- the Jacobian's 1/h, sqrt(g h), 1/(l3 - l1) once per cell and direction); the up-going parts wait one row
//                 in registers, the right- and left-going parts reach the neighbour columns by warp shuffles; G~' of the lower
//                 edge, F~' of the left edge (the right one from the next lane), then the update of cell r-1, clean-up, friction.
// Every expression in the order of the specification (bit-identical to the oracle, tests/test_gpu_unsplit.py).
#include <mutex>
#include <string>
#include "gc_internal.h"
#include "gc_scheme.cuh"

#define UNS_SEG 32          // edges / cells per marching segment
#define UNS_WIN 126         // finished x-edges per window of 128 solved ones
#define UNS_WPB 8           // windows per block of k_uns_xedges

struct UnsArgs {
    const PatchDesc *pat;
    const double *h, *hu, *hv, *b;          // Q^n and bathymetry
    double *oh, *ohu, *ohv;                 // Q^{n+1}
    double *T;                              // 18 planes of `tot`: am_x, ap_x, F_x, bm_y, bp_y, G_y, 3 components each
    int64_t tot;
    const double *rdx, *rdy, *ey, *kappa;
    double ex, g, eps, dt, dxdy;
    int coord, limiter, write_out;
    double gn2, fdepth; int friction;
    DevStats *stats;
};

__device__ __forceinline__ RState uns_cell(const UnsArgs &a, int64_t o, int dir)
{
    RState S; S.h = a.h[o]; S.b = a.b[o];
    if (dir == 0) { S.p = a.hu[o]; S.t = a.hv[o]; } else { S.p = a.hv[o]; S.t = a.hu[o]; }
    S.u = 0.0; S.v = 0.0; S.phi = 0.0; S.c = 0.0;
    return S;
}

// solve one edge: the guarded open-ocean code where it applies, else the general code (same bits where both apply).
// Returns true for a "standard" edge (guarded code: s[0] < 0 < s[2]), which the control-flow-free gc_edge_terms_std may finish.
__device__ __forceinline__ bool uns_solve(const UnsArgs &a, const RState &L0, const RState &R0, double ef, Waves &W)
{
    RState L = L0, R = R0;
    const double hlo = a.eps > 0x1p-100 ? a.eps : 0x1p-100;
    const bool okL = gc_prim_fast(L, a.g, 0.5 * a.g, hlo);
    const bool okR = gc_prim_fast(R, a.g, 0.5 * a.g, hlo);
    const bool ok = gc_riemann_fast(a.g, L, R, W.Z, W.s) & okL & okR & (a.g >= 0x1p-20) & (a.g <= 0x1p20);
    if (!ok) {
        MathIeee mi;
        L = L0; R = R0;
        gc_prim(mi, L, a.g, a.eps); gc_prim(mi, R, a.g, a.eps);
        gc_riemann(mi, a.g, a.eps, L, R, W.Z, W.s);
    }
    if (a.coord == 1) {
#pragma unroll
        for (int w = 0; w < 3; w++) { W.s[w] = W.s[w] * ef; W.Z[w][0] = W.Z[w][0] * ef; W.Z[w][1] = W.Z[w][1] * ef; W.Z[w][2] = W.Z[w][2] * ef; }
    }
    return ok;
}

// (3)-(5) of one edge and its three planes of each kind, at offset o of plane set T
__device__ __forceinline__ void uns_finish(const UnsArgs &a, const Waves &We, bool stdE, const double (&dlo)[3], const double (&dhi)[3],
                                           double rdL, double rdR, double *T)
{
    double am[3], ap[3], F[3];
    bool done = false;
    if (stdE && a.limiter != 0) done = gc_edge_terms_std(We, dlo, dhi, 0.5 * __fma_rn(a.dt, rdL, a.dt * rdR), am, ap, F);
    if (!done) { MathIeee mi; gc_edge_terms(mi, We, dlo, dhi, a.limiter, a.dt, rdL, rdR, am, ap, F); }
#pragma unroll
    for (int k = 0; k < 3; k++) { T[(int64_t)k * a.tot] = am[k]; T[(int64_t)(3 + k) * a.tot] = ap[k]; T[(int64_t)(6 + k) * a.tot] = F[k]; }
}

__device__ __forceinline__ void uns_cpa8(unsigned sdst, const double *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" :: "r"(sdst), "l"(gsrc) : "memory");
}

__device__ __forceinline__ void uns_cfl_out(const UnsArgs &a, double cfl)
{
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) cfl = dmax(cfl, __longlong_as_double(__shfl_xor_sync(0xffffffffu, __double_as_longlong(cfl), s)));
    if ((threadIdx.x & 31) == 0 && cfl > 0.0) atomicMax(&a.stats->sdx_bits, (unsigned long long)__double_as_longlong(cfl));
}

// grid = patches x groups of UNS_WPB windows.  Flat index t of a solved edge: row 1 + t / (nx+3), edge e = 1 + t % (nx+3).
__global__ void __launch_bounds__(128) k_uns_xedges(UnsArgs a)
{
    __shared__ double sZ[2][9][128];
    const PatchDesc pd = a.pat[blockIdx.x];
    const int k = threadIdx.x;
    const int ne2 = pd.nx + 3, nflat = (pd.ny + 2) * ne2;
    const int nwin = (nflat + UNS_WIN - 1) / UNS_WIN;
    const int w0 = blockIdx.y * UNS_WPB, w1 = min(nwin, w0 + UNS_WPB);
    double cfl = 0.0;
    // where thread k stands in window w; a thread outside the sequence loads the patch's first edge and solves nothing
    auto locate = [&](int w, int &line, int &e, int64_t &o) -> bool {
        const int t = UNS_WIN * w - 1 + k;
        const bool act = t >= 0 && t < nflat;
        line = act ? 1 + t / ne2 : 1;
        e = act ? 1 + (t - (line - 1) * ne2) : 1;
        o = pd.off + (int64_t)line * pd.pitch + e;
        return act;
    };
    int line, e; int64_t o;
    bool active = locate(w0, line, e, o);
    RState cL = uns_cell(a, o - 1, 0), cR = uns_cell(a, o, 0);
    double rd = a.rdx[pd.j0 + line];
    for (int w = w0; w < w1; w++) {
        const int buf = w & 1;
        int line2 = line, e2 = e; int64_t o2 = o; bool act2 = false;
        RState nL = cL, nR = cR;
        double rd2 = rd;
        if (w + 1 < w1) {                                       // the next window's cells, loaded a window ahead of their use
            act2 = locate(w + 1, line2, e2, o2);
            nL = uns_cell(a, o2 - 1, 0); nR = uns_cell(a, o2, 0);
            rd2 = a.rdx[pd.j0 + line2];
        }
        Waves We;
        bool stdE = false;
        if (active) stdE = uns_solve(a, cL, cR, a.ex, We);
        else gc_waves_zero(We);
#pragma unroll
        for (int q = 0; q < 3; q++) { sZ[buf][3 * q][k] = We.Z[q][0]; sZ[buf][3 * q + 1][k] = We.Z[q][1]; sZ[buf][3 * q + 2][k] = We.Z[q][2]; }
        __syncthreads();
        if (active && k >= 1 && k <= UNS_WIN && e >= 2 && e <= pd.nx + 2) {
            double dlo[3], dhi[3];
#pragma unroll
            for (int q = 0; q < 3; q++) {                      // gc_wave_dots with the neighbour's waves read from shared memory
                dlo[q] = __fma_rn(We.Z[q][2], sZ[buf][3 * q + 2][k - 1], __fma_rn(We.Z[q][1], sZ[buf][3 * q + 1][k - 1], We.Z[q][0] * sZ[buf][3 * q][k - 1]));
                dhi[q] = __fma_rn(sZ[buf][3 * q + 2][k + 1], We.Z[q][2], __fma_rn(sZ[buf][3 * q + 1][k + 1], We.Z[q][1], sZ[buf][3 * q][k + 1] * We.Z[q][0]));
            }
            uns_finish(a, We, stdE, dlo, dhi, rd, rd, a.T + o);
            if (line >= 2 && line < pd.ny + 2) cfl = dmax(cfl, gc_edge_cfl(We, rd, rd));
        }
        active = act2; line = line2; e = e2; o = o2; cL = nL; cR = nR; rd = rd2;
    }
    uns_cfl_out(a, cfl);
}

// grid = patches x groups of 4 tasks (one per warp); task = (32 columns of 1..nx+2) x (UNS_SEG edges of e = 2..ny+2)
__global__ void __launch_bounds__(128) k_uns_yedges(UnsArgs a)
{
    const PatchDesc pd = a.pat[blockIdx.x];
    const int lane = threadIdx.x & 31;
    const int ncw = (pd.nx + 2 + 31) / 32, nsg = (pd.ny + 1 + UNS_SEG - 1) / UNS_SEG;
    const int task = blockIdx.y * 4 + (threadIdx.x >> 5);
    if (task >= ncw * nsg) return;
    const int cw = task % ncw, sg = task / ncw;
    const int col0 = 1 + cw * 32 + lane;
    const bool valid = col0 <= pd.nx + 2;
    const int col = valid ? col0 : pd.nx + 2;                   // lanes past the patch repeat its last column and store nothing
    const int ea = 2 + sg * UNS_SEG, eb = min(ea + UNS_SEG, pd.ny + 3);
    const bool counted = valid && col >= 2 && col < pd.nx + 2;
    // the column's cells are staged three rows ahead of their use, 8 bytes per lane and plane by cp.async into the warp's ring
    // of four rows (a DRAM round trip under this load outlasts an iteration, and plain loads two ahead would still be waited
    // for at the top of every iteration: they share a scoreboard); metric terms are loaded one iteration ahead
    __shared__ double ring[4][4][4][32];                        // warp, stage, plane (h, hu, hv, b), lane
    const int wp = threadIdx.x >> 5;
    const unsigned sl = (unsigned)__cvta_generic_to_shared(&ring[wp][0][0][lane]);
    int64_t o = pd.off + (int64_t)(ea - 2) * pd.pitch + col;
    RState cprev = uns_cell(a, o, 1);
#pragma unroll
    for (int q = 0; q < 3; q++) {                               // rows ea-1, ea, ea+1 into stages 0, 1, 2
        if (ea - 1 + q <= eb) {
            const int64_t oq = o + (int64_t)(q + 1) * pd.pitch;
            uns_cpa8(sl + q * 1024u, a.h + oq); uns_cpa8(sl + q * 1024u + 256u, a.hu + oq);
            uns_cpa8(sl + q * 1024u + 512u, a.hv + oq); uns_cpa8(sl + q * 1024u + 768u, a.b + oq);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    double efn = a.ey[pd.j0 + ea - 1], rd0 = a.rdy[pd.j0 + ea - 3 >= 0 ? pd.j0 + ea - 3 : 0], rd1 = a.rdy[pd.j0 + ea - 2], rdn = a.rdy[pd.j0 + ea - 1];
    Waves Wc;
    gc_waves_zero(Wc);
    double dlo[3] = {0.0, 0.0, 0.0};
    bool stdc = false;
    double cfl = 0.0;
    int st = 0;                                                 // ring stage of row m
    for (int m = ea - 1; m <= eb; m++) {                        // solves edge m (cells m-1 | m); finishes edge m-1
        o += pd.pitch;
        {
            const int s3 = (st + 3) & 3;
            if (m + 3 <= eb) {
                const int64_t oq = o + 3 * (int64_t)pd.pitch;
                uns_cpa8(sl + s3 * 1024u, a.h + oq); uns_cpa8(sl + s3 * 1024u + 256u, a.hu + oq);
                uns_cpa8(sl + s3 * 1024u + 512u, a.hv + oq); uns_cpa8(sl + s3 * 1024u + 768u, a.b + oq);
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
            asm volatile("cp.async.wait_group 3;" ::: "memory"); // row m has arrived
        }
        RState cnew;
        cnew.h = ring[wp][st][0][lane]; cnew.p = ring[wp][st][2][lane]; cnew.t = ring[wp][st][1][lane]; cnew.b = ring[wp][st][3][lane];
        cnew.u = 0.0; cnew.v = 0.0; cnew.phi = 0.0; cnew.c = 0.0;
        const double ef = efn, rdL = rd0, rdR = rd1;            // ey[j0 + m], rdy[j0 + m - 2], rdy[j0 + m - 1]
        rd0 = rd1; rd1 = rdn;
        if (m < eb) { efn = a.ey[pd.j0 + m + 1]; rdn = a.rdy[pd.j0 + m + 1]; }
        Waves Wn;
        const bool stdn = uns_solve(a, cprev, cnew, ef, Wn);
        double dhi[3];
        gc_wave_dots(Wn, Wc, dhi);
        if (m >= ea + 1) {
            if (valid) uns_finish(a, Wc, stdc, dlo, dhi, rdL, rdR, a.T + 9 * a.tot + (o - pd.pitch));
            if (counted) cfl = dmax(cfl, gc_edge_cfl(Wc, rdL, rdR));
        }
        Wc = Wn; stdc = stdn; cprev = cnew;
#pragma unroll
        for (int q = 0; q < 3; q++) dlo[q] = dhi[q];
        st = (st + 1) & 3;
    }
    uns_cfl_out(a, cfl);
}

// the target direction's Jacobian at the cell state (h, pn, pt): what its split needs, once per cell and
// direction; IEEE operators, the specification's order
struct UnsJac { double l1, l2, l3, z, rho; bool n1, p1, n2, p2, n3, p3; };     // the sign flags are false in a dry cell
// Both Jacobians of a cell (x: along hu, y: along hv) share 1/h and sqrt(g h).  FAST: the reciprocals and the root by the
// unchecked correctly rounded sequences of gc_math.cuh; returns false if a wet cell has an operand outside their window (the
// caller then calls the IEEE version: same bits wherever both apply).
template <bool FAST>
__device__ __forceinline__ bool uns_jac2(double g, double eps, double h, double hu, double hv, UnsJac &Jx, UnsJac &Jy)
{
    const bool wet = h > eps;
    const double gh = g * h;
    const double rh = FAST ? gc_frcp(h) : 1.0 / h;
    const double c = FAST ? gc_fsqrt(gh) : sqrt(gh);
    const double wx = hu * rh, wy = hv * rh;
    Jx.z = wy; Jy.z = wx;
    Jx.l1 = wx - c; Jx.l2 = wx; Jx.l3 = wx + c;
    Jy.l1 = wy - c; Jy.l2 = wy; Jy.l3 = wy + c;
    const double dx = Jx.l3 - Jx.l1, dy = Jy.l3 - Jy.l1;
    Jx.rho = FAST ? gc_frcp(dx) : 1.0 / dx;
    Jy.rho = FAST ? gc_frcp(dy) : 1.0 / dy;
    Jx.n1 = wet & (Jx.l1 < 0.0); Jx.p1 = wet & (Jx.l1 > 0.0); Jx.n2 = wet & (Jx.l2 < 0.0); Jx.p2 = wet & (Jx.l2 > 0.0);
    Jx.n3 = wet & (Jx.l3 < 0.0); Jx.p3 = wet & (Jx.l3 > 0.0);
    Jy.n1 = wet & (Jy.l1 < 0.0); Jy.p1 = wet & (Jy.l1 > 0.0); Jy.n2 = wet & (Jy.l2 < 0.0); Jy.p2 = wet & (Jy.l2 > 0.0);
    Jy.n3 = wet & (Jy.l3 < 0.0); Jy.p3 = wet & (Jy.l3 > 0.0);
    return !wet | (gc_in_window(h) & gc_in_window(gh) & (gh > 0.0) & gc_in_window(dx) & gc_in_window(dy));
}
// split of a (target frame: depth, momentum along the target direction, momentum across it) into the parts travelling down
// (bm) and up (bp) the target direction; a dry cell passes nothing on.  Written without control flow: the specification adds
// family p's vector to bm if lambda_p < 0, to bp if lambda_p > 0, in the order p = 1, 2, 3, starting from +0.0; here a family
// that does not take part (every family of a dry cell) is added as +0.0, which changes no bit (a partial sum that starts at +0.0 is never -0.0), and family
// 2's vector (0, 0, l2 b2) is left out of components 0 and 1 for the same reason.  A dry cell's numbers (1/h of a tiny or zero
// h) are computed and never selected.
__device__ __forceinline__ void uns_split(const UnsJac &J, const double (&a)[3], double (&bm)[3], double (&bp)[3])
{
    const double b1 = __fma_rn(J.l3, a[0], -a[1]) * J.rho;
    const double b3 = __fma_rn(-J.l1, a[0], a[1]) * J.rho;
    const double b2 = __fma_rn(-J.z, a[0], a[2]);
    double V0[3], V2[3];
    V0[0] = J.l1 * b1; V0[1] = V0[0] * J.l1; V0[2] = V0[0] * J.z;
    V2[0] = J.l3 * b3; V2[1] = V2[0] * J.l3; V2[2] = V2[0] * J.z;
    const double V12 = J.l2 * b2;
#pragma unroll
    for (int k = 0; k < 3; k++) {
        double m = 0.0 + (J.n1 ? V0[k] : 0.0), q = 0.0 + (J.p1 ? V0[k] : 0.0);
        if (k == 2) { m = m + (J.n2 ? V12 : 0.0); q = q + (J.p2 ? V12 : 0.0); }
        m = m + (J.n3 ? V2[k] : 0.0); q = q + (J.p3 ? V2[k] : 0.0);
        bm[k] = m; bp[k] = q;
    }
}

// the vector an edge sends into one of its two cells: part 0: a- = A-dQ + F~ (cell on the low side), part 1: a+ = A+dQ - F~,
// returned in the frame of the transverse (target) direction: components 1 and 2 swapped
__device__ __forceinline__ void uns_vec(const double *T, int64_t tot, int64_t o, int part, double (&at)[3])
{
    double a[3];
#pragma unroll
    for (int k = 0; k < 3; k++)
        a[k] = part == 0 ? T[(int64_t)k * tot + o] + T[(int64_t)(6 + k) * tot + o] : T[(int64_t)(3 + k) * tot + o] - T[(int64_t)(6 + k) * tot + o];
    at[0] = a[0]; at[1] = a[2]; at[2] = a[1];
}

__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_dn1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }

// ---- k_uns_update -------------------------------------------------------------------------------------------------
// What a lane needs of row r sits in 21 planes at its own cell: h, hu, hv, and (A-dQ, A+dQ, F~) of the cell's left x-edge and
// lower y-edge.  Rows are staged two ahead of their use in a ring of three, 8 bytes per lane and plane by cp.async (each warp
// its own ring: 3 x 21 x 256 bytes), so that the march never waits for memory; the right x-edge's values are the next lane's.
#define UNS_UPD_WARPS 2
#define UNS_NPL 21
#define UNS_RING_DOUBLES (3 * UNS_NPL * 32)
__device__ __forceinline__ void uns_stage_row(const UnsArgs &a, int64_t o, unsigned sdst)
{
    uns_cpa8(sdst, a.h + o); uns_cpa8(sdst + 256u, a.hu + o); uns_cpa8(sdst + 512u, a.hv + o);
    const double *T = a.T + o;
#pragma unroll
    for (int p = 0; p < 18; p++) uns_cpa8(sdst + (unsigned)(3 + p) * 256u, T + (int64_t)p * a.tot);
}

// grid = patches x groups of UNS_UPD_WARPS tasks; task = (30 updating columns, a halo lane on each side) x (UNS_SEG rows of 2..ny+1).
// Every row does the same work with no branch around the shuffles (the first and the last row of a segment compute a few numbers
// nobody uses); SPH: latitude-longitude grid (edge factors applied).
template <int SPH>
__global__ void __launch_bounds__(32 * UNS_UPD_WARPS) k_uns_update(UnsArgs a)
{
    extern __shared__ double uns_sm[];
    const PatchDesc pd = a.pat[blockIdx.x];
    const int lane = threadIdx.x & 31;
    const int ncw = (pd.nx + 29) / 30, nsg = (pd.ny + UNS_SEG - 1) / UNS_SEG;
    const int task = blockIdx.y * UNS_UPD_WARPS + (threadIdx.x >> 5);
    if (task >= ncw * nsg) return;
    const int cw = task % ncw, sg = task / ncw;
    const int col0 = 1 + cw * 30 + lane;                        // lane 0: the column left of the 30; lane 31: the one right of them
    const int col = min(col0, pd.nx + 2);                       // lanes past the patch repeat its last column and store nothing
    const bool upd = lane >= 1 && lane <= 30 && col0 <= pd.nx + 1;
    const int ja = 2 + sg * UNS_SEG, jb = min(ja + UNS_SEG, pd.ny + 2);
    const double *S = uns_sm + (threadIdx.x >> 5) * UNS_RING_DOUBLES;                       // this warp's ring
    const unsigned sl = (unsigned)__cvta_generic_to_shared(S) + (unsigned)lane * 8u;        // ... and this lane's column of it
    const int ln1 = min(lane + 1, 31);
    int64_t o = pd.off + (int64_t)(ja - 1) * pd.pitch + col;
    uns_stage_row(a, o, sl);
    asm volatile("cp.async.commit_group;" ::: "memory");
    uns_stage_row(a, o + pd.pitch, sl + (unsigned)(UNS_NPL * 256));
    asm volatile("cp.async.commit_group;" ::: "memory");
    double bpq[2][3] = {{0.0, 0.0, 0.0}, {0.0, 0.0, 0.0}};      // up-going parts of row r-1
    double dfx[3] = {0.0, 0.0, 0.0}, gp[3] = {0.0, 0.0, 0.0}, qh = 0.0, qu = 0.0, qv = 0.0;   // of cell r-1
    int st = 0;                                                 // ring stage of row r
    // metric terms of rows r-1, r (and the edge factors of edges r, r+1), loaded a row ahead of their use
    double ey0 = a.ey[pd.j0 + ja - 1], ey1 = a.ey[pd.j0 + ja], rxm = a.rdx[pd.j0 + ja - 2], rx0 = a.rdx[pd.j0 + ja - 1],
           rym = a.rdy[pd.j0 + ja - 2], ry0 = a.rdy[pd.j0 + ja - 1];
    for (int r = ja - 1; r <= jb; r++, o += pd.pitch) {
        const double ey2 = a.ey[pd.j0 + r + 2], rx1 = a.rdx[pd.j0 + r + 1], ry1 = a.rdy[pd.j0 + r + 1];
        const int st1 = st == 2 ? 0 : st + 1, st2 = st1 == 2 ? 0 : st1 + 1;
        __syncwarp();                                           // every lane has finished with row r-1, whose stage is refilled
        if (r + 2 <= jb) uns_stage_row(a, o + 2 * (int64_t)pd.pitch, sl + (unsigned)(st2 * UNS_NPL * 256));
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 1;" ::: "memory");    // rows r and r+1 have arrived
        __syncwarp();
        const double *R0 = S + st * (UNS_NPL * 32), *R1 = S + st1 * (UNS_NPL * 32);
        const double h = R0[lane], hu = R0[32 + lane], hv = R0[64 + lane];
        double amx1[3], apx[3], Fx[3], Fx1[3], amy[3], apy[3], Gy[3], amu[3], Gu[3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            amx1[k] = R0[(3 + k) * 32 + ln1]; apx[k] = R0[(6 + k) * 32 + lane]; Fx[k] = R0[(9 + k) * 32 + lane]; Fx1[k] = R0[(9 + k) * 32 + ln1];
            amy[k] = R0[(12 + k) * 32 + lane]; apy[k] = R0[(15 + k) * 32 + lane]; Gy[k] = R0[(18 + k) * 32 + lane];
            amu[k] = R1[(12 + k) * 32 + lane]; Gu[k] = R1[(18 + k) * 32 + lane];      // of the cell's upper y-edge: the next row's
        }
        UnsJac Jx, Jy;
        if (!uns_jac2<true>(a.g, a.eps, h, hu, hv, Jx, Jy)) uns_jac2<false>(a.g, a.eps, h, hu, hv, Jx, Jy);
        // a+ of the cell's left and a- of its right x-edge (target frame: components 1 and 2 swapped), split by the y-Jacobian;
        // b+ of its lower and b- of its upper y-edge, split by the x-Jacobian
        double bm[2][3], bp[2][3], cm[2][3], cp[2][3];
        {
            const double a0[3] = { apx[0] - Fx[0], apx[2] - Fx[2], apx[1] - Fx[1] };
            const double a1[3] = { amx1[0] + Fx1[0], amx1[2] + Fx1[2], amx1[1] + Fx1[1] };
            const double b0[3] = { apy[0] - Gy[0], apy[2] - Gy[2], apy[1] - Gy[1] };
            const double b1[3] = { amu[0] + Gu[0], amu[2] + Gu[2], amu[1] + Gu[1] };
            uns_split(Jy, a0, bm[0], bp[0]);
            uns_split(Jy, a1, bm[1], bp[1]);
            uns_split(Jx, b0, cm[0], cp[0]);
            uns_split(Jx, b1, cm[1], cp[1]);
        }
        if (SPH) {
            const double e0 = ey0, e1 = ey1;
#pragma unroll
            for (int q = 0; q < 2; q++)
#pragma unroll
                for (int k = 0; k < 3; k++) { bm[q][k] = bm[q][k] * e0; bp[q][k] = bp[q][k] * e1; cm[q][k] = cm[q][k] * a.ex; cp[q][k] = cp[q][k] * a.ex; }
        }
        // F~' of the cell's left x-edge: F~, the right-going parts from the column to the left (the lane below), the left-going
        // parts from this column; the right edge's F~' is the next lane's
        const double hf = 0.5 * (a.dt * ry0);
        double F2[3], dfn[3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            double v = Fx[k];
            v = __fma_rn(-hf, shfl_up1(cp[0][k]), v); v = __fma_rn(-hf, shfl_up1(cp[1][k]), v);
            v = __fma_rn(-hf, cm[0][k], v);           v = __fma_rn(-hf, cm[1][k], v);
            F2[k] = v;
        }
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const double fm = shfl_dn1(F2[k]) + amx1[k], fp = F2[k] - apx[k];
            dfn[k] = fm - fp;
        }
        // G~' of the y-edge below cell r: G~, the up-going parts from row r-1, the down-going parts from row r (3.13's order)
        double G2[3];
        const double hb = 0.5 * (a.dt * rxm), hr = 0.5 * (a.dt * rx0);
#pragma unroll
        for (int k = 0; k < 3; k++) {
            double v = Gy[k];
            v = __fma_rn(-hb, bpq[0][k], v); v = __fma_rn(-hb, bpq[1][k], v);
            v = __fma_rn(-hr, bm[0][k], v);  v = __fma_rn(-hr, bm[1][k], v);
            G2[k] = v;
        }
        if (r > ja) {                                           // it closes cell r-1
            const int j = r - 1;
            double dgy[3];
#pragma unroll
            for (int k = 0; k < 3; k++) { const double gm = G2[k] + amy[k]; dgy[k] = gm - gp[k]; }
            const double dtdx = a.dt * rxm, dtdy = a.dt * rym;
            double hh = __fma_rn(-dtdy, dgy[0], __fma_rn(-dtdx, dfx[0], qh));
            double uu = __fma_rn(-dtdy, dgy[2], __fma_rn(-dtdx, dfx[1], qu));
            double vv = __fma_rn(-dtdy, dgy[1], __fma_rn(-dtdx, dfx[2], qv));
            if (upd) {
                if (hh < a.eps && a.write_out) {                                             // dry clean-up (S-9)
                    if (hh < 0.0) {
                        atomicAdd(&a.stats->nclip, 1ull);
                        atomicAdd(&a.stats->clipped, (-hh) * (a.kappa[pd.j0 + j] * a.dxdy));
                    }
                    hh = dmax(hh, 0.0); uu = 0.0; vv = 0.0;
                }
                if (a.friction && a.write_out) {
                    const double2 q = gc_friction_apply(a.gn2, a.eps, a.fdepth, a.dt, hh, uu, vv);
                    uu = q.x; vv = q.y;
                }
                if (hh != hh || uu != uu || vv != vv) a.stats->nan_seen = 1;
                if (a.write_out) { const int64_t oc = o - pd.pitch; a.oh[oc] = hh; a.ohu[oc] = uu; a.ohv[oc] = vv; }
            }
        }
#pragma unroll
        for (int k = 0; k < 3; k++) { gp[k] = G2[k] - apy[k]; dfx[k] = dfn[k]; bpq[0][k] = bp[0][k]; bpq[1][k] = bp[1][k]; }
        qh = h; qu = hu; qv = hv;
        ey0 = ey1; ey1 = ey2; rxm = rx0; rx0 = rx1; rym = ry0; ry0 = ry1;
        st = st1;
    }
}

// the three launches of one unsplit step with the 18 scratch planes at T (plane stride L->tot doubles)
static void uns_run(gc_level *L, double dt, int write_out, double *T)
{
    const gc_params &P = L->ctx->P;
    const int cur = L->cur, nxt = 1 - cur;
    UnsArgs a;
    a.pat = L->d_pat; a.h = L->q[cur][0]; a.hu = L->q[cur][1]; a.hv = L->q[cur][2]; a.b = L->b;
    a.oh = L->q[nxt][0]; a.ohu = L->q[nxt][1]; a.ohv = L->q[nxt][2];
    a.T = T; a.tot = L->tot;
    a.rdx = L->d_rdx; a.rdy = L->d_rdy; a.ey = L->d_ey; a.kappa = L->d_kappa;
    a.ex = L->ex; a.g = P.g; a.eps = P.dry_tol; a.dt = dt; a.dxdy = L->dx * L->dy;
    a.coord = P.coord; a.limiter = P.limiter; a.write_out = write_out;
    a.gn2 = P.g * (P.manning_n * P.manning_n); a.fdepth = P.friction_depth; a.friction = P.manning_n > 0.0 ? 1 : 0;
    a.stats = L->d_stats;
    int64_t wx = 1, ty = 1, tu = 1;                            // windows of k_uns_xedges, tasks of k_uns_yedges / k_uns_update
    for (const gc_patch &Q : L->pat) {
        wx = std::max<int64_t>(wx, ((int64_t)(Q.ny + 2) * (Q.nx + 3) + UNS_WIN - 1) / UNS_WIN);
        ty = std::max<int64_t>(ty, (int64_t)((Q.nx + 2 + 31) / 32) * ((Q.ny + 1 + UNS_SEG - 1) / UNS_SEG));
        tu = std::max<int64_t>(tu, (int64_t)((Q.nx + 29) / 30) * ((Q.ny + UNS_SEG - 1) / UNS_SEG));
    }
    const dim3 gx((unsigned)L->np, (unsigned)((wx + UNS_WPB - 1) / UNS_WPB)), gy((unsigned)L->np, (unsigned)((ty + 3) / 4)),
               gu((unsigned)L->np, (unsigned)((tu + UNS_UPD_WARPS - 1) / UNS_UPD_WARPS));
    { ProfScope ps(L->ctx, GC_SLOT_XSWEEP); k_uns_xedges<<<gx, 128, 0, L->ctx->stream>>>(a); }
    { ProfScope ps(L->ctx, GC_SLOT_YSWEEP); k_uns_yedges<<<gy, 128, 0, L->ctx->stream>>>(a); }
    { ProfScope ps(L->ctx, GC_SLOT_FUSED); const size_t sm = UNS_UPD_WARPS * UNS_RING_DOUBLES * sizeof(double);
      if (P.coord == 1) k_uns_update<1><<<gu, 32 * UNS_UPD_WARPS, sm, L->ctx->stream>>>(a);
      else k_uns_update<0><<<gu, 32 * UNS_UPD_WARPS, sm, L->ctx->stream>>>(a); }
}

int gc_launch_unsplit(gc_level *L, double dt, int write_out)
{
    if (!L->d_uns) {                                            // 18 planes of scratch, allocated at the first unsplit step
        L->d_uns = (double *)gc_dev_alloc(L->ctx, (size_t)18 * (size_t)L->tot * sizeof(double));
        if (!L->d_uns) return GC_ERR_NOMEM;
        L->allocs.push_back(L->d_uns);
    }
    if (L->np == 0) return GC_OK;
    uns_run(L, dt, write_out, L->d_uns);
    return GC_OK;
}

// ---- gc_level_step_unsplit_static: the same step for callers that may not allocate (CUDA graph capture, serving loops) ------
// The 18 scratch planes live in a file-scope device array of GC_UNS_STATIC_MAX_CELLS storage cells per plane (gc.h): 37.75 MB that
// every GPU which loads the library holds until the process exits.  In host code `g_uns_static` is a host-side stand-in, not a
// device address; the address is resolved with cudaGetSymbolAddress once per device, with that device current (at gc_ctx_create;
// here, should the device not have seen one), and that pointer goes to the kernels.  Nothing in the array has to start at zero:
// every value k_uns_update uses was written by the two edge kernels of the same call (what it reads beyond that -- the x-edge
// planes of column 1, the y-edge planes of row 1 -- feeds halo lanes and rows whose results are discarded), so the previous call's
// contents do no harm.  Every call on a device shares the array: calls that overlap on the GPU (two streams, two contexts) race.
static __device__ __align__(256) double g_uns_static[(size_t)18 * GC_UNS_STATIC_MAX_CELLS];

#define GC_UNS_MAX_DEV 64
static double *g_uns_static_addr[GC_UNS_MAX_DEV];       // per device: the array's device address, resolved once
static cudaError_t g_uns_static_rc[GC_UNS_MAX_DEV];
static bool g_uns_static_tried[GC_UNS_MAX_DEV];
static std::mutex g_uns_static_mx;

// resolves the array's address on the CURRENT device; returns it, or nullptr (the CUDA error kept for the entry point's message)
static double *uns_static_resolve(cudaError_t *rc_out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= GC_UNS_MAX_DEV) { cudaGetLastError(); if (rc_out) *rc_out = e != cudaSuccess ? e : cudaErrorInvalidDevice; return nullptr; }
    std::lock_guard<std::mutex> lk(g_uns_static_mx);
    if (!g_uns_static_tried[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_uns_static);
        if (e != cudaSuccess) { cudaGetLastError(); p = nullptr; }
        g_uns_static_addr[dev] = (double *)p; g_uns_static_rc[dev] = e; g_uns_static_tried[dev] = true;
    }
    if (rc_out) *rc_out = g_uns_static_rc[dev];
    return g_uns_static_addr[dev];
}

void gc_unsplit_static_setup(void) { uns_static_resolve(nullptr); }   // gc_ctx_create: set-up time, the context's device current

extern "C" int64_t gc_unsplit_static_max_cells(void) { return (int64_t)GC_UNS_STATIC_MAX_CELLS; }

extern "C" int gc_level_step_unsplit_static(gc_level *L, double dt, gc_step_stats *out)
{
    if (!L || !(dt >= 0.0)) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_step_unsplit_static: bad argument");
    if (L->reg_fine || L->reg_coarse)
        return gc_fail(L->ctx, GC_ERR_STATE, "gc_level_step_unsplit_static: flux registers are defined for the split step only");
    if (L->tot > (int64_t)GC_UNS_STATIC_MAX_CELLS)
        return gc_fail(L->ctx, GC_ERR_BADARG, "gc_level_step_unsplit_static: level larger than GC_UNS_STATIC_MAX_CELLS storage cells "
                                              "(patch cells incl. ghost cells and row padding); use gc_level_step_unsplit");
    cudaError_t e = cudaSuccess;
    double *T = uns_static_resolve(&e);
    if (!T) {
        L->ctx->err = std::string("gc_level_step_unsplit_static: cudaGetSymbolAddress of the static scratch failed: ") + cudaGetErrorString(e);
        return GC_ERR_CUDA;
    }
    gc_launch_stats_reset(L);
    if (L->np > 0) uns_run(L, dt, dt > 0.0 ? 1 : 0, T);
    if (dt > 0.0) L->cur = 1 - L->cur;
    int rc = gc_cuda_check(L->ctx, "gc_level_step_unsplit_static");
    if (rc) return rc;
    if (out) {
        rc = gc_level_stats(L, out);
        if (rc) return rc;
        out->cfl_max = dt * out->s_over_dx_max;
        if (out->nan_seen) return gc_fail(L->ctx, GC_ERR_NAN, "gc_level_step_unsplit_static: NaN in the updated state");
    }
    return GC_OK;
}
