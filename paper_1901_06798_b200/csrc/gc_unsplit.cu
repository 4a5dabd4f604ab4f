// gc_unsplit.cu -- the unsplit wave-propagation step with transverse Riemann solves.
//
// P:309 and P:371 name it ("the original GeoClaw ... with the unsplit algorithm"); the paper's GPU code simplifies it to
// dimensional splitting.  DESIGN.md 3.13 (reading S-21) fixes the formulas.  Two kernels per step, both reading Q^n only:
//   k_uns_edges<DIR>  thread <-> edge: fluctuations A-dQ, A+dQ and limited correction flux F~ of every x-edge of rows 1..ny+2
//                     (every y-edge of columns 1..nx+2), by the device functions of the split sweeps (three Riemann problems per
//                     edge for the limiter: redundant, simple), stored per edge; eq. 15 over interior lines
//   k_uns_update      thread <-> interior cell: the transverse splits that reach the cell's four edges (16 per cell, in the
//                     order DESIGN.md 3.13 fixes), the modified correction fluxes, the update, clean-up, friction
// A first correct version of a "next" row: every expression in the order of the specification (bit-identical to the oracle,
// tests/test_gpu_unsplit.py); it stores 18 doubles per cell between the two kernels and is not tuned.
#include "gc_internal.h"
#include "gc_scheme.cuh"

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

// solve one edge: the guarded open-ocean code where it applies, else the general code (same bits where both apply)
__device__ __forceinline__ void uns_solve(const UnsArgs &a, const RState &L0, const RState &R0, double ef, Waves &W)
{
    RState L = L0, R = R0;
    const bool okL = gc_prim_fast(L, a.g, 0.5 * a.g, a.eps > 0x1p-100 ? a.eps : 0x1p-100);
    const bool okR = gc_prim_fast(R, a.g, 0.5 * a.g, a.eps > 0x1p-100 ? a.eps : 0x1p-100);
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
}

// grid = patches x chunks of 4096 edges.  DIR 0: edge (j, e), j = 1..ny+2, e = 2..nx+2; DIR 1: edge (e, i), i = 1..nx+2, e = 2..ny+2
template <int DIR>
__global__ void __launch_bounds__(128) k_uns_edges(UnsArgs a)
{
    const PatchDesc pd = a.pat[blockIdx.x];
    const int nl = (DIR == 0 ? pd.ny : pd.nx) + 2;            // lines
    const int ne = (DIR == 0 ? pd.nx : pd.ny) + 1;            // edges per line
    const int n = nl * ne;
    double cfl = 0.0;
    for (int t = blockIdx.y * 4096 + threadIdx.x; t < min(n, (int)(blockIdx.y + 1) * 4096); t += blockDim.x) {
        int line, e;
        if (DIR == 0) { line = 1 + t / ne; e = 2 + t % ne; } else { e = 2 + t / nl; line = 1 + t % nl; }   // x: e fastest; y: column fastest
        const int64_t str = DIR == 0 ? 1 : pd.pitch;
        const int64_t o = DIR == 0 ? pd.off + (int64_t)line * pd.pitch + e : pd.off + (int64_t)e * pd.pitch + line;
        const RState c0 = uns_cell(a, o - 2 * str, DIR), c1 = uns_cell(a, o - str, DIR), c2 = uns_cell(a, o, DIR), c3 = uns_cell(a, o + str, DIR);
        double ef0, ef1, ef2, rdL, rdR;
        if (DIR == 0) { ef0 = ef1 = ef2 = a.ex; rdL = rdR = a.rdx[pd.j0 + line]; }
        else { ef0 = a.ey[pd.j0 + e - 1]; ef1 = a.ey[pd.j0 + e]; ef2 = a.ey[pd.j0 + e + 1]; rdL = a.rdy[pd.j0 + e - 1]; rdR = a.rdy[pd.j0 + e]; }
        Waves Wl, We, Wh;
        uns_solve(a, c0, c1, ef0, Wl); uns_solve(a, c1, c2, ef1, We); uns_solve(a, c2, c3, ef2, Wh);
        double dlo[3], dhi[3], am[3], ap[3], F[3];
        gc_wave_dots(We, Wl, dlo);
        gc_wave_dots(Wh, We, dhi);
        MathIeee mi;
        gc_edge_terms(mi, We, dlo, dhi, a.limiter, a.dt, rdL, rdR, am, ap, F);
        double *T = a.T + (int64_t)(DIR == 0 ? 0 : 9) * a.tot + o;
#pragma unroll
        for (int k = 0; k < 3; k++) { T[(int64_t)k * a.tot] = am[k]; T[(int64_t)(3 + k) * a.tot] = ap[k]; T[(int64_t)(6 + k) * a.tot] = F[k]; }
        const bool interior = DIR == 0 ? (line >= 2 && line < pd.ny + 2) : (line >= 2 && line < pd.nx + 2);
        if (interior) cfl = dmax(cfl, gc_edge_cfl(We, rdL, rdR));
    }
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) cfl = dmax(cfl, __longlong_as_double(__shfl_xor_sync(0xffffffffu, __double_as_longlong(cfl), s)));
    if ((threadIdx.x & 31) == 0 && cfl > 0.0) atomicMax(&a.stats->sdx_bits, (unsigned long long)__double_as_longlong(cfl));
}

// split of a (target frame: depth, momentum along the target direction, momentum across it) by the target
// direction's Jacobian at the cell state (h, pn, pt); IEEE operators, the specification's order
__device__ __forceinline__ void gc_transverse(double g, double eps, double h, double pn, double pt, const double (&a)[3],
                                              double (&bm)[3], double (&bp)[3])
{
#pragma unroll
    for (int k = 0; k < 3; k++) { bm[k] = 0.0; bp[k] = 0.0; }
    if (!(h > eps)) return;
    const double rh = 1.0 / h;
    const double w = pn * rh, z = pt * rh, c = sqrt(g * h);
    const double l1 = w - c, l2 = w, l3 = w + c;
    const double rho = 1.0 / (l3 - l1);
    const double b1 = __fma_rn(l3, a[0], -a[1]) * rho;
    const double b3 = __fma_rn(-l1, a[0], a[1]) * rho;
    const double b2 = __fma_rn(-z, a[0], a[2]);
    double lam[3] = { l1, l2, l3 };
    double V[3][3];
    V[0][0] = l1 * b1; V[0][1] = V[0][0] * l1; V[0][2] = V[0][0] * z;
    V[1][0] = 0.0;     V[1][1] = 0.0;          V[1][2] = l2 * b2;
    V[2][0] = l3 * b3; V[2][1] = V[2][0] * l3; V[2][2] = V[2][0] * z;
#pragma unroll
    for (int p = 0; p < 3; p++)
#pragma unroll
        for (int k = 0; k < 3; k++) {
            if (lam[p] < 0.0) bm[k] = bm[k] + V[p][k];
            else if (lam[p] > 0.0) bp[k] = bp[k] + V[p][k];
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

// G~' of the y-edge at the lower side of cell (row e, column i) [offset o]: G~, then the up-going parts from row e-1, then the
// down-going parts from row e, each row's x-edges in the order (a+ of the cell's left edge, a- of its right edge)
__device__ __forceinline__ void uns_G2(const UnsArgs &a, const PatchDesc &pd, int64_t o, int e, double (&G2)[3])
{
    const double *Tx = a.T, *Ty = a.T + 9 * a.tot;
#pragma unroll
    for (int k = 0; k < 3; k++) G2[k] = Ty[(int64_t)(6 + k) * a.tot + o];
#pragma unroll
    for (int r = 0; r < 2; r++) {                               // r = 0: row e-1 (its bp), r = 1: row e (its bm)
        const int j = e - 1 + r;
        const int64_t c = o - (int64_t)(1 - r) * pd.pitch;      // the cell of that row in this column
        const double half = 0.5 * (a.dt * a.rdx[pd.j0 + j]);
        const double h = a.h[c], pn = a.hv[c], pt = a.hu[c];
#pragma unroll
        for (int q = 0; q < 2; q++) {                           // q = 0: a+ of x-edge (j, i) ; q = 1: a- of x-edge (j, i+1)
            double at[3], bm[3], bp[3];
            uns_vec(Tx, a.tot, c + q, q == 0 ? 1 : 0, at);
            gc_transverse(a.g, a.eps, h, pn, pt, at, bm, bp);
            if (a.coord == 1) {
#pragma unroll
                for (int k = 0; k < 3; k++) { bm[k] = bm[k] * a.ey[pd.j0 + j]; bp[k] = bp[k] * a.ey[pd.j0 + j + 1]; }
            }
#pragma unroll
            for (int k = 0; k < 3; k++) G2[k] = __fma_rn(-half, r == 0 ? bp[k] : bm[k], G2[k]);
        }
    }
}

// F~' of the x-edge at the left side of cell (row j, column e) [offset o]: F~, then the right-going parts from column e-1,
// then the left-going parts from column e, each column's y-edges in the order (b+ of the cell's lower edge, b- of its upper edge)
__device__ __forceinline__ void uns_F2(const UnsArgs &a, const PatchDesc &pd, int64_t o, int j, double (&F2)[3])
{
    const double *Tx = a.T, *Ty = a.T + 9 * a.tot;
#pragma unroll
    for (int k = 0; k < 3; k++) F2[k] = Tx[(int64_t)(6 + k) * a.tot + o];
    const double half = 0.5 * (a.dt * a.rdy[pd.j0 + j]);
#pragma unroll
    for (int r = 0; r < 2; r++) {                               // r = 0: column e-1 (its cp), r = 1: column e (its cm)
        const int64_t c = o - (1 - r);
        const double h = a.h[c], pn = a.hu[c], pt = a.hv[c];
#pragma unroll
        for (int q = 0; q < 2; q++) {                           // q = 0: b+ of y-edge (j, .) ; q = 1: b- of y-edge (j+1, .)
            double at[3], cm[3], cp[3];
            uns_vec(Ty, a.tot, c + (int64_t)q * pd.pitch, q == 0 ? 1 : 0, at);
            gc_transverse(a.g, a.eps, h, pn, pt, at, cm, cp);
            if (a.coord == 1) {
#pragma unroll
                for (int k = 0; k < 3; k++) { cm[k] = cm[k] * a.ex; cp[k] = cp[k] * a.ex; }
            }
#pragma unroll
            for (int k = 0; k < 3; k++) F2[k] = __fma_rn(-half, r == 0 ? cp[k] : cm[k], F2[k]);
        }
    }
}

__global__ void __launch_bounds__(128) k_uns_update(UnsArgs a)
{
    const PatchDesc pd = a.pat[blockIdx.x];
    const int n = pd.nx * pd.ny;
    const double *Tx = a.T, *Ty = a.T + 9 * a.tot;
    for (int t = blockIdx.y * 4096 + threadIdx.x; t < min(n, (int)(blockIdx.y + 1) * 4096); t += blockDim.x) {
        const int j = 2 + t / pd.nx, i = 2 + t % pd.nx;
        const int64_t o = pd.off + (int64_t)j * pd.pitch + i;
        double Fl[3], Fr[3], Gl[3], Gu[3];
        uns_F2(a, pd, o, j, Fl); uns_F2(a, pd, o + 1, j, Fr);
        uns_G2(a, pd, o, j, Gl); uns_G2(a, pd, o + pd.pitch, j + 1, Gu);
        double dfx[3], dgy[3];
#pragma unroll
        for (int k = 0; k < 3; k++) {
            const double fm = Fr[k] + Tx[(int64_t)k * a.tot + o + 1], fp = Fl[k] - Tx[(int64_t)(3 + k) * a.tot + o];
            const double gm = Gu[k] + Ty[(int64_t)k * a.tot + o + pd.pitch], gp = Gl[k] - Ty[(int64_t)(3 + k) * a.tot + o];
            dfx[k] = fm - fp; dgy[k] = gm - gp;
        }
        const double dtdx = a.dt * a.rdx[pd.j0 + j], dtdy = a.dt * a.rdy[pd.j0 + j];
        double hh = __fma_rn(-dtdy, dgy[0], __fma_rn(-dtdx, dfx[0], a.h[o]));
        double uu = __fma_rn(-dtdy, dgy[2], __fma_rn(-dtdx, dfx[1], a.hu[o]));
        double vv = __fma_rn(-dtdy, dgy[1], __fma_rn(-dtdx, dfx[2], a.hv[o]));
        if (hh < a.eps && a.write_out) {                                                 // dry clean-up (S-9)
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
        if (a.write_out) { a.oh[o] = hh; a.ohu[o] = uu; a.ohv[o] = vv; }
    }
}

int gc_launch_unsplit(gc_level *L, double dt, int write_out)
{
    const gc_params &P = L->ctx->P;
    if (!L->d_uns) {                                            // 18 planes of scratch, allocated at the first unsplit step
        L->d_uns = (double *)gc_dev_alloc(L->ctx, (size_t)18 * (size_t)L->tot * sizeof(double));
        if (!L->d_uns) return GC_ERR_NOMEM;
        L->allocs.push_back(L->d_uns);
    }
    if (L->np == 0) return GC_OK;
    const int cur = L->cur, nxt = 1 - cur;
    UnsArgs a;
    a.pat = L->d_pat; a.h = L->q[cur][0]; a.hu = L->q[cur][1]; a.hv = L->q[cur][2]; a.b = L->b;
    a.oh = L->q[nxt][0]; a.ohu = L->q[nxt][1]; a.ohv = L->q[nxt][2];
    a.T = L->d_uns; a.tot = L->tot;
    a.rdx = L->d_rdx; a.rdy = L->d_rdy; a.ey = L->d_ey; a.kappa = L->d_kappa;
    a.ex = L->ex; a.g = P.g; a.eps = P.dry_tol; a.dt = dt; a.dxdy = L->dx * L->dy;
    a.coord = P.coord; a.limiter = P.limiter; a.write_out = write_out;
    a.gn2 = P.g * (P.manning_n * P.manning_n); a.fdepth = P.friction_depth; a.friction = P.manning_n > 0.0 ? 1 : 0;
    a.stats = L->d_stats;
    int64_t me = 1, mc = 1;
    for (const gc_patch &Q : L->pat) {
        me = std::max<int64_t>(me, std::max<int64_t>((int64_t)(Q.ny + 2) * (Q.nx + 1), (int64_t)(Q.nx + 2) * (Q.ny + 1)));
        mc = std::max<int64_t>(mc, (int64_t)Q.nx * Q.ny);
    }
    const dim3 ge((unsigned)L->np, (unsigned)((me + 4095) / 4096)), gc((unsigned)L->np, (unsigned)((mc + 4095) / 4096));
    { ProfScope ps(L->ctx, GC_SLOT_XSWEEP); k_uns_edges<0><<<ge, 128, 0, L->ctx->stream>>>(a); }
    { ProfScope ps(L->ctx, GC_SLOT_YSWEEP); k_uns_edges<1><<<ge, 128, 0, L->ctx->stream>>>(a); }
    { ProfScope ps(L->ctx, GC_SLOT_FUSED); k_uns_update<<<gc, 128, 0, L->ctx->stream>>>(a); }
    return GC_OK;
}
