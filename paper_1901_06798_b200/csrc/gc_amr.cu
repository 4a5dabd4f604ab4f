// gc_amr.cu -- level-transfer kernels: coarse-to-fine interpolation in space and time (A3, A11),
// fine-to-coarse averaging (A9), refinement flags with buffer (A10) and the
// flux registers with the conservative fix-up (A8).  Formulas: DESIGN.md 3.6-3.8.
//
// The paper keeps all of these on the CPU; here each is ONE launch over host-built work lists covering
// every patch of the level, so the parallelism is O(perimeter) or O(cells), not O(patch side).
#include <algorithm>
#include "gc_internal.h"
#include "gc_scheme.cuh"

// thread t -> (rectangle k, cell c inside it): start[] holds the exclusive prefix sums of the cell counts
__device__ __forceinline__ int find_rect(const int64_t *start, int n, int64_t t)
{
    int lo = 0, hi = n - 1;
    while (lo < hi) {
        int mid = (lo + hi + 1) >> 1;
        if (start[mid] <= t) lo = mid; else hi = mid - 1;
    }
    return lo;
}

// minmod of two one-sided differences
__device__ __forceinline__ double minmod2(double a, double b)
{
    if (a * b <= 0.0) return 0.0;
    return (fabs(a) < fabs(b)) ? a : b;
}

// ---- A3 / A11: one thread per fine cell
struct CoarseFillArgs {
    const CoarseFillRect *rects; const int64_t *start; int n; int64_t ncells;
    const double *cn0, *cn1, *cn2;     // coarse current buffer
    const double *co0, *co1, *co2;     // coarse previous buffer (use_old)
    const double *cb, *fb;             // coarse / fine bathymetry
    double *f0, *f1, *f2;              // fine state planes
    double alpha, eps;
    int r, use_old;
};

__global__ void __launch_bounds__(128) k_coarse_fill(CoarseFillArgs a)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= a.ncells) return;
    const int k = find_rect(a.start, a.n, t);
    const CoarseFillRect R = a.rects[k];
    const int c = (int)(t - a.start[k]);
    const int y = c / R.w, x = c - y * R.w;
    const int fi = R.ii0 + x, fj = R.jj0 + y;
    const int ci = fi / a.r, cj = fj / a.r;
    const int ii = fi - ci * a.r, jj = fj - cj * a.r;
    const int64_t dst = R.dst + (int64_t)y * R.dpitch + x;
    const int64_t c0 = R.csrc + (int64_t)cj * R.cpitch + ci;
    const int64_t nb[5] = { c0, c0 - 1, c0 + 1, c0 - R.cpitch, c0 + R.cpitch };   // C, W, E, S, N
    double eta[5], u[5], v[5], hh[5];
    bool anydry = false;
#pragma unroll
    for (int m = 0; m < 5; m++) {
        double q0 = a.cn0[nb[m]], q1 = a.cn1[nb[m]], q2 = a.cn2[nb[m]];
        if (a.use_old) {                                   // Q = Q_old + alpha (Q_new - Q_old)
            const double o0 = a.co0[nb[m]], o1 = a.co1[nb[m]], o2 = a.co2[nb[m]];
            q0 = o0 + a.alpha * (q0 - o0); q1 = o1 + a.alpha * (q1 - o1); q2 = o2 + a.alpha * (q2 - o2);
        }
        hh[m] = q0;
        eta[m] = q0 + a.cb[nb[m]];
        if (q0 > a.eps) { const double rh = 1.0 / q0; u[m] = q1 * rh; v[m] = q2 * rh; }
        else { u[m] = 0.0; v[m] = 0.0; anydry = true; }
    }
    double o0 = 0.0, o1 = 0.0, o2 = 0.0;
    if (hh[0] > a.eps) {
        const double xi = ((double)ii + 0.5) / (double)a.r - 0.5;
        const double ze = ((double)jj + 0.5) / (double)a.r - 0.5;
        double sx0 = 0.0, sx1 = 0.0, sx2 = 0.0, sy0 = 0.0, sy1 = 0.0, sy2 = 0.0;
        if (!anydry) {
            sx0 = minmod2(eta[0] - eta[1], eta[2] - eta[0]); sy0 = minmod2(eta[0] - eta[3], eta[4] - eta[0]);
            sx1 = minmod2(u[0] - u[1], u[2] - u[0]);         sy1 = minmod2(u[0] - u[3], u[4] - u[0]);
            sx2 = minmod2(v[0] - v[1], v[2] - v[0]);         sy2 = minmod2(v[0] - v[3], v[4] - v[0]);
        }
        const double ef = (eta[0] + xi * sx0) + ze * sy0;
        const double uf = (u[0] + xi * sx1) + ze * sy1;
        const double vf = (v[0] + xi * sx2) + ze * sy2;
        const double hf = dmax(0.0, ef - a.fb[dst]);
        double huf = hf * uf, hvf = hf * vf;
        if (hf < a.eps) { huf = 0.0; hvf = 0.0; }          // clean-up rule
        o0 = hf; o1 = huf; o2 = hvf;
    }
    a.f0[dst] = o0; a.f1[dst] = o1; a.f2[dst] = o2;
}

void gc_launch_coarse_fill(gc_level *L, const gc_level *C, const CoarseFillRect *rects, const int64_t *start, int n, int64_t ncells,
                           double alpha, int use_old, int slot)
{
    if (ncells <= 0) return;
    CoarseFillArgs a;
    a.rects = rects; a.start = start; a.n = n; a.ncells = ncells;
    a.cn0 = C->q[C->cur][0]; a.cn1 = C->q[C->cur][1]; a.cn2 = C->q[C->cur][2];
    a.co0 = C->q[1 - C->cur][0]; a.co1 = C->q[1 - C->cur][1]; a.co2 = C->q[1 - C->cur][2];
    a.cb = C->b; a.fb = L->b;
    a.f0 = L->q[L->cur][0]; a.f1 = L->q[L->cur][1]; a.f2 = L->q[L->cur][2];
    a.alpha = alpha; a.eps = L->ctx->P.dry_tol; a.r = L->ratio; a.use_old = use_old;
    ProfScope ps(L->ctx, slot);
    k_coarse_fill<<<(unsigned)((ncells + 127) / 128), 128, 0, L->ctx->stream>>>(a);
}

// ---- A11: copy from the old fine level where it overlapped (different pools: separate source planes)
__global__ void k_copy_overlap(const CopyRect *rects, int n, double *d0, double *d1, double *d2,
                               const double *s0, const double *s1, const double *s2)
{
    int warp = (int)((blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5);
    int lane = threadIdx.x & 31;
    if (warp >= n) return;
    CopyRect r = rects[warp];
    int cells = r.w * r.h;
    for (int c = lane; c < cells; c += 32) {
        int y = c / r.w, x = c - y * r.w;
        int64_t d = r.dst + (int64_t)y * r.dpitch + x, s = r.src + (int64_t)y * r.spitch + x;
        d0[d] = s0[s]; d1[d] = s1[s]; d2[d] = s2[s];
    }
}

void gc_launch_copy_overlap(gc_level *N, const gc_level *O, const CopyRect *rects, int n)
{
    if (n <= 0) return;
    ProfScope ps(N->ctx, GC_SLOT_AVG);
    int64_t blocks = ((int64_t)n * 32 + 255) / 256;
    k_copy_overlap<<<(unsigned)blocks, 256, 0, N->ctx->stream>>>(rects, n, N->q[N->cur][0], N->q[N->cur][1], N->q[N->cur][2],
                                                                  O->q[O->cur][0], O->q[O->cur][1], O->q[O->cur][2]);
}

// ---- A9: one thread per covered coarse cell; the r*r fine cells are summed in row-major order
struct AvgArgs {
    const AvgRect *rects; const int64_t *start; int n; int64_t ncells;
    const double *f0, *f1, *f2, *fb, *fkappa;
    double *c0, *c1, *c2; const double *cb;
    double eps; int r;
};

__global__ void __launch_bounds__(128) k_average_down(AvgArgs a)
{
    const int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (t >= a.ncells) return;
    const int k = find_rect(a.start, a.n, t);
    const AvgRect R = a.rects[k];
    const int c = (int)(t - a.start[k]);
    const int y = c / R.w, x = c - y * R.w;
    const int64_t cc = R.cdst + (int64_t)y * R.cpitch + x;
    const int64_t f00 = R.fsrc + (int64_t)(y * a.r) * R.fpitch + x * a.r;
    double sw = 0.0, se = 0.0, sh = 0.0, su = 0.0, sv = 0.0;
    bool allwet = true;
    for (int jj = 0; jj < a.r; jj++) {
        const double w = a.fkappa[R.frow + y * a.r + jj];
        for (int ii = 0; ii < a.r; ii++) {
            const int64_t f = f00 + (int64_t)jj * R.fpitch + ii;
            const double h = a.f0[f];
            if (!(h > a.eps)) allwet = false;
            sw = sw + w;
            se = se + w * (h + a.fb[f]);
            sh = sh + w * h;
            su = su + w * a.f1[f];
            sv = sv + w * a.f2[f];
        }
    }
    double hc = allwet ? dmax(0.0, se / sw - a.cb[cc]) : sh / sw;
    double huc = su / sw, hvc = sv / sw;
    if (hc < a.eps) { hc = dmax(hc, 0.0); huc = 0.0; hvc = 0.0; }
    a.c0[cc] = hc; a.c1[cc] = huc; a.c2[cc] = hvc;
}

void gc_launch_average_down(gc_level *C, const gc_level *F, const AvgRect *rects, const int64_t *start, int n, int64_t ncells)
{
    if (ncells <= 0) return;
    AvgArgs a;
    a.rects = rects; a.start = start; a.n = n; a.ncells = ncells;
    a.f0 = F->q[F->cur][0]; a.f1 = F->q[F->cur][1]; a.f2 = F->q[F->cur][2]; a.fb = F->b; a.fkappa = F->d_kappa;
    a.c0 = C->q[C->cur][0]; a.c1 = C->q[C->cur][1]; a.c2 = C->q[C->cur][2]; a.cb = C->b;
    a.eps = C->ctx->P.dry_tol; a.r = F->ratio;
    ProfScope ps(C->ctx, GC_SLOT_AVG);
    k_average_down<<<(unsigned)((ncells + 127) / 128), 128, 0, C->ctx->stream>>>(a);
}

// ---- A10: flags.  Pass 1 (k_flag_raw): the criteria per interior cell.  Pass 2 (k_flag_dilate): a cell is flagged
// if any raw-flagged cell of the level lies within `buffer` cells (Chebyshev distance): gather over the patch's
// own cells and those of the neighbour patches listed by the host.  One block per patch.
// grid = (patches, chunks of FLAG_CHUNK cells of a patch): a level that is one large patch spreads over the chip, not over one SM
#define FLAG_CHUNK 4096
__global__ void k_flag_raw(const PatchDesc *pat, const double *h, const double *b, double eps, double sea, double tol_eta,
                           double tol_slope, int offshore_only, int nboxes, const double *boxes, double t,
                           double xlo, double ylo, double dx, double dy, uint8_t *raw)
{
    const PatchDesc pd = pat[blockIdx.x];
    const int n = pd.nx * pd.ny;
    const int q1 = min(n, (int)(blockIdx.y + 1) * FLAG_CHUNK);
    for (int q = (int)blockIdx.y * FLAG_CHUNK + threadIdx.x; q < q1; q += blockDim.x) {
        const int j = q / pd.nx, i = q - j * pd.nx;
        const int64_t c = pd.off + (int64_t)(j + 2) * pd.pitch + i + 2;
        const double hc = h[c], bc = b[c];
        int fl = 0;
        const bool wet = hc > eps;
        const bool wave_ok = wet && (!offshore_only || bc < 0.0);
        if (wave_ok && tol_eta > 0.0 && fabs((hc + bc) - sea) > tol_eta) fl = 1;
        if (wave_ok && tol_slope > 0.0) {
            const int64_t lo[2] = { c - 1, c - pd.pitch }, hi[2] = { c + 1, c + pd.pitch };
#pragma unroll
            for (int k = 0; k < 2; k++)
                if (h[lo[k]] > eps && h[hi[k]] > eps) {
                    const double sl = 0.5 * fabs((h[hi[k]] + b[hi[k]]) - (h[lo[k]] + b[lo[k]]));
                    if (sl > tol_slope) fl = 1;
                }
        }
        if (!fl && nboxes > 0) {
            const double xc = xlo + ((double)((int64_t)pd.i0 + i) + 0.5) * dx;
            const double yc = ylo + ((double)((int64_t)pd.j0 + j) + 0.5) * dy;
            for (int k = 0; k < nboxes; k++) {
                const double *B = boxes + 6 * k;
                if (xc >= B[0] && xc <= B[1] && yc >= B[2] && yc <= B[3] && t >= B[4] && t <= B[5]) fl = 1;
            }
        }
        raw[pd.ioff + q] = (uint8_t)fl;
    }
}

__device__ __forceinline__ bool any_raw_in(const PatchDesc &Q, const uint8_t *raw, int64_t gi, int64_t gj, int bw)
{
    const int64_t a0 = max(gi - bw, (int64_t)Q.i0), a1 = min(gi + bw, (int64_t)Q.i0 + Q.nx - 1);
    const int64_t b0 = max(gj - bw, (int64_t)Q.j0), b1 = min(gj + bw, (int64_t)Q.j0 + Q.ny - 1);
    for (int64_t y = b0; y <= b1; y++)
        for (int64_t x = a0; x <= a1; x++)
            if (raw[Q.ioff + (y - Q.j0) * Q.nx + (x - Q.i0)]) return true;
    return false;
}

__global__ void k_flag_dilate(const PatchDesc *pat, const uint8_t *raw, uint8_t *flags, int bw,
                              const int32_t *nbr_start, const int32_t *nbr_list, unsigned long long *count)
{
    __shared__ unsigned sc;
    if (threadIdx.x == 0) sc = 0u;
    __syncthreads();
    const int p = blockIdx.x;
    const PatchDesc pd = pat[p];
    const int n = pd.nx * pd.ny;
    const int q1 = min(n, (int)(blockIdx.y + 1) * FLAG_CHUNK);
    unsigned mine = 0;
    for (int q = (int)blockIdx.y * FLAG_CHUNK + threadIdx.x; q < q1; q += blockDim.x) {
        const int j = q / pd.nx, i = q - j * pd.nx;
        const int64_t gi = (int64_t)pd.i0 + i, gj = (int64_t)pd.j0 + j;
        bool fl = raw[pd.ioff + q] != 0;
        if (!fl && bw > 0) {
            fl = any_raw_in(pd, raw, gi, gj, bw);
            // only cells within bw of the patch border can be reached from another patch
            if (!fl && (i < bw || j < bw || i >= pd.nx - bw || j >= pd.ny - bw))
                for (int k = nbr_start[p]; k < nbr_start[p + 1] && !fl; k++) fl = any_raw_in(pat[nbr_list[k]], raw, gi, gj, bw);
        }
        flags[pd.ioff + q] = fl ? 1 : 0;
        mine += fl ? 1u : 0u;
    }
    mine = __reduce_add_sync(0xffffffffu, mine);
    if ((threadIdx.x & 31) == 0 && mine) atomicAdd(&sc, mine);
    __syncthreads();
    if (threadIdx.x == 0 && sc) atomicAdd(count, (unsigned long long)sc);
}

void gc_launch_flags(const gc_level *L, const gc_flag_params *fp, const double *d_boxes, double t, uint8_t *raw, uint8_t *flags,
                     const int32_t *nbr_start, const int32_t *nbr_list, unsigned long long *d_count)
{
    if (L->np == 0) return;
    const gc_params &P = L->ctx->P;
    ProfScope ps(L->ctx, GC_SLOT_FLAG, 2);
    int64_t maxn = 1;
    for (const gc_patch &pp : L->pat) maxn = std::max<int64_t>(maxn, (int64_t)pp.nx * pp.ny);
    const dim3 grid((unsigned)L->np, (unsigned)((maxn + FLAG_CHUNK - 1) / FLAG_CHUNK));
    k_flag_raw<<<grid, 256, 0, L->ctx->stream>>>(L->d_pat, L->q[L->cur][0], L->b, P.dry_tol, P.sea_level, fp->tol_eta, fp->tol_slope,
                                                  fp->offshore_only, fp->nboxes, d_boxes, t, L->xlo, L->ylo, L->dx, L->dy, raw);
    k_flag_dilate<<<grid, 256, 0, L->ctx->stream>>>(L->d_pat, raw, flags, fp->buffer > 0 ? fp->buffer : 0, nbr_start, nbr_list, d_count);
}

// ---- A8: flux registers.  The sweeps keep nothing per edge; a register re-derives the flux-like
// quantity of its edge from the state the sweep saw (Q^n for x-edges, Q* for y-edges; both are still in the pool
// after the step): three Riemann problems (edges e-1, e, e+1 for the limiter) and gc_edge_flux -- the same
// device functions in the same order as the sweep kernels, hence the same bits.
struct LineAcc {            // one grid line of a patch: planes in (h, normal, transverse, b) order, element stride along the line
    const double *h, *p, *t, *b;
    int64_t str;
};

__device__ __forceinline__ RState load_cell(const LineAcc &A, int64_t o)
{
    RState S; S.h = A.h[o]; S.p = A.p[o]; S.t = A.t[o]; S.b = A.b[o];
    S.u = 0.0; S.v = 0.0; S.phi = 0.0; S.c = 0.0;
    return S;
}

// fm, fp of the edge on the low side of cell `o` (offset of that cell); ef[0..2] = edge factors of edges e-1, e, e+1;
// rdL, rdR = 1/(kappa dx) of cells e-1, e
__device__ __forceinline__ void edge_fmfp(const LineAcc &A, int64_t o, double g, double eps, int coord, int limiter, double dt,
                                          const double (&ef)[3], double rdL, double rdR, double (&fm)[3], double (&fp)[3])
{
    MathIeee mi;
    RState c0 = load_cell(A, o - 2 * A.str), c1 = load_cell(A, o - A.str), c2 = load_cell(A, o), c3 = load_cell(A, o + A.str);
    gc_prim(mi, c0, g, eps); gc_prim(mi, c1, g, eps); gc_prim(mi, c2, g, eps); gc_prim(mi, c3, g, eps);
    Waves Wl, We, Wh;
    gc_solve_edge_prim(mi, g, eps, c0, c1, coord, ef[0], Wl);
    gc_solve_edge_prim(mi, g, eps, c1, c2, coord, ef[1], We);
    gc_solve_edge_prim(mi, g, eps, c2, c3, coord, ef[2], Wh);
    double dlo[3], dhi[3];
    gc_wave_dots(We, Wl, dlo);
    gc_wave_dots(Wh, We, dhi);
    gc_edge_flux(mi, We, dlo, dhi, limiter, dt, rdL, rdR, fm, fp);
}

struct FluxArgs {
    const FluxReg *reg; int nreg;
    double *delta, *base;
    const PatchDesc *pat;
    const double *qn0, *qn1, *qn2;     // Q^n of the stepping level (previous buffer after the swap)
    const double *qs0, *qs1, *qs2;     // Q*
    const double *b;
    const double *rdx, *rdy, *ey;
    double ex, dx, dy, g, eps;
    double dt; const double *dt_dev;
    int coord, limiter, r;
};

// the coarse level has just stepped: delta += dt l F, F = fm (fine region on the high side) or fp; remember the state of C
__global__ void __launch_bounds__(64) k_flux_coarse(FluxArgs a)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    if (n >= a.nreg) return;
    const FluxReg R = a.reg[n];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;
    const int64_t c = R.ccell;
    double fm[3], fp[3], len;
    LineAcc A;
    if (R.dir == 0) {
        A.h = a.qn0; A.p = a.qn1; A.t = a.qn2; A.b = a.b; A.str = 1;
        const double ef[3] = { a.ex, a.ex, a.ex };
        const double rd = a.rdx[R.crow];
        edge_fmfp(A, R.side > 0 ? c + 1 : c, a.g, a.eps, a.coord, a.limiter, dt, ef, rd, rd, fm, fp);
        len = a.dy;
        a.base[4 * n + 0] = a.qn0[c]; a.base[4 * n + 1] = a.qn1[c]; a.base[4 * n + 2] = a.qn2[c];
    } else {
        A.h = a.qs0; A.p = a.qs2; A.t = a.qs1; A.b = a.b; A.str = R.cpitch;
        const int er = R.side > 0 ? R.crow + 1 : R.crow;       // table index of the row above the edge
        const double ef[3] = { a.ey[er - 1], a.ey[er], a.ey[er + 1] };
        edge_fmfp(A, R.side > 0 ? c + R.cpitch : c, a.g, a.eps, a.coord, a.limiter, dt, ef, a.rdy[er - 1], a.rdy[er], fm, fp);
        len = a.dx;
        a.base[4 * n + 0] = a.qs0[c]; a.base[4 * n + 1] = a.qs2[c]; a.base[4 * n + 2] = a.qs1[c];
    }
    a.base[4 * n + 3] = a.b[c];
#pragma unroll
    for (int k = 0; k < 3; k++) {
        const double F = R.side > 0 ? fm[k] : fp[k];
        a.delta[3 * n + k] = a.delta[3 * n + k] + dt * len * F;
    }
}

__device__ __forceinline__ double p_used(double h, double p, double eps) { return (h <= eps) ? 0.0 : p; }

// the fine level has just stepped: delta -= dt l (F_k + e J_k) for the r fine cells along the coarse edge, in order.
// Thread <-> (register, fine cell k): the r terms of a register -- four Riemann problems each -- are computed side by side,
// then the register's first thread subtracts them in order.  Block = FLUX_FINE_BLOCK threads = floor(block / r) registers.
#define FLUX_FINE_BLOCK 128
__global__ void __launch_bounds__(FLUX_FINE_BLOCK) k_flux_fine(FluxArgs a)
{
    __shared__ double term[3][FLUX_FINE_BLOCK];
    const int per = FLUX_FINE_BLOCK / a.r;
    const int li = threadIdx.x / a.r, m = threadIdx.x - li * a.r;
    const int n = blockIdx.x * per + li;
    const bool act = li < per && n < a.nreg;
    if (act) {
        const FluxReg R = a.reg[n];
        const double dt = a.dt_dev ? *a.dt_dev : a.dt;
        RState B; B.h = a.base[4 * n + 0]; B.p = a.base[4 * n + 1]; B.t = a.base[4 * n + 2]; B.b = a.base[4 * n + 3];
        B.u = 0.0; B.v = 0.0; B.phi = 0.0; B.c = 0.0;
        const double sg = (R.side > 0) ? 1.0 : -1.0;
        LineAcc A;
        if (R.dir == 0) { A.h = a.qn0; A.p = a.qn1; A.t = a.qn2; A.b = a.b; A.str = 1; }
        else            { A.h = a.qs0; A.p = a.qs2; A.t = a.qs1; A.b = a.b; A.str = R.fpitch; }
        const int64_t c = R.fcell + (R.dir == 0 ? (int64_t)m * R.fpitch : (int64_t)m);
        double fm[3], fp[3], len, efJ;
        if (R.dir == 0) {
            const double ef[3] = { a.ex, a.ex, a.ex };
            const double rd = a.rdx[R.frow + m];
            edge_fmfp(A, R.side > 0 ? c : c + 1, a.g, a.eps, a.coord, a.limiter, dt, ef, rd, rd, fm, fp);
            len = a.dy; efJ = (a.coord == 1) ? a.ex : 1.0;
        } else {
            const int er = R.side > 0 ? R.frow : R.frow + 1;   // table index of the row above the shared edge
            const double ef[3] = { a.ey[er - 1], a.ey[er], a.ey[er + 1] };
            edge_fmfp(A, R.side > 0 ? c : c + R.fpitch, a.g, a.eps, a.coord, a.limiter, dt, ef, a.rdy[er - 1], a.rdy[er], fm, fp);
            len = a.dx; efJ = (a.coord == 1) ? a.ey[er] : 1.0;
        }
        const RState S = load_cell(A, c);
        MathIeee mi;
        double Z[3][3], s[3];
        {
            RState L = (R.side > 0) ? B : S, Rr = (R.side > 0) ? S : B;     // geometric order
            gc_prim(mi, L, a.g, a.eps); gc_prim(mi, Rr, a.g, a.eps);
            gc_riemann(mi, a.g, a.eps, L, Rr, Z, s);
        }
        const double J0 = p_used(S.h, S.p, a.eps) - p_used(B.h, B.p, a.eps);
        const double J1 = sg * ((Z[0][1] + Z[1][1]) + Z[2][1]);
        const double J2 = sg * ((Z[0][2] + Z[1][2]) + Z[2][2]);
        const double F0 = R.side > 0 ? fp[0] : fm[0], F1 = R.side > 0 ? fp[1] : fm[1], F2 = R.side > 0 ? fp[2] : fm[2];
        term[0][threadIdx.x] = dt * len * (F0 + efJ * J0);
        term[1][threadIdx.x] = dt * len * (F1 + efJ * J1);
        term[2][threadIdx.x] = dt * len * (F2 + efJ * J2);
    }
    __syncthreads();
    if (act && m == 0) {
        double d0 = a.delta[3 * n + 0], d1 = a.delta[3 * n + 1], d2 = a.delta[3 * n + 2];
        for (int k = 0; k < a.r; k++) {
            d0 = d0 - term[0][threadIdx.x + k]; d1 = d1 - term[1][threadIdx.x + k]; d2 = d2 - term[2][threadIdx.x + k];
        }
        a.delta[3 * n + 0] = d0; a.delta[3 * n + 1] = d1; a.delta[3 * n + 2] = d2;
    }
}

static void fill_flux_args(FluxArgs &a, const gc_level *S, const gc_level *Creg, double dt, const double *dt_dev)
{
    const gc_params &P = S->ctx->P;
    a.reg = Creg->d_reg; a.nreg = Creg->nreg; a.delta = Creg->d_delta; a.base = Creg->d_base;
    a.pat = S->d_pat;
    const int old = 1 - S->cur;
    a.qn0 = S->q[old][0]; a.qn1 = S->q[old][1]; a.qn2 = S->q[old][2];
    a.qs0 = S->qs[0]; a.qs1 = S->qs[1]; a.qs2 = S->qs[2];
    a.b = S->b; a.rdx = S->d_rdx; a.rdy = S->d_rdy; a.ey = S->d_ey;
    a.ex = S->ex; a.dx = S->dx; a.dy = S->dy; a.g = P.g; a.eps = P.dry_tol;
    a.dt = dt; a.dt_dev = dt_dev; a.coord = P.coord; a.limiter = P.limiter; a.r = Creg->r_reg;
}

void gc_launch_flux_coarse(gc_level *C, double dt, const double *dt_dev)
{
    if (C->nreg == 0) return;
    FluxArgs a; fill_flux_args(a, C, C, dt, dt_dev);
    ProfScope ps(C->ctx, GC_SLOT_FLUX);
    k_flux_coarse<<<(C->nreg + 63) / 64, 64, 0, C->ctx->stream>>>(a);
}

void gc_launch_flux_fine(gc_level *F, double dt, const double *dt_dev)
{
    gc_level *C = F->reg_coarse;
    if (!C || C->nreg == 0) return;
    FluxArgs a; fill_flux_args(a, F, C, dt, dt_dev);
    ProfScope ps(F->ctx, GC_SLOT_FLUX);
    const int per = FLUX_FINE_BLOCK / a.r;                      // registers per block (a.r <= FLUX_FINE_BLOCK: checked at attach)
    k_flux_fine<<<(C->nreg + per - 1) / per, FLUX_FINE_BLOCK, 0, F->ctx->stream>>>(a);
}

// fix-up: one thread per corrected coarse cell, its registers applied in list order, then the clean-up rule
__global__ void k_flux_fixup(const FluxReg *reg, const int32_t *fixstart, const int32_t *fixreg, int nfix, double *delta,
                             double *q0, double *q1, double *q2, const double *kappa, double dx, double dy, double eps)
{
    const int gidx = blockIdx.x * blockDim.x + threadIdx.x;
    if (gidx >= nfix) return;
    const int k0 = fixstart[gidx], k1 = fixstart[gidx + 1];
    const int64_t c = reg[fixreg[k0]].ccell;
    double h = q0[c], hu = q1[c], hv = q2[c];
    for (int k = k0; k < k1; k++) {
        const int n = fixreg[k];
        const FluxReg R = reg[n];
        const double area = kappa[R.crow] * dx * dy;
        const double sg = (double)R.side;
        const double a0 = sg * delta[3 * n + 0] / area, a1 = sg * delta[3 * n + 1] / area, a2 = sg * delta[3 * n + 2] / area;
        h = h + a0;
        if (R.dir == 0) { hu = hu + a1; hv = hv + a2; } else { hv = hv + a1; hu = hu + a2; }
        delta[3 * n + 0] = 0.0; delta[3 * n + 1] = 0.0; delta[3 * n + 2] = 0.0;
    }
    if (h < eps) { h = dmax(h, 0.0); hu = 0.0; hv = 0.0; }
    q0[c] = h; q1[c] = hu; q2[c] = hv;
}

void gc_launch_flux_fixup(gc_level *C)
{
    if (C->nfix == 0) return;
    ProfScope ps(C->ctx, GC_SLOT_FLUX);
    k_flux_fixup<<<(C->nfix + 127) / 128, 128, 0, C->ctx->stream>>>(C->d_reg, C->d_fixstart, C->d_fixreg, C->nfix, C->d_delta,
                                                                   C->q[C->cur][0], C->q[C->cur][1], C->q[C->cur][2],
                                                                   C->d_kappa, C->dx, C->dy, C->ctx->P.dry_tol);
}


// ---- gauges (reading S-19): thread per bound gauge.  Offsets and weights were fixed on the host at bind
// time; the sample is the bilinear form in the cell centres, in DESIGN.md's order, or the containing cell if the stencil is not all wet.
__global__ void k_gauges_sample(const GaugeLoc *g, int n, const double *h, const double *hu, const double *hv, const double *b,
                                double eps, double *out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const GaugeLoc G = g[k];
    double v[4][4];
    bool dry = false;
#pragma unroll
    for (int m = 0; m < 4; m++) {
        const int64_t c = G.c00 + (m & 1) + (int64_t)(m >> 1) * G.pitch;
        const double hh = h[c];
        v[0][m] = hh; v[1][m] = hu[c]; v[2][m] = hv[c]; v[3][m] = hh + b[c];
        dry = dry || !(hh > eps);
    }
    if (dry) {
        const double hh = h[G.cc];
        out[4 * k] = hh; out[4 * k + 1] = hu[G.cc]; out[4 * k + 2] = hv[G.cc]; out[4 * k + 3] = hh + b[G.cc];
    } else {
        const double a = G.a, bw = G.b;
#pragma unroll
        for (int f = 0; f < 4; f++)
            out[4 * k + f] = (1.0 - bw) * ((1.0 - a) * v[f][0] + a * v[f][1]) + bw * ((1.0 - a) * v[f][2] + a * v[f][3]);
    }
}

void gc_launch_gauges(const gc_level *L, double *out)
{
    if (L->ngauge <= 0) return;
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    k_gauges_sample<<<(L->ngauge + 127) / 128, 128, 0, L->ctx->stream>>>(L->d_gauge, L->ngauge, L->q[L->cur][0], L->q[L->cur][1],
                                                                         L->q[L->cur][2], L->b, L->ctx->P.dry_tol, out);
}
