// gc_ghost.cu -- ghost-cell fill kernels: same-level copy (A2) and physical boundary (A4), plus the
// field transfer, wet-mask and mass kernels.  P:143 (step 2 of the AMR algorithm); DESIGN.md 3.6.
// The paper keeps ghost filling on the CPU because a per-patch kernel has only O(a) parallelism;
// here ONE launch covers every patch of the level through host-built work lists, so the parallelism is
// O(total perimeter).
#include <algorithm>
#include "gc_internal.h"

// ---- A2: same-level copy.  The host lists, per patch, the rectangles its ghost cells take from the interiors of its
// neighbours (two x faces of width 2, two y faces of height 2, four 2 x 2 corners on a regular tiling).  A patch is served by
// `wpp` warps (one for small patches, several when the perimeter is long) that walk its rectangles together: a wide rectangle
// row by row with the lanes along x (coalesced), a narrow one several rows per pass (lane -> (row, column): one division per
// rectangle, none per cell).  Two rows are in flight per lane and plane before anything is stored.  Pure data movement:
// every ghost cell written once, 48 bytes of algorithmic traffic per cell (3 planes read + written).
// (the cells read are interior cells, the cells written ghost cells: the two sets are disjoint, so the loads may take the
// read-only path and move ahead of the stores)
template <int NF>
__device__ __forceinline__ void copy_pair(double *f0, double *f1, double *f2, int64_t d0, int64_t s0, int64_t d1, int64_t s1, bool two)
{
    double a0 = __ldg(f0 + s0), a1 = 0.0, a2 = 0.0, b0 = 0.0, b1 = 0.0, b2 = 0.0;
    if (NF > 1) { a1 = __ldg(f1 + s0); a2 = __ldg(f2 + s0); }
    if (two) { b0 = __ldg(f0 + s1); if (NF > 1) { b1 = __ldg(f1 + s1); b2 = __ldg(f2 + s1); } }
    f0[d0] = a0; if (NF > 1) { f1[d0] = a1; f2[d0] = a2; }
    if (two) { f0[d1] = b0; if (NF > 1) { f1[d1] = b1; f2[d1] = b2; } }
}

__device__ __forceinline__ CopyRect rect_from_lane(const CopyRect &mine, int i)
{
    CopyRect r;
    r.dst = __shfl_sync(0xffffffffu, mine.dst, i); r.src = __shfl_sync(0xffffffffu, mine.src, i);
    r.w = __shfl_sync(0xffffffffu, mine.w, i); r.h = __shfl_sync(0xffffffffu, mine.h, i);
    r.dpitch = __shfl_sync(0xffffffffu, mine.dpitch, i); r.spitch = __shfl_sync(0xffffffffu, mine.spitch, i);
    return r;
}
// lane -> (row, column) inside one pass over a rectangle narrower than 32 cells; rpp = rows per pass (0: a wide rectangle)
__device__ __forceinline__ void narrow_map(int w, int lane, int &rpp, int &ly, int &lx)
{
    if (w == 2) { rpp = 16; ly = lane >> 1; lx = lane & 1; }                     // x faces, corners: no division
    else if (w == 16) { rpp = 2; ly = lane >> 4; lx = lane & 15; }
    else if (w < 32) { rpp = 32 / w; ly = lane / w; lx = lane - ly * w; }
    else { rpp = 0; ly = 0; lx = 0; }
}

template <int NF>
__global__ void __launch_bounds__(256, 2) k_copy_rects(const CopyRect *rects, const int2 *range, int np, int wpp, double *f0, double *f1, double *f2)
{
    const int gw = (int)((blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5);
    const int lane = threadIdx.x & 31;
    const int patch = gw / wpp, sub = gw - patch * wpp;
    if (patch >= np) return;
    const int2 pr = range[patch];
    for (int i0 = 0; i0 < pr.y; i0 += 32) {
        // the patch's rectangle descriptors arrive with one load (lane k takes rectangle i0 + k) and are handed round by shuffles:
        // one memory round trip instead of one per rectangle
        CopyRect mine; mine.dst = 0; mine.src = 0; mine.w = 0; mine.h = 0; mine.dpitch = 0; mine.spitch = 0;
        if (i0 + lane < pr.y) mine = rects[pr.x + i0 + lane];
        const int cnt = min(32, pr.y - i0);
        for (int i = 0; i < cnt; i += 4) {
            // Narrow rectangles (faces and corners of small patches) four at a time: the first two passes of each -- all of it
            // for a patch of side <= 32 -- are loaded before anything is stored, 24 loads in flight per lane.  One rectangle
            // after the other left a warp waiting one DRAM round trip per rectangle (side 16: 8 of them per patch).
            int64_t da[4], sa[4], db[4], sb[4];
            bool va[4], vb[4];
            bool more = false;                                                     // some rectangle of the four is wide, or taller than two passes of the patch's warps
#pragma unroll
            for (int k = 0; k < 4; k++) {
                const CopyRect r = rect_from_lane(mine, min(i + k, cnt - 1));      // past the end: the last one again, masked out
                int rpp, ly, lx;
                narrow_map(r.w, lane, rpp, ly, lx);
                more |= (rpp == 0) | (r.h > 2 * wpp * rpp);                        // the same for every lane: it depends on the rectangle only
                const int y = 2 * sub * rpp + ly;
                va[k] = (i + k < cnt) & (ly < rpp) & (y < r.h);
                vb[k] = va[k] & (y + rpp < r.h);
                da[k] = r.dst + (int64_t)y * r.dpitch + lx; sa[k] = r.src + (int64_t)y * r.spitch + lx;
                db[k] = da[k] + (int64_t)rpp * r.dpitch; sb[k] = sa[k] + (int64_t)rpp * r.spitch;
            }
            double a[4][3], b[4][3];
#pragma unroll
            for (int k = 0; k < 4; k++) {
                a[k][0] = va[k] ? __ldg(f0 + sa[k]) : 0.0; b[k][0] = vb[k] ? __ldg(f0 + sb[k]) : 0.0;
                if (NF > 1) {
                    a[k][1] = va[k] ? __ldg(f1 + sa[k]) : 0.0; a[k][2] = va[k] ? __ldg(f2 + sa[k]) : 0.0;
                    b[k][1] = vb[k] ? __ldg(f1 + sb[k]) : 0.0; b[k][2] = vb[k] ? __ldg(f2 + sb[k]) : 0.0;
                }
            }
#pragma unroll
            for (int k = 0; k < 4; k++) {
                if (va[k]) { f0[da[k]] = a[k][0]; if (NF > 1) { f1[da[k]] = a[k][1]; f2[da[k]] = a[k][2]; } }
                if (vb[k]) { f0[db[k]] = b[k][0]; if (NF > 1) { f1[db[k]] = b[k][1]; f2[db[k]] = b[k][2]; } }
            }
            // what is left: the later passes of a tall narrow rectangle, and the wide rectangles
            if (!more) continue;
            for (int k = 0; k < 4 && i + k < cnt; k++) {
                const CopyRect r = rect_from_lane(mine, i + k);
                if (r.w >= 32) {                                           // (row pair, 32-column chunk) items dealt round the patch's warps
                    const int nxc = (r.w + 31) >> 5;
                    int y = 0, xc = sub;                                   // item sub, sub + wpp, ...: no division
                    while (xc >= nxc) { xc -= nxc; y += 2; }
                    while (y < r.h) {
                        const int x = xc * 32 + lane;
                        if (x < r.w)
                            copy_pair<NF>(f0, f1, f2, r.dst + (int64_t)y * r.dpitch + x, r.src + (int64_t)y * r.spitch + x,
                                          r.dst + (int64_t)(y + 1) * r.dpitch + x, r.src + (int64_t)(y + 1) * r.spitch + x, y + 1 < r.h);
                        xc += wpp;
                        while (xc >= nxc) { xc -= nxc; y += 2; }
                    }
                } else {
                    int rpp, ly, lx;
                    narrow_map(r.w, lane, rpp, ly, lx);
                    if (ly < rpp) {
                        for (int y = 2 * (sub + wpp) * rpp + ly; y < r.h; y += 2 * wpp * rpp) {
                            const bool two = y + rpp < r.h;
                            copy_pair<NF>(f0, f1, f2, r.dst + (int64_t)y * r.dpitch + lx, r.src + (int64_t)y * r.spitch + lx,
                                          r.dst + (int64_t)(y + rpp) * r.dpitch + lx, r.src + (int64_t)(y + rpp) * r.spitch + lx, two);
                        }
                    }
                }
            }
        }
    }
}

void gc_launch_copy_rects(gc_level *L, double *f0, double *f1, double *f2, int nf, bool for_step)
{
    const bool red = for_step && L->ncopy_red >= 0;
    if ((red ? L->ncopy_red : L->ncopy) == 0) return;
    const CopyRect *rects = red ? L->d_copy_red : L->d_copy;
    const int2 *range = red ? L->d_copy_range_red : L->d_copy_range;
    const int threads = 256, wpp = L->copy_wpp;
    const int64_t blocks = ((int64_t)L->np * wpp * 32 + threads - 1) / threads;
    ProfScope ps(L->ctx, GC_SLOT_COPY);
    if (nf > 1) k_copy_rects<3><<<(unsigned)blocks, threads, 0, L->ctx->stream>>>(rects, range, L->np, wpp, f0, f1, f2);
    else k_copy_rects<1><<<(unsigned)blocks, threads, 0, L->ctx->stream>>>(rects, range, L->np, wpp, f0, f1, f2);
}

// ---- A4: physical boundary.  pass 0: x faces over rows inside the domain; pass 1: y faces over all columns; pass 2: both, one
// block per patch doing the one after the other.
// Wall: mirror cell, normal momentum negated (is_state: f1 = hu, f2 = hv); extrapolation: nearest interior cell.
__global__ void k_bc(const PatchDesc *pat, const int32_t *list, double *f0, double *f1, double *f2, int nf, int is_state,
                     int pass, int64_t nxl, int64_t nyl, int bc0, int bc1, int bc2, int bc3)
{
    PatchDesc pd = pat[list[blockIdx.x]];
    int rows = pd.ny + 4;
    if (pass != 1) {
        // up to 4 ghost columns (2 per side) x rows
        for (int t = threadIdx.x; t < rows * 4; t += blockDim.x) {
            int j = t >> 2, c = t & 3;
            int i = (c < 2) ? c : pd.nx + c;            // storage columns 0,1, nx+2, nx+3
            int64_t gi = (int64_t)pd.i0 + i - 2, gj = (int64_t)pd.j0 + j - 2;
            if (gj < 0 || gj >= nyl) continue;
            int wall; int64_t gs;
            if (gi < 0) { wall = bc0; gs = wall ? -1 - gi : 0; }
            else if (gi >= nxl) { wall = bc1; gs = wall ? 2 * nxl - 1 - gi : nxl - 1; }
            else continue;
            int is = (int)(gs - pd.i0 + 2);
            int64_t d = pd.off + (int64_t)j * pd.pitch + i, s = pd.off + (int64_t)j * pd.pitch + is;
            f0[d] = f0[s];
            if (nf > 1) {
                double a = f1[s];
                f1[d] = (wall && is_state) ? -1.0 * a : a;
                f2[d] = f2[s];
            }
        }
    }
    if (pass == 2) __syncthreads();      // both passes in one launch: the y faces read this patch's own x faces, written by this block
    if (pass != 0) {
        const int W = pd.nx + 4;
        for (int t = threadIdx.x; t < W * 4; t += blockDim.x) {
            int c = t / W, i = t - c * W;
            int j = (c < 2) ? c : pd.ny + c;
            int64_t gj = (int64_t)pd.j0 + j - 2;
            int wall; int64_t gs;
            if (gj < 0) { wall = bc2; gs = wall ? -1 - gj : 0; }
            else if (gj >= nyl) { wall = bc3; gs = wall ? 2 * nyl - 1 - gj : nyl - 1; }
            else continue;
            int js = (int)(gs - pd.j0 + 2);
            int64_t d = pd.off + (int64_t)j * pd.pitch + i, s = pd.off + (int64_t)js * pd.pitch + i;
            f0[d] = f0[s];
            if (nf > 1) {
                f1[d] = f1[s];
                double a = f2[s];
                f2[d] = (wall && is_state) ? -1.0 * a : a;
            }
        }
    }
}

void gc_launch_bc(gc_level *L, double *f0, double *f1, double *f2, int nf, int is_state)
{
    if (L->nbcp == 0) return;
    const int *bc = L->ctx->P.bc;
    ProfScope ps(L->ctx, GC_SLOT_BC, 1);
    k_bc<<<L->nbcp, 128, 0, L->ctx->stream>>>(L->d_pat, L->d_bcp, f0, f1, f2, nf, is_state, 2, L->nxl, L->nyl, bc[0], bc[1], bc[2], bc[3]);
}

// ---- field transfer.  Grids are patches x chunks of GC_CHUNK cells, so that a level that is one large patch spreads over the
// chip (a block per patch ran config 4's 1800 x 900 coarse level on one SM)
#define GC_CHUNK 8192
static dim3 gc_chunk_grid(const gc_level *L, int grow)
{
    int64_t mx = 1;
    for (const gc_patch &P : L->pat) mx = std::max<int64_t>(mx, (int64_t)(P.nx + grow) * (P.ny + grow));
    return dim3((unsigned)L->np, (unsigned)((mx + GC_CHUNK - 1) / GC_CHUNK));
}
__global__ void k_set_global(const PatchDesc *pat, double *plane, const double *src, int64_t ld,
                             int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    PatchDesc pd = pat[blockIdx.x];
    const int W = pd.nx + 4;
    int n = W * (pd.ny + 4);
    const int t1 = min(n, (int)(blockIdx.y + 1) * GC_CHUNK);
    for (int t = blockIdx.y * GC_CHUNK + threadIdx.x; t < t1; t += blockDim.x) {
        int j = t / W, i = t - j * W;
        int64_t gi = (int64_t)pd.i0 + i - 2 - gi0, gj = (int64_t)pd.j0 + j - 2 - gj0;
        if (gi < 0 || gi >= gnx || gj < 0 || gj >= gny) continue;
        plane[pd.off + (int64_t)j * pd.pitch + i] = src[gj * ld + gi];
    }
}

// every patch at once from a packed source: patch p's (ny + 4) x (nx + 4) block, ghost cells included, starts at goff[p];
// cells outside the level are left alone (the boundary fill owns them), as k_set_global leaves them
__global__ void k_set_patches(const PatchDesc *pat, const int64_t *goff, double *plane, const double *src, int64_t nxl, int64_t nyl)
{
    const PatchDesc pd = pat[blockIdx.x];
    const double *sp = src + goff[blockIdx.x];
    const int W = pd.nx + 4;
    const int n = W * (pd.ny + 4);
    const int t1 = min(n, (int)(blockIdx.y + 1) * GC_CHUNK);
    for (int t = blockIdx.y * GC_CHUNK + threadIdx.x; t < t1; t += blockDim.x) {
        const int j = t / W, i = t - j * W;
        const int64_t gi = (int64_t)pd.i0 + i - 2, gj = (int64_t)pd.j0 + j - 2;
        if (gi < 0 || gi >= nxl || gj < 0 || gj >= nyl) continue;
        plane[pd.off + (int64_t)j * pd.pitch + i] = sp[t];
    }
}
void gc_launch_set_patches(gc_level *L, double *plane, const int64_t *goff, const double *src)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_set_patches<<<gc_chunk_grid(L, 4), 256, 0, L->ctx->stream>>>(L->d_pat, goff, plane, src, L->nxl, L->nyl);
}

__global__ void k_get_global(const PatchDesc *pat, const double *plane, double *dst, int64_t ld,
                             int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    PatchDesc pd = pat[blockIdx.x];
    int n = pd.nx * pd.ny;
    const int t1 = min(n, (int)(blockIdx.y + 1) * GC_CHUNK);
    for (int t = blockIdx.y * GC_CHUNK + threadIdx.x; t < t1; t += blockDim.x) {
        int j = t / pd.nx, i = t - j * pd.nx;
        int64_t gi = (int64_t)pd.i0 + i - gi0, gj = (int64_t)pd.j0 + j - gj0;
        if (gi < 0 || gi >= gnx || gj < 0 || gj >= gny) continue;
        dst[gj * ld + gi] = plane[pd.off + (int64_t)(j + 2) * pd.pitch + i + 2];
    }
}

void gc_launch_set_global(gc_level *L, double *plane, const double *src, int64_t ld, int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_set_global<<<gc_chunk_grid(L, 4), 256, 0, L->ctx->stream>>>(L->d_pat, plane, src, ld, gi0, gj0, gnx, gny);
}
void gc_launch_get_global(const gc_level *L, const double *plane, double *dst, int64_t ld, int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_get_global<<<gc_chunk_grid(L, 0), 256, 0, L->ctx->stream>>>(L->d_pat, plane, dst, ld, gi0, gj0, gnx, gny);
}

__global__ void k_copy2d(double *dst, int64_t dld, const double *src, int64_t sld, int w, int h)
{
    int64_t n = (int64_t)w * h;
    for (int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; t < n; t += (int64_t)gridDim.x * blockDim.x) {
        int64_t j = t / w, i = t - j * w;
        dst[j * dld + i] = src[j * sld + i];
    }
}
void gc_launch_copy2d(cudaStream_t s, double *dst, int64_t dld, const double *src, int64_t sld, int w, int h)
{
    int64_t n = (int64_t)w * h;
    int blocks = (int)((n + 255) / 256 < 4096 ? (n + 255) / 256 : 4096);
    if (n > 0) k_copy2d<<<blocks, 256, 0, s>>>(dst, dld, src, sld, w, h);
}

// ---- time-dependent bathymetry (P:52 B(x, y, t); P:273, P:333 deformation on uniform grids, reading S-20):
// b <- fma(w, dz(cell centre), b) on every storage cell whose centre lies inside the domain; dz bilinear between the nodes of
// the deformation grid, 0 outside it.  Same expressions in the same order as the specification (IEEE divide, no contraction
// but the one fma).  Grid = patches x chunks.
struct DeformArgs { double x0, y0, ddx, ddy; long long mx, my; const double *dz; };
__device__ __forceinline__ double gc_deform_at(const DeformArgs &D, double x, double y)
{
    const double s = (x - D.x0) / D.ddx, t = (y - D.y0) / D.ddy;
    if (!(s >= 0.0) || !(t >= 0.0) || !(s <= (double)(D.mx - 1)) || !(t <= (double)(D.my - 1))) return 0.0;
    long long m = (long long)floor(s), n = (long long)floor(t);
    if (m > D.mx - 2) m = D.mx - 2;
    if (n > D.my - 2) n = D.my - 2;
    const double a = s - (double)m, c = t - (double)n;
    const double *z = D.dz + n * D.mx + m;
    const double lo = (1.0 - a) * z[0] + a * z[1];
    const double hi = (1.0 - a) * z[D.mx] + a * z[D.mx + 1];
    return (1.0 - c) * lo + c * hi;
}
__global__ void k_bathy_update(const PatchDesc *pat, double *b, DeformArgs D, double w, double xlo, double ylo, double dx, double dy,
                               int64_t nxl, int64_t nyl)
{
    const PatchDesc pd = pat[blockIdx.x];
    const int W = pd.nx + 4;
    const int n = W * (pd.ny + 4);
    const int t1 = min(n, (int)(blockIdx.y + 1) * GC_CHUNK);
    for (int t = blockIdx.y * GC_CHUNK + threadIdx.x; t < t1; t += blockDim.x) {
        const int j = t / W, i = t - j * W;
        const int64_t gi = (int64_t)pd.i0 + i - 2, gj = (int64_t)pd.j0 + j - 2;
        if (gi < 0 || gi >= nxl || gj < 0 || gj >= nyl) continue;
        const double x = xlo + ((double)gi + 0.5) * dx, y = ylo + ((double)gj + 0.5) * dy;
        const int64_t c = pd.off + (int64_t)j * pd.pitch + i;
        b[c] = __fma_rn(w, gc_deform_at(D, x, y), b[c]);
    }
}
void gc_launch_bathy_update(gc_level *L, double x0, double y0, double ddx, double ddy, int64_t mx, int64_t my, const double *d_dz, double w)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    DeformArgs D; D.x0 = x0; D.y0 = y0; D.ddx = ddx; D.ddy = ddy; D.mx = mx; D.my = my; D.dz = d_dz;
    if (L->np) k_bathy_update<<<gc_chunk_grid(L, 4), 256, 0, L->ctx->stream>>>(L->d_pat, L->b, D, w, L->xlo, L->ylo, L->dx, L->dy, L->nxl, L->nyl);
}

// ---- wet mask (h > eps), interior-packed
__global__ void k_wet_mask(const PatchDesc *pat, const double *h, double eps, uint8_t *mask)
{
    PatchDesc pd = pat[blockIdx.x];
    int n = pd.nx * pd.ny;
    const int t1 = min(n, (int)(blockIdx.y + 1) * GC_CHUNK);
    for (int t = blockIdx.y * GC_CHUNK + threadIdx.x; t < t1; t += blockDim.x) {
        int j = t / pd.nx, i = t - j * pd.nx;
        mask[pd.ioff + t] = h[pd.off + (int64_t)(j + 2) * pd.pitch + i + 2] > eps ? 1 : 0;
    }
}
void gc_launch_wet_mask(const gc_level *L, uint8_t *mask)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_wet_mask<<<gc_chunk_grid(L, 0), 256, 0, L->ctx->stream>>>(L->d_pat, L->q[L->cur][0], L->ctx->P.dry_tol, mask);
}

// ---- mass: grid = patches x chunks of GC_CHUNK cells; each block reduces its chunk in a fixed order (thread-strided partial
// sums, then a fixed tree) into partial[patch * nchunk + chunk]; the host adds the partials in index order.  Deterministic for
// a given patch list.
__global__ void k_mass(const PatchDesc *pat, const double *h, const double *kappa, double dxdy, double *partial)
{
    __shared__ double sm[256];
    PatchDesc pd = pat[blockIdx.x];
    int n = pd.nx * pd.ny;
    const int t1 = min(n, (int)(blockIdx.y + 1) * GC_CHUNK);
    double acc = 0.0;
    for (int t = blockIdx.y * GC_CHUNK + threadIdx.x; t < t1; t += 256) {
        int j = t / pd.nx, i = t - j * pd.nx;
        acc += h[pd.off + (int64_t)(j + 2) * pd.pitch + i + 2] * (kappa[pd.j0 + j + 2] * dxdy);
    }
    sm[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[(size_t)blockIdx.x * gridDim.y + blockIdx.y] = sm[0];
}
int gc_mass_partials(const gc_level *L) { const dim3 g = gc_chunk_grid(L, 0); return (int)(g.x * g.y); }
void gc_launch_mass(const gc_level *L)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_mass<<<gc_chunk_grid(L, 0), 256, 0, L->ctx->stream>>>(L->d_pat, L->q[L->cur][0], L->d_kappa, L->dx * L->dy, L->d_partial);
}
