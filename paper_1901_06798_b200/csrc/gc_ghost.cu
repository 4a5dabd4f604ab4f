// gc_ghost.cu -- ghost-cell fill kernels: same-level copy (A2) and physical boundary (A4), plus the
// field transfer, wet-mask and mass kernels.  P:143 (step 2 of the AMR algorithm); DESIGN.md 3.6.
// The paper keeps ghost filling on the CPU because a per-patch kernel has only O(a) parallelism;
// here ONE launch covers every patch of the level through host-built work lists, so the parallelism is
// O(total perimeter).
#include "gc_internal.h"

// ---- A2: one warp per rectangle (w x h cells), up to three planes
__global__ void k_copy_rects(const CopyRect *rects, int n, double *f0, double *f1, double *f2, int nf)
{
    int warp = (int)((blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5);
    int lane = threadIdx.x & 31;
    if (warp >= n) return;
    CopyRect r = rects[warp];
    int cells = r.w * r.h;
    for (int c = lane; c < cells; c += 32) {
        int y = c / r.w, x = c - y * r.w;
        int64_t d = r.dst + (int64_t)y * r.dpitch + x, s = r.src + (int64_t)y * r.spitch + x;
        f0[d] = f0[s];
        if (nf > 1) { f1[d] = f1[s]; f2[d] = f2[s]; }
    }
}

void gc_launch_copy_rects(gc_level *L, double *f0, double *f1, double *f2, int nf)
{
    if (L->ncopy == 0) return;
    int threads = 256;
    int64_t blocks = ((int64_t)L->ncopy * 32 + threads - 1) / threads;
    ProfScope ps(L->ctx, GC_SLOT_COPY);
    k_copy_rects<<<(unsigned)blocks, threads, 0, L->ctx->stream>>>(L->d_copy, L->ncopy, f0, f1, f2, nf);
}

// ---- A4: physical boundary.  pass 0: x faces over rows inside the domain; pass 1: y faces over all columns.
// Wall: mirror cell, normal momentum negated (is_state: f1 = hu, f2 = hv); extrapolation: nearest interior cell.
__global__ void k_bc(const PatchDesc *pat, const int32_t *list, double *f0, double *f1, double *f2, int nf, int is_state,
                     int pass, int64_t nxl, int64_t nyl, int bc0, int bc1, int bc2, int bc3)
{
    PatchDesc pd = pat[list[blockIdx.x]];
    int rows = pd.ny + 4;
    if (pass == 0) {
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
    } else {
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
    ProfScope ps(L->ctx, GC_SLOT_BC, 2);
    for (int pass = 0; pass < 2; pass++)
        k_bc<<<L->nbcp, 128, 0, L->ctx->stream>>>(L->d_pat, L->d_bcp, f0, f1, f2, nf, is_state, pass, L->nxl, L->nyl,
                                                  bc[0], bc[1], bc[2], bc[3]);
}

// ---- field transfer
__global__ void k_set_global(const PatchDesc *pat, double *plane, const double *src, int64_t ld,
                             int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    PatchDesc pd = pat[blockIdx.x];
    const int W = pd.nx + 4;
    int n = W * (pd.ny + 4);
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
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
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
        const int j = t / W, i = t - j * W;
        const int64_t gi = (int64_t)pd.i0 + i - 2, gj = (int64_t)pd.j0 + j - 2;
        if (gi < 0 || gi >= nxl || gj < 0 || gj >= nyl) continue;
        plane[pd.off + (int64_t)j * pd.pitch + i] = sp[t];
    }
}
void gc_launch_set_patches(gc_level *L, double *plane, const int64_t *goff, const double *src)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_set_patches<<<L->np, 256, 0, L->ctx->stream>>>(L->d_pat, goff, plane, src, L->nxl, L->nyl);
}

__global__ void k_get_global(const PatchDesc *pat, const double *plane, double *dst, int64_t ld,
                             int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    PatchDesc pd = pat[blockIdx.x];
    int n = pd.nx * pd.ny;
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
        int j = t / pd.nx, i = t - j * pd.nx;
        int64_t gi = (int64_t)pd.i0 + i - gi0, gj = (int64_t)pd.j0 + j - gj0;
        if (gi < 0 || gi >= gnx || gj < 0 || gj >= gny) continue;
        dst[gj * ld + gi] = plane[pd.off + (int64_t)(j + 2) * pd.pitch + i + 2];
    }
}

void gc_launch_set_global(gc_level *L, double *plane, const double *src, int64_t ld, int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_set_global<<<L->np, 256, 0, L->ctx->stream>>>(L->d_pat, plane, src, ld, gi0, gj0, gnx, gny);
}
void gc_launch_get_global(const gc_level *L, const double *plane, double *dst, int64_t ld, int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_get_global<<<L->np, 256, 0, L->ctx->stream>>>(L->d_pat, plane, dst, ld, gi0, gj0, gnx, gny);
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

// ---- wet mask (h > eps), interior-packed
__global__ void k_wet_mask(const PatchDesc *pat, const double *h, double eps, uint8_t *mask)
{
    PatchDesc pd = pat[blockIdx.x];
    int n = pd.nx * pd.ny;
    for (int t = threadIdx.x; t < n; t += blockDim.x) {
        int j = t / pd.nx, i = t - j * pd.nx;
        mask[pd.ioff + t] = h[pd.off + (int64_t)(j + 2) * pd.pitch + i + 2] > eps ? 1 : 0;
    }
}
void gc_launch_wet_mask(const gc_level *L, uint8_t *mask)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_wet_mask<<<L->np, 256, 0, L->ctx->stream>>>(L->d_pat, L->q[L->cur][0], L->ctx->P.dry_tol, mask);
}

// ---- mass: per patch, fixed-order reduction (thread-strided partial sums, then a fixed tree); the host adds
// the per-patch partials in patch order.  Deterministic for a given patch list.
__global__ void k_mass(const PatchDesc *pat, const double *h, const double *kappa, double dxdy, double *partial)
{
    __shared__ double sm[256];
    PatchDesc pd = pat[blockIdx.x];
    int n = pd.nx * pd.ny;
    double acc = 0.0;
    for (int t = threadIdx.x; t < n; t += 256) {
        int j = t / pd.nx, i = t - j * pd.nx;
        acc += h[pd.off + (int64_t)(j + 2) * pd.pitch + i + 2] * (kappa[pd.j0 + j + 2] * dxdy);
    }
    sm[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sm[0];
}
void gc_launch_mass(const gc_level *L)
{
    ProfScope ps(L->ctx, GC_SLOT_MISC);
    if (L->np) k_mass<<<L->np, 256, 0, L->ctx->stream>>>(L->d_pat, L->q[L->cur][0], L->d_kappa, L->dx * L->dy, L->d_partial);
}
