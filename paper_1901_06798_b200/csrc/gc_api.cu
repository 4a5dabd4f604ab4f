// gc_api.cu -- C ABI entry points (include/gc.h) and the host-side level runtime: pool layout, patch
// descriptors, metric tables, work lists.  All arithmetic of the method runs in the kernels; the host only
// builds index lists ("only clustering and bookkeeping stay on the host") and the per-row metric tables
// (sin/cos evaluated once on the host).
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <algorithm>
#include <atomic>
#include "gc_internal.h"

static std::atomic<uint64_t> g_gen{1};

int gc_fail(gc_ctx *c, int code, const char *msg) { if (c) c->err = msg; return code; }

int gc_cuda_check(gc_ctx *c, const char *what)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) {
        if (c) c->err = std::string(what) + ": " + cudaGetErrorString(e);
        return GC_ERR_CUDA;
    }
    return GC_OK;
}

void *gc_dev_alloc(gc_ctx *c, size_t bytes)
{
    if (bytes == 0) bytes = 8;
    if (c->alloc) return c->alloc(bytes, c->user);
    void *p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}
void gc_dev_free(gc_ctx *c, void *p)
{
    if (!p) return;
    if (c->free_) c->free_(p, c->user); else if (!c->alloc) cudaFree(p);
}

#define GC_STAGE_KEEP_MAX ((size_t)64 << 20)
void *gc_stage_get(gc_ctx *c, size_t bytes, bool *transient)
{
    *transient = bytes > GC_STAGE_KEEP_MAX;
    if (*transient) return gc_dev_alloc(c, bytes);
    if (bytes > c->stage_bytes) {
        // every host-pointer call ends with a stream synchronisation, so nothing queued still uses the old buffer
        if (c->stage) { cudaStreamSynchronize(c->stream); gc_dev_free(c, c->stage); c->stage = nullptr; c->stage_bytes = 0; }
        size_t cap = (size_t)1 << 20;
        while (cap < bytes) cap <<= 1;
        c->stage = gc_dev_alloc(c, cap);
        if (!c->stage) return nullptr;
        c->stage_bytes = cap;
    }
    return c->stage;
}

extern "C" const char *gc_last_error(const gc_ctx *c) { return c ? c->err.c_str() : "null context"; }

extern "C" int gc_ctx_create(const gc_params *P, void *stream, gc_alloc_fn alloc, gc_free_fn free_, void *user, gc_ctx **out)
{
    if (!P || !out) return GC_ERR_BADARG;
    if (!(P->g > 0.0) || !(P->dry_tol >= 0.0) || (P->coord != 0 && P->coord != 1)) return GC_ERR_BADARG;
    if (!(P->manning_n >= 0.0) || (P->manning_n > 0.0 && !(P->dry_tol > 0.0))) return GC_ERR_BADARG;   // friction divides by h^(7/3), h > dry_tol
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return GC_ERR_CUDA; }   // no CPU fallback
    gc_ctx *c = new gc_ctx();
    c->P = *P; c->stream = (cudaStream_t)stream; c->alloc = alloc; c->free_ = free_; c->user = user;
    gc_unsplit_static_setup();        // gc_level_step_unsplit_static: address of its scratch array, once per device (a failure is reported there)
    *out = c;
    return GC_OK;
}
extern "C" int gc_ctx_destroy(gc_ctx *c)
{
    if (c && c->stage) { cudaStreamSynchronize(c->stream); gc_dev_free(c, c->stage); }
    delete c;
    return GC_OK;
}

extern "C" int gc_ctx_set_option(gc_ctx *c, int key, int64_t value)
{
    if (!c) return GC_ERR_BADARG;
    if (key == GC_OPT_SWEEP_FAMILY && value >= 0 && value <= 2) { c->opt_family = (int)value; return GC_OK; }
    if (key == GC_OPT_CHAINS && (value == 0 || value == 1 || (value >= 8 && value <= 1000000))) { c->opt_chains = (int)value; return GC_OK; }
    if (key == GC_OPT_MARCH_SEG && (value == 0 || (value >= 4 && value <= 4096))) { c->opt_seg = (int)value; return GC_OK; }
    return gc_fail(c, GC_ERR_BADARG, "gc_ctx_set_option: unknown key or value out of range");
}

extern "C" int64_t gc_launch_count(const gc_ctx *c) { return c ? (int64_t)c->launches : 0; }
extern "C" int gc_profile_enable(gc_ctx *c, int on) { if (!c) return GC_ERR_BADARG; c->prof = on != 0; c->prof_last = nullptr; return GC_OK; }
extern "C" int gc_profile_read(gc_ctx *c, double *ms, int64_t *count)
{
    if (!c || !ms || !count) return GC_ERR_BADARG;
    cudaStreamSynchronize(c->stream);
    for (int s = 0; s < GC_NSLOT; s++) {
        ms[s] = 0.0; count[s] = (int64_t)c->ev[s].size();
        for (auto &p : c->ev[s]) {
            float t = 0.f;
            cudaEventElapsedTime(&t, p.first, p.second);
            ms[s] += t;
        }
        c->ev[s].clear();
    }
    for (cudaEvent_t e : c->ev_own) cudaEventDestroy(e);
    c->ev_own.clear(); c->prof_last = nullptr;
    return gc_cuda_check(c, "gc_profile_read");
}

template <class T> static T *upload(gc_level *L, const std::vector<T> &v)
{
    T *d = (T *)gc_dev_alloc(L->ctx, v.size() * sizeof(T));
    if (!d) return nullptr;
    L->allocs.push_back(d);
    if (!v.empty()) cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, L->ctx->stream);
    return d;
}

static inline int64_t bkey(int64_t bx, int64_t by) { return (bx << 32) ^ (by & 0xffffffffll); }

int gc_find_patch_host(const gc_level *L, int64_t gi, int64_t gj)
{
    if (gi < 0 || gj < 0 || gi >= L->nxl || gj >= L->nyl) return -1;
    auto it = L->buckets.find(bkey(gi / L->bsize, gj / L->bsize));
    if (it == L->buckets.end()) return -1;
    for (int32_t q : it->second) {
        const gc_patch &Q = L->pat[q];
        if (gi >= Q.i0 && gi < (int64_t)Q.i0 + Q.nx && gj >= Q.j0 && gj < (int64_t)Q.j0 + Q.ny) return q;
    }
    return -1;
}

// DESIGN.md 3.5 metric tables over global rows -2..ny+1 (index +2) and edges -2..ny+2
static void build_metric(gc_level *L)
{
    const gc_params &P = L->ctx->P;
    int64_t ny = L->nyl, nr = ny + 4, ne = ny + 5;
    L->kappa.assign(nr, 1.0); L->rdx.assign(nr, 0.0); L->rdy.assign(nr, 0.0); L->ey.assign(ne, 1.0);
    L->ex = 1.0;
    if (P.coord == 1) {
        const double pi = 3.14159265358979323846;
        const double d2r = pi / 180.0;
        double R = P.earth_radius;
        L->ex = R * d2r;
        for (int64_t j = -2; j <= ny + 2; j++) {
            double lat = (L->ylo + (double)j * L->dy) * d2r;
            L->ey[j + 2] = R * cos(lat) * d2r;
        }
        for (int64_t j = -2; j <= ny + 1; j++) {
            double lat0 = (L->ylo + (double)j * L->dy) * d2r;
            double lat1 = (L->ylo + (double)(j + 1) * L->dy) * d2r;
            L->kappa[j + 2] = d2r * (R * R) * (sin(lat1) - sin(lat0)) / L->dy;
        }
        if (P.bc[2] == 1) { L->kappa[1] = L->kappa[2]; L->kappa[0] = L->kappa[3]; L->ey[1] = L->ey[3]; L->ey[0] = L->ey[4]; }
        if (P.bc[3] == 1) {
            L->kappa[ny + 2] = L->kappa[ny + 1]; L->kappa[ny + 3] = L->kappa[ny];
            L->ey[ny + 3] = L->ey[ny + 1]; L->ey[ny + 4] = L->ey[ny];
        }
    }
    for (int64_t j = 0; j < nr; j++) {
        L->rdx[j] = 1.0 / (L->kappa[j] * L->dx);
        L->rdy[j] = 1.0 / (L->kappa[j] * L->dy);
    }
}

static void build_tiles(gc_level *L, std::vector<SweepTile> &xt, std::vector<SweepTile> &yt)
{
    const int B = 256, YW = 8;
    for (int p = 0; p < L->np; p++) {
        const gc_patch &P = L->pat[p];
        // x-sweep: all rows 0..ny+3; whole rows if nx+3 <= B, else balanced chunks of <= B-3 cells
        int nchunk = (P.nx + (B - 3) - 1) / (B - 3);
        {   // pick the chunking with the most updated cells per thread: R rows of (nc + 3) edges fill a block of B threads
            int best = 0;
            for (int m = nchunk; m <= std::max(nchunk, P.nx / 8); m++) {
                int nc = (P.nx + m - 1) / m, R = B / (nc + 3);
                if (R < 1) continue;
                int useful = std::min(R, P.ny + 4) * nc;
                if (useful > best) { best = useful; nchunk = m; }
            }
        }
        for (int c = 0; c < nchunk; c++) {
            int c0 = (int)((int64_t)P.nx * c / nchunk), c1 = (int)((int64_t)P.nx * (c + 1) / nchunk);
            int nc = c1 - c0, R = B / (nc + 3);
            for (int r0 = 0; r0 < P.ny + 4; r0 += R)
                xt.push_back(SweepTile{p, r0, std::min(R, P.ny + 4 - r0), 2 + c0, nc});
        }
        // y-sweep: interior columns in groups of YW, segments of <= B/YW - 3 cells along y
        int E = B / YW, nseg = (P.ny + (E - 3) - 1) / (E - 3);
        for (int s = 0; s < nseg; s++) {
            int r0 = (int)((int64_t)P.ny * s / nseg), r1 = (int)((int64_t)P.ny * (s + 1) / nseg);
            for (int i0 = 0; i0 < P.nx; i0 += YW)
                yt.push_back(SweepTile{p, 2 + i0, std::min(YW, P.nx - i0), 2 + r0, r1 - r0});
        }
    }
}

// ---- chains (gc_internal.h): succ[p] = the patch that continues p along `dir`, or -1.  A patch continues another when it has
// the same extent across the sweep and starts where the other ends.  Pieces shorter than 8 cells are not chained (the kernels keep
// the bases of two pieces only, and the output runs 5 cells behind the input); along x every piece but the last must be a multiple
// of 4 cells long so that the 16-byte loads and the 32-byte stores of the x-sweep keep their alignment across pieces.
// GC_OPT_CHAINS = k >= 8 keeps pieces of k cells or more on their own (measurements).
static void build_chains(gc_level *L, int dir, std::vector<int32_t> &succ, std::vector<int32_t> &pred)
{
    succ.assign((size_t)std::max(L->np, 1), -1); pred.assign((size_t)std::max(L->np, 1), -1);
    if (L->ctx->opt_chains == 1) return;
    const int maxp = L->ctx->opt_chains >= 8 ? L->ctx->opt_chains : 2147483647;
    for (int p = 0; p < L->np; p++) {
        const gc_patch &P = L->pat[p];
        const int n = dir == 0 ? P.nx : P.ny;
        if (n < 8 || n >= maxp || (dir == 0 && n % 4 != 0)) continue;
        const int q = dir == 0 ? gc_find_patch_host(L, (int64_t)P.i0 + P.nx, P.j0) : gc_find_patch_host(L, P.i0, (int64_t)P.j0 + P.ny);
        if (q < 0) continue;
        const gc_patch &Q = L->pat[q];
        if ((dir == 0 ? Q.nx : Q.ny) < 8 || (dir == 0 ? Q.nx : Q.ny) >= maxp) continue;
        const bool fits = dir == 0 ? (Q.i0 == P.i0 + P.nx && Q.j0 == P.j0 && Q.ny == P.ny) : (Q.j0 == P.j0 + P.ny && Q.i0 == P.i0 && Q.nx == P.nx);
        if (!fits) continue;
        succ[(size_t)p] = q; pred[(size_t)q] = p;
    }
}

// marching lines (k_marchp): every row (x) / interior column (y) of every chain of patches, cut into balanced segments of about
// `seg` cells whose boundaries are multiples of 4 cells, so that an x segment starts on a 32-byte boundary of its row.
// xl_red: the x lines without the ghost rows that no y line reads (patches continued inside a y chain on that side).
// need[p]: which parts of patch p's ghost ring some line reads -- bit 0 the left ghost columns (p heads its x chain), bit 1 the right
// ones (p ends it), bit 2 the bottom ghost rows (some piece of p's x chain has no patch below in its y chain, so the chain's ghost
// rows are swept), bit 3 the top ones.  Everything else is reached through the neighbour's interior (gc_fill_ghost_step).
static void build_lines(gc_level *L, int seg, std::vector<LineDesc> &xl, std::vector<LineDesc> &yl, std::vector<LineDesc> &xl_red,
                        std::vector<ChainLink> &xlink, std::vector<ChainLink> &ylink, std::vector<uint8_t> &need)
{
    std::vector<int32_t> succ[2], pred[2];
    build_chains(L, 0, succ[0], pred[0]); build_chains(L, 1, succ[1], pred[1]);
    xlink.resize((size_t)std::max(L->np, 1)); ylink.resize((size_t)std::max(L->np, 1));
    {
        size_t nx_ = 0, ny_ = 0;
        for (const gc_patch &P : L->pat) {
            nx_ += (size_t)(P.ny + 4) * (size_t)std::max(1, (P.nx + seg - 1) / seg);
            ny_ += (size_t)P.nx * (size_t)std::max(1, (P.ny + seg - 1) / seg);
        }
        xl.reserve(nx_); yl.reserve(ny_);
    }
    L->chained = 0;
    std::vector<int32_t> piece; std::vector<int64_t> shift;
    for (int dir = 0; dir < 2; dir++) {
        std::vector<ChainLink> &link = dir == 0 ? xlink : ylink;
        for (int h = 0; h < L->np; h++) {
            if (pred[dir][(size_t)h] >= 0) continue;                                   // chains start at their heads
            piece.clear(); shift.clear();
            int64_t n = 0;                                                               // cells along the sweep (<= 2e9: gc_level_create)
            bool lo_ghost = false, hi_ghost = false;                                     // x chains: some piece's ghost rows are read by y lines
            for (int p = h; p >= 0; p = succ[dir][(size_t)p]) {
                const gc_patch &P = L->pat[p];
                piece.push_back(p); shift.push_back(n);
                n += dir == 0 ? P.nx : P.ny;
                if (dir == 0) { lo_ghost |= pred[1][(size_t)p] < 0; hi_ghost |= succ[1][(size_t)p] < 0; }
            }
            if (piece.size() > 1) L->chained = 1;
            if (dir == 0)
                for (size_t k = 0; k < piece.size(); k++)
                    need[(size_t)piece[k]] = (uint8_t)((k == 0 ? 1 : 0) | (k + 1 == piece.size() ? 2 : 0) | (lo_ghost ? 4 : 0) | (hi_ghost ? 8 : 0));
            for (size_t k = 0; k < piece.size(); k++) {
                const PatchDesc &D = L->hpat[(size_t)piece[k]];
                ChainLink &K = link[(size_t)piece[k]];
                const bool last = k + 1 == piece.size();
                K.A = dir == 0 ? D.off - shift[k] : D.off - shift[k] * D.pitch;
                K.end = last ? 2147483647 : (int32_t)(shift[k] + 2 + (dir == 0 ? D.nx : D.ny));
                K.next = last ? -1 : piece[k + 1];
                K.pitch = D.pitch;
                K.org = dir == 0 ? D.j0 : (int32_t)(D.j0 - shift[k]);
            }
            const gc_patch &H = L->pat[h];
            const int nlines = dir == 0 ? H.ny + 4 : H.nx;                               // x: all rows (S-5); y: interior columns
            const int line0 = dir == 0 ? 0 : 2;
            const int nch = (int)std::max<int64_t>(1, (n + seg - 1) / seg);
            size_t k0 = 0;
            for (int k = 0; k < nch; k++) {
                int64_t b0 = k == 0 ? 0 : ((n * k / nch + 3) / 4 * 4);
                int64_t b1 = k == nch - 1 ? n : ((n * (k + 1) / nch + 3) / 4 * 4);
                b0 = std::min(b0, n); b1 = std::min(b1, n);
                if (b1 <= b0) continue;
                // the piece holding position b0 (= c0 - 2): piece k0 owns positions [shift + 2, shift + 2 + its cells), the head from 0
                while (k0 + 1 < piece.size() && b0 >= shift[k0 + 1] + 2) k0++;
                const int32_t sp = piece[k0];
                for (int l = 0; l < nlines; l++) {
                    const LineDesc d{sp, line0 + l, (int32_t)(2 + b0), (int32_t)(b1 - b0)};
                    if (dir == 0) {
                        xl.push_back(d); L->sweep_cells[0] += d.nc;
                        const bool ghost_row = l < 2 || l >= H.ny + 2;
                        if (!ghost_row || (l < 2 ? lo_ghost : hi_ghost)) { xl_red.push_back(d); L->sweep_cells[1] += d.nc; }
                    } else { yl.push_back(d); L->sweep_cells[2] += d.nc; }
                }
            }
        }
    }
}

extern "C" int gc_level_create(gc_ctx *ctx, int level, double xlo, double ylo, double dx, double dy,
                               int64_t nxl, int64_t nyl, int ratio, int np, const gc_patch *pat, gc_level **out)
{
    if (!ctx || !out || np < 0 || (np > 0 && !pat) || nxl < 1 || nyl < 1 || !(dx > 0.0) || !(dy > 0.0) || ratio < 1 || level < 1)
        return gc_fail(ctx, GC_ERR_BADARG, "gc_level_create: bad argument");
    if (nxl > 2000000000ll || nyl > 2000000000ll) return gc_fail(ctx, GC_ERR_BADARG, "gc_level_create: level too large");
    int maxdim = 1;
    for (int p = 0; p < np; p++) {
        const gc_patch &P = pat[p];
        if (P.nx < 2 || P.ny < 2 || P.i0 < 0 || P.j0 < 0 || (int64_t)P.i0 + P.nx > nxl || (int64_t)P.j0 + P.ny > nyl)
            return gc_fail(ctx, GC_ERR_BADARG, "gc_level_create: patch outside the level or smaller than 2 cells");
        if (level > 1 && (P.i0 % ratio || P.j0 % ratio || P.nx % ratio || P.ny % ratio))
            return gc_fail(ctx, GC_ERR_BADARG, "gc_level_create: fine patch not aligned with coarse cells");
        maxdim = std::max(maxdim, std::max(P.nx, P.ny));
    }
    gc_level *L = new gc_level();
    L->ctx = ctx; L->level = level; L->ratio = ratio; L->np = np; L->cur = 0;
    L->xlo = xlo; L->ylo = ylo; L->dx = dx; L->dy = dy; L->nxl = nxl; L->nyl = nyl;
    L->gen = g_gen.fetch_add(1);
    L->pat.assign(pat, pat + np);
    L->bsize = std::max(maxdim, 8);
    L->hpat.resize(np);
    // Every patch starts 2 elements (16 bytes) past a 32-byte boundary and its pitch is a multiple of 4, so that storage column 2
    // -- the first interior cell -- of every row starts a 32-byte sector: interior rows are read and written as whole sectors
    // (with ghost width 2 the other choice, rows starting on a sector, leaves both ends of every interior row on half sectors,
    // which small patches pay in DRAM traffic: 5 sectors touched for a 16-cell row instead of 4, read-modify-write at both ends)
    int64_t off = 2, ioff = 0;
    for (int p = 0; p < np; p++) {
        const gc_patch &P = L->pat[p];
        PatchDesc &D = L->hpat[p];
        D.i0 = P.i0; D.j0 = P.j0; D.nx = P.nx; D.ny = P.ny; D.off = off; D.ioff = ioff; D.pitch = ((P.nx + 4 + 3) / 4) * 4;
        D.bcmask = (P.i0 - 2 < 0 ? 1 : 0) | ((int64_t)P.i0 + P.nx + 2 > nxl ? 2 : 0) | (P.j0 - 2 < 0 ? 4 : 0) | ((int64_t)P.j0 + P.ny + 2 > nyl ? 8 : 0);
        off += (int64_t)D.pitch * (P.ny + 4);   // multiple of 4 elements
        ioff += (int64_t)P.nx * P.ny;
        for (int64_t by = P.j0 / L->bsize; by <= (P.j0 + P.ny - 1) / L->bsize; by++)
            for (int64_t bx = P.i0 / L->bsize; bx <= (P.i0 + P.nx - 1) / L->bsize; bx++)
                L->buckets[bkey(bx, by)].push_back(p);
    }
    L->tot = off; L->ncells = ioff;
    // overlap check (patches of a level are disjoint)
    for (int p = 0; p < np; p++) {
        const gc_patch &P = L->pat[p];
        for (int64_t by = P.j0 / L->bsize; by <= (P.j0 + P.ny - 1) / L->bsize; by++)
            for (int64_t bx = P.i0 / L->bsize; bx <= (P.i0 + P.nx - 1) / L->bsize; bx++)
                for (int32_t q : L->buckets[bkey(bx, by)]) {
                    if (q <= p) continue;
                    const gc_patch &Q = L->pat[q];
                    if (std::max(P.i0, Q.i0) < std::min(P.i0 + P.nx, Q.i0 + Q.nx) && std::max(P.j0, Q.j0) < std::min(P.j0 + P.ny, Q.j0 + Q.ny)) {
                        delete L;
                        return gc_fail(ctx, GC_ERR_BADARG, "gc_level_create: patches overlap");
                    }
                }
    }
    // pool: q[0][3], q[1][3], b, qs[3] = 10 planes, one allocation
    int64_t plane = ((L->tot + 31) / 32) * 32 + 32;
    L->pool = (double *)gc_dev_alloc(ctx, (size_t)plane * 10 * sizeof(double));
    if (!L->pool) { delete L; return gc_fail(ctx, GC_ERR_NOMEM, "gc_level_create: pool allocation failed"); }
    L->allocs.push_back(L->pool);
    cudaMemsetAsync(L->pool, 0, (size_t)plane * 10 * sizeof(double), ctx->stream);
    for (int w = 0; w < 2; w++) for (int f = 0; f < 3; f++) L->q[w][f] = L->pool + (int64_t)(w * 3 + f) * plane;
    L->b = L->pool + 6 * plane;
    for (int f = 0; f < 3; f++) L->qs[f] = L->pool + (int64_t)(7 + f) * plane;

    std::vector<uint8_t> need((size_t)std::max(np, 1), 15);   // parts of each ghost ring a sweep reads (build_lines): all of it unless chained
    build_metric(L);
    L->d_kappa = upload(L, L->kappa); L->d_rdx = upload(L, L->rdx); L->d_rdy = upload(L, L->rdy); L->d_ey = upload(L, L->ey);
    L->d_pat = upload(L, L->hpat);
    {   // sweep kernel family: marching lines for large levels, edge-parallel tiles for small ones (gc_ctx_set_option overrides);
        // only the family's own work list is built
        L->use_march = L->ncells >= (int64_t)GC_MARCH_MIN_CELLS;
        if (ctx->opt_family == 1) L->use_march = 0;
        if (ctx->opt_family == 2) L->use_march = 1;
        std::vector<SweepTile> xt, yt;
        if (!L->use_march) build_tiles(L, xt, yt);
        L->nxt = (int)xt.size(); L->nyt = (int)yt.size();
        L->d_xt = upload(L, xt); L->d_yt = upload(L, yt);
        int seg = (int)std::min<int64_t>(128, std::max<int64_t>(16, (L->ncells / 400000 + 3) / 4 * 4));
        if (ctx->opt_seg >= 4) seg = ctx->opt_seg / 4 * 4;
        std::vector<LineDesc> xl, yl, xl_red;
        std::vector<ChainLink> xlink, ylink;
        if (L->use_march) build_lines(L, seg, xl, yl, xl_red, xlink, ylink, need);
        if (xl_red.size() == xl.size()) xl_red.clear();                  // nothing to leave out: one list
        L->nxl_lines = (int64_t)xl.size(); L->nyl_lines = (int64_t)yl.size(); L->nxl_red = (int64_t)xl_red.size();
        L->d_xl = upload(L, xl); L->d_yl = upload(L, yl); L->d_xl_red = upload(L, xl_red);
        L->d_xlink = upload(L, xlink); L->d_ylink = upload(L, ylink);
        cudaStreamSynchronize(ctx->stream);
    }

    // same-level copy rectangles: grown box of p  x  interior of q (A2, incl. corners)
    std::vector<CopyRect> rects, rects_red;                   // all of them; the ones a split step reads (gc_fill_ghost_step)
    std::vector<int2> rrange((size_t)std::max(np, 1)), rrange_red((size_t)std::max(np, 1));
    int64_t ghost_cells = 0;
    std::vector<int32_t> bcp;
    std::vector<uint8_t> mask;
    for (int p = 0; p < np; p++) {
        const gc_patch &P = L->pat[p];
        const PatchDesc &D = L->hpat[p];
        if (D.bcmask) bcp.push_back(p);
        int64_t gx0 = (int64_t)P.i0 - 2, gx1 = (int64_t)P.i0 + P.nx + 2, gy0 = (int64_t)P.j0 - 2, gy1 = (int64_t)P.j0 + P.ny + 2;
        bool need_mask = level > 1;
        if (need_mask) mask.assign((size_t)D.pitch * (P.ny + 4), 0);
        size_t first = rects.size(), first_red = rects_red.size();
        int64_t bx0 = std::max<int64_t>(gx0, 0) / L->bsize, bx1 = std::min<int64_t>(gx1 - 1, nxl - 1) / L->bsize;
        int64_t by0 = std::max<int64_t>(gy0, 0) / L->bsize, by1 = std::min<int64_t>(gy1 - 1, nyl - 1) / L->bsize;
        for (int64_t by = by0; by <= by1; by++) for (int64_t bx = bx0; bx <= bx1; bx++) {
            auto it = L->buckets.find(bkey(bx, by));
            if (it == L->buckets.end()) continue;
            for (int32_t q : it->second) {
                if (q == p) continue;
                const gc_patch &Q = L->pat[q];
                int64_t x0 = std::max<int64_t>(gx0, Q.i0), x1 = std::min<int64_t>(gx1, (int64_t)Q.i0 + Q.nx);
                int64_t y0 = std::max<int64_t>(gy0, Q.j0), y1 = std::min<int64_t>(gy1, (int64_t)Q.j0 + Q.ny);
                if (x0 >= x1 || y0 >= y1) continue;
                const PatchDesc &DQ = L->hpat[q];
                CopyRect r;
                r.dst = D.off + (y0 - P.j0 + 2) * D.pitch + (x0 - P.i0 + 2);
                r.src = DQ.off + (y0 - Q.j0 + 2) * DQ.pitch + (x0 - Q.i0 + 2);
                r.w = (int)(x1 - x0); r.h = (int)(y1 - y0); r.dpitch = D.pitch; r.spitch = DQ.pitch;
                // a patch spanning several buckets is met more than once: keep the first
                bool dup = false;
                for (size_t k = first; k < rects.size(); k++) if (rects[k].dst == r.dst) { dup = true; break; }
                if (dup) continue;
                rects.push_back(r);
                ghost_cells += (int64_t)r.w * r.h;
                {   // does a sweep line read any cell of it?  (storage coordinates of p; interior = columns 2..nx+1, rows 2..ny+1)
                    const int64_t rx0 = x0 - P.i0 + 2, rx1 = x1 - P.i0 + 2, ry0 = y0 - P.j0 + 2, ry1 = y1 - P.j0 + 2;
                    const uint8_t nd = need[(size_t)p];
                    const bool sideL = rx0 < 2 && (nd & 1), sideR = rx1 > P.nx + 2 && (nd & 2);
                    const bool cols_in = rx0 < P.nx + 2 && rx1 > 2, rows_in = ry0 < P.ny + 2 && ry1 > 2;
                    const bool used = (rows_in && (sideL || sideR)) || (ry0 < 2 && (nd & 4) && (cols_in || sideL || sideR))
                                      || (ry1 > P.ny + 2 && (nd & 8) && (cols_in || sideL || sideR));
                    if (used) rects_red.push_back(r);
                }
                if (need_mask)
                    for (int64_t y = y0; y < y1; y++) for (int64_t x = x0; x < x1; x++)
                        mask[(size_t)(y - P.j0 + 2) * D.pitch + (x - P.i0 + 2)] = 1;
            }
        }
        rrange[(size_t)p] = make_int2((int)first, (int)(rects.size() - first));
        rrange_red[(size_t)p] = make_int2((int)first_red, (int)(rects_red.size() - first_red));
        if (need_mask) {   // in-domain ghost cells without a same-level source come from the coarser level (A3)
            for (int j = 0; j < P.ny + 4; j++) for (int i = 0; i < P.nx + 4; i++) {
                if (i == 2 && j >= 2 && j < P.ny + 2) i = P.nx + 2;              // the ghost ring only: skip the row's interior
                int64_t gi = (int64_t)P.i0 + i - 2, gj = (int64_t)P.j0 + j - 2;
                if (gi < 0 || gi >= nxl || gj < 0 || gj >= nyl) continue;
                if (mask[(size_t)j * D.pitch + i]) continue;
                L->coarse_ghost.push_back(D.off + (int64_t)j * D.pitch + i);
                L->coarse_ghost_ij.push_back((int32_t)gi); L->coarse_ghost_ij.push_back((int32_t)gj);
            }
        }
    }
    L->ncopy = (int)rects.size(); L->d_copy = upload(L, rects);
    L->d_copy_range = upload(L, rrange);
    L->ncopy_red = -1;                                            // -1: every rectangle is read by the step, one list
    if (rects_red.size() < rects.size()) {
        L->ncopy_red = (int)rects_red.size(); L->d_copy_red = upload(L, rects_red); L->d_copy_range_red = upload(L, rrange_red);
        if (!L->d_copy_red || !L->d_copy_range_red) L->ncopy_red = -1;
    }
    {   // warps per patch: about 256 ghost cells per warp, at most 16
        const int64_t per = np > 0 ? ghost_cells / np : 0;
        L->copy_wpp = (int)std::min<int64_t>(16, std::max<int64_t>(1, per / 256));
    }
    L->nbcp = (int)bcp.size(); L->d_bcp = upload(L, bcp);
    L->d_stats = (DevStats *)gc_dev_alloc(ctx, sizeof(DevStats)); L->allocs.push_back(L->d_stats);
    if (L->d_stats) cudaMemsetAsync(L->d_stats, 0, sizeof(DevStats), ctx->stream);
    L->d_partial = (double *)gc_dev_alloc(ctx, sizeof(double) * (size_t)std::max(gc_mass_partials(L), 1)); L->allocs.push_back(L->d_partial);
    L->cf_for = nullptr; L->cf_gen = 0; L->d_cf = nullptr; L->d_cfstart = nullptr; L->ncf = 0; L->ncfcells = 0;
    L->avg_gen = 0; L->d_avg = nullptr; L->d_avgstart = nullptr; L->navg = 0; L->navgcells = 0;
    L->nbr_buffer = -1; L->d_nbrstart = nullptr; L->d_nbrlist = nullptr; L->r_reg = 1;
    L->reg_fine = nullptr; L->reg_coarse = nullptr; L->d_reg = nullptr; L->nreg = 0;
    L->d_delta = nullptr; L->d_base = nullptr; L->d_fixstart = nullptr; L->d_fixreg = nullptr; L->nfix = 0;
    if (!L->d_pat || !L->d_xt || !L->d_yt || !L->d_xl || !L->d_yl || !L->d_xl_red || !L->d_xlink || !L->d_ylink || !L->d_copy || !L->d_copy_range || !L->d_bcp || !L->d_stats || !L->d_partial || !L->d_kappa) {
        gc_level_destroy(L);
        return gc_fail(ctx, GC_ERR_NOMEM, "gc_level_create: table allocation failed");
    }
    gc_launch_stats_reset(L);
    cudaStreamSynchronize(ctx->stream);   // host vectors used by the uploads go out of scope
    int rc = gc_cuda_check(ctx, "gc_level_create");
    if (rc) { gc_level_destroy(L); return rc; }
    *out = L;
    return GC_OK;
}

void gc_amr_on_destroy(gc_level *L);

extern "C" int gc_level_destroy(gc_level *L)
{
    if (!L) return GC_OK;
    gc_amr_on_destroy(L);
    cudaStreamSynchronize(L->ctx->stream);
    for (cudaEvent_t e : {L->ev_up_copied, L->ev_up_free, L->ev_dn_ready, L->ev_dn_free}) if (e) { cudaEventSynchronize(e); cudaEventDestroy(e); }
    for (void *p : L->allocs) gc_dev_free(L->ctx, p);
    delete L;
    return GC_OK;
}

extern "C" int64_t gc_level_ncells(const gc_level *L) { return L ? L->ncells : 0; }

static double *plane_of(const gc_level *L, int field, int which)
{
    if (field == GC_FIELD_B) return L->b;
    return L->q[which == GC_NEW ? L->cur : 1 - L->cur][field];
}

extern "C" int gc_level_set_field(gc_level *L, int p, int field, const double *src, int is_device, int64_t ld)
{
    if (!L || p < 0 || p >= L->np || field < 0 || field > 3 || !src || ld < L->pat[p].nx + 4) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_set_field: bad argument");
    const PatchDesc &D = L->hpat[p];
    double *dst = plane_of(L, field, GC_NEW) + D.off;
    cudaMemcpy2DAsync(dst, (size_t)D.pitch * 8, src, (size_t)ld * 8, (size_t)(D.nx + 4) * 8, D.ny + 4,
                      is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, L->ctx->stream);
    if (!is_device) cudaStreamSynchronize(L->ctx->stream);
    return gc_cuda_check(L->ctx, "gc_level_set_field");
}

extern "C" int gc_level_get_field(const gc_level *L, int p, int field, int which, double *dst, int is_device, int64_t ld)
{
    if (!L || p < 0 || p >= L->np || field < 0 || field > 3 || !dst || ld < L->pat[p].nx + 4) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_get_field: bad argument");
    const PatchDesc &D = L->hpat[p];
    const double *src = plane_of(L, field, which) + D.off;
    cudaMemcpy2DAsync(dst, (size_t)ld * 8, src, (size_t)D.pitch * 8, (size_t)(D.nx + 4) * 8, D.ny + 4,
                      is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, L->ctx->stream);
    if (!is_device) cudaStreamSynchronize(L->ctx->stream);
    return gc_cuda_check(L->ctx, "gc_level_get_field");
}

extern "C" int gc_level_set_global(gc_level *L, int field, const double *src, int is_device, int64_t ld,
                                   int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    if (!L || field < 0 || field > 3 || !src || gnx < 1 || gny < 1 || ld < gnx) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_set_global: bad argument");
    gc_ctx *c = L->ctx;
    const double *dsrc = src; int64_t dld = ld; double *tmp = nullptr; bool transient = false;
    if (!is_device) {
        tmp = (double *)gc_stage_get(c, (size_t)gnx * gny * 8, &transient);
        if (!tmp) return gc_fail(c, GC_ERR_NOMEM, "gc_level_set_global: staging allocation failed");
        cudaMemcpy2DAsync(tmp, (size_t)gnx * 8, src, (size_t)ld * 8, (size_t)gnx * 8, gny, cudaMemcpyHostToDevice, c->stream);
        dsrc = tmp; dld = gnx;
    }
    gc_launch_set_global(L, plane_of(L, field, GC_NEW), dsrc, dld, gi0, gj0, gnx, gny);
    if (tmp) { cudaStreamSynchronize(c->stream); if (transient) gc_dev_free(c, tmp); }   // the caller's array is free on return
    return gc_cuda_check(c, "gc_level_set_global");
}

extern "C" int gc_level_set_patches(gc_level *L, int field, const double *src, int is_device)
{
    if (!L || field < 0 || field > 3 || !src) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_set_patches: bad argument");
    gc_ctx *c = L->ctx;
    if (!L->d_goff) {                                 // packed layout: patch p starts at the sum of (nx + 4)(ny + 4) of the patches before it
        std::vector<int64_t> goff((size_t)std::max(L->np, 1));
        int64_t o = 0;
        for (int p = 0; p < L->np; p++) { goff[(size_t)p] = o; o += (int64_t)(L->pat[p].nx + 4) * (L->pat[p].ny + 4); }
        L->gtot = o;
        L->d_goff = (int64_t *)gc_dev_alloc(c, goff.size() * sizeof(int64_t));
        if (!L->d_goff) return gc_fail(c, GC_ERR_NOMEM, "gc_level_set_patches: table allocation failed");
        L->allocs.push_back(L->d_goff);
        cudaMemcpyAsync(L->d_goff, goff.data(), goff.size() * sizeof(int64_t), cudaMemcpyHostToDevice, c->stream);
        cudaStreamSynchronize(c->stream);
    }
    const double *dsrc = src; double *tmp = nullptr; bool transient = false;
    if (!is_device) {
        tmp = (double *)gc_stage_get(c, (size_t)std::max<int64_t>(L->gtot, 1) * 8, &transient);
        if (!tmp) return gc_fail(c, GC_ERR_NOMEM, "gc_level_set_patches: staging allocation failed");
        cudaMemcpyAsync(tmp, src, (size_t)L->gtot * 8, cudaMemcpyHostToDevice, c->stream);
        dsrc = tmp;
    }
    gc_launch_set_patches(L, plane_of(L, field, GC_NEW), L->d_goff, dsrc);
    if (tmp) { cudaStreamSynchronize(c->stream); if (transient) gc_dev_free(c, tmp); }   // the caller's array is free on return
    return gc_cuda_check(c, "gc_level_set_patches");
}

// ---- asynchronous whole-level state transfer (copies overlapped with kernels)
static int xfer_prepare(gc_level *L, bool up)
{
    gc_ctx *c = L->ctx;
    double **st = up ? L->xfer_up : L->xfer_dn;
    if (!st[0]) {
        const size_t bytes = (size_t)L->nxl * (size_t)L->nyl * 8;
        for (int f = 0; f < 3; f++) {
            st[f] = (double *)gc_dev_alloc(c, bytes);
            if (!st[f]) return gc_fail(c, GC_ERR_NOMEM, "state transfer: staging allocation failed");
            L->allocs.push_back(st[f]);
        }
    }
    cudaEvent_t *ev[2] = { up ? &L->ev_up_copied : &L->ev_dn_ready, up ? &L->ev_up_free : &L->ev_dn_free };
    for (int k = 0; k < 2; k++)
        if (!*ev[k] && cudaEventCreateWithFlags(ev[k], cudaEventDisableTiming) != cudaSuccess) return gc_cuda_check(c, "state transfer: event");
    return GC_OK;
}

extern "C" int gc_level_upload_state_async(gc_level *L, const double *const host[3], void *copy_stream)
{
    if (!L || !host || !host[0] || !host[1] || !host[2]) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_upload_state_async: bad argument");
    gc_ctx *c = L->ctx;
    const bool first = L->xfer_up[0] == nullptr;
    int rc = xfer_prepare(L, true);
    if (rc) return rc;
    cudaStream_t cs = (cudaStream_t)copy_stream;
    const size_t bytes = (size_t)L->nxl * (size_t)L->nyl * 8;
    if (!first) cudaStreamWaitEvent(cs, L->ev_up_free, 0);          // the previous upload's scatter has read the staging planes
    for (int f = 0; f < 3; f++) cudaMemcpyAsync(L->xfer_up[f], host[f], bytes, cudaMemcpyHostToDevice, cs);
    cudaEventRecord(L->ev_up_copied, cs);
    cudaStreamWaitEvent(c->stream, L->ev_up_copied, 0);
    for (int f = 0; f < 3; f++) gc_launch_set_global(L, L->q[L->cur][f], L->xfer_up[f], L->nxl, 0, 0, L->nxl, L->nyl);
    cudaEventRecord(L->ev_up_free, c->stream);
    return gc_cuda_check(c, "gc_level_upload_state_async");
}

extern "C" int gc_level_download_state_async(gc_level *L, double *const host[3], void *copy_stream)
{
    if (!L || !host || !host[0] || !host[1] || !host[2]) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_download_state_async: bad argument");
    gc_ctx *c = L->ctx;
    const bool first = L->xfer_dn[0] == nullptr;
    int rc = xfer_prepare(L, false);
    if (rc) return rc;
    cudaStream_t cs = (cudaStream_t)copy_stream;
    const size_t bytes = (size_t)L->nxl * (size_t)L->nyl * 8;
    if (!first) cudaStreamWaitEvent(c->stream, L->ev_dn_free, 0);   // the previous download's copies have left the staging planes
    for (int f = 0; f < 3; f++) {
        if (L->ncells != L->nxl * L->nyl) cudaMemsetAsync(L->xfer_dn[f], 0, bytes, c->stream);   // cells no patch covers read as 0
        gc_launch_get_global(L, L->q[L->cur][f], L->xfer_dn[f], L->nxl, 0, 0, L->nxl, L->nyl);
    }
    cudaEventRecord(L->ev_dn_ready, c->stream);
    cudaStreamWaitEvent(cs, L->ev_dn_ready, 0);
    for (int f = 0; f < 3; f++) cudaMemcpyAsync(host[f], L->xfer_dn[f], bytes, cudaMemcpyDeviceToHost, cs);
    cudaEventRecord(L->ev_dn_free, cs);
    return gc_cuda_check(c, "gc_level_download_state_async");
}

extern "C" int gc_level_get_global(const gc_level *L, int field, int which, double *dst, int is_device, int64_t ld,
                                   int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny)
{
    if (!L || field < 0 || field > 3 || !dst || gnx < 1 || gny < 1 || ld < gnx) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_get_global: bad argument");
    gc_ctx *c = L->ctx;
    double *ddst = dst; int64_t dld = ld; double *tmp = nullptr; bool transient = false;
    if (!is_device) {
        tmp = (double *)gc_stage_get(c, (size_t)gnx * gny * 8, &transient);
        if (!tmp) return gc_fail(c, GC_ERR_NOMEM, "gc_level_get_global: staging allocation failed");
        // cells not covered by a patch keep the caller's values
        cudaMemcpy2DAsync(tmp, (size_t)gnx * 8, dst, (size_t)ld * 8, (size_t)gnx * 8, gny, cudaMemcpyHostToDevice, c->stream);
        ddst = tmp; dld = gnx;
    }
    gc_launch_get_global(L, plane_of(L, field, which), ddst, dld, gi0, gj0, gnx, gny);
    if (tmp) {
        cudaMemcpy2DAsync(dst, (size_t)ld * 8, tmp, (size_t)gnx * 8, (size_t)gnx * 8, gny, cudaMemcpyDeviceToHost, c->stream);
        cudaStreamSynchronize(c->stream);
        if (transient) gc_dev_free(c, tmp);
    }
    return gc_cuda_check(c, "gc_level_get_global");
}

extern "C" int gc_fill_ghost_b(gc_level *L)
{
    if (!L) return GC_ERR_BADARG;
    gc_launch_copy_rects(L, L->b, nullptr, nullptr, 1, false);
    gc_launch_bc(L, L->b, nullptr, nullptr, 1, 0);
    return gc_cuda_check(L->ctx, "gc_fill_ghost_b");
}

extern "C" int gc_bathy_update(gc_level *L, const gc_deform *D, double w)
{
    if (!L || !D || !D->dz || D->mx < 2 || D->my < 2 || !(D->ddx > 0.0) || !(D->ddy > 0.0) || !(w == w))
        return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_bathy_update: bad argument");
    gc_ctx *c = L->ctx;
    const double *dz = D->dz; double *tmp = nullptr; bool transient = false;
    const size_t bytes = (size_t)D->mx * (size_t)D->my * 8;
    if (!D->dz_is_device) {
        tmp = (double *)gc_stage_get(c, bytes, &transient);
        if (!tmp) return gc_fail(c, GC_ERR_NOMEM, "gc_bathy_update: staging allocation failed");
        cudaMemcpyAsync(tmp, D->dz, bytes, cudaMemcpyHostToDevice, c->stream);
        dz = tmp;
    }
    gc_launch_bathy_update(L, D->x0, D->y0, D->ddx, D->ddy, D->mx, D->my, dz, w);
    if (tmp) { cudaStreamSynchronize(c->stream); if (transient) gc_dev_free(c, tmp); }   // the caller's array is free on return
    return gc_cuda_check(c, "gc_bathy_update");
}

int gc_fill_coarse_ghosts(gc_level *L, const gc_level *C, double alpha);   // gc_api_amr.cu
void gc_amr_on_destroy(gc_level *L);                                       // gc_api_amr.cu
int gc_flux_after_step(gc_level *L, double dt, const double *dt_dev);     // gc_api_amr.cu

static int fill_ghost(gc_level *L, const gc_level *coarser, double alpha, bool for_step)
{
    if (!L) return GC_ERR_BADARG;
    double **q = L->q[L->cur];
    // for_step: only the rectangles a sweep line of the split step reads.  A flux register reads ghost cells of its own, and then
    // the x-sweep takes every ghost row (gc_launch_sweeps): everything is filled.
    const bool regs = (L->nreg > 0 && L->reg_fine) || L->reg_coarse;
    gc_launch_copy_rects(L, q[0], q[1], q[2], 3, for_step && !regs);
    if (coarser) {
        int rc = gc_fill_coarse_ghosts(L, coarser, alpha);
        if (rc) return rc;
    } else if (!L->coarse_ghost.empty()) {
        return gc_fail(L->ctx, GC_ERR_STATE, "gc_fill_ghost: ghost cells need a coarser level");
    }
    gc_launch_bc(L, q[0], q[1], q[2], 3, 1);
    return gc_cuda_check(L->ctx, "gc_fill_ghost");
}

extern "C" int gc_fill_ghost(gc_level *L, const gc_level *coarser, double alpha) { return fill_ghost(L, coarser, alpha, false); }
extern "C" int gc_fill_ghost_step(gc_level *L, const gc_level *coarser, double alpha) { return fill_ghost(L, coarser, alpha, true); }

extern "C" int gc_level_stats(const gc_level *L, gc_step_stats *out)
{
    if (!L || !out) return GC_ERR_BADARG;
    DevStats s;
    cudaMemcpyAsync(&s, L->d_stats, sizeof s, cudaMemcpyDeviceToHost, L->ctx->stream);
    cudaStreamSynchronize(L->ctx->stream);
    int rc = gc_cuda_check(L->ctx, "gc_level_stats");
    if (rc) return rc;
    double sdx; memcpy(&sdx, &s.sdx_bits, 8);
    out->s_over_dx_max = sdx; out->cfl_max = 0.0; out->clipped_mass = s.clipped; out->n_clipped = (int64_t)s.nclip; out->nan_seen = s.nan_seen;
    return GC_OK;
}

extern "C" int gc_level_sweep_cells(const gc_level *L, int64_t out[3])
{
    if (!L || !out) return GC_ERR_BADARG;
    for (int k = 0; k < 3; k++) out[k] = L->sweep_cells[k];
    return GC_OK;
}

extern "C" int gc_level_fallback_counts(const gc_level *L, int64_t out[4])
{
    if (!L || !out) return GC_ERR_BADARG;
    DevStats s;
    cudaMemcpyAsync(&s, L->d_stats, sizeof s, cudaMemcpyDeviceToHost, L->ctx->stream);
    cudaStreamSynchronize(L->ctx->stream);
    int rc = gc_cuda_check(L->ctx, "gc_level_fallback_counts");
    if (rc) return rc;
    out[0] = (int64_t)s.warp_iters; out[1] = (int64_t)s.fb_warp_iters; out[2] = (int64_t)s.fb_solves; out[3] = (int64_t)s.fb_fluxes;
    return GC_OK;
}

extern "C" int gc_level_step(gc_level *L, double dt, gc_step_stats *out)
{
    if (!L || !(dt >= 0.0)) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_step: bad argument");
    gc_launch_stats_reset(L);
    gc_launch_sweeps(L, dt, nullptr, dt > 0.0 ? 1 : 0);
    if (dt > 0.0) {
        L->cur = 1 - L->cur;
        int rc = gc_flux_after_step(L, dt, nullptr);
        if (rc) return rc;
    }
    int rc = gc_cuda_check(L->ctx, "gc_level_step");
    if (rc) return rc;
    if (out) {
        rc = gc_level_stats(L, out);
        if (rc) return rc;
        out->cfl_max = dt * out->s_over_dx_max;
        if (out->nan_seen) return gc_fail(L->ctx, GC_ERR_NAN, "gc_level_step: NaN in the updated state");
    }
    return GC_OK;
}

extern "C" int gc_level_stats_reset(gc_level *L)
{
    if (!L) return GC_ERR_BADARG;
    gc_launch_stats_reset(L);
    return gc_cuda_check(L->ctx, "gc_level_stats_reset");
}

extern "C" int gc_level_step_accum(gc_level *L, double dt)
{
    if (!L || !(dt > 0.0)) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_step_accum: bad argument");
    gc_launch_sweeps(L, dt, nullptr, 1);
    L->cur = 1 - L->cur;
    int rc = gc_flux_after_step(L, dt, nullptr);
    if (rc) return rc;
    return gc_cuda_check(L->ctx, "gc_level_step_accum");
}

extern "C" int gc_level_step_unsplit(gc_level *L, double dt, gc_step_stats *out)
{
    if (!L || !(dt >= 0.0)) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_step_unsplit: bad argument");
    if (L->reg_fine || L->reg_coarse) return gc_fail(L->ctx, GC_ERR_STATE, "gc_level_step_unsplit: flux registers are defined for the split step only");
    gc_launch_stats_reset(L);
    int rc = gc_launch_unsplit(L, dt, dt > 0.0 ? 1 : 0);
    if (rc) return gc_fail(L->ctx, rc, "gc_level_step_unsplit: scratch allocation failed");
    if (dt > 0.0) L->cur = 1 - L->cur;
    rc = gc_cuda_check(L->ctx, "gc_level_step_unsplit");
    if (rc) return rc;
    if (out) {
        rc = gc_level_stats(L, out);
        if (rc) return rc;
        out->cfl_max = dt * out->s_over_dx_max;
        if (out->nan_seen) return gc_fail(L->ctx, GC_ERR_NAN, "gc_level_step_unsplit: NaN in the updated state");
    }
    return GC_OK;
}

extern "C" int gc_level_step_auto(gc_level *L, double *dt_dev, double cfl_target)
{
    if (!L || !dt_dev || !(cfl_target > 0.0)) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_level_step_auto: bad argument");
    gc_launch_stats_reset(L);
    gc_launch_sweeps(L, 0.0, dt_dev, 1);
    L->cur = 1 - L->cur;
    int rc = gc_flux_after_step(L, 0.0, dt_dev);
    if (rc) return rc;
    gc_launch_next_dt(L, dt_dev, cfl_target);
    return gc_cuda_check(L->ctx, "gc_level_step_auto");
}

extern "C" int gc_wet_mask(const gc_level *L, uint8_t *mask, int is_device)
{
    if (!L || !mask) return GC_ERR_BADARG;
    gc_ctx *c = L->ctx;
    uint8_t *d = mask;
    if (!is_device) { d = (uint8_t *)gc_dev_alloc(c, (size_t)L->ncells); if (!d) return gc_fail(c, GC_ERR_NOMEM, "gc_wet_mask: allocation failed"); }
    gc_launch_wet_mask(L, d);
    if (!is_device) {
        cudaMemcpyAsync(mask, d, (size_t)L->ncells, cudaMemcpyDeviceToHost, c->stream);
        cudaStreamSynchronize(c->stream);
        gc_dev_free(c, d);
    }
    return gc_cuda_check(c, "gc_wet_mask");
}

extern "C" double gc_level_mass(const gc_level *L)
{
    if (!L) return NAN;
    gc_launch_mass(L);
    const int npart = L->np > 0 ? gc_mass_partials(L) : 0;
    std::vector<double> part((size_t)std::max(npart, 1), 0.0);
    cudaMemcpyAsync(part.data(), L->d_partial, sizeof(double) * npart, cudaMemcpyDeviceToHost, L->ctx->stream);
    cudaStreamSynchronize(L->ctx->stream);
    if (gc_cuda_check(L->ctx, "gc_level_mass")) return NAN;
    double m = 0.0;
    for (int p = 0; p < npart; p++) m += part[p];
    return m;
}

extern "C" int gc_selftest_math(gc_ctx *c, const double *a, const double *b, int64_t n, int64_t *nmismatch, int64_t *nfallback)
{
    if (!c || !a || !b || n < 0 || !nmismatch || !nfallback) return GC_ERR_BADARG;
    double *d = (double *)gc_dev_alloc(c, (size_t)(2 * n + 2) * 8);
    if (!d) return gc_fail(c, GC_ERR_NOMEM, "gc_selftest_math: allocation failed");
    unsigned long long *cnt = (unsigned long long *)(d + 2 * n), h[2] = {0, 0};
    cudaMemcpyAsync(d, a, (size_t)n * 8, cudaMemcpyHostToDevice, c->stream);
    cudaMemcpyAsync(d + n, b, (size_t)n * 8, cudaMemcpyHostToDevice, c->stream);
    cudaMemsetAsync(cnt, 0, 16, c->stream);
    gc_launch_math_selftest(c->stream, d, d + n, n, cnt);
    cudaMemcpyAsync(h, cnt, 16, cudaMemcpyDeviceToHost, c->stream);
    cudaStreamSynchronize(c->stream);
    gc_dev_free(c, d);
    *nmismatch = (int64_t)h[0]; *nfallback = (int64_t)h[1];
    return gc_cuda_check(c, "gc_selftest_math");
}

extern "C" int gc_probe_fp64_peak(gc_ctx *c, double *flops_out)
{
    if (!c || !flops_out) return GC_ERR_BADARG;
    double *d = (double *)gc_dev_alloc(c, 64);
    if (!d) return gc_fail(c, GC_ERR_NOMEM, "gc_probe_fp64_peak: allocation failed");
    int dev = 0, nsm = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
    const int iters = 1 << 16, threads = 512, blocks = nsm * 4;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    gc_launch_fp64_probe(c->stream, d, 1024, blocks, threads);   // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3; rep++) {
        cudaEventRecord(e0, c->stream);
        gc_launch_fp64_probe(c->stream, d, iters, blocks, threads);
        cudaEventRecord(e1, c->stream);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    gc_dev_free(c, d);
    int rc = gc_cuda_check(c, "gc_probe_fp64_peak");
    if (rc) return rc;
    *flops_out = 2.0 * 8.0 * (double)iters * threads * blocks / (best * 1e-3);
    return GC_OK;
}
