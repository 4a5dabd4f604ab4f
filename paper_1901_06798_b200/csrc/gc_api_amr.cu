// gc_api_amr.cu -- level-transfer entry points (A3, A8-A11): host list building + launches.
// The host only intersects boxes and builds index lists (bookkeeping); every value is computed in gc_amr.cu.
#include <math.h>
#include <string.h>
#include <algorithm>
#include <map>
#include "gc_internal.h"

struct Box { int64_t x0, y0, x1, y1; };   // half-open [x0,x1) x [y0,y1)

template <class T> static T *upload_tmp(gc_ctx *c, const std::vector<T> &v)
{
    T *d = (T *)gc_dev_alloc(c, std::max<size_t>(v.size(), 1) * sizeof(T));
    if (d && !v.empty()) cudaMemcpyAsync(d, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, c->stream);
    return d;
}

static void drop_alloc(gc_level *L, void *p)
{
    if (!p) return;
    auto it = std::find(L->allocs.begin(), L->allocs.end(), p);
    if (it != L->allocs.end()) L->allocs.erase(it);
    gc_dev_free(L->ctx, p);
}

// patches of L whose interior intersects the box (each once)
static void patches_in(const gc_level *L, const Box &b, std::vector<int32_t> &out)
{
    out.clear();
    int64_t x0 = std::max<int64_t>(b.x0, 0), x1 = std::min<int64_t>(b.x1, L->nxl), y0 = std::max<int64_t>(b.y0, 0), y1 = std::min<int64_t>(b.y1, L->nyl);
    if (x0 >= x1 || y0 >= y1) return;
    for (int64_t by = y0 / L->bsize; by <= (y1 - 1) / L->bsize; by++)
        for (int64_t bx = x0 / L->bsize; bx <= (x1 - 1) / L->bsize; bx++) {
            auto it = L->buckets.find((bx << 32) ^ (by & 0xffffffffll));
            if (it == L->buckets.end()) continue;
            for (int32_t q : it->second) {
                const gc_patch &Q = L->pat[q];
                if (std::max<int64_t>(x0, Q.i0) < std::min<int64_t>(x1, (int64_t)Q.i0 + Q.nx) &&
                    std::max<int64_t>(y0, Q.j0) < std::min<int64_t>(y1, (int64_t)Q.j0 + Q.ny) &&
                    std::find(out.begin(), out.end(), q) == out.end()) out.push_back(q);
            }
        }
    std::sort(out.begin(), out.end());
}

// a box of FINE cells inside fine patch p -> coarse-fill rectangles, one per coarse patch under it.  false: not nested.
static bool add_fill_rects(const gc_level *L, int p, const Box &b, const gc_level *C, std::vector<CoarseFillRect> &rects,
                           std::vector<int64_t> &start, int64_t &ncells)
{
    const int r = L->ratio;
    const PatchDesc &D = L->hpat[p];
    Box cb{ b.x0 / r, b.y0 / r, (b.x1 - 1) / r + 1, (b.y1 - 1) / r + 1 };
    std::vector<int32_t> cps;
    patches_in(C, cb, cps);
    int64_t covered = 0;
    for (int32_t cp : cps) {
        const gc_patch &Q = C->pat[cp];
        const PatchDesc &DQ = C->hpat[cp];
        int64_t x0 = std::max<int64_t>(b.x0, (int64_t)Q.i0 * r), x1 = std::min<int64_t>(b.x1, ((int64_t)Q.i0 + Q.nx) * r);
        int64_t y0 = std::max<int64_t>(b.y0, (int64_t)Q.j0 * r), y1 = std::min<int64_t>(b.y1, ((int64_t)Q.j0 + Q.ny) * r);
        if (x0 >= x1 || y0 >= y1) continue;
        CoarseFillRect R;
        R.dst = D.off + (y0 - D.j0 + 2) * D.pitch + (x0 - D.i0 + 2);
        int64_t I0 = x0 / r, J0 = y0 / r;
        R.csrc = DQ.off + (J0 - Q.j0 + 2) * DQ.pitch + (I0 - Q.i0 + 2);
        R.dpitch = D.pitch; R.cpitch = DQ.pitch; R.w = (int32_t)(x1 - x0); R.h = (int32_t)(y1 - y0);
        R.ii0 = (int32_t)(x0 - I0 * r); R.jj0 = (int32_t)(y0 - J0 * r);
        rects.push_back(R); start.push_back(ncells);
        ncells += (int64_t)R.w * R.h; covered += (int64_t)R.w * R.h;
    }
    return covered == (b.x1 - b.x0) * (b.y1 - b.y0);
}

// A3: ghost cells of L without a same-level source <- coarser level C at time fraction alpha
int gc_fill_coarse_ghosts(gc_level *L, const gc_level *C, double alpha)
{
    if (L->coarse_ghost.empty()) return GC_OK;
    if (C->ctx != L->ctx || L->ratio < 1) return gc_fail(L->ctx, GC_ERR_BADARG, "gc_fill_ghost: coarser level of another context");
    if (L->cf_for != C || L->cf_gen != C->gen) {
        std::vector<CoarseFillRect> rects; std::vector<int64_t> start; int64_t ncells = 0;
        const size_t n = L->coarse_ghost.size();
        size_t k = 0;
        while (k < n) {   // runs of consecutive ghost cells in one row of one patch
            size_t e = k + 1;
            while (e < n && L->coarse_ghost[e] == L->coarse_ghost[e - 1] + 1 && L->coarse_ghost_ij[2 * e + 1] == L->coarse_ghost_ij[2 * k + 1] &&
                   L->coarse_ghost_ij[2 * e] == L->coarse_ghost_ij[2 * (e - 1)] + 1) e++;
            // the run lies in one fine patch; recover it from the offset
            int64_t gi0 = L->coarse_ghost_ij[2 * k], gj = L->coarse_ghost_ij[2 * k + 1];
            int p = (int)(std::upper_bound(L->hpat.begin(), L->hpat.end(), L->coarse_ghost[k],
                                           [](int64_t o, const PatchDesc &d) { return o < d.off; }) - L->hpat.begin()) - 1;
            Box b{ gi0, gj, gi0 + (int64_t)(e - k), gj + 1 };
            if (!add_fill_rects(L, p, b, C, rects, start, ncells))
                return gc_fail(L->ctx, GC_ERR_STATE, "gc_fill_ghost: fine level not properly nested in the coarser level");
            k = e;
        }
        drop_alloc(L, L->d_cf); drop_alloc(L, L->d_cfstart);
        L->d_cf = upload_tmp(L->ctx, rects); L->d_cfstart = upload_tmp(L->ctx, start);
        if (!L->d_cf || !L->d_cfstart) return gc_fail(L->ctx, GC_ERR_NOMEM, "gc_fill_ghost: list allocation failed");
        L->allocs.push_back(L->d_cf); L->allocs.push_back(L->d_cfstart);
        cudaStreamSynchronize(L->ctx->stream);
        L->ncf = (int)rects.size(); L->ncfcells = ncells; L->cf_for = C; L->cf_gen = C->gen;
    }
    gc_launch_coarse_fill(L, C, L->d_cf, L->d_cfstart, L->ncf, L->ncfcells, alpha, 1, GC_SLOT_COARSE);
    return GC_OK;
}

// A8: accumulate into the registers after a step of L (as the coarse side of its own registers, as the fine side of its
// coarser level's registers)
int gc_flux_after_step(gc_level *L, double dt, const double *dt_dev)
{
    if (L->nreg > 0 && L->reg_fine) gc_launch_flux_coarse(L, dt, dt_dev);
    if (L->reg_coarse && L->reg_coarse->reg_fine == L) gc_launch_flux_fine(L, dt, dt_dev);
    return GC_OK;
}

void gc_amr_on_destroy(gc_level *L)
{
    if (L->reg_fine) { gc_level *F = const_cast<gc_level *>(L->reg_fine); if (F->reg_coarse == L) F->reg_coarse = nullptr; }
    if (L->reg_coarse && L->reg_coarse->reg_fine == L) { L->reg_coarse->reg_fine = nullptr; L->reg_coarse->nreg = 0; L->reg_coarse->nfix = 0; }
}

// b minus c -> up to four boxes appended to out
static void subtract(const Box &b, const Box &c, std::vector<Box> &out)
{
    int64_t x0 = std::max(b.x0, c.x0), x1 = std::min(b.x1, c.x1), y0 = std::max(b.y0, c.y0), y1 = std::min(b.y1, c.y1);
    if (x0 >= x1 || y0 >= y1) { out.push_back(b); return; }
    if (b.y0 < y0) out.push_back(Box{ b.x0, b.y0, b.x1, y0 });
    if (y1 < b.y1) out.push_back(Box{ b.x0, y1, b.x1, b.y1 });
    if (b.x0 < x0) out.push_back(Box{ b.x0, y0, x0, y1 });
    if (x1 < b.x1) out.push_back(Box{ x1, y0, b.x1, y1 });
}

// A11: interior of N <- old fine level O where it overlapped, else interpolation from C's current buffer
extern "C" int gc_level_init_from(gc_level *N, const gc_level *O, const gc_level *C)
{
    if (!N || !C || N->ctx != C->ctx || (O && O->ctx != N->ctx)) return gc_fail(N ? N->ctx : nullptr, GC_ERR_BADARG, "gc_level_init_from: bad argument");
    gc_ctx *ctx = N->ctx;
    std::vector<CopyRect> copies;
    std::vector<CoarseFillRect> rects; std::vector<int64_t> start; int64_t ncells = 0;
    std::vector<int32_t> qs;
    std::vector<Box> rest, next;
    for (int p = 0; p < N->np; p++) {
        const gc_patch &P = N->pat[p];
        const PatchDesc &D = N->hpat[p];
        Box pb{ P.i0, P.j0, (int64_t)P.i0 + P.nx, (int64_t)P.j0 + P.ny };
        rest.assign(1, pb);
        if (O) {
            patches_in(O, pb, qs);
            for (int32_t q : qs) {
                const gc_patch &Q = O->pat[q];
                const PatchDesc &DQ = O->hpat[q];
                Box qb{ Q.i0, Q.j0, (int64_t)Q.i0 + Q.nx, (int64_t)Q.j0 + Q.ny };
                int64_t x0 = std::max(pb.x0, qb.x0), x1 = std::min(pb.x1, qb.x1), y0 = std::max(pb.y0, qb.y0), y1 = std::min(pb.y1, qb.y1);
                CopyRect r;
                r.dst = D.off + (y0 - P.j0 + 2) * D.pitch + (x0 - P.i0 + 2);
                r.src = DQ.off + (y0 - Q.j0 + 2) * DQ.pitch + (x0 - Q.i0 + 2);
                r.w = (int)(x1 - x0); r.h = (int)(y1 - y0); r.dpitch = D.pitch; r.spitch = DQ.pitch;
                copies.push_back(r);
                next.clear();
                for (const Box &b : rest) subtract(b, qb, next);
                rest.swap(next);
            }
        }
        for (const Box &b : rest)
            if (!add_fill_rects(N, p, b, C, rects, start, ncells))
                return gc_fail(ctx, GC_ERR_STATE, "gc_level_init_from: new level not properly nested in the coarser level");
    }
    CopyRect *d_copies = upload_tmp(ctx, copies);
    CoarseFillRect *d_rects = upload_tmp(ctx, rects);
    int64_t *d_start = upload_tmp(ctx, start);
    int rc = GC_OK;
    if (!d_copies || !d_rects || !d_start) rc = gc_fail(ctx, GC_ERR_NOMEM, "gc_level_init_from: list allocation failed");
    else {
        if (O) gc_launch_copy_overlap(N, O, d_copies, (int)copies.size());
        gc_launch_coarse_fill(N, C, d_rects, d_start, (int)rects.size(), ncells, 1.0, 0, GC_SLOT_AVG);
        cudaStreamSynchronize(ctx->stream);
        rc = gc_cuda_check(ctx, "gc_level_init_from");
    }
    gc_dev_free(ctx, d_copies); gc_dev_free(ctx, d_rects); gc_dev_free(ctx, d_start);
    return rc;
}

// A9: covered coarse cells <- average of the fine cells on top
extern "C" int gc_average_down(gc_level *C, const gc_level *F)
{
    if (!C || !F || C->ctx != F->ctx) return gc_fail(C ? C->ctx : nullptr, GC_ERR_BADARG, "gc_average_down: bad argument");
    gc_ctx *ctx = C->ctx;
    if (C->avg_gen != F->gen) {
        const int r = F->ratio;
        std::vector<AvgRect> rects; std::vector<int64_t> start; int64_t ncells = 0;
        std::vector<int32_t> cps;
        for (int p = 0; p < F->np; p++) {
            const gc_patch &P = F->pat[p];
            const PatchDesc &D = F->hpat[p];
            Box cb{ P.i0 / r, P.j0 / r, ((int64_t)P.i0 + P.nx) / r, ((int64_t)P.j0 + P.ny) / r };
            patches_in(C, cb, cps);
            int64_t covered = 0;
            for (int32_t cp : cps) {
                const gc_patch &Q = C->pat[cp];
                const PatchDesc &DQ = C->hpat[cp];
                int64_t x0 = std::max<int64_t>(cb.x0, Q.i0), x1 = std::min<int64_t>(cb.x1, (int64_t)Q.i0 + Q.nx);
                int64_t y0 = std::max<int64_t>(cb.y0, Q.j0), y1 = std::min<int64_t>(cb.y1, (int64_t)Q.j0 + Q.ny);
                if (x0 >= x1 || y0 >= y1) continue;
                AvgRect R;
                R.cdst = DQ.off + (y0 - Q.j0 + 2) * DQ.pitch + (x0 - Q.i0 + 2);
                R.fsrc = D.off + (y0 * r - P.j0 + 2) * D.pitch + (x0 * r - P.i0 + 2);
                R.cpitch = DQ.pitch; R.fpitch = D.pitch; R.w = (int32_t)(x1 - x0); R.h = (int32_t)(y1 - y0);
                R.frow = (int32_t)(y0 * r + 2); R.pad = 0;
                rects.push_back(R); start.push_back(ncells);
                ncells += (int64_t)R.w * R.h; covered += (int64_t)R.w * R.h;
            }
            if (covered != (cb.x1 - cb.x0) * (cb.y1 - cb.y0))
                return gc_fail(ctx, GC_ERR_STATE, "gc_average_down: fine level not properly nested in the coarser level");
        }
        drop_alloc(C, C->d_avg); drop_alloc(C, C->d_avgstart);
        C->d_avg = upload_tmp(ctx, rects); C->d_avgstart = upload_tmp(ctx, start);
        if (!C->d_avg || !C->d_avgstart) return gc_fail(ctx, GC_ERR_NOMEM, "gc_average_down: list allocation failed");
        C->allocs.push_back(C->d_avg); C->allocs.push_back(C->d_avgstart);
        cudaStreamSynchronize(ctx->stream);
        C->navg = (int)rects.size(); C->navgcells = ncells; C->avg_gen = F->gen;
    }
    gc_launch_average_down(C, F, C->d_avg, C->d_avgstart, C->navg, C->navgcells);
    return gc_cuda_check(ctx, "gc_average_down");
}

// A10
extern "C" int gc_flag_cells(const gc_level *Lc, const gc_flag_params *fp, double t, uint8_t *flags, int is_device, int64_t *nflag)
{
    if (!Lc || !fp || !flags || fp->nboxes < 0 || (fp->nboxes > 0 && !fp->boxes)) return gc_fail(Lc ? Lc->ctx : nullptr, GC_ERR_BADARG, "gc_flag_cells: bad argument");
    gc_level *L = const_cast<gc_level *>(Lc);     // the cached neighbour lists live in the level
    gc_ctx *ctx = L->ctx;
    if (nflag) *nflag = 0;
    if (L->ncells == 0) return GC_OK;
    const int bw = fp->buffer > 0 ? fp->buffer : 0;
    if (L->nbr_buffer != bw || !L->d_nbrstart) {
        std::vector<int32_t> nstart(L->np + 1, 0), nlist, qs;
        for (int p = 0; p < L->np; p++) {
            const gc_patch &P = L->pat[p];
            Box gb{ (int64_t)P.i0 - bw, (int64_t)P.j0 - bw, (int64_t)P.i0 + P.nx + bw, (int64_t)P.j0 + P.ny + bw };
            patches_in(L, gb, qs);
            for (int32_t q : qs) if (q != p) nlist.push_back(q);
            nstart[p + 1] = (int32_t)nlist.size();
        }
        drop_alloc(L, L->d_nbrstart); drop_alloc(L, L->d_nbrlist);
        L->d_nbrstart = upload_tmp(ctx, nstart); L->d_nbrlist = upload_tmp(ctx, nlist);
        if (!L->d_nbrstart || !L->d_nbrlist) return gc_fail(ctx, GC_ERR_NOMEM, "gc_flag_cells: list allocation failed");
        L->allocs.push_back(L->d_nbrstart); L->allocs.push_back(L->d_nbrlist);
        cudaStreamSynchronize(ctx->stream);
        L->nbr_buffer = bw;
    }
    std::vector<double> boxes(fp->boxes, fp->boxes + 6 * (size_t)fp->nboxes);
    double *d_boxes = upload_tmp(ctx, boxes);
    // scratch: raw flags, (host output: flags), counter
    uint8_t *d_raw = (uint8_t *)gc_dev_alloc(ctx, (size_t)L->ncells);
    uint8_t *d_flags = is_device ? flags : (uint8_t *)gc_dev_alloc(ctx, (size_t)L->ncells);
    unsigned long long *d_count = (unsigned long long *)gc_dev_alloc(ctx, 8);
    int rc = GC_OK;
    if (!d_boxes || !d_raw || !d_flags || !d_count) rc = gc_fail(ctx, GC_ERR_NOMEM, "gc_flag_cells: allocation failed");
    else {
        cudaMemsetAsync(d_count, 0, 8, ctx->stream);
        gc_launch_flags(L, fp, d_boxes, t, d_raw, d_flags, L->d_nbrstart, L->d_nbrlist, d_count);
        unsigned long long cnt = 0;
        cudaMemcpyAsync(&cnt, d_count, 8, cudaMemcpyDeviceToHost, ctx->stream);
        if (!is_device) cudaMemcpyAsync(flags, d_flags, (size_t)L->ncells, cudaMemcpyDeviceToHost, ctx->stream);
        cudaStreamSynchronize(ctx->stream);
        rc = gc_cuda_check(ctx, "gc_flag_cells");
        if (nflag) *nflag = (int64_t)cnt;
    }
    gc_dev_free(ctx, d_boxes); gc_dev_free(ctx, d_raw); gc_dev_free(ctx, d_count);
    if (!is_device) gc_dev_free(ctx, d_flags);
    return rc;
}

// A8: registers on the boundary of the fine region, in the order fine patch / side xlo, xhi, ylo, yhi / position
extern "C" int gc_flux_attach(gc_level *C, gc_level *F)
{
    if (!C || !F || C->ctx != F->ctx || C == F) return gc_fail(C ? C->ctx : nullptr, GC_ERR_BADARG, "gc_flux_attach: bad argument");
    gc_ctx *ctx = C->ctx;
    const int r = F->ratio;
    if (r < 1 || r > 128) return gc_fail(ctx, GC_ERR_BADARG, "gc_flux_attach: refinement ratio outside 1..128");
    std::vector<FluxReg> regs;
    for (int p = 0; p < F->np; p++) {
        const gc_patch &P = F->pat[p];
        const PatchDesc &D = F->hpat[p];
        const int64_t I0 = P.i0 / r, I1 = ((int64_t)P.i0 + P.nx) / r, J0 = P.j0 / r, J1 = ((int64_t)P.j0 + P.ny) / r;
        for (int side = 0; side < 4; side++) {
            const int dir = side / 2;
            const int64_t n = dir == 0 ? J1 - J0 : I1 - I0;
            for (int64_t m = 0; m < n; m++) {
                int64_t I, J;
                if (side == 0) { I = I0 - 1; J = J0 + m; } else if (side == 1) { I = I1; J = J0 + m; }
                else if (side == 2) { I = I0 + m; J = J0 - 1; } else { I = I0 + m; J = J1; }
                if (I < 0 || J < 0 || I >= C->nxl || J >= C->nyl) continue;      // physical boundary
                if (gc_find_patch_host(F, I * r, J * r) >= 0) continue;           // fine-fine boundary
                const int cp = gc_find_patch_host(C, I, J);
                if (cp < 0) return gc_fail(ctx, GC_ERR_STATE, "gc_flux_attach: fine level not properly nested in the coarser level");
                const gc_patch &Q = C->pat[cp];
                const PatchDesc &DQ = C->hpat[cp];
                FluxReg R;
                const int ci = (int)(I - Q.i0 + 2), cj = (int)(J - Q.j0 + 2);
                R.ccell = DQ.off + (int64_t)cj * DQ.pitch + ci;
                R.cpitch = DQ.pitch; R.fpitch = D.pitch;
                R.crow = Q.j0 + cj;                                               // table index = global row + 2
                R.dir = dir;
                R.side = (side == 0 || side == 2) ? +1 : -1;                      // fine region on the high side of C for lo sides
                int fi, fj;
                if (side == 0) { fi = 2; fj = (int)(2 + m * r); }
                else if (side == 1) { fi = P.nx + 1; fj = (int)(2 + m * r); }
                else if (side == 2) { fi = (int)(2 + m * r); fj = 2; }
                else { fi = (int)(2 + m * r); fj = P.ny + 1; }
                R.fcell = D.off + (int64_t)fj * D.pitch + fi;
                R.frow = P.j0 + fj;
                regs.push_back(R);
            }
        }
    }
    // fix-up groups: registers of the same coarse cell, in list order; groups in order of first appearance
    std::map<int64_t, int> gid;
    std::vector<std::vector<int32_t>> groups;
    for (size_t n = 0; n < regs.size(); n++) {
        auto it = gid.find(regs[n].ccell);
        if (it == gid.end()) { gid[regs[n].ccell] = (int)groups.size(); groups.push_back({ (int32_t)n }); }
        else groups[it->second].push_back((int32_t)n);
    }
    std::vector<int32_t> fstart(1, 0), freg;
    for (auto &gr : groups) { for (int32_t n : gr) freg.push_back(n); fstart.push_back((int32_t)freg.size()); }

    // allocate the new arrays first and swap on success: a failed attach leaves the previous attachment as it was
    FluxReg *n_reg = upload_tmp(ctx, regs); int32_t *n_fixstart = upload_tmp(ctx, fstart), *n_fixreg = upload_tmp(ctx, freg);
    double *n_delta = (double *)gc_dev_alloc(ctx, std::max<size_t>(regs.size(), 1) * 3 * sizeof(double));
    double *n_base = (double *)gc_dev_alloc(ctx, std::max<size_t>(regs.size(), 1) * 4 * sizeof(double));
    if (!n_reg || !n_fixstart || !n_fixreg || !n_delta || !n_base) {
        cudaStreamSynchronize(ctx->stream);
        gc_dev_free(ctx, n_reg); gc_dev_free(ctx, n_fixstart); gc_dev_free(ctx, n_fixreg); gc_dev_free(ctx, n_delta); gc_dev_free(ctx, n_base);
        return gc_fail(ctx, GC_ERR_NOMEM, "gc_flux_attach: allocation failed");
    }
    drop_alloc(C, C->d_reg); drop_alloc(C, C->d_delta); drop_alloc(C, C->d_base); drop_alloc(C, C->d_fixstart); drop_alloc(C, C->d_fixreg);
    C->d_reg = n_reg; C->d_fixstart = n_fixstart; C->d_fixreg = n_fixreg; C->d_delta = n_delta; C->d_base = n_base;
    C->allocs.push_back(C->d_reg); C->allocs.push_back(C->d_fixstart); C->allocs.push_back(C->d_fixreg);
    C->allocs.push_back(C->d_delta); C->allocs.push_back(C->d_base);
    cudaMemsetAsync(C->d_delta, 0, std::max<size_t>(regs.size(), 1) * 3 * sizeof(double), ctx->stream);
    cudaMemsetAsync(C->d_base, 0, std::max<size_t>(regs.size(), 1) * 4 * sizeof(double), ctx->stream);
    cudaStreamSynchronize(ctx->stream);
    if (C->reg_fine && C->reg_fine != F) { gc_level *Fo = const_cast<gc_level *>(C->reg_fine); if (Fo->reg_coarse == C) Fo->reg_coarse = nullptr; }
    C->nreg = (int)regs.size(); C->nfix = (int)groups.size(); C->r_reg = r;
    C->reg_fine = F; F->reg_coarse = C;
    return gc_cuda_check(ctx, "gc_flux_attach");
}

extern "C" int gc_flux_fixup(gc_level *C, gc_level *F)
{
    if (!C || !F || C->reg_fine != F) return gc_fail(C ? C->ctx : nullptr, GC_ERR_BADARG, "gc_flux_fixup: levels are not attached");
    gc_launch_flux_fixup(C);
    return gc_cuda_check(C->ctx, "gc_flux_fixup");
}


// ---- gauges
extern "C" int gc_gauges_bind(gc_level *L, int n, const int32_t *patch, const double *xy)
{
    if (!L || n < 0 || (n > 0 && (!patch || !xy))) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_gauges_bind: bad argument");
    std::vector<GaugeLoc> loc((size_t)n);
    for (int k = 0; k < n; k++) {
        if (patch[k] < 0 || patch[k] >= L->np) return gc_fail(L->ctx, GC_ERR_BADARG, "gc_gauges_bind: no such patch");
        const PatchDesc &D = L->hpat[patch[k]];
        const double gx = (xy[2 * k] - L->xlo) / L->dx, gy = (xy[2 * k + 1] - L->ylo) / L->dy;
        if (!(gx >= (double)D.i0 && gx < (double)D.i0 + D.nx && gy >= (double)D.j0 && gy < (double)D.j0 + D.ny))
            return gc_fail(L->ctx, GC_ERR_BADARG, "gc_gauges_bind: gauge outside the interior of its patch");
        const int64_t ic = (int64_t)floor(gx), jc = (int64_t)floor(gy);       // the cell that contains the point
        const double xi = gx - 0.5, et = gy - 0.5;
        const int64_t i = (int64_t)floor(xi), j = (int64_t)floor(et);
        GaugeLoc &G = loc[(size_t)k];
        G.a = xi - (double)i; G.b = et - (double)j;
        G.pitch = D.pitch; G.pad = 0;
        G.c00 = D.off + (j - D.j0 + 2) * (int64_t)D.pitch + (i - D.i0 + 2);
        G.cc = D.off + (jc - D.j0 + 2) * (int64_t)D.pitch + (ic - D.i0 + 2);
    }
    if (L->d_gauge) { cudaStreamSynchronize(L->ctx->stream); drop_alloc(L, L->d_gauge); L->d_gauge = nullptr; }
    L->ngauge = 0;
    if (n > 0) {
        L->d_gauge = upload_tmp(L->ctx, loc);
        if (!L->d_gauge) return gc_fail(L->ctx, GC_ERR_NOMEM, "gc_gauges_bind: allocation failed");
        L->allocs.push_back(L->d_gauge);
        L->ngauge = n;
        cudaStreamSynchronize(L->ctx->stream);                                   // loc goes out of scope
    }
    return gc_cuda_check(L->ctx, "gc_gauges_bind");
}

extern "C" int gc_gauges_sample(const gc_level *L, double *out, int out_is_device)
{
    if (!L || (L->ngauge > 0 && !out)) return gc_fail(L ? L->ctx : nullptr, GC_ERR_BADARG, "gc_gauges_sample: bad argument");
    if (L->ngauge == 0) return GC_OK;
    gc_ctx *c = L->ctx;
    if (out_is_device) { gc_launch_gauges(L, out); return gc_cuda_check(c, "gc_gauges_sample"); }   // asynchronous
    bool transient = false;
    const size_t bytes = (size_t)L->ngauge * 4 * sizeof(double);
    double *d = (double *)gc_stage_get(c, bytes, &transient);
    if (!d) return gc_fail(c, GC_ERR_NOMEM, "gc_gauges_sample: staging allocation failed");
    gc_launch_gauges(L, d);
    cudaMemcpyAsync(out, d, bytes, cudaMemcpyDeviceToHost, c->stream);
    cudaStreamSynchronize(c->stream);
    if (transient) gc_dev_free(c, d);
    return gc_cuda_check(c, "gc_gauges_sample");
}
