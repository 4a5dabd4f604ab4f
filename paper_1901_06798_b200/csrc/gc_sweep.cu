// gc_sweep.cu -- x-sweep and y-sweep kernels (A5, A6) with the CFL max-reduction (A7).
//
// P:65-120 (eqs. 4-14) in f-wave form, DESIGN.md 3.4.  Two-pass variant: the x-sweep reads Q^n (ghosts
// filled) and writes Q* for columns 2..nx+1 on ALL rows; the y-sweep reads Q*, writes Q^{n+1} on the interior
// and applies the dry clean-up.  Thread <-> edge for the Riemann solve and the limiter, then thread <-> cell
// for the update (the paper's re-assignment), neighbour waves through shared memory.
//
// Two kernel families compute the same bits:
//  * k_sweep  (edge-parallel): thread <-> edge, neighbour waves through shared memory.  Much parallelism per
//    cell, used for small levels where the GPU would otherwise be empty.
//  * k_march  (line-marching): thread <-> line segment, walking along the sweep with the waves of the previous
//    edge, the primitive variables of the previous cell and the pending fluxes in registers.  No shared
//    memory, no barriers, each cell's primitive variables computed once, 3 redundant edges per segment only.
//    The x-sweep reads 4 cells of its row per 256-bit load (rows are 32-byte aligned); the y-sweep reads
//    one row of 32 adjacent columns per warp (coalesced).  Used for large levels (fp64-pipe bound).
#include "gc_internal.h"
#include "gc_scheme.cuh"

#define SW_BLOCK 256
#ifndef MARCH_BLOCK
#define MARCH_BLOCK 128
#endif
#ifndef MARCH_MINB
#define MARCH_MINB 3     // resident blocks per SM the register allocation is bounded for
#endif
#ifndef MARCH_UNROLL
#define MARCH_UNROLL 1
#endif
#define SW_YW 8       // columns per y-sweep block (8 doubles = 2 full 32-byte sectors per row access)

struct SweepArgs {
    const PatchDesc *pat;
    const SweepTile *tiles;
    const LineDesc *lines; int64_t nlines;
    const double *h, *hu, *hv, *b;   // input planes
    double *oh, *ohu, *ohv;          // output planes
    const double *rd;                // rdx (x-sweep) or rdy (y-sweep), per global row (+2)
    const double *ey;                // y edge factors per global edge (+2)
    double ex;
    double g, eps;
    double dt; const double *dt_dev; // dt_dev != NULL: read dt from device memory
    int coord, limiter, write_out;
    DevStats *stats;
    double dxdy;                     // dx*dy (cell area = kappa*dx*dy)
    const double *kappa;
};

__device__ __forceinline__ double warp_max(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        double w = __longlong_as_double(__shfl_xor_sync(0xffffffffu, __double_as_longlong(v), o));
        v = dmax(v, w);
    }
    return v;
}

template <int DIR>
__global__ void __launch_bounds__(SW_BLOCK) k_sweep(SweepArgs a)
{
    __shared__ double sZ[9][SW_BLOCK];
    __shared__ double sF[3][SW_BLOCK];
    __shared__ double sred[SW_BLOCK / 32];
    __shared__ unsigned long long sclip[SW_BLOCK / 32];
    __shared__ double sclipm[SW_BLOCK / 32];

    const SweepTile T = a.tiles[blockIdx.x];
    const PatchDesc pd = a.pat[T.patch];
    const int k = threadIdx.x;
    const int ne = T.nc + 3;                  // edges solved along the sweep
    int e, line, dk;
    bool active;
    if (DIR == 0) { int r = k / ne; e = k - r * ne; line = T.line0 + r; active = r < T.nlines; dk = 1; }
    else          { e = k / T.nlines; int ic = k - e * T.nlines; line = T.line0 + ic; active = e < ne; dk = T.nlines; }
    const int ce = T.c0 - 1 + e;              // storage index (along the sweep) of the cell right of / above this edge
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;

    Waves W;
    double (&Z)[3][3] = W.Z; double (&s)[3] = W.s;
    double rdR = 0.0, rdL = 0.0;              // 1/(kappa dx) of the right and the left cell of the edge
    int64_t idx = 0, str = 1;
    double qh = 0.0, qp = 0.0, qt = 0.0;      // state of the right cell (the one this thread updates)
    bool stdE = false;                        // "standard" edge: solved by the straight-line open-ocean code, s[0] < 0 < s[2]
    if (active) {
        RState L, R;
        if (DIR == 0) { idx = pd.off + (int64_t)line * pd.pitch + ce; str = 1; }
        else          { idx = pd.off + (int64_t)ce * pd.pitch + line; str = pd.pitch; }
        L.h = a.h[idx - str]; R.h = a.h[idx];
        L.b = a.b[idx - str]; R.b = a.b[idx];
        if (DIR == 0) { L.p = a.hu[idx - str]; L.t = a.hv[idx - str]; R.p = a.hu[idx]; R.t = a.hv[idx]; }
        else          { L.p = a.hv[idx - str]; L.t = a.hu[idx - str]; R.p = a.hv[idx]; R.t = a.hu[idx]; }
        qh = R.h; qp = R.p; qt = R.t;
        {   // straight-line code for an open-ocean edge first; any other edge is redone with the general code (same bits)
            MathFast mf;
            RState Lf = L, Rf = R;
            gc_prim_fast(mf, Lf, a.g, a.eps);
            gc_prim_fast(mf, Rf, a.g, a.eps);
            stdE = gc_riemann_fast(mf, a.g, a.eps, Lf, Rf, Z, s);
        }
        if (!stdE) {
            MathIeee mi;
            gc_prim(mi, L, a.g, a.eps);
            gc_prim(mi, R, a.g, a.eps);
            gc_riemann(mi, a.g, a.eps, L, R, Z, s);
        }
        if (DIR == 0) { rdR = a.rd[pd.j0 + line]; rdL = rdR; }
        else          { rdR = a.rd[pd.j0 + ce]; rdL = a.rd[pd.j0 + ce - 1]; }
        if (a.coord == 1) {                   // scale by the edge factor
            double ef = (DIR == 0) ? a.ex : a.ey[pd.j0 + ce];
#pragma unroll
            for (int w = 0; w < 3; w++) { s[w] = s[w] * ef; Z[w][0] = Z[w][0] * ef; Z[w][1] = Z[w][1] * ef; Z[w][2] = Z[w][2] * ef; }
        }
    } else {
        gc_waves_zero(W);
    }
#pragma unroll
    for (int w = 0; w < 3; w++) { sZ[3 * w + 0][k] = Z[w][0]; sZ[3 * w + 1][k] = Z[w][1]; sZ[3 * w + 2][k] = Z[w][2]; }
    __syncthreads();

    const bool limited = active && e >= 1 && e <= ne - 2;   // both neighbour edges are in this tile
    double fm[3] = {0.0, 0.0, 0.0}, fp[3] = {0.0, 0.0, 0.0};
    double cflm = 0.0;
    if (limited) {
        double zi[3];                                          // Z_I . Z_e with the upwind neighbour I of eq. 11
#pragma unroll
        for (int w = 0; w < 3; w++) {
            const int kn = (s[w] > 0.0) ? k - dk : k + dk;
            zi[w] = (sZ[3 * w + 0][kn] * Z[w][0] + sZ[3 * w + 1][kn] * Z[w][1]) + sZ[3 * w + 2][kn] * Z[w][2];
        }
        bool done = false;
        if (stdE) { MathFast mf; gc_edge_flux_std(mf, W, zi, zi, a.limiter, dt, rdL, rdR, fm, fp); done = !mf.failed(); }
        if (!done) { MathIeee mi; gc_edge_flux(mi, W, zi, zi, a.limiter, dt, rdL, rdR, fm, fp); }
        // eq. 15: right-going waves enter the right cell, left-going the left cell; interior lines only
        const bool count = (DIR == 1) || (line >= 2 && line < pd.ny + 2);
        if (count) cflm = stdE ? gc_edge_cfl_std(W, rdL, rdR) : gc_edge_cfl(W, rdL, rdR);
    }
    sF[0][k] = fm[0]; sF[1][k] = fm[1]; sF[2][k] = fm[2];
    __syncthreads();

    unsigned long long nclip = 0; double clipm = 0.0; int nanf = 0;
    if (limited && e <= ne - 3) {             // thread <-> cell ce: Q_c <- Q_c - dt rdx_c (fm_{c+1} - fp_c)
        double dtdx = dt * rdR;
        int kr = k + dk;
        double nh = qh - dtdx * (sF[0][kr] - fp[0]);
        double np_ = qp - dtdx * (sF[1][kr] - fp[1]);
        double nt = qt - dtdx * (sF[2][kr] - fp[2]);
        if (DIR == 0) {
            a.oh[idx] = nh; a.ohu[idx] = np_; a.ohv[idx] = nt;
        } else {
            if (nh < a.eps && a.write_out) {           // dry clean-up (S-9)
                if (nh < 0.0) { nclip = 1; clipm = (-nh) * (a.kappa[pd.j0 + ce] * a.dxdy); }
                nh = dmax(nh, 0.0); np_ = 0.0; nt = 0.0;
            }
            if (nh != nh || np_ != np_ || nt != nt) nanf = 1;
            if (a.write_out) { a.oh[idx] = nh; a.ohv[idx] = np_; a.ohu[idx] = nt; }
        }
    }

    // A7: exact, order-independent max: warp shuffle -> block -> one atomicMax on the bit image (values >= 0)
    cflm = warp_max(cflm);
    if (DIR == 1) {
        nclip = __reduce_add_sync(0xffffffffu, (unsigned)nclip);
        nanf = __any_sync(0xffffffffu, nanf);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) clipm += __shfl_xor_sync(0xffffffffu, clipm, o);
    }
    if ((k & 31) == 0) { sred[k >> 5] = cflm; if (DIR == 1) { sclip[k >> 5] = nclip; sclipm[k >> 5] = clipm; if (nanf) a.stats->nan_seen = 1; } }
    __syncthreads();
    if (k == 0) {
        double m = sred[0];
#pragma unroll
        for (int w = 1; w < SW_BLOCK / 32; w++) m = dmax(m, sred[w]);
        if (m > 0.0) atomicMax(&a.stats->sdx_bits, (unsigned long long)__double_as_longlong(m));
        if (DIR == 1) {
            unsigned long long n = 0; double cm = 0.0;
#pragma unroll
            for (int w = 0; w < SW_BLOCK / 32; w++) { n += sclip[w]; cm += sclipm[w]; }
            if (n) { atomicAdd(&a.stats->nclip, n); atomicAdd(&a.stats->clipped, cm); }
        }
    }
}

// ---- line-marching sweep ------------------------------------------------------------------------------------
__device__ __forceinline__ void ld4(const double *p, double &x, double &y, double &z, double &w)
{
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(x), "=d"(y), "=d"(z), "=d"(w) : "l"(p));
}

// x-sweep staging: each thread copies the next 4 cells (32 bytes) of its row, per plane, into its own slots of a
// two-stage shared-memory buffer with cp.async, one group ahead of their use
__device__ __forceinline__ void cp16(const double *sdst, const double *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"((unsigned)__cvta_generic_to_shared(sdst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void stage_group(const SweepArgs &a, const double *sb, int64_t o)
{
    cp16(sb, a.h + o);                        cp16(sb + 2, a.h + o + 2);
    cp16(sb + MARCH_BLOCK * 4, a.hu + o);     cp16(sb + MARCH_BLOCK * 4 + 2, a.hu + o + 2);
    cp16(sb + 2 * MARCH_BLOCK * 4, a.hv + o); cp16(sb + 2 * MARCH_BLOCK * 4 + 2, a.hv + o + 2);
    cp16(sb + 3 * MARCH_BLOCK * 4, a.b + o);  cp16(sb + 3 * MARCH_BLOCK * 4 + 2, a.b + o + 2);
    asm volatile("cp.async.commit_group;" ::: "memory");
}
#define MARCH_STAGE_BYTES (2 * 4 * MARCH_BLOCK * 4 * 8)   // [stage][plane][thread][4 cells] doubles

template <int DIR>
__global__ void __launch_bounds__(MARCH_BLOCK, MARCH_MINB) k_march(SweepArgs a)
{
    __shared__ double sred[MARCH_BLOCK / 32];
    __shared__ unsigned long long sclip[MARCH_BLOCK / 32];
    __shared__ double sclipm[MARCH_BLOCK / 32];

    const int64_t lid = (int64_t)blockIdx.x * MARCH_BLOCK + threadIdx.x;
    const bool active = lid < a.nlines;
    LineDesc ln; ln.patch = 0; ln.line = 0; ln.c0 = 2; ln.nc = -4;
    if (active) { int4 v = *reinterpret_cast<const int4 *>(a.lines + lid); ln.patch = v.x; ln.line = v.y; ln.c0 = v.z; ln.nc = v.w; }
    const PatchDesc pd = a.pat[ln.patch];
    const double dt = a.dt_dev ? *a.dt_dev : a.dt;
    const int nst = ln.nc + 4;                                   // cells read by this line
    const int nst_warp = __reduce_max_sync(0xffffffffu, nst);
    const int cfirst = ln.c0 - 2;                                // storage index (along the sweep) of the first cell read
    int64_t base; int64_t str;
    if (DIR == 0) { base = pd.off + (int64_t)ln.line * pd.pitch + cfirst; str = 1; }
    else          { base = pd.off + (int64_t)cfirst * pd.pitch + ln.line; str = pd.pitch; }
    const bool count = (DIR == 1) || (ln.line >= 2 && ln.line < pd.ny + 2);   // eq. 15 over interior lines only
    const double rdrow = (DIR == 0 && active) ? a.rd[pd.j0 + ln.line] : 0.0;

    Waves Wc; gc_waves_zero(Wc);                                 // waves of the previous edge (r-1)
    double dlo[3] = {0.0, 0.0, 0.0};                             // Z_{r-2} . Z_{r-1}
    double fpp[3] = {0.0, 0.0, 0.0};                             // fp of edge r-2
    RState Lst; Lst.h = 0.0; Lst.p = 0.0; Lst.t = 0.0; Lst.b = 0.0; Lst.u = 0.0; Lst.v = 0.0; Lst.phi = 0.0; Lst.c = 0.0;
    double q1h = 0.0, q1p = 0.0, q1t = 0.0, q2h = 0.0, q2p = 0.0, q2t = 0.0;   // raw state of cells r-1, r-2
    double rd1 = 0.0, rd2 = 0.0;                                 // 1/(kappa dx) of cells r-1, r-2
    double cflm = 0.0, clipm = 0.0; unsigned nclip = 0; int nanf = 0;
    bool stdc = false;                                           // the previous edge is "standard" (gc_edge_flux_std)

    extern __shared__ __align__(16) double stage[];              // x-sweep: MARCH_STAGE_BYTES of staging slots
    if (DIR == 0 && nst > 0) stage_group(a, stage + threadIdx.x * 4, base);
    double nh_ = 0.0, np_ = 0.0, nt_ = 0.0, nb_ = 0.0;           // y-sweep: next row, loaded one step ahead
    if (DIR == 1 && nst > 0) {
        nh_ = a.h[base]; nb_ = a.b[base]; np_ = a.hv[base]; nt_ = a.hu[base];
    }

    constexpr int kMarchUnroll = MARCH_UNROLL;
#pragma unroll kMarchUnroll
    for (int r = 0; r < nst_warp; r++) {
        const bool live = r < nst;
        double qh, qp, qt, qb;
        if (DIR == 0) {
            // the 4 cells of a group were requested one group ago (cp.async.cg into this thread's own staging slots: no
            // register is tied up while the request is in flight and nothing is allocated in L1, which the spilled
            // loop invariants need); each cell is read from its slot when its turn comes
            if ((r & 3) == 0) {
                asm volatile("cp.async.wait_group 0;" ::: "memory");
                if (r + 4 < nst) stage_group(a, stage + (size_t)(((r >> 2) + 1) & 1) * (4 * MARCH_BLOCK * 4) + threadIdx.x * 4, base + r + 4);
            }
            const double *sb = stage + (size_t)((r >> 2) & 1) * (4 * MARCH_BLOCK * 4) + threadIdx.x * 4 + (r & 3);
            qh = live ? sb[0] : 0.0; qp = live ? sb[MARCH_BLOCK * 4] : 0.0;
            qt = live ? sb[2 * MARCH_BLOCK * 4] : 0.0; qb = live ? sb[3 * MARCH_BLOCK * 4] : 0.0;
        } else {
            qh = nh_; qp = np_; qt = nt_; qb = nb_;
            if (r + 1 < nst) {
                const int64_t o = base + (int64_t)(r + 1) * str;
                nh_ = a.h[o]; nb_ = a.b[o]; np_ = a.hv[o]; nt_ = a.hu[o];
            }
        }
        const int c = cfirst + r;                                // storage index of this cell = index of the edge on its low side
        double rd0, ef;
        if (DIR == 0) { rd0 = rdrow; ef = a.ex; }
        else          { rd0 = live ? a.rd[pd.j0 + c] : 0.0; ef = live ? a.ey[pd.j0 + c] : 1.0; }

        RState R; R.h = qh; R.p = qp; R.t = qt; R.b = qb;
        Waves Wn;
        bool stdn = false;
        {   // straight-line code for an open-ocean edge first (gc_riemann_fast); any other kind of edge, or a fast-math
            // operand outside its window (gc_math.cuh), redoes this cell + edge with the general code and IEEE operators
            MathFast mf;
            const RState R0 = R;
            gc_prim_fast(mf, R, a.g, a.eps);
            bool ok = !mf.failed();
            if (r >= 1 && live) ok = gc_riemann_fast(mf, a.g, a.eps, Lst, R, Wn.Z, Wn.s) && ok;
            else gc_waves_zero(Wn);
            stdn = ok && (r >= 1) && live;
            if (!ok) {
                MathIeee mi;
                R = R0;
                gc_prim(mi, R, a.g, a.eps);
                if (r >= 1 && live) gc_riemann(mi, a.g, a.eps, Lst, R, Wn.Z, Wn.s);
            }
            if (a.coord == 1) {                                   // scale by the edge factor
#pragma unroll
                for (int w = 0; w < 3; w++) { Wn.s[w] = Wn.s[w] * ef; Wn.Z[w][0] = Wn.Z[w][0] * ef; Wn.Z[w][1] = Wn.Z[w][1] * ef; Wn.Z[w][2] = Wn.Z[w][2] * ef; }
            }
        }
        double dhi[3];
        gc_wave_dots(Wn, Wc, dhi);                                                      // Z_r . Z_{r-1}
        double fm[3], fp[3];
        {   // edge r-1: a standard edge (s[0] < 0 < s[2], solved by the fast path) needs no sign tests for families 1 and 3
            MathFast mf;
            if (stdc) gc_edge_flux_std(mf, Wc, dlo, dhi, a.limiter, dt, rd2, rd1, fm, fp);
            else gc_edge_flux_fast(mf, Wc, dlo, dhi, a.limiter, dt, rd2, rd1, fm, fp);
            if (mf.failed()) { MathIeee mi; gc_edge_flux(mi, Wc, dlo, dhi, a.limiter, dt, rd2, rd1, fm, fp); }
        }
        if (live && r >= 3 && count) cflm = dmax(cflm, stdc ? gc_edge_cfl_std(Wc, rd2, rd1) : gc_edge_cfl(Wc, rd2, rd1));
        if (live && r >= 4) {                                                           // cell r-2
            const double dtdx = dt * rd2;
            double uh = q2h - dtdx * (fm[0] - fpp[0]);
            double up = q2p - dtdx * (fm[1] - fpp[1]);
            double ut = q2t - dtdx * (fm[2] - fpp[2]);
            const int64_t o = base + (int64_t)(r - 2) * str;
            if (DIR == 0) {
                a.oh[o] = uh; a.ohu[o] = up; a.ohv[o] = ut;
            } else {
                if (uh < a.eps && a.write_out) {                                        // dry clean-up (S-9)
                    if (uh < 0.0) { nclip++; clipm += (-uh) * (a.kappa[pd.j0 + c - 2] * a.dxdy); }
                    uh = dmax(uh, 0.0); up = 0.0; ut = 0.0;
                }
                if (uh != uh || up != up || ut != ut) nanf = 1;
                if (a.write_out) { a.oh[o] = uh; a.ohv[o] = up; a.ohu[o] = ut; }
            }
        }
#pragma unroll
        for (int k = 0; k < 3; k++) { fpp[k] = fp[k]; dlo[k] = dhi[k]; }
        Wc = Wn; Lst = R; stdc = stdn;
        q2h = q1h; q2p = q1p; q2t = q1t; q1h = qh; q1p = qp; q1t = qt;
        rd2 = rd1; rd1 = rd0;
    }

    cflm = warp_max(cflm);
    if (DIR == 1) {
        nclip = __reduce_add_sync(0xffffffffu, nclip);
        nanf = __any_sync(0xffffffffu, nanf);
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) clipm += __shfl_xor_sync(0xffffffffu, clipm, o);
    }
    const int k = threadIdx.x;
    if ((k & 31) == 0) { sred[k >> 5] = cflm; if (DIR == 1) { sclip[k >> 5] = nclip; sclipm[k >> 5] = clipm; if (nanf) a.stats->nan_seen = 1; } }
    __syncthreads();
    if (k == 0) {
        double m = sred[0];
#pragma unroll
        for (int w = 1; w < MARCH_BLOCK / 32; w++) m = dmax(m, sred[w]);
        if (m > 0.0) atomicMax(&a.stats->sdx_bits, (unsigned long long)__double_as_longlong(m));
        if (DIR == 1) {
            unsigned long long n = 0; double cm = 0.0;
#pragma unroll
            for (int w = 0; w < MARCH_BLOCK / 32; w++) { n += sclip[w]; cm += sclipm[w]; }
            if (n) { atomicAdd(&a.stats->nclip, n); atomicAdd(&a.stats->clipped, cm); }
        }
    }
}

__global__ void k_stats_reset(DevStats *s) { s->sdx_bits = 0ull; s->nclip = 0ull; s->clipped = 0.0; s->nan_seen = 0; }

__global__ void k_next_dt(const DevStats *s, double *dt_dev, double cfl)
{
    double sdx = __longlong_as_double((long long)s->sdx_bits);
    *dt_dev = cfl / sdx;
}

void gc_launch_stats_reset(gc_level *L) { ProfScope ps(L->ctx, GC_SLOT_MISC); k_stats_reset<<<1, 1, 0, L->ctx->stream>>>(L->d_stats); }

void gc_launch_next_dt(gc_level *L, double *dt_dev, double cfl) { ProfScope ps(L->ctx, GC_SLOT_MISC); k_next_dt<<<1, 1, 0, L->ctx->stream>>>(L->d_stats, dt_dev, cfl); }

void gc_launch_sweeps(gc_level *L, double dt, const double *dt_dev, int write_out)
{
    const gc_params &P = L->ctx->P;
    int cur = L->cur, nxt = 1 - cur;
    SweepArgs a;
    a.pat = L->d_pat; a.g = P.g; a.eps = P.dry_tol; a.dt = dt; a.dt_dev = dt_dev;
    a.coord = P.coord; a.limiter = P.limiter; a.write_out = write_out; a.stats = L->d_stats;
    a.lines = nullptr; a.nlines = 0;
    a.ex = L->ex; a.ey = L->d_ey; a.dxdy = L->dx * L->dy; a.kappa = L->d_kappa; a.b = L->b;
    // x-sweep: Q^n -> Q*
    a.tiles = L->d_xt; a.h = L->q[cur][0]; a.hu = L->q[cur][1]; a.hv = L->q[cur][2];
    a.oh = L->qs[0]; a.ohu = L->qs[1]; a.ohv = L->qs[2]; a.rd = L->d_rdx;
    if (L->use_march) {
        a.lines = L->d_xl; a.nlines = L->nxl_lines;
        if (a.nlines > 0) { ProfScope ps(L->ctx, GC_SLOT_XSWEEP); k_march<0><<<(unsigned)((a.nlines + MARCH_BLOCK - 1) / MARCH_BLOCK), MARCH_BLOCK, MARCH_STAGE_BYTES, L->ctx->stream>>>(a); }
    } else if (L->nxt > 0) { ProfScope ps(L->ctx, GC_SLOT_XSWEEP); k_sweep<0><<<L->nxt, SW_BLOCK, 0, L->ctx->stream>>>(a); }
    // y-sweep: Q* -> Q^{n+1}
    a.tiles = L->d_yt; a.h = L->qs[0]; a.hu = L->qs[1]; a.hv = L->qs[2];
    a.oh = L->q[nxt][0]; a.ohu = L->q[nxt][1]; a.ohv = L->q[nxt][2]; a.rd = L->d_rdy;
    if (L->use_march) {
        a.lines = L->d_yl; a.nlines = L->nyl_lines;
        if (a.nlines > 0) { ProfScope ps(L->ctx, GC_SLOT_YSWEEP); k_march<1><<<(unsigned)((a.nlines + MARCH_BLOCK - 1) / MARCH_BLOCK), MARCH_BLOCK, 0, L->ctx->stream>>>(a); }
    } else if (L->nyt > 0) { ProfScope ps(L->ctx, GC_SLOT_YSWEEP); k_sweep<1><<<L->nyt, SW_BLOCK, 0, L->ctx->stream>>>(a); }
}

// ---- self-test of gc_math.cuh: MathFast against the IEEE operators on caller-supplied operands
__global__ void k_math_selftest(const double *a, const double *b, int64_t n, unsigned long long *out)
{
    int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    double x = a[i], y = b[i];
    MathIeee mi;
    { MathFast mf; double q = mf.div(x, y);
      if (mf.failed()) atomicAdd(out + 1, 1ull);
      else if (__double_as_longlong(q) != __double_as_longlong(mi.div(x, y))) atomicAdd(out, 1ull); }
    { MathFast mf; double q = mf.rcp(y);
      if (mf.failed()) atomicAdd(out + 1, 1ull);
      else if (__double_as_longlong(q) != __double_as_longlong(mi.rcp(y))) atomicAdd(out, 1ull); }
    { MathFast mf; double q = mf.sqrt_(x);
      if (mf.failed()) atomicAdd(out + 1, 1ull);
      else if (__double_as_longlong(q) != __double_as_longlong(mi.sqrt_(x))) atomicAdd(out, 1ull); }
}
void gc_launch_math_selftest(cudaStream_t s, const double *a, const double *b, int64_t n, unsigned long long *out)
{
    if (n > 0) k_math_selftest<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(a, b, n, out);
}

// ---- fp64 ALU peak probe: dependent DFMA chains, 8 independent accumulators per thread
__global__ void k_fp64_probe(double *out, int iters)
{
    double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3;
    double a4 = a0 + 4e-3, a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
    const double m = 0.999999999, c = 1e-12;
    for (int i = 0; i < iters; i++) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    double r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123.456) out[0] = r;
}

void gc_launch_fp64_probe(cudaStream_t s, double *out, int iters, int blocks, int threads)
{
    k_fp64_probe<<<blocks, threads, 0, s>>>(out, iters);
}
