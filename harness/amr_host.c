/* amr_host.c -- native versions of the AMR harness's host bookkeeping (harness/driver.py): Berger-Rigoutsos clustering of
 * refinement flags, the proper-nesting mask and the unpacking of interior-packed flags.  Bookkeeping only: no arithmetic
 * of the method.  Shared by both backends AFTER their flags have been compared bit for bit; the Python functions of
 * driver.py stay as the definition, and tests/test_harness_pins.py holds these to the same boxes / masks.
 * Built by harness/build.py: gcc -O2 -shared -fPIC. */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* interior-packed per-patch bytes -> 2-D array over bbox = [bi, ei) x [bj, ej); pat: np x 4 (i0, j0, nx, ny) */
void amr_unpack(const uint8_t *packed, const int32_t *pat, int np, int bi, int bj, int ei, int ej, uint8_t *out)
{
    int64_t W = ei - bi, o = 0;
    memset(out, 0, (size_t)W * (size_t)(ej - bj));
    for (int p = 0; p < np; p++) {
        int i0 = pat[4 * p], j0 = pat[4 * p + 1], nx = pat[4 * p + 2], ny = pat[4 * p + 3];
        for (int j = 0; j < ny; j++) memcpy(out + (int64_t)(j0 - bj + j) * W + (i0 - bi), packed + o + (int64_t)j * nx, (size_t)nx);
        o += (int64_t)nx * ny;
    }
}

/* cells of the level (inside bbox) whose 3 x 3 neighbourhood, clipped to the domain nxl x nyl, lies inside the level's patches */
void amr_nesting_mask(const int32_t *pat, int np, int bi, int bj, int ei, int ej, int nxl, int nyl, uint8_t *ok)
{
    int W = ei - bi, H = ej - bj, CW = W + 2, CH = H + 2;
    uint8_t *cov = calloc((size_t)CW * CH, 1);           /* index (j - bj + 1, i - bi + 1) */
    if (bj == 0) memset(cov, 1, (size_t)CW);               /* outside the domain counts as fine (physical BC) */
    if (ej == nyl) memset(cov + (size_t)(CH - 1) * CW, 1, (size_t)CW);
    if (bi == 0) for (int j = 0; j < CH; j++) cov[(size_t)j * CW] = 1;
    if (ei == nxl) for (int j = 0; j < CH; j++) cov[(size_t)j * CW + CW - 1] = 1;
    for (int p = 0; p < np; p++) {
        int i0 = pat[4 * p], j0 = pat[4 * p + 1], nx = pat[4 * p + 2], ny = pat[4 * p + 3];
        int a0 = i0 - bi + 1, a1 = a0 + nx, c0 = j0 - bj + 1, c1 = c0 + ny;
        if (a0 < 0) a0 = 0; if (a1 > CW) a1 = CW; if (c0 < 0) c0 = 0; if (c1 > CH) c1 = CH;
        for (int j = c0; j < c1; j++) if (a0 < a1) memset(cov + (size_t)j * CW + a0, 1, (size_t)(a1 - a0));
    }
    for (int j = 0; j < H; j++) for (int i = 0; i < W; i++) {
        const uint8_t *c = cov + (size_t)j * CW + i;
        ok[(size_t)j * W + i] = c[0] & c[1] & c[2] & c[CW] & c[CW + 1] & c[CW + 2] & c[2 * CW] & c[2 * CW + 1] & c[2 * CW + 2];
    }
    free(cov);
}

/* cut position (1..n-1) of a 1-D signature, or -1: a hole nearest the centre, else the strongest Laplacian inflection */
static int signature_cut(const int64_t *sig, int n)
{
    int bestk = -1;
    double bd = 0.0;
    for (int k = 1; k < n - 1; k++) if (sig[k] == 0) {
        double d = k - n / 2.0; if (d < 0) d = -d;
        if (bestk < 0 || d < bd) { bestk = k; bd = d; }    /* ties: the lower index (it comes first) */
    }
    if (bestk >= 0) return bestk;
    if (n < 4) return -1;
    int64_t best = 0;
    for (int k = 0; k + 1 < n - 2; k++) {
        int64_t l0 = sig[k] - 2 * sig[k + 1] + sig[k + 2], l1 = sig[k + 1] - 2 * sig[k + 2] + sig[k + 3];
        if ((l0 < 0 && l1 > 0) || (l0 > 0 && l1 < 0)) {
            int64_t mag = l0 - l1; if (mag < 0) mag = -mag;
            double dn = k + 2 - n / 2.0, db = bestk - n / 2.0;
            if (dn < 0) dn = -dn; if (db < 0) db = -db;
            if (mag > best || (mag == best && bestk >= 0 && dn < db)) { best = mag; bestk = k + 2; }
        }
    }
    return bestk;
}

static int box_cmp(const void *a, const void *b)
{
    const int32_t *x = a, *y = b;
    if (x[1] != y[1]) return x[1] < y[1] ? -1 : 1;
    if (x[0] != y[0]) return x[0] < y[0] ? -1 : 1;
    return 0;
}

/* fl, valid (nullable): NY x NX bytes.  out: up to cap boxes (i0, j0, nx, ny), sorted by (j0, i0).  Returns the number of boxes,
 * or -1 if cap is too small. */
int amr_cluster(const uint8_t *fl, const uint8_t *valid, int NY, int NX, double efficiency, int max_side, int32_t *out, int cap)
{
    int64_t *cy = calloc((size_t)(NY + 1) * NX, sizeof(int64_t));          /* cy[j][i]: flags in column i below row j */
    int64_t *cx = calloc((size_t)NY * (NX + 1), sizeof(int64_t));          /* cx[j][i]: flags in row j left of column i */
    int64_t *bad = valid ? calloc((size_t)(NY + 1) * (NX + 1), sizeof(int64_t)) : NULL;
    for (int j = 0; j < NY; j++) for (int i = 0; i < NX; i++) {
        int f = fl[(size_t)j * NX + i] != 0;
        cy[(size_t)(j + 1) * NX + i] = cy[(size_t)j * NX + i] + f;
        cx[(size_t)j * (NX + 1) + i + 1] = cx[(size_t)j * (NX + 1) + i] + f;
        if (bad) bad[(size_t)(j + 1) * (NX + 1) + i + 1] = bad[(size_t)j * (NX + 1) + i + 1] + bad[(size_t)(j + 1) * (NX + 1) + i]
                                                          - bad[(size_t)j * (NX + 1) + i] + (valid[(size_t)j * NX + i] == 0);
    }
    int scap = 64, sn = 0, n = 0;
    int32_t *stack = malloc(sizeof(int32_t) * 4 * scap);
    int64_t *sx = malloc(sizeof(int64_t) * (NX + 1)), *sy = malloc(sizeof(int64_t) * (NY + 1));
    stack[0] = 0; stack[1] = 0; stack[2] = NX; stack[3] = NY; sn = 1;
    while (sn > 0) {
        sn--;
        int i0 = stack[4 * sn], j0 = stack[4 * sn + 1], nx = stack[4 * sn + 2], ny = stack[4 * sn + 3];
        int x0 = -1, x1 = -1, y0 = -1, y1 = -1;
        for (int i = 0; i < nx; i++) {
            sx[i] = cy[(size_t)(j0 + ny) * NX + i0 + i] - cy[(size_t)j0 * NX + i0 + i];
            if (sx[i]) { if (x0 < 0) x0 = i; x1 = i; }
        }
        if (x0 < 0) continue;
        for (int j = 0; j < ny; j++) {
            sy[j] = cx[(size_t)(j0 + j) * (NX + 1) + i0 + nx] - cx[(size_t)(j0 + j) * (NX + 1) + i0];
            if (sy[j]) { if (y0 < 0) y0 = j; y1 = j; }
        }
        i0 += x0; nx = x1 - x0 + 1; j0 += y0; ny = y1 - y0 + 1;
        const int64_t *bx = sx + x0, *by = sy + y0;
        int64_t tot = 0;
        for (int i = 0; i < nx; i++) tot += bx[i];
        int ok_valid = 1;
        if (bad) ok_valid = (bad[(size_t)(j0 + ny) * (NX + 1) + i0 + nx] - bad[(size_t)j0 * (NX + 1) + i0 + nx]
                             - bad[(size_t)(j0 + ny) * (NX + 1) + i0] + bad[(size_t)j0 * (NX + 1) + i0]) == 0;
        double eff = (double)tot / (double)((int64_t)nx * ny);
        int accept = eff >= efficiency && ok_valid && nx <= max_side && ny <= max_side;
        int cdir = -1, cpos = 0;                           /* 0: cut in x, 1: cut in y */
        if (!accept) {
            if (nx > max_side || ny > max_side) { cdir = nx >= ny ? 0 : 1; cpos = nx >= ny ? nx / 2 : ny / 2; }
            else {
                int kx = signature_cut(bx, nx), ky = signature_cut(by, ny);
                int hx = kx >= 0 && bx[kx] == 0, hy = ky >= 0 && by[ky] == 0;
                if (hx || hy) { if (hx && (!hy || nx >= ny)) { cdir = 0; cpos = kx; } else { cdir = 1; cpos = ky; } }
                else if (kx >= 0 || ky >= 0) { if (kx >= 0 && (ky < 0 || nx >= ny)) { cdir = 0; cpos = kx; } else { cdir = 1; cpos = ky; } }
                else if (nx > 1 || ny > 1) { cdir = nx >= ny ? 0 : 1; cpos = nx >= ny ? nx / 2 : ny / 2; }
            }
        }
        if (accept || cdir < 0) {
            if (n >= cap) { n = -1; break; }
            out[4 * n] = i0; out[4 * n + 1] = j0; out[4 * n + 2] = nx; out[4 * n + 3] = ny; n++;
            continue;
        }
        if (sn + 2 > scap) { scap *= 2; stack = realloc(stack, sizeof(int32_t) * 4 * scap); }
        if (cdir == 0) {
            stack[4 * sn] = i0 + cpos; stack[4 * sn + 1] = j0; stack[4 * sn + 2] = nx - cpos; stack[4 * sn + 3] = ny; sn++;
            stack[4 * sn] = i0; stack[4 * sn + 1] = j0; stack[4 * sn + 2] = cpos; stack[4 * sn + 3] = ny; sn++;
        } else {
            stack[4 * sn] = i0; stack[4 * sn + 1] = j0 + cpos; stack[4 * sn + 2] = nx; stack[4 * sn + 3] = ny - cpos; sn++;
            stack[4 * sn] = i0; stack[4 * sn + 1] = j0; stack[4 * sn + 2] = nx; stack[4 * sn + 3] = cpos; sn++;
        }
    }
    if (n > 0) qsort(out, (size_t)n, 4 * sizeof(int32_t), box_cmp);
    free(cy); free(cx); free(bad); free(stack); free(sx); free(sy);
    return n;
}

/* Packs the storage-shaped blocks ((ny + 4) rows of (nx + 4) doubles, ghost width 2) of every patch of a level, back to back,
 * from a cache of square tiles of T x T cells aligned to the level's global cell indices (workloads.Workload.bathy_box keeps
 * such tiles).  tiles: ntx x nty table of pointers (row-major over tile row tj, then ti), NULL where no tile is held -- every
 * tile a patch touches inside the level must be present.  Cells outside the level (nxl x nyl) are written as 0.  Pure copying. */
int amr_pack_from_tiles(const double *const *tiles, int ntx, int nty, int T, const int32_t *pat, int np, int nxl, int nyl, double *out)
{
    int64_t o = 0;
    for (int p = 0; p < np; p++) {
        int i0 = pat[4 * p], j0 = pat[4 * p + 1], nx = pat[4 * p + 2], ny = pat[4 * p + 3];
        int W = nx + 4;
        for (int j = 0; j < ny + 4; j++) {
            int gj = j0 + j - 2;
            double *row = out + o + (int64_t)j * W;
            if (gj < 0 || gj >= nyl) { memset(row, 0, sizeof(double) * (size_t)W); continue; }
            int tj = gj / T, lj = gj - tj * T;
            int i = 0;
            while (i < W) {
                int gi = i0 + i - 2;
                if (gi < 0 || gi >= nxl) { row[i++] = 0.0; continue; }
                int ti = gi / T, li = gi - ti * T;
                int run = T - li;                                   /* cells left in this tile row */
                if (run > W - i) run = W - i;
                if (gi + run > nxl) run = nxl - gi;
                if (tj >= nty || ti >= ntx) return -1;
                const double *t = tiles[(size_t)tj * ntx + ti];
                if (!t) return -1;
                memcpy(row + i, t + (size_t)lj * T + li, sizeof(double) * (size_t)run);
                i += run;
            }
        }
        o += (int64_t)W * (ny + 4);
    }
    return 0;
}
