/* gco.h -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow fp64 CPU implementation (single-threaded unless gco_set_threads says otherwise) of the per-level time step of
 * GPU GeoClaw ("Efficient Tsunami Modeling on Adaptive Grids with GPUs", arXiv 1901.06798;
 * PAPER.md = P:<line>), written from the paper and from DESIGN.md section 3 (the readings of
 * every point the paper leaves open).  It shares no code with paper_1901_06798_b200/ (the CUDA
 * path) and neither includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math (see oracle/gco.py).  C99 fma() exactly where DESIGN.md 3.3-3.4 write it, no
 * other contraction, IEEE
 * sqrt and divide; min/max are written as ternaries (max2/min2) so that signed zeros and
 * ties behave identically everywhere.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): lake at rest, closed-basin mass balance,
 * Stoker / Ritter dam breaks, d'Alembert pulse (2nd order), cell-centric brute force recomputation,
 * y-independent 2-D == 1-D, tiling invariance, full-cover fine level == single level, constant /
 * rest states through interpolation, averaging and regrid, sphere band area closed form,
 * flux-register mass conservation across a coarse-fine interface.
 * Parity unpinned: none of the functions below is without a pin; the Riemann solver's choice
 * of branch thresholds (tau, one Newton / secant step) is a DESIGN.md reading, pinned only
 * through the convergence tests.
 */
#ifndef GCO_H
#define GCO_H
#include <stdint.h>
#include <stddef.h>

#define GCO_G 2 /* ghost width */

enum { GCO_H_ = 0, GCO_HU = 1, GCO_HV = 2, GCO_B = 3 };
enum { GCO_OK = 0, GCO_ERR_BADARG = -1, GCO_ERR_NOMEM = -2, GCO_ERR_STATE = -6 };

typedef struct {
    int coord;            /* 0 Cartesian (m), 1 spherical lon/lat (deg) */
    double g, dry_tol, sea_level, earth_radius;
    int limiter;          /* 0 none (first order), 1 MC */
    int bc[4];            /* xlo, xhi, ylo, yhi: 0 extrapolation, 1 wall */
    double manning_n;     /* Manning coefficient n of P:52-57 eq. 2 (the paper uses 0.025); 0 = friction off */
    double friction_depth;/* friction acts in cells with dry_tol < h <= friction_depth */
} gco_params;

typedef struct { int32_t i0, j0, nx, ny; } gco_patch; /* interior box, global cell indices of the level */

typedef struct {
    double tol_eta, tol_slope; /* <= 0: criterion off */
    int offshore_only;         /* wave criteria need b < 0 */
    int buffer;                /* dilation width in cells */
    int nboxes;
    const double *boxes;       /* x0,x1,y0,y1,t0,t1 per forced box */
} gco_flag_params;

typedef struct {
    double cfl_max, s_over_dx_max, clipped_mass;
    int64_t n_clipped;
    int32_t nan_seen;
} gco_step_stats;

typedef struct gco_ctx gco_ctx;
typedef struct gco_level gco_level;

/* ---- Manning friction (gco_level.c), eq. 1b-1c, 2; DESIGN.md 3.9 (reading S-16) ---- */
/* cube root of a positive normal double by the fixed sequence of DESIGN.md 3.9 (bit seed + three Halley steps) */
double gco_cbrt(double x);
/* semi-implicit friction step of one cell over dt: hu, hv <- hu / d, hv / d, d = 1 + dt g n^2 |hu, hv| / h^(7/3);
 * acts only if manning_n > 0 and dry_tol < h <= friction_depth */
void gco_friction(const gco_params *P, double dt, double h, double *hu, double *hv);

/* ---- Riemann solver (gco_riemann.c), DESIGN.md 3.3 ---- */
/* inputs: depth, normal momentum, transverse momentum, bathymetry on each side.
 * outputs: f-waves Z[p][k] (p = family 0..2; k = 0:h, 1:normal, 2:transverse), speeds s[p]. */
void gco_riemann(double g, double eps, double hL, double pL, double tL, double bL,
                 double hR, double pR, double tR, double bR, double Z[3][3], double s[3]);
void gco_middle_state(double g, double eps, double hL, double hR, double uL, double uR,
                      double cL, double cR, double *hm, double *s1m, double *s2m);

/* ---- 1-D line sweep (gco_sweep.c), DESIGN.md 3.4 ----
 * Cells c = 0..n+3 (ghost width 2); edge e lies between cells e-1 and e.
 * rdx[c] = 1/(kappa_c*dx); efac[e] = edge scale factor (1 in Cartesian).
 * Updates cells 2..n+1 into (ho,po,to).  fm/fp (nullable) receive the flux-like
 * quantities at edges 2..n+2 (3 doubles each, index [e*3+k]).  *sdx is max-updated with
 * max_e,p |s|*rdx (eq. 15) when count_cfl != 0. */
void gco_sweep_line(const gco_params *P, int n, const double *h, const double *p, const double *t,
                    const double *b, const double *rdx, const double *efac, double dt,
                    double *ho, double *po, double *to, double *fm, double *fp,
                    int count_cfl, double *sdx);

void gco_line_terms(const gco_params *P, int n, const double *h, const double *p, const double *t,
                    const double *b, const double *rdx, const double *efac, double dt,
                    double *am, double *ap, double *F, double *s);

/* ---- level API (gco_level.c / gco_amr.c); mirrors include/gc.h with host pointers ---- */
int gco_ctx_create(const gco_params *, gco_ctx **out);
int gco_ctx_destroy(gco_ctx *);
int gco_level_create(gco_ctx *, int level, double xlo, double ylo, double dx, double dy,
                     int64_t nx_level, int64_t ny_level, int ratio_to_coarser, int npatch,
                     const gco_patch *, gco_level **out);
int gco_level_destroy(gco_level *);
/* per-patch storage-shaped arrays: (ny+4) rows of (nx+4), leading dimension ld */
int gco_level_set_field(gco_level *, int patch, int field, const double *src, int64_t ld);
int gco_level_get_field(const gco_level *, int patch, int field, int which /*0 new(current), 1 old*/,
                        double *dst, int64_t ld);
/* level-global arrays: src covers global cells [gi0,gi0+gnx) x [gj0,gj0+gny); every storage cell
 * (ghosts included) of every patch that falls inside is set / every interior cell is read. */
int gco_level_set_global(gco_level *, int field, const double *src, int64_t ld,
                         int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny);
int gco_level_get_global(const gco_level *, int field, int which, double *dst, int64_t ld,
                         int64_t gi0, int64_t gj0, int64_t gnx, int64_t gny);
int gco_fill_ghost_b(gco_level *);
int gco_fill_ghost(gco_level *L, const gco_level *coarser, double alpha);
int gco_level_step(gco_level *L, double dt, gco_step_stats *out);
/* ---- unsplit step with transverse Riemann solves (gco_unsplit.c); DESIGN.md 3.13 (reading S-21) ---- */
void gco_transverse(double g, double eps, double h, double pn, double pt, const double a[3], double bm[3], double bp[3]);
int gco_level_step_unsplit(gco_level *L, double dt, gco_step_stats *out);
/* threads for gco_level_step's loop over patches (default 1; no result bit depends on it: patches are independent inside a step,
 * SURVEY 8(d) "patch-level omp parallel for"); used by bench.py's N-core baseline and by the long parity runs */
int gco_set_threads(int n);
int gco_get_threads(void);
/* ---- time-dependent bathymetry (gco_bathy.c); DESIGN.md 3.12 (reading S-20) ---- */
typedef struct {
    double x0, y0, ddx, ddy;   /* node (m, n) at (x0 + m ddx, y0 + n ddy), in the level's coordinates */
    int64_t mx, my;            /* nodes per direction, >= 2 */
    const double *dz;          /* my rows of mx values: vertical seafloor displacement in metres, + up */
} gco_deform;
double gco_deform_at(const gco_deform *D, double x, double y);     /* bilinear between nodes, 0 outside the grid */
/* b <- fma(w, dz(cell centre), b) on every storage cell inside the domain; h, hu, hv untouched (eta moves with the seafloor) */
int gco_bathy_update(gco_level *L, const gco_deform *D, double w);
/* ---- gauges (gco_amr.c); DESIGN.md 3.10 (reading S-19) ---- */
/* Samples n points from the current state of L (ghost cells as they are): point k = (xy[2k], xy[2k+1]) must lie in the interior
 * of patch patch[k] (else GCO_ERR_BADARG).  out: 4 per point -- h, hu, hv, eta = h + b; bilinear between the four cell centres
 * around the point when all four are wet, else the value of the cell containing the point. */
int gco_gauges_sample(const gco_level *L, int n, const int32_t *patch, const double *xy, double *out);
int gco_wet_mask(const gco_level *, uint8_t *mask /* interior-packed per patch */);
double gco_level_mass(const gco_level *);
int64_t gco_level_ncells(const gco_level *);
int gco_flag_cells(const gco_level *L, const gco_flag_params *, double t, uint8_t *flags, int64_t *nflag);
int gco_average_down(gco_level *coarse, const gco_level *fine);
int gco_level_init_from(gco_level *newfine, const gco_level *oldfine, const gco_level *coarse);
int gco_flux_attach(gco_level *coarse, gco_level *fine);
int gco_flux_fixup(gco_level *coarse, gco_level *fine);
/* metric tables as the oracle computes them (for the sphere pins); n = ny_level + 4 rows / + 5 edges */
int gco_level_metric(const gco_level *, double *kappa, double *rdx, double *rdy, double *ey);

#endif
