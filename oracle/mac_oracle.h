/*
 * mac_oracle.h -- CPU fp64 ORACLE for the MAESTROeX MAC projection (TEST INFRASTRUCTURE).
 *
 * This is test infrastructure, not the product.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code with the CUDA
 * path under paper_1910_12979_b200/csrc/ and neither includes the other.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, "P:n" = line n):
 *   the velocity constraint   div(beta0 U) = beta0 (S - ...)            P:49  (Sec. 2, Eq. 6)
 *   with the pressure term    (beta0/rho) grad(pi/beta0)                P:35  (Sec. 2, Eq. 2)
 *   on a 1-D base state       rho0(r), p0(r), beta0(r)                  P:29, P:39, P:45 (Eq. 4-5)
 *   solved by "multigrid linear solvers" inside a "second order projection method"  P:63 (Sec. 3)
 * i.e.  solve  L phi = rhs,  L phi = D((beta0/rho) G phi),  rhs = D(beta0 U_edge) - beta0 S,
 *       then   U <- U_edge - (1/rho_face) G phi.
 * The paper gives no discretisation; every concrete choice is a reading listed in DESIGN.md
 * ("Readings", R1..) and SURVEY.md Sec. 8(c) (O1..O10, A1..A25).  The steps are written out in the
 * order of SURVEY.md Sec. 8(c) with no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): dense direct solve (P1), symmetry and row
 * sums (P2), manufactured-solution order (P3), constraint identity (P4/P5), red-black property
 * (P6), Fourier closed form (P7), scaling laws (P8), idempotence (P9), transfer invariants (P10),
 * convergence factor (P11), independent D*B*G Kronecker assembly.
 * PARITY UNPINNED: the absolute scale of phi relative to the paper's pi (needs the time-step
 * factor the paper does not give; irrelevant to U).
 *
 * Layout (x fastest):  cell  i + nx*(j + ny*k)
 *                      u     i + (nx+1)*(j + ny*k),  i in [0,nx]   (x-face i-1/2)
 *                      v     i + nx*(j + (ny+1)*k),  j in [0,ny]
 *                      w     i + nx*(j + ny*k),      k in [0,nz]
 * Face-coefficient arrays bx,by,bz have the layout of u,v,w and hold b = beta0/rho_face.
 */
#ifndef MAC_ORACLE_H
#define MAC_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_PERIODIC = 0, ORC_WALL = 1, ORC_OUTFLOW = 2 };
enum { ORC_PLANAR = 0, ORC_SPHERICAL = 1 };

/* Grid of one multigrid level: cells n[3], spacing h[3], boundary types per side. */
typedef struct {
    int n[3];
    double h[3];
    int bc_lo[3], bc_hi[3];
    int rho_mean;             /* face density: 0 arithmetic mean of rho (default), 1 harmonic (mean of 1/rho); A3 */
} orc_grid;

/* 1-D base-state sampling: nr samples at r_m = (m + 1/2) dr.  Planar: r = z. */
typedef struct {
    int geometry;
    int nr;
    double dr;
    double center[3];
} orc_base;

typedef struct {
    int nu_pre, nu_post;      /* RBGS sweeps before / after the coarse correction  (2, 2) */
    int max_cycles;           /* 100 */
    double rel_tol;           /* 1e-10 on ||r||inf / ||rhs||inf ; 0 = run max_cycles   */
    int coarsest_n;           /* 4 */
    int prolongation;         /* 0 trilinear, 1 piecewise constant */
} orc_mg;

typedef struct {
    int cycles, singular, levels, converged;
    double rhs_norm_inf, res_norm_inf, rhs_mean_removed;
    double res_history[128];
} orc_stats;

int orc_num_threads(void);
void orc_set_num_threads(int n);

/* O1  profile evaluation at radius r (piecewise linear, constant beyond the end samples) */
double orc_profile(const double *f, int nr, double dr, double r);
/* radius of a point for the base state: planar r = z, spherical r = |x - center| */
double orc_radius(const orc_base *b, double x, double y, double z);

/* O2+O3  face coefficients b = beta0(face centre) / rho_face  on level 0 */
void orc_face_coeff(const orc_grid *g, const orc_base *b, const double *beta0,
                    const double *rho, double *bx, double *by, double *bz);
/* rho at cell centres from the rho0 profile (used when the caller passes rho == NULL) */
void orc_rho_from_profile(const orc_grid *g, const orc_base *b, const double *rho0, double *rho);

/* O4  rhs = D(beta0_face U_edge) - beta0_cell S   (S may be NULL = 0).  No mean removal here. */
void orc_rhs(const orc_grid *g, const orc_base *b, const double *beta0,
             const double *u, const double *v, const double *w, const double *S, double *rhs);
double orc_norm_inf(const double *a, long long n);
double orc_mean(const double *a, long long n);
void orc_shift(double *a, long long n, double c);      /* a -= c */
int orc_is_singular(const orc_grid *g);                /* 1 if no OUTFLOW side anywhere */

/* O5  operator and its diagonal */
void orc_apply(const orc_grid *g, const double *bx, const double *by, const double *bz,
               const double *phi, double *out);
void orc_diag(const orc_grid *g, const double *bx, const double *by, const double *bz,
              double *diag);
void orc_residual(const orc_grid *g, const double *bx, const double *by, const double *bz,
                  const double *phi, const double *rhs, double *res);

/* O6  smoother: one colour pass (colour 0 = red = (i+j+k) even), one sweep = red then black */
void orc_rbgs_color(const orc_grid *g, const double *bx, const double *by, const double *bz,
                    const double *rhs, double *phi, int color);
void orc_rbgs_sweep(const orc_grid *g, const double *bx, const double *by, const double *bz,
                    const double *rhs, double *phi);

/* O7  hierarchy */
int orc_can_coarsen(const orc_grid *g, int coarsest_n);
void orc_coarsen_grid(const orc_grid *f, orc_grid *c);
void orc_coarsen_coeff(const orc_grid *f, const double *bx, const double *by, const double *bz,
                       double *cbx, double *cby, double *cbz);
/* O8  transfers.  restrict: coarse = mean of 8 children.  prolong: fine += P coarse */
void orc_restrict(const orc_grid *f, const double *fine, double *coarse);
void orc_prolong_add(const orc_grid *f, const double *coarse, double *fine, int prolongation);
/* O8  bottom: dense Gaussian elimination with partial pivoting (bordered if singular).
 * Returns 0, or -1 if the matrix is numerically singular / too large. */
int orc_bottom_solve(const orc_grid *g, const double *bx, const double *by, const double *bz,
                     const double *f, double *e);
/* O8  one V-cycle on (phi, rhs) of level g; coefficient arrays are built by coarsening. */
int orc_vcycle(const orc_grid *g, const double *bx, const double *by, const double *bz,
               const double *rhs, double *phi, const orc_mg *mg);

/* O10  velocity correction, in place */
void orc_correct(const orc_grid *g, const double *rho, const double *phi,
                 double *u, double *v, double *w);

/* O9  the whole projection.  rho may be NULL (then rho := rho0 profile at cell centres);
 * S may be NULL; phi may be NULL.  u,v,w are corrected in place.
 * Returns 0 converged, 1 max_cycles reached, <0 error (-2 unsupported hierarchy, -5 nonfinite). */
int orc_project(const orc_grid *g, const orc_base *b, const orc_mg *mg,
                const double *beta0, const double *rho0, const double *rho,
                double *u, double *v, double *w, const double *S, double *phi,
                orc_stats *stats);

/* O11 (Eq. 5): beta0 on the profile samples r_m = (m + 1/2) dr from p0 and Gamma1bar.
 *   beta0_0 = rho0_0 (the innermost sample stands for r = 0; a constant factor of beta0 does not change U, pin P8),
 *   ln beta0_{m+1} = ln beta0_m + (ln p0_{m+1} - ln p0_m) / (0.5 (Gamma1bar_m + Gamma1bar_{m+1}))
 * i.e. the integrand (1/(Gamma1bar p0)) dp0/dr integrated as d(ln p0)/Gamma1bar with Gamma1bar taken at the
 * midpoint; exact where Gamma1bar is constant (readings A26, A27). */
void orc_make_beta0(int nr, const double *rho0, const double *p0, const double *gamma1bar, double *beta0);
/* O12 (Eq. 6): the base-state term of the constraint on the samples,
 *   q_m = dp0dt_m / (Gamma1bar_m p0_m),
 * and the effective source  S_eff = S - q(r_cell)  (q evaluated at cell centres by O1; S may be NULL = 0),
 * so that  rhs = D(beta0 U_edge) - beta0 (S - (1/(Gamma1bar p0)) dp0/dt)  (reading A28). */
void orc_dpdt_term(int nr, const double *p0, const double *gamma1bar, const double *dp0dt, double *q);
void orc_effective_source(const orc_grid *g, const orc_base *b, const double *S, const double *q, double *S_eff);

/* O13 ("rho0 ... represents the lateral average"): the base-state density from the cell density.
 * Cell (i,j,k) with centre radius r (planar: r = z) belongs to sample m = min(nr - 1, floor(r / dr)), i.e. to the
 * shell [m dr, (m+1) dr) around r_m = (m + 1/2) dr; rho0[m] = mean of rho over the cells of sample m.  Samples
 * without a cell (spherical geometry with dr < dx has many near the centre) are filled by linear interpolation in
 * m between the nearest samples that have cells, constant beyond the first / last such sample (readings A29, A30,
 * DESIGN.md).  count[m] (may be NULL) receives the number of cells of sample m.  Planar with nr = nz, dr = dz:
 * rho0[k] is the mean of plane k. */
void orc_lateral_average(const orc_grid *g, const orc_base *b, const double *rho, double *rho0, long long *count);

/* Constraint residual  D(beta0 U) - beta0 S  (same discrete operators as orc_rhs). */
void orc_constraint(const orc_grid *g, const orc_base *b, const double *beta0,
                    const double *u, const double *v, const double *w, const double *S,
                    double *out);

#ifdef __cplusplus
}
#endif
#endif
