/*
 * mac_oracle.c -- CPU fp64 ORACLE for the MAESTROeX MAC projection (TEST INFRASTRUCTURE).
 * See mac_oracle.h for scope, citations, layout and the list of pins.
 *
 * Plain loops, one function per step of SURVEY.md Sec. 8(c) (O1..O10).  OpenMP pragmas sit only on
 * loops whose iterations are independent (pointwise passes, one colour of the smoother) and on
 * max-reductions, so results do not depend on the thread count.  Sums are taken plane by plane
 * and then added serially for the same reason.
 */
#include "mac_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long long ll;

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ---------- indexing ------------------------------------------------------------------------ */

static inline ll cidx(const orc_grid *g, int i, int j, int k)
{
    return (ll)i + (ll)g->n[0] * ((ll)j + (ll)g->n[1] * (ll)k);
}
/* face of axis d, index (i,j,k) with the face index running 0..n[d] along d */
static inline ll fidx(const orc_grid *g, int d, int i, int j, int k)
{
    ll sx = g->n[0] + (d == 0), sy = g->n[1] + (d == 1);
    return (ll)i + sx * ((ll)j + sy * (ll)k);
}
static inline ll ncells(const orc_grid *g) { return (ll)g->n[0] * g->n[1] * g->n[2]; }
static inline ll nfaces(const orc_grid *g, int d)
{
    return (ll)(g->n[0] + (d == 0)) * (g->n[1] + (d == 1)) * (g->n[2] + (d == 2));
}
static inline int is_periodic(const orc_grid *g, int d) { return g->bc_lo[d] == ORC_PERIODIC; }

/* ---------- O1: base-state profile ---------------------------------------------------------- */

/* P:29, P:39, P:45 say only that the base state is a function of r.  Reading:
 * samples at r_m = (m+1/2) dr, linear between samples, constant beyond the first and last. */
double orc_profile(const double *f, int nr, double dr, double r)
{
    double s = r / dr - 0.5;
    if (s <= 0.0) return f[0];
    if (s >= (double)(nr - 1)) return f[nr - 1];
    int m = (int)floor(s);
    double t = s - (double)m;
    return (1.0 - t) * f[m] + t * f[m + 1];
}

/* planar or spherical geometry.  Reading A5: the true radius of the point. */
double orc_radius(const orc_base *b, double x, double y, double z)
{
    if (b->geometry == ORC_PLANAR) return z;
    double ax = x - b->center[0], ay = y - b->center[1], az = z - b->center[2];
    return sqrt(ax * ax + ay * ay + az * az);
}

/* position of the centre of cell (i,j,k) */
static void cell_pos(const orc_grid *g, int i, int j, int k, double p[3])
{
    p[0] = (i + 0.5) * g->h[0];
    p[1] = (j + 0.5) * g->h[1];
    p[2] = (k + 0.5) * g->h[2];
}
/* position of the centre of the face of axis d with face index (i,j,k).  On a periodic axis the
 * face n[d] is the face 0 (reading A18: evaluated at the low-side position). */
static void face_pos(const orc_grid *g, int d, int i, int j, int k, double p[3])
{
    int id[3] = {i, j, k};
    if (is_periodic(g, d) && id[d] == g->n[d]) id[d] = 0;
    for (int a = 0; a < 3; ++a) p[a] = (a == d) ? id[a] * g->h[a] : (id[a] + 0.5) * g->h[a];
}
static double beta_cell(const orc_grid *g, const orc_base *b, const double *beta0, int i, int j, int k)
{
    double p[3];
    cell_pos(g, i, j, k, p);
    return orc_profile(beta0, b->nr, b->dr, orc_radius(b, p[0], p[1], p[2]));
}
static double beta_face(const orc_grid *g, const orc_base *b, const double *beta0, int d, int i, int j, int k)
{
    double p[3];
    face_pos(g, d, i, j, k, p);
    return orc_profile(beta0, b->nr, b->dr, orc_radius(b, p[0], p[1], p[2]));
}

/* ---------- O2: density on a face ----------------------------------------------------------- */

/* rho_face = (rho_L + rho_R)/2 ; periodic axis wraps; non-periodic boundary face takes the one
 * interior cell (readings A3, A17).  g->rho_mean == 1 (the harmonic variant of A3): the face takes the mean of
 * 1/rho instead, rho_face = 2 / (1/rho_L + 1/rho_R); coefficient (O3) and correction (O10) both use it. */
static double rho_face(const orc_grid *g, const double *rho, int d, int i, int j, int k)
{
    int id[3] = {i, j, k};
    int n = g->n[d];
    int f = id[d];
    int lo[3] = {i, j, k}, hi[3] = {i, j, k};
    if (f == 0 || f == n) {
        if (is_periodic(g, d)) {
            lo[d] = n - 1;
            hi[d] = 0;
        } else if (f == 0) {
            lo[d] = hi[d] = 0;
        } else {
            lo[d] = hi[d] = n - 1;
        }
    } else {
        lo[d] = f - 1;
        hi[d] = f;
    }
    const double rl = rho[cidx(g, lo[0], lo[1], lo[2])], rh = rho[cidx(g, hi[0], hi[1], hi[2])];
    if (g->rho_mean == 1) return 2.0 / (1.0 / rl + 1.0 / rh);
    return 0.5 * (rl + rh);
}

/* ---------- O3: face coefficient b = beta0 / rho  (Eq. 2: the factor beta0/rho) --------- */

void orc_face_coeff(const orc_grid *g, const orc_base *b, const double *beta0,
                    const double *rho, double *bx, double *by, double *bz)
{
    double *out[3] = {bx, by, bz};
    for (int d = 0; d < 3; ++d) {
        int mx = g->n[0] + (d == 0), my = g->n[1] + (d == 1), mz = g->n[2] + (d == 2);
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < mz; ++k)
            for (int j = 0; j < my; ++j)
                for (int i = 0; i < mx; ++i)
                    out[d][fidx(g, d, i, j, k)] =
                        beta_face(g, b, beta0, d, i, j, k) / rho_face(g, rho, d, i, j, k);
    }
}

void orc_rho_from_profile(const orc_grid *g, const orc_base *b, const double *rho0, double *rho)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i)
                rho[cidx(g, i, j, k)] = beta_cell(g, b, rho0, i, j, k);
}

/* ---------- O11, O12: the base state of Eq. 5 and the dp0/dt term of Eq. 6 -------------------- */

void orc_make_beta0(int nr, const double *rho0, const double *p0, const double *gamma1bar, double *beta0)
{
    double lnb = log(rho0[0]);                       /* beta0(0) = rho0(0)  (Eq. 5) */
    beta0[0] = rho0[0];
    for (int m = 0; m + 1 < nr; ++m) {
        const double gmid = 0.5 * (gamma1bar[m] + gamma1bar[m + 1]);
        lnb += (log(p0[m + 1]) - log(p0[m])) / gmid; /* int (1/(Gamma1bar p0)) dp0/dr dr over [r_m, r_m+1] */
        beta0[m + 1] = exp(lnb);
    }
}

void orc_dpdt_term(int nr, const double *p0, const double *gamma1bar, const double *dp0dt, double *q)
{
    for (int m = 0; m < nr; ++m) q[m] = dp0dt[m] / (gamma1bar[m] * p0[m]);
}

void orc_effective_source(const orc_grid *g, const orc_base *b, const double *S, const double *q, double *S_eff)
{
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                const ll c = cidx(g, i, j, k);
                S_eff[c] = (S ? S[c] : 0.0) - beta_cell(g, b, q, i, j, k);   /* beta_cell: any profile at the cell centre */
            }
}

/* ---------- O13: lateral average  rho -> rho0(r) -------------------------------------- */

void orc_lateral_average(const orc_grid *g, const orc_base *b, const double *rho, double *rho0, long long *count)
{
    const int nr = b->nr;
    double *sum = (double *)calloc((size_t)nr, sizeof(double));
    ll *cnt = (ll *)calloc((size_t)nr, sizeof(ll));
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                double p[3];
                cell_pos(g, i, j, k, p);
                const double r = orc_radius(b, p[0], p[1], p[2]);
                int m = (int)floor(r / b->dr);
                if (m > nr - 1) m = nr - 1;
                if (m < 0) m = 0;
                sum[m] += rho[cidx(g, i, j, k)];
                cnt[m] += 1;
            }
    /* means of the samples that have cells */
    for (int m = 0; m < nr; ++m)
        if (cnt[m] > 0) rho0[m] = sum[m] / (double)cnt[m];
    /* samples without cells: linear in m between the nearest filled samples, constant beyond the ends */
    int prev = -1;
    for (int m = 0; m < nr; ++m) {
        if (cnt[m] == 0) continue;
        if (prev < 0)
            for (int q = 0; q < m; ++q) rho0[q] = rho0[m];
        else
            for (int q = prev + 1; q < m; ++q) {
                const double t = (double)(q - prev) / (double)(m - prev);
                rho0[q] = (1.0 - t) * rho0[prev] + t * rho0[m];
            }
        prev = m;
    }
    if (prev >= 0)
        for (int q = prev + 1; q < nr; ++q) rho0[q] = rho0[prev];
    if (count)
        for (int m = 0; m < nr; ++m) count[m] = cnt[m];
    free(sum);
    free(cnt);
}

/* ---------- O4: right-hand side  D(beta0 U_edge) - beta0 S   (Eq. 6) ------------------- */

/* velocity on face (i,j,k) of axis d; on a periodic axis face n reads entry 0 */
static double face_val(const orc_grid *g, const double *a, int d, int i, int j, int k)
{
    int id[3] = {i, j, k};
    if (is_periodic(g, d) && id[d] == g->n[d]) id[d] = 0;
    return a[fidx(g, d, id[0], id[1], id[2])];
}

void orc_constraint(const orc_grid *g, const orc_base *b, const double *beta0,
                    const double *u, const double *v, const double *w, const double *S,
                    double *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                double fxl = beta_face(g, b, beta0, 0, i, j, k) * face_val(g, u, 0, i, j, k);
                double fxh = beta_face(g, b, beta0, 0, i + 1, j, k) * face_val(g, u, 0, i + 1, j, k);
                double fyl = beta_face(g, b, beta0, 1, i, j, k) * face_val(g, v, 1, i, j, k);
                double fyh = beta_face(g, b, beta0, 1, i, j + 1, k) * face_val(g, v, 1, i, j + 1, k);
                double fzl = beta_face(g, b, beta0, 2, i, j, k) * face_val(g, w, 2, i, j, k);
                double fzh = beta_face(g, b, beta0, 2, i, j, k + 1) * face_val(g, w, 2, i, j, k + 1);
                double div = (fxh - fxl) / g->h[0] + (fyh - fyl) / g->h[1] + (fzh - fzl) / g->h[2];
                double src = S ? beta_cell(g, b, beta0, i, j, k) * S[cidx(g, i, j, k)] : 0.0;
                out[cidx(g, i, j, k)] = div - src;
            }
}

void orc_rhs(const orc_grid *g, const orc_base *b, const double *beta0,
             const double *u, const double *v, const double *w, const double *S, double *rhs)
{
    orc_constraint(g, b, beta0, u, v, w, S, rhs);
}

double orc_norm_inf(const double *a, ll n)
{
    double m = 0.0;
    int bad = 0;
#pragma omp parallel for reduction(max : m) reduction(| : bad) schedule(static)
    for (ll q = 0; q < n; ++q) {
        double v = fabs(a[q]);
        if (!(v <= 1.79769313486231570e308)) bad = 1; /* NaN or Inf */
        if (v > m) m = v;
    }
    return bad ? NAN : m;
}

/* mean: sums over chunks of 4096 entries, then a serial sum of the chunk sums, so the value does
 * not depend on the thread count */
double orc_mean(const double *a, ll n)
{
    const ll chunk = 4096;
    ll nchunk = (n + chunk - 1) / chunk;
    double *part = (double *)malloc(sizeof(double) * (size_t)(nchunk > 0 ? nchunk : 1));
#pragma omp parallel for schedule(static)
    for (ll c = 0; c < nchunk; ++c) {
        ll lo = c * chunk, hi = lo + chunk < n ? lo + chunk : n;
        double s = 0.0;
        for (ll q = lo; q < hi; ++q) s += a[q];
        part[c] = s;
    }
    double s = 0.0;
    for (ll c = 0; c < nchunk; ++c) s += part[c];
    free(part);
    return n > 0 ? s / (double)n : 0.0;
}

void orc_shift(double *a, ll n, double c)
{
#pragma omp parallel for schedule(static)
    for (ll q = 0; q < n; ++q) a[q] -= c;
}

/* reading A10: the problem is singular when no side is OUTFLOW (constants are in the null space) */
int orc_is_singular(const orc_grid *g)
{
    for (int d = 0; d < 3; ++d)
        if (g->bc_lo[d] == ORC_OUTFLOW || g->bc_hi[d] == ORC_OUTFLOW) return 0;
    return 1;
}

/* ---------- O5: operator  L phi = D(b G phi) ------------------------------------------------- */

/* phi at (i,j,k), any index possibly one outside the grid.  Ghost rule: periodic wraps; WALL
 * phi_ghost = +phi_0 (zero flux); OUTFLOW phi_ghost = -phi_0 (phi = 0 on the face). A7, A8. */
static double phi_ghost(const orc_grid *g, const double *phi, int i, int j, int k)
{
    int id[3] = {i, j, k};
    double sign = 1.0;
    for (int d = 0; d < 3; ++d) {
        int n = g->n[d];
        if (id[d] < 0) {
            if (g->bc_lo[d] == ORC_PERIODIC) {
                id[d] += n;
            } else {
                id[d] = -1 - id[d]; /* mirror: -1 -> 0 */
                if (g->bc_lo[d] == ORC_OUTFLOW) sign = -sign;
            }
        } else if (id[d] >= n) {
            if (g->bc_hi[d] == ORC_PERIODIC) {
                id[d] -= n;
            } else {
                id[d] = 2 * n - 1 - id[d]; /* mirror: n -> n-1 */
                if (g->bc_hi[d] == ORC_OUTFLOW) sign = -sign;
            }
        }
    }
    return sign * phi[cidx(g, id[0], id[1], id[2])];
}

/* coefficient on face (i,j,k) of axis d; periodic face n is face 0 */
static double bface(const orc_grid *g, const double *b, int d, int i, int j, int k)
{
    return face_val(g, b, d, i, j, k);
}

static double apply_at(const orc_grid *g, const double *bx, const double *by, const double *bz,
                       const double *phi, int i, int j, int k)
{
    double p0 = phi[cidx(g, i, j, k)];
    double hx2 = g->h[0] * g->h[0], hy2 = g->h[1] * g->h[1], hz2 = g->h[2] * g->h[2];
    double lx = (bface(g, bx, 0, i + 1, j, k) * (phi_ghost(g, phi, i + 1, j, k) - p0) -
                 bface(g, bx, 0, i, j, k) * (p0 - phi_ghost(g, phi, i - 1, j, k))) / hx2;
    double ly = (bface(g, by, 1, i, j + 1, k) * (phi_ghost(g, phi, i, j + 1, k) - p0) -
                 bface(g, by, 1, i, j, k) * (p0 - phi_ghost(g, phi, i, j - 1, k))) / hy2;
    double lz = (bface(g, bz, 2, i, j, k + 1) * (phi_ghost(g, phi, i, j, k + 1) - p0) -
                 bface(g, bz, 2, i, j, k) * (p0 - phi_ghost(g, phi, i, j, k - 1))) / hz2;
    return lx + ly + lz;
}

/* c_f = 1 interior or periodic face, 0 WALL face, 2 OUTFLOW face */
static double face_weight(const orc_grid *g, int d, int f)
{
    if (f == 0 && g->bc_lo[d] != ORC_PERIODIC) return g->bc_lo[d] == ORC_WALL ? 0.0 : 2.0;
    if (f == g->n[d] && g->bc_hi[d] != ORC_PERIODIC) return g->bc_hi[d] == ORC_WALL ? 0.0 : 2.0;
    return 1.0;
}

static double diag_at(const orc_grid *g, const double *bx, const double *by, const double *bz,
                      int i, int j, int k)
{
    double hx2 = g->h[0] * g->h[0], hy2 = g->h[1] * g->h[1], hz2 = g->h[2] * g->h[2];
    double s = 0.0;
    s += face_weight(g, 0, i) * bface(g, bx, 0, i, j, k) / hx2;
    s += face_weight(g, 0, i + 1) * bface(g, bx, 0, i + 1, j, k) / hx2;
    s += face_weight(g, 1, j) * bface(g, by, 1, i, j, k) / hy2;
    s += face_weight(g, 1, j + 1) * bface(g, by, 1, i, j + 1, k) / hy2;
    s += face_weight(g, 2, k) * bface(g, bz, 2, i, j, k) / hz2;
    s += face_weight(g, 2, k + 1) * bface(g, bz, 2, i, j, k + 1) / hz2;
    return -s;
}

void orc_apply(const orc_grid *g, const double *bx, const double *by, const double *bz,
               const double *phi, double *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i)
                out[cidx(g, i, j, k)] = apply_at(g, bx, by, bz, phi, i, j, k);
}

void orc_diag(const orc_grid *g, const double *bx, const double *by, const double *bz, double *diag)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i)
                diag[cidx(g, i, j, k)] = diag_at(g, bx, by, bz, i, j, k);
}

void orc_residual(const orc_grid *g, const double *bx, const double *by, const double *bz,
                  const double *phi, const double *rhs, double *res)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i)
                res[cidx(g, i, j, k)] = rhs[cidx(g, i, j, k)] - apply_at(g, bx, by, bz, phi, i, j, k);
}

/* ---------- O6: red-black Gauss-Seidel ------------------------------------------------------- */

/* One colour: phi_0 <- phi_0 + (rhs_0 - (L phi)_0) / L_diag, omega = 1.  A cell of one colour has
 * only neighbours of the other colour (also across periodic seams when n is even; when n is odd
 * the seam couples equal colours and the plain sequential order of this loop is what is defined,
 * hence no OpenMP in that case). */
void orc_rbgs_color(const orc_grid *g, const double *bx, const double *by, const double *bz,
                    const double *rhs, double *phi, int color)
{
    int odd_periodic = 0;
    for (int d = 0; d < 3; ++d)
        if (is_periodic(g, d) && (g->n[d] & 1)) odd_periodic = 1;
    if (odd_periodic) {
        for (int k = 0; k < g->n[2]; ++k)
            for (int j = 0; j < g->n[1]; ++j)
                for (int i = 0; i < g->n[0]; ++i) {
                    if (((i + j + k) & 1) != color) continue;
                    ll c = cidx(g, i, j, k);
                    phi[c] += (rhs[c] - apply_at(g, bx, by, bz, phi, i, j, k)) / diag_at(g, bx, by, bz, i, j, k);
                }
        return;
    }
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                if (((i + j + k) & 1) != color) continue;
                ll c = cidx(g, i, j, k);
                phi[c] += (rhs[c] - apply_at(g, bx, by, bz, phi, i, j, k)) / diag_at(g, bx, by, bz, i, j, k);
            }
}

void orc_rbgs_sweep(const orc_grid *g, const double *bx, const double *by, const double *bz,
                    const double *rhs, double *phi)
{
    orc_rbgs_color(g, bx, by, bz, rhs, phi, 0); /* red: (i+j+k) even */
    orc_rbgs_color(g, bx, by, bz, rhs, phi, 1); /* black */
}

/* ---------- O7: hierarchy -------------------------------------------------------------------- */

int orc_can_coarsen(const orc_grid *g, int coarsest_n)
{
    for (int d = 0; d < 3; ++d)
        if ((g->n[d] & 1) || g->n[d] / 2 < coarsest_n) return 0;
    return 1;
}

void orc_coarsen_grid(const orc_grid *f, orc_grid *c)
{
    for (int d = 0; d < 3; ++d) {
        c->n[d] = f->n[d] / 2;
        c->h[d] = 2.0 * f->h[d];
        c->bc_lo[d] = f->bc_lo[d];
        c->bc_hi[d] = f->bc_hi[d];
    }
    c->rho_mean = f->rho_mean;
}

/* coarse face coefficient = arithmetic mean of the 4 fine faces that tile it (reading A11) */
void orc_coarsen_coeff(const orc_grid *f, const double *bx, const double *by, const double *bz,
                       double *cbx, double *cby, double *cbz)
{
    orc_grid c;
    orc_coarsen_grid(f, &c);
    const double *in[3] = {bx, by, bz};
    double *out[3] = {cbx, cby, cbz};
    for (int d = 0; d < 3; ++d) {
        int mx = c.n[0] + (d == 0), my = c.n[1] + (d == 1), mz = c.n[2] + (d == 2);
#pragma omp parallel for collapse(2) schedule(static)
        for (int K = 0; K < mz; ++K)
            for (int J = 0; J < my; ++J)
                for (int I = 0; I < mx; ++I) {
                    int base[3] = {2 * I, 2 * J, 2 * K};
                    int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
                    double s = 0.0;
                    for (int a = 0; a < 2; ++a)
                        for (int bq = 0; bq < 2; ++bq) {
                            int id[3] = {base[0], base[1], base[2]};
                            id[t1] += a;
                            id[t2] += bq;
                            s += in[d][fidx(f, d, id[0], id[1], id[2])];
                        }
                    out[d][fidx(&c, d, I, J, K)] = 0.25 * s;
                }
    }
}

/* ---------- O8: transfers -------------------------------------------------------------------- */

void orc_restrict(const orc_grid *f, const double *fine, double *coarse)
{
    orc_grid c;
    orc_coarsen_grid(f, &c);
#pragma omp parallel for collapse(2) schedule(static)
    for (int K = 0; K < c.n[2]; ++K)
        for (int J = 0; J < c.n[1]; ++J)
            for (int I = 0; I < c.n[0]; ++I) {
                double s = 0.0;
                for (int dk = 0; dk < 2; ++dk)
                    for (int dj = 0; dj < 2; ++dj)
                        for (int di = 0; di < 2; ++di)
                            s += fine[cidx(f, 2 * I + di, 2 * J + dj, 2 * K + dk)];
                coarse[cidx(&c, I, J, K)] = 0.125 * s;
            }
}

/* fine += P coarse.  Trilinear, cell centred: along each axis a fine cell takes 3/4 of its parent
 * and 1/4 of the parent's neighbour on the fine cell's own side.  Coarse neighbours outside the
 * grid follow the ghost rule of O5.  prolongation == 1: piecewise constant. (reading A12) */
void orc_prolong_add(const orc_grid *f, const double *coarse, double *fine, int prolongation)
{
    orc_grid c;
    orc_coarsen_grid(f, &c);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < f->n[2]; ++k)
        for (int j = 0; j < f->n[1]; ++j)
            for (int i = 0; i < f->n[0]; ++i) {
                int I = i / 2, J = j / 2, K = k / 2;
                double val;
                if (prolongation == 1) {
                    val = coarse[cidx(&c, I, J, K)];
                } else {
                    int si = (i & 1) ? 1 : -1, sj = (j & 1) ? 1 : -1, sk = (k & 1) ? 1 : -1;
                    val = 0.0;
                    for (int a = 0; a < 2; ++a)
                        for (int bq = 0; bq < 2; ++bq)
                            for (int cq = 0; cq < 2; ++cq) {
                                double wgt = (a ? 0.25 : 0.75) * (bq ? 0.25 : 0.75) * (cq ? 0.25 : 0.75);
                                val += wgt * phi_ghost(&c, coarse, I + a * si, J + bq * sj, K + cq * sk);
                            }
                }
                fine[cidx(f, i, j, k)] += val;
            }
}

/* ---------- O8: bottom solve by dense elimination ------------------------------------------- */

int orc_bottom_solve(const orc_grid *g, const double *bx, const double *by, const double *bz,
                     const double *f, double *e)
{
    ll n = ncells(g);
    if (n > 4096) return -1;
    int singular = orc_is_singular(g);
    int m = (int)n + (singular ? 1 : 0);
    double *A = (double *)calloc((size_t)m * (size_t)m, sizeof(double));
    double *rhs = (double *)calloc((size_t)m, sizeof(double));
    double *unit = (double *)calloc((size_t)n, sizeof(double));
    double *col = (double *)calloc((size_t)n, sizeof(double));
    /* column q of L = L applied to the q-th unit vector */
    for (int q = 0; q < (int)n; ++q) {
        unit[q] = 1.0;
        orc_apply(g, bx, by, bz, unit, col);
        unit[q] = 0.0;
        for (int r = 0; r < (int)n; ++r) A[(size_t)r * m + q] = col[r];
    }
    double fm = singular ? orc_mean(f, n) : 0.0;
    for (int r = 0; r < (int)n; ++r) rhs[r] = f[r] - fm;
    if (singular) { /* bordered system [L 1; 1^T 0] gives the zero-mean solution */
        for (int r = 0; r < (int)n; ++r) {
            A[(size_t)r * m + n] = 1.0;
            A[(size_t)n * m + r] = 1.0;
        }
        rhs[n] = 0.0;
    }
    int status = 0;
    for (int p = 0; p < m && status == 0; ++p) {
        int piv = p;
        double best = fabs(A[(size_t)p * m + p]);
        for (int r = p + 1; r < m; ++r)
            if (fabs(A[(size_t)r * m + p]) > best) {
                best = fabs(A[(size_t)r * m + p]);
                piv = r;
            }
        if (!(best > 0.0)) {
            status = -1;
            break;
        }
        if (piv != p) {
            for (int cc = 0; cc < m; ++cc) {
                double t = A[(size_t)p * m + cc];
                A[(size_t)p * m + cc] = A[(size_t)piv * m + cc];
                A[(size_t)piv * m + cc] = t;
            }
            double t = rhs[p];
            rhs[p] = rhs[piv];
            rhs[piv] = t;
        }
        for (int r = p + 1; r < m; ++r) {
            double fct = A[(size_t)r * m + p] / A[(size_t)p * m + p];
            if (fct == 0.0) continue;
            for (int cc = p; cc < m; ++cc) A[(size_t)r * m + cc] -= fct * A[(size_t)p * m + cc];
            rhs[r] -= fct * rhs[p];
        }
    }
    if (status == 0) {
        for (int r = m - 1; r >= 0; --r) {
            double s = rhs[r];
            for (int cc = r + 1; cc < m; ++cc) s -= A[(size_t)r * m + cc] * rhs[cc];
            rhs[r] = s / A[(size_t)r * m + r];
        }
        for (int r = 0; r < (int)n; ++r) e[r] = rhs[r];
    }
    free(A);
    free(rhs);
    free(unit);
    free(col);
    return status;
}

/* ---------- O8: V-cycle ---------------------------------------------------------------------- */

typedef struct {
    int nlev;
    orc_grid grid[32];
    double *bx[32], *by[32], *bz[32]; /* level 0 entries are borrowed, the rest owned */
    double *phi[32], *rhs[32], *res[32];
} hierarchy;

static int hier_build(hierarchy *H, const orc_grid *g, const double *bx, const double *by,
                      const double *bz, int coarsest_n)
{
    memset(H, 0, sizeof(*H));
    H->grid[0] = *g;
    H->bx[0] = (double *)bx;
    H->by[0] = (double *)by;
    H->bz[0] = (double *)bz;
    H->nlev = 1;
    while (orc_can_coarsen(&H->grid[H->nlev - 1], coarsest_n) && H->nlev < 32) {
        int l = H->nlev;
        orc_coarsen_grid(&H->grid[l - 1], &H->grid[l]);
        H->bx[l] = (double *)malloc(sizeof(double) * (size_t)nfaces(&H->grid[l], 0));
        H->by[l] = (double *)malloc(sizeof(double) * (size_t)nfaces(&H->grid[l], 1));
        H->bz[l] = (double *)malloc(sizeof(double) * (size_t)nfaces(&H->grid[l], 2));
        orc_coarsen_coeff(&H->grid[l - 1], H->bx[l - 1], H->by[l - 1], H->bz[l - 1], H->bx[l], H->by[l], H->bz[l]);
        H->phi[l] = (double *)malloc(sizeof(double) * (size_t)ncells(&H->grid[l]));
        H->rhs[l] = (double *)malloc(sizeof(double) * (size_t)ncells(&H->grid[l]));
        H->nlev++;
    }
    for (int l = 0; l < H->nlev; ++l)
        H->res[l] = (double *)malloc(sizeof(double) * (size_t)ncells(&H->grid[l]));
    if (ncells(&H->grid[H->nlev - 1]) > 4096) return -2;
    return 0;
}

static void hier_free(hierarchy *H)
{
    for (int l = 0; l < H->nlev; ++l) {
        if (l > 0) {
            free(H->bx[l]);
            free(H->by[l]);
            free(H->bz[l]);
            free(H->phi[l]);
            free(H->rhs[l]);
        }
        free(H->res[l]);
    }
}

/* V-cycle on level l: nu_pre sweeps; r = f - L phi; f_c = mean of 8 children; e_c = 0; recurse;
 * phi += P e_c; nu_post sweeps.  Bottom level: exact solve. */
static int vcycle_level(hierarchy *H, int l, double *phi, const double *rhs, const orc_mg *mg)
{
    const orc_grid *g = &H->grid[l];
    if (l == H->nlev - 1) return orc_bottom_solve(g, H->bx[l], H->by[l], H->bz[l], rhs, phi);
    for (int s = 0; s < mg->nu_pre; ++s) orc_rbgs_sweep(g, H->bx[l], H->by[l], H->bz[l], rhs, phi);
    orc_residual(g, H->bx[l], H->by[l], H->bz[l], phi, rhs, H->res[l]);
    orc_restrict(g, H->res[l], H->rhs[l + 1]);
    memset(H->phi[l + 1], 0, sizeof(double) * (size_t)ncells(&H->grid[l + 1]));
    int st = vcycle_level(H, l + 1, H->phi[l + 1], H->rhs[l + 1], mg);
    if (st != 0) return st;
    orc_prolong_add(g, H->phi[l + 1], phi, mg->prolongation);
    for (int s = 0; s < mg->nu_post; ++s) orc_rbgs_sweep(g, H->bx[l], H->by[l], H->bz[l], rhs, phi);
    return 0;
}

int orc_vcycle(const orc_grid *g, const double *bx, const double *by, const double *bz,
               const double *rhs, double *phi, const orc_mg *mg)
{
    hierarchy H;
    int st = hier_build(&H, g, bx, by, bz, mg->coarsest_n);
    if (st == 0) st = vcycle_level(&H, 0, phi, rhs, mg);
    hier_free(&H);
    return st;
}

/* ---------- O10: velocity correction  U <- U_edge - (1/rho_face) G phi  (Eq. 2) --------- */

void orc_correct(const orc_grid *g, const double *rho, const double *phi,
                 double *u, double *v, double *w)
{
    double *vel[3] = {u, v, w};
    for (int d = 0; d < 3; ++d) {
        int mx = g->n[0] + (d == 0), my = g->n[1] + (d == 1), mz = g->n[2] + (d == 2);
        int n = g->n[d];
        double h = g->h[d];
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < mz; ++k)
            for (int j = 0; j < my; ++j)
                for (int i = 0; i < mx; ++i) {
                    int id[3] = {i, j, k};
                    int f = id[d];
                    if (f == n && is_periodic(g, d)) continue; /* copied from face 0 below */
                    int lo[3] = {i, j, k}, hi[3] = {i, j, k};
                    lo[d] = f - 1;
                    hi[d] = f;
                    double grad;
                    if (f == 0 && !is_periodic(g, d)) {
                        if (g->bc_lo[d] == ORC_WALL) continue;
                        grad = 2.0 * phi[cidx(g, hi[0], hi[1], hi[2])] / h; /* (phi_0 - (-phi_0))/h */
                    } else if (f == n) {
                        if (g->bc_hi[d] == ORC_WALL) continue;
                        grad = -2.0 * phi[cidx(g, lo[0], lo[1], lo[2])] / h;
                    } else {
                        grad = (phi_ghost(g, phi, hi[0], hi[1], hi[2]) - phi_ghost(g, phi, lo[0], lo[1], lo[2])) / h;
                    }
                    vel[d][fidx(g, d, i, j, k)] -= grad / rho_face(g, rho, d, i, j, k);
                }
        if (is_periodic(g, d)) {
#pragma omp parallel for collapse(2) schedule(static)
            for (int k = 0; k < mz; ++k)
                for (int j = 0; j < my; ++j)
                    for (int i = 0; i < mx; ++i) {
                        int id[3] = {i, j, k};
                        if (id[d] != n) continue;
                        int z[3] = {i, j, k};
                        z[d] = 0;
                        vel[d][fidx(g, d, i, j, k)] = vel[d][fidx(g, d, z[0], z[1], z[2])];
                    }
        }
    }
}

/* ---------- O9: driver ----------------------------------------------------------------------- */

int orc_project(const orc_grid *g, const orc_base *b, const orc_mg *mg,
                const double *beta0, const double *rho0, const double *rho_in,
                double *u, double *v, double *w, const double *S, double *phi_out,
                orc_stats *stats)
{
    ll nc = ncells(g);
    orc_stats st;
    memset(&st, 0, sizeof(st));
    int ret = 0;
    double *rho_own = NULL;
    const double *rho = rho_in;
    if (!rho) {
        rho_own = (double *)malloc(sizeof(double) * (size_t)nc);
        orc_rho_from_profile(g, b, rho0, rho_own);
        rho = rho_own;
    }
    double *bx = (double *)malloc(sizeof(double) * (size_t)nfaces(g, 0));
    double *by = (double *)malloc(sizeof(double) * (size_t)nfaces(g, 1));
    double *bz = (double *)malloc(sizeof(double) * (size_t)nfaces(g, 2));
    double *rhs = (double *)malloc(sizeof(double) * (size_t)nc);
    double *phi = (double *)calloc((size_t)nc, sizeof(double)); /* A16: phi = 0 */
    hierarchy H;
    memset(&H, 0, sizeof(H));

    /* every density must be positive and finite */
    int bad_rho = 0;
#pragma omp parallel for reduction(| : bad_rho) schedule(static)
    for (ll q = 0; q < nc; ++q)
        if (!(rho[q] > 0.0) || !(rho[q] <= 1.79769313486231570e308)) bad_rho = 1;

    orc_face_coeff(g, b, beta0, rho, bx, by, bz);
    orc_rhs(g, b, beta0, u, v, w, S, rhs);
    st.singular = orc_is_singular(g);
    if (st.singular) { /* A10: remove the mean so the system is solvable */
        st.rhs_mean_removed = orc_mean(rhs, nc);
        orc_shift(rhs, nc, st.rhs_mean_removed);
    }
    st.rhs_norm_inf = orc_norm_inf(rhs, nc);
    if (bad_rho || isnan(st.rhs_norm_inf) || isinf(st.rhs_norm_inf)) {
        ret = -5;
        goto done;
    }
    ret = hier_build(&H, g, bx, by, bz, mg->coarsest_n);
    st.levels = H.nlev;
    if (ret != 0) goto done;

    if (st.rhs_norm_inf == 0.0) { /* nothing to project: phi = 0, U untouched */
        st.converged = 1;
    } else {
        ret = 1;
        while (st.cycles < mg->max_cycles) {
            int vs = vcycle_level(&H, 0, phi, rhs, mg);
            if (vs != 0) {
                ret = -5;
                goto done;
            }
            orc_residual(g, bx, by, bz, phi, rhs, H.res[0]);
            st.res_norm_inf = orc_norm_inf(H.res[0], nc);
            double rel = st.res_norm_inf / st.rhs_norm_inf;
            if (st.cycles < 128) st.res_history[st.cycles] = rel;
            st.cycles++;
            if (isnan(rel)) {
                ret = -5;
                goto done;
            }
            if (mg->rel_tol > 0.0 && rel <= mg->rel_tol) { /* A14 */
                st.converged = 1;
                ret = 0;
                break;
            }
        }
        if (mg->rel_tol <= 0.0) ret = 0; /* fixed cycle count requested */
        if (st.singular) orc_shift(phi, nc, orc_mean(phi, nc));
        orc_correct(g, rho, phi, u, v, w);
    }
    if (phi_out) memcpy(phi_out, phi, sizeof(double) * (size_t)nc);

done:
    hier_free(&H);
    free(bx);
    free(by);
    free(bz);
    free(rhs);
    free(phi);
    free(rho_own);
    if (stats) *stats = st;
    return ret;
}
