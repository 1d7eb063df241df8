/*
 * nodal_oracle.c -- CPU fp64 ORACLE for the end-of-step (nodal) projection (TEST INFRASTRUCTURE).
 * See nodal_oracle.h for scope, citations (Eq. 2, Eq. 6), the readings N1..N10 and the pins.
 *
 * Plain loops in the order of the readings; the operator is written element by element (for every node the up
 * to 8 cells around it, for every cell its 8 corners) with no stencil precomputation.  OpenMP only on loops
 * whose iterations are independent; sums are taken plane by plane and added serially, so results do not
 * depend on the thread count.
 */
#include "nodal_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef long long ll;

/* ---------- indexing ------------------------------------------------------------------------ */

static inline ll cidx(const orc_grid *g, int i, int j, int k)
{
    return (ll)i + (ll)g->n[0] * ((ll)j + (ll)g->n[1] * (ll)k);
}
static inline ll nidx(const orc_grid *g, int i, int j, int k)
{
    return (ll)i + (ll)(g->n[0] + 1) * ((ll)j + (ll)(g->n[1] + 1) * (ll)k);
}
static inline ll ncells(const orc_grid *g) { return (ll)g->n[0] * g->n[1] * g->n[2]; }
static inline ll nnodes(const orc_grid *g) { return (ll)(g->n[0] + 1) * (g->n[1] + 1) * (g->n[2] + 1); }
static inline int is_periodic(const orc_grid *g, int d) { return g->bc_lo[d] == ORC_PERIODIC; }

/* N4: kind of node index t along axis d: 0 unknown, 1 OUTFLOW node, 2 periodic duplicate */
static inline int axis_kind(const orc_grid *g, int d, int t)
{
    if (is_periodic(g, d)) return t == g->n[d] ? 2 : 0;
    if (t == 0 && g->bc_lo[d] == ORC_OUTFLOW) return 1;
    if (t == g->n[d] && g->bc_hi[d] == ORC_OUTFLOW) return 1;
    return 0;
}
static inline int node_kind(const orc_grid *g, int i, int j, int k)
{
    int a = axis_kind(g, 0, i), b = axis_kind(g, 1, j), c = axis_kind(g, 2, k);
    if (a == 1 || b == 1 || c == 1) return 1;
    if (a == 2 || b == 2 || c == 2) return 2;
    return 0;
}
void nod_node_kind(const orc_grid *g, int *kind)
{
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i) kind[nidx(g, i, j, k)] = node_kind(g, i, j, k);
}
/* phi at node (i,j,k) under the node rules of N4 */
static inline double node_val(const orc_grid *g, const double *phi, int i, int j, int k)
{
    if (node_kind(g, i, j, k) == 1) return 0.0;
    if (is_periodic(g, 0) && i == g->n[0]) i = 0;
    if (is_periodic(g, 1) && j == g->n[1]) j = 0;
    if (is_periodic(g, 2) && k == g->n[2]) k = 0;
    return phi[nidx(g, i, j, k)];
}
/* the cell at offset o in {-1, 0} from node index t along axis d: its index, or -1 if it does not exist */
static inline int cell_of_node(const orc_grid *g, int d, int t, int o)
{
    int c = t + o;
    if (c < 0) return is_periodic(g, d) ? g->n[d] - 1 : -1;
    if (c >= g->n[d]) return -1; /* t == n on a non-periodic axis (periodic duplicates are never visited) */
    return c;
}

/* N7 */
double nod_omega(const orc_grid *g)
{
    double gd[3], sum = 0.0, mx = 0.0;
    for (int d = 0; d < 3; ++d) {
        gd[d] = 1.0 / (g->h[d] * g->h[d]);
        sum += gd[d];
        if (gd[d] > mx) mx = gd[d];
    }
    return sum / (3.0 * mx);
}

/* N2: K^c_ab / V for corners sa, sb of a cell */
static inline double kelem(const orc_grid *g, const int sa[3], const int sb[3])
{
    double s = 0.0;
    for (int d = 0; d < 3; ++d) {
        double t = (sa[d] == sb[d] ? 1.0 : -1.0) / (g->h[d] * g->h[d]);
        for (int e = 0; e < 3; ++e)
            if (e != d) t *= (sa[e] == sb[e]) ? (1.0 / 3.0) : (1.0 / 6.0);
        s += t;
    }
    return s;
}

void nod_weights(const orc_grid *g, double *wgt)
{
#pragma omp parallel for schedule(static)
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i) {
                double w = 0.0;
                if (node_kind(g, i, j, k) == 0)
                    for (int ok = -1; ok <= 0; ++ok)
                        for (int oj = -1; oj <= 0; ++oj)
                            for (int oi = -1; oi <= 0; ++oi)
                                if (cell_of_node(g, 0, i, oi) >= 0 && cell_of_node(g, 1, j, oj) >= 0 &&
                                    cell_of_node(g, 2, k, ok) >= 0)
                                    w += 0.125;
                wgt[nidx(g, i, j, k)] = w;
            }
}

/* N3 */
void nod_sigma(const orc_grid *g, const orc_base *b, const double *beta0, const double *rho, double *sigma)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                double r = orc_radius(b, (i + 0.5) * g->h[0], (j + 0.5) * g->h[1], (k + 0.5) * g->h[2]);
                sigma[cidx(g, i, j, k)] = orc_profile(beta0, b->nr, b->dr, r) / rho[cidx(g, i, j, k)];
            }
}

/* ---------- N1/N2: operator ------------------------------------------------------------------ */

/* (L phi)_a at node (i,j,k); diag_only: L_aa */
static double apply_at(const orc_grid *g, const double *sigma, const double *phi, int i, int j, int k, int diag_only)
{
    double acc = 0.0;
    for (int ok = -1; ok <= 0; ++ok)
        for (int oj = -1; oj <= 0; ++oj)
            for (int oi = -1; oi <= 0; ++oi) {
                int ci = cell_of_node(g, 0, i, oi), cj = cell_of_node(g, 1, j, oj), ck = cell_of_node(g, 2, k, ok);
                if (ci < 0 || cj < 0 || ck < 0) continue;
                const int sa[3] = {-oi, -oj, -ok}; /* which corner of the cell node a is */
                double cell = 0.0;
                if (diag_only) {
                    cell = kelem(g, sa, sa);
                } else {
                    for (int tk = 0; tk <= 1; ++tk)
                        for (int tj = 0; tj <= 1; ++tj)
                            for (int ti = 0; ti <= 1; ++ti) {
                                const int sb[3] = {ti, tj, tk};
                                cell += kelem(g, sa, sb) * node_val(g, phi, ci + ti, cj + tj, ck + tk);
                            }
                }
                acc += sigma[cidx(g, ci, cj, ck)] * cell;
            }
    return -acc;
}

void nod_apply(const orc_grid *g, const double *sigma, const double *phi, double *out)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i)
                out[nidx(g, i, j, k)] = node_kind(g, i, j, k) == 0 ? apply_at(g, sigma, phi, i, j, k, 0) : 0.0;
}

void nod_diag(const orc_grid *g, const double *sigma, double *diag)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i)
                diag[nidx(g, i, j, k)] = node_kind(g, i, j, k) == 0 ? apply_at(g, sigma, NULL, i, j, k, 1) : 0.0;
}

void nod_residual(const orc_grid *g, const double *sigma, const double *phi, const double *rhs, double *res)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i) {
                ll a = nidx(g, i, j, k);
                res[a] = node_kind(g, i, j, k) == 0 ? rhs[a] - apply_at(g, sigma, phi, i, j, k, 0) : 0.0;
            }
}

/* ---------- N1: right-hand side --------------------------------------------------------------- */

void nod_rhs(const orc_grid *g, const orc_base *b, const double *beta0, const double *u, const double *v,
             const double *w, const double *S, double *rhs)
{
    const double *vel[3] = {u, v, w};
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i) {
                double acc = 0.0;
                if (node_kind(g, i, j, k) == 0)
                    for (int ok = -1; ok <= 0; ++ok)
                        for (int oj = -1; oj <= 0; ++oj)
                            for (int oi = -1; oi <= 0; ++oi) {
                                int ci = cell_of_node(g, 0, i, oi), cj = cell_of_node(g, 1, j, oj), ck = cell_of_node(g, 2, k, ok);
                                if (ci < 0 || cj < 0 || ck < 0) continue;
                                const int sa[3] = {-oi, -oj, -ok};
                                ll c = cidx(g, ci, cj, ck);
                                double r = orc_radius(b, (ci + 0.5) * g->h[0], (cj + 0.5) * g->h[1], (ck + 0.5) * g->h[2]);
                                double bc = orc_profile(beta0, b->nr, b->dr, r);
                                for (int d = 0; d < 3; ++d) /* (D F)_a: -(2 s_d - 1) F_c,d / (4 h_d) */
                                    acc -= (2 * sa[d] - 1) * (bc * vel[d][c]) / (4.0 * g->h[d]);
                                if (S) acc -= 0.125 * (bc * S[c]); /* (M f)_a */
                            }
                rhs[nidx(g, i, j, k)] = acc;
            }
}

void nod_constraint(const orc_grid *g, const orc_base *b, const double *beta0, const double *u, const double *v,
                    const double *w, const double *S, double *out)
{
    nod_rhs(g, b, beta0, u, v, w, S, out);
}

/* ---------- reductions over the unknowns ------------------------------------------------------ */

double nod_norm_inf(const orc_grid *g, const double *f)
{
    double m = 0.0;
    int nan_seen = 0;
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i)
                if (node_kind(g, i, j, k) == 0) {
                    double a = fabs(f[nidx(g, i, j, k)]);
                    if (a != a) nan_seen = 1;
                    if (a > m) m = a;
                }
    return nan_seen ? NAN : m;
}

/* sum over the unknowns of w_a f_a (wgt != NULL) or of f_a: plane sums added serially */
static double node_sum(const orc_grid *g, const double *f, const double *wgt)
{
    int nzp = g->n[2] + 1;
    double *pl = (double *)calloc((size_t)nzp, sizeof(double));
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nzp; ++k) {
        double s = 0.0;
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i)
                if (node_kind(g, i, j, k) == 0) {
                    ll a = nidx(g, i, j, k);
                    s += wgt ? wgt[a] * f[a] : f[a];
                }
        pl[k] = s;
    }
    double tot = 0.0;
    for (int k = 0; k < nzp; ++k) tot += pl[k];
    free(pl);
    return tot;
}

double nod_weighted_mean(const orc_grid *g, const double *f)
{
    double *wgt = (double *)malloc(sizeof(double) * (size_t)nnodes(g));
    nod_weights(g, wgt);
    double s = node_sum(g, f, wgt);
    free(wgt);
    return s / (double)ncells(g); /* sum_a w_a = number of cells */
}

/* ---------- N7: Jacobi ------------------------------------------------------------------------ */

void nod_jacobi(const orc_grid *g, const double *sigma, const double *rhs, double *phi, double omega)
{
    ll nn = nnodes(g);
    double *nw = (double *)malloc(sizeof(double) * (size_t)nn);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k <= g->n[2]; ++k)
        for (int j = 0; j <= g->n[1]; ++j)
            for (int i = 0; i <= g->n[0]; ++i) {
                ll a = nidx(g, i, j, k);
                if (node_kind(g, i, j, k) != 0) {
                    nw[a] = 0.0;
                    continue;
                }
                double lp = apply_at(g, sigma, phi, i, j, k, 0);
                double dg = apply_at(g, sigma, NULL, i, j, k, 1);
                nw[a] = phi[a] + omega * (rhs[a] - lp) / dg;
            }
    memcpy(phi, nw, sizeof(double) * (size_t)nn);
    free(nw);
}

/* ---------- N6: transfers --------------------------------------------------------------------- */

void nod_coarsen_sigma(const orc_grid *f, const double *sf, double *sc)
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
                        for (int di = 0; di < 2; ++di) s += sf[cidx(f, 2 * I + di, 2 * J + dj, 2 * K + dk)];
                sc[cidx(&c, I, J, K)] = 0.125 * s;
            }
}

/* fine node index 2 T + o along axis d mapped to a stored unknown index, or -1 if there is no such node */
static inline int fine_of_coarse(const orc_grid *f, int d, int T, int o)
{
    int t = 2 * T + o;
    if (is_periodic(f, d)) {
        if (t < 0) t += f->n[d];
        if (t >= f->n[d]) t -= f->n[d];
        return t;
    }
    if (t < 0 || t > f->n[d]) return -1;
    return t;
}

/* coarse = (1/8) P^T fine: weights 1, 1/2 per axis over the 27 fine nodes around the coincident one */
void nod_restrict(const orc_grid *f, const double *fine, double *coarse)
{
    orc_grid c;
    orc_coarsen_grid(f, &c);
#pragma omp parallel for collapse(2) schedule(static)
    for (int K = 0; K <= c.n[2]; ++K)
        for (int J = 0; J <= c.n[1]; ++J)
            for (int I = 0; I <= c.n[0]; ++I) {
                double s = 0.0;
                if (node_kind(&c, I, J, K) == 0)
                    for (int ok = -1; ok <= 1; ++ok)
                        for (int oj = -1; oj <= 1; ++oj)
                            for (int oi = -1; oi <= 1; ++oi) {
                                int i = fine_of_coarse(f, 0, I, oi), j = fine_of_coarse(f, 1, J, oj), k = fine_of_coarse(f, 2, K, ok);
                                if (i < 0 || j < 0 || k < 0) continue;
                                if (node_kind(f, i, j, k) != 0) continue; /* OUTFLOW nodes carry no residual */
                                double wt = (oi ? 0.5 : 1.0) * (oj ? 0.5 : 1.0) * (ok ? 0.5 : 1.0);
                                s += wt * fine[nidx(f, i, j, k)];
                            }
                coarse[nidx(&c, I, J, K)] = 0.125 * s;
            }
}

/* fine += P coarse at the fine unknowns: trilinear interpolation from the coarse nodes (node rules of N4) */
void nod_prolong_add(const orc_grid *f, const double *coarse, double *fine)
{
    orc_grid c;
    orc_coarsen_grid(f, &c);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k <= f->n[2]; ++k)
        for (int j = 0; j <= f->n[1]; ++j)
            for (int i = 0; i <= f->n[0]; ++i) {
                if (node_kind(f, i, j, k) != 0) continue;
                int lo[3] = {i >> 1, j >> 1, k >> 1};
                int odd[3] = {i & 1, j & 1, k & 1};
                double s = 0.0;
                for (int tk = 0; tk <= odd[2]; ++tk)
                    for (int tj = 0; tj <= odd[1]; ++tj)
                        for (int ti = 0; ti <= odd[0]; ++ti) {
                            double wt = (odd[0] ? 0.5 : 1.0) * (odd[1] ? 0.5 : 1.0) * (odd[2] ? 0.5 : 1.0);
                            s += wt * node_val(&c, coarse, lo[0] + ti, lo[1] + tj, lo[2] + tk);
                        }
                fine[nidx(f, i, j, k)] += s;
            }
}

/* ---------- N8: bottom solve ------------------------------------------------------------------ */

int nod_bottom_solve(const orc_grid *g, const double *sigma, const double *f, double *e)
{
    ll nn = nnodes(g);
    int *kind = (int *)malloc(sizeof(int) * (size_t)nn);
    int *list = (int *)malloc(sizeof(int) * (size_t)nn);
    nod_node_kind(g, kind);
    int n = 0;
    for (ll a = 0; a < nn; ++a)
        if (kind[a] == 0) list[n++] = (int)a;
    if (n > 6000) {
        free(kind);
        free(list);
        return -1;
    }
    int singular = orc_is_singular(g);
    int m = n + (singular ? 1 : 0);
    double *A = (double *)calloc((size_t)m * (size_t)m, sizeof(double));
    double *rhs = (double *)calloc((size_t)m, sizeof(double));
    double *unit = (double *)calloc((size_t)nn, sizeof(double));
    double *col = (double *)calloc((size_t)nn, sizeof(double));
    for (int q = 0; q < n; ++q) { /* column q of L = L applied to the q-th unit vector */
        unit[list[q]] = 1.0;
        nod_apply(g, sigma, unit, col);
        unit[list[q]] = 0.0;
        for (int r = 0; r < n; ++r) A[(size_t)r * m + q] = col[list[r]];
    }
    double fm = 0.0;
    if (singular) {
        for (int r = 0; r < n; ++r) fm += f[list[r]];
        fm /= (double)n;
    }
    for (int r = 0; r < n; ++r) rhs[r] = f[list[r]] - fm;
    if (singular) { /* bordered system [L 1; 1^T 0]: the solution with zero plain mean */
        for (int r = 0; r < n; ++r) {
            A[(size_t)r * m + n] = 1.0;
            A[(size_t)n * m + r] = 1.0;
        }
    }
    int status = 0;
    for (int p = 0; p < m && status == 0; ++p) { /* Gaussian elimination with partial pivoting */
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
        memset(e, 0, sizeof(double) * (size_t)nn);
        for (int r = 0; r < n; ++r) e[list[r]] = rhs[r];
    }
    free(A);
    free(rhs);
    free(unit);
    free(col);
    free(kind);
    free(list);
    return status;
}

/* ---------- N6/N8: V-cycle -------------------------------------------------------------------- */

#define NOD_MAXLEV 32
typedef struct {
    int nlev;
    orc_grid grid[NOD_MAXLEV];
    double *sigma[NOD_MAXLEV], *phi[NOD_MAXLEV], *rhs[NOD_MAXLEV], *res[NOD_MAXLEV];
    double omega;
} nod_hier;

static void nhier_free(nod_hier *H)
{
    for (int l = 0; l < H->nlev; ++l) {
        if (l > 0) free(H->sigma[l]);
        free(H->phi[l]);
        free(H->rhs[l]);
        free(H->res[l]);
    }
    H->nlev = 0;
}

static int nhier_build(nod_hier *H, const orc_grid *g, const double *sigma, int coarsest_n)
{
    memset(H, 0, sizeof(*H));
    H->grid[0] = *g;
    H->sigma[0] = (double *)sigma;
    H->omega = nod_omega(g);
    int l = 0;
    for (;;) {
        ll nn = nnodes(&H->grid[l]);
        H->phi[l] = (double *)calloc((size_t)nn, sizeof(double));
        H->rhs[l] = (double *)calloc((size_t)nn, sizeof(double));
        H->res[l] = (double *)calloc((size_t)nn, sizeof(double));
        H->nlev = l + 1;
        if (!orc_can_coarsen(&H->grid[l], coarsest_n) || l + 1 >= NOD_MAXLEV) break;
        orc_coarsen_grid(&H->grid[l], &H->grid[l + 1]);
        H->sigma[l + 1] = (double *)malloc(sizeof(double) * (size_t)ncells(&H->grid[l + 1]));
        nod_coarsen_sigma(&H->grid[l], H->sigma[l], H->sigma[l + 1]);
        ++l;
    }
    if (ncells(&H->grid[H->nlev - 1]) > 4096) return -2;
    return 0;
}

static int nvcycle_level(nod_hier *H, int l, double *phi, const double *rhs, const orc_mg *mg)
{
    const orc_grid *g = &H->grid[l];
    if (l == H->nlev - 1) return nod_bottom_solve(g, H->sigma[l], rhs, phi);
    for (int s = 0; s < mg->nu_pre; ++s) nod_jacobi(g, H->sigma[l], rhs, phi, H->omega);
    nod_residual(g, H->sigma[l], phi, rhs, H->res[l]);
    nod_restrict(g, H->res[l], H->rhs[l + 1]);
    memset(H->phi[l + 1], 0, sizeof(double) * (size_t)nnodes(&H->grid[l + 1]));
    int st = nvcycle_level(H, l + 1, H->phi[l + 1], H->rhs[l + 1], mg);
    if (st != 0) return st;
    nod_prolong_add(g, H->phi[l + 1], phi);
    for (int s = 0; s < mg->nu_post; ++s) nod_jacobi(g, H->sigma[l], rhs, phi, H->omega);
    return 0;
}

int nod_vcycle(const orc_grid *g, const double *sigma, const double *rhs, double *phi, const orc_mg *mg)
{
    nod_hier H;
    int st = nhier_build(&H, g, sigma, mg->coarsest_n);
    if (st == 0) st = nvcycle_level(&H, 0, phi, rhs, mg);
    nhier_free(&H);
    return st;
}

/* ---------- N10: correction ------------------------------------------------------------------- */

void nod_correct(const orc_grid *g, const double *rho, const double *phi, double *u, double *v, double *w)
{
    double *vel[3] = {u, v, w};
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->n[2]; ++k)
        for (int j = 0; j < g->n[1]; ++j)
            for (int i = 0; i < g->n[0]; ++i) {
                ll c = cidx(g, i, j, k);
                double grad[3] = {0.0, 0.0, 0.0};
                for (int tk = 0; tk <= 1; ++tk)
                    for (int tj = 0; tj <= 1; ++tj)
                        for (int ti = 0; ti <= 1; ++ti) {
                            const int sb[3] = {ti, tj, tk};
                            double p = node_val(g, phi, i + ti, j + tj, k + tk);
                            for (int d = 0; d < 3; ++d) grad[d] += (2 * sb[d] - 1) * p / (4.0 * g->h[d]);
                        }
                for (int d = 0; d < 3; ++d) vel[d][c] -= grad[d] / rho[c];
            }
}

/* ---------- driver ---------------------------------------------------------------------------- */

int nod_project(const orc_grid *g, const orc_base *b, const orc_mg *mg, const double *beta0, const double *rho0,
                const double *rho_in, double *u, double *v, double *w, const double *S, double *phi_out,
                orc_stats *stats)
{
    ll nc = ncells(g), nn = nnodes(g);
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
    double *sigma = (double *)malloc(sizeof(double) * (size_t)nc);
    double *rhs = (double *)malloc(sizeof(double) * (size_t)nn);
    double *wgt = (double *)malloc(sizeof(double) * (size_t)nn);
    double *phi = (double *)calloc((size_t)nn, sizeof(double)); /* N9: phi = 0 */
    nod_hier H;
    memset(&H, 0, sizeof(H));

    int bad_rho = 0;
#pragma omp parallel for reduction(| : bad_rho) schedule(static)
    for (ll q = 0; q < nc; ++q)
        if (!(rho[q] > 0.0) || !(rho[q] <= 1.79769313486231570e308)) bad_rho = 1;

    nod_sigma(g, b, beta0, rho, sigma);
    nod_rhs(g, b, beta0, u, v, w, S, rhs);
    nod_weights(g, wgt);
    st.singular = orc_is_singular(g);
    if (st.singular) { /* N5 */
        st.rhs_mean_removed = node_sum(g, rhs, NULL) / (double)nc;
        for (ll a = 0; a < nn; ++a) rhs[a] -= st.rhs_mean_removed * wgt[a];
    }
    st.rhs_norm_inf = nod_norm_inf(g, rhs);
    if (bad_rho || isnan(st.rhs_norm_inf) || isinf(st.rhs_norm_inf)) {
        ret = -5;
        goto done;
    }
    ret = nhier_build(&H, g, sigma, mg->coarsest_n);
    st.levels = H.nlev;
    if (ret != 0) goto done;

    if (st.rhs_norm_inf == 0.0) {
        st.converged = 1;
    } else {
        ret = 1;
        while (st.cycles < mg->max_cycles) {
            int vs = nvcycle_level(&H, 0, phi, rhs, mg);
            if (vs != 0) {
                ret = -5;
                goto done;
            }
            nod_residual(g, sigma, phi, rhs, H.res[0]);
            st.res_norm_inf = nod_norm_inf(g, H.res[0]);
            double rel = st.res_norm_inf / st.rhs_norm_inf;
            if (st.cycles < 128) st.res_history[st.cycles] = rel;
            st.cycles++;
            if (rel != rel) {
                ret = -5;
                goto done;
            }
            if (mg->rel_tol > 0.0 && rel <= mg->rel_tol) {
                ret = 0;
                st.converged = 1;
                break;
            }
        }
        if (mg->rel_tol == 0.0) ret = 0;
        if (st.singular) { /* N5: zero w-weighted mean */
            double mean = node_sum(g, phi, wgt) / (double)nc;
            for (ll a = 0; a < nn; ++a) phi[a] -= mean;
        }
        /* N4: OUTFLOW nodes are 0, periodic duplicates equal their image */
        for (int k = 0; k <= g->n[2]; ++k)
            for (int j = 0; j <= g->n[1]; ++j)
                for (int i = 0; i <= g->n[0]; ++i)
                    if (node_kind(g, i, j, k) != 0) phi[nidx(g, i, j, k)] = node_val(g, phi, i, j, k);
        nod_correct(g, rho, phi, u, v, w);
    }
    if (phi_out) memcpy(phi_out, phi, sizeof(double) * (size_t)nn);
done:
    if (stats) *stats = st;
    nhier_free(&H);
    free(rho_own);
    free(sigma);
    free(rhs);
    free(wgt);
    free(phi);
    return ret;
}
