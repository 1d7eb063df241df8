/*
 * nodal_oracle.h -- CPU fp64 ORACLE for the end-of-step (nodal) projection of MAESTROeX (TEST INFRASTRUCTURE).
 *
 * This is test infrastructure, not the product.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load it.  It shares no code with the CUDA path under
 * paper_1910_12979_b200/csrc/ and neither includes the other.  (It uses orc_grid, orc_base, orc_mg, orc_stats,
 * orc_profile and orc_radius of mac_oracle.h, the MAC projection's oracle: same grid, same base state.)
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, "P:n" = line n).  The paper integrates velocity by a
 * "second order projection method" with "multigrid linear solvers for the pressure projection steps" -- plural,
 * P:63 (Sec. 3): besides the MAC projection of the face velocities there is the projection of the CELL-CENTRED
 * velocity at the end of the step.  It enforces the same constraint
 *        div(beta0 U) = beta0 (S - (1/(Gamma1bar p0)) dp0/dt)           P:49 (Sec. 2, Eq. 6)
 * (the dp0/dt term folded into S by the caller) with the same weighting beta0/rho of the pressure term
 *        (beta0/rho) grad(pi/beta0)                                     P:35 (Sec. 2, Eq. 2)
 * on the same one-dimensional base state.  The paper describes neither projection; every
 * concrete choice is a reading, listed in DESIGN.md ("Nodal projection: readings", N1..N10):
 *
 *  N1  phi lives on the NODES (corners) of the cells, (nx+1)(ny+1)(nz+1) values; U = (u, v, w), rho, S and
 *      sigma = beta0(r_cell)/rho are cell-centred.  Find phi with, for every trilinear nodal hat function psi_a,
 *          int sigma grad(phi).grad(psi_a) = int beta0 U.grad(psi_a) + int beta0 S psi_a
 *      (the weak form of div(beta0 (U - (1/rho) grad phi)) = beta0 S; phi trilinear, sigma / beta0 U / beta0 S
 *      constant per cell, integrals exact), then U <- U - (1/rho) G phi with G the cell-mean gradient.
 *      Written like the MAC system, L phi = rhs with a negative semi-definite L, both sides divided by the cell
 *      volume V = dx dy dz:
 *          (L phi)_a = -(1/V) sum_c sigma_c sum_b K^c_ab phi_b,      K^c_ab = int_c grad psi_a . grad psi_b
 *          rhs_a     = (D(beta0 U))_a - (M(beta0 S))_a
 *          (D F)_a   = -(1/V) sum_c F_c . int_c grad psi_a = sum_c sum_d -(2 s_d - 1) F_c,d / (4 h_d)
 *          (M f)_a   = (1/V) sum_c f_c int_c psi_a = (1/8) sum_c f_c
 *      (c: the up to 8 cells around node a; s_d in {0,1}: the corner of cell c that a is, along axis d).
 *      This is the approximate nodal projection with the 27-point finite-element stencil (Almgren, Bell, Szymczak
 *      1996; the one-point-quadrature operator D sigma G would be an exact projection but decouples into
 *      checkerboard modes).
 *  N2  K^c_ab / V = sum_d (1/h_d^2) k(sa_d, sb_d) prod_{e != d} m(sa_e, sb_e),   k = +1 same corner / -1 other,
 *      m = 1/3 same / 1/6 other.  Unit cube, sigma = 1: centre 8/3, face neighbours 0, edge neighbours -1/6, corner
 *      neighbours -1/12 (the textbook Q1 stencil).
 *  N3  beta0 at a cell centre: the profile at the centre's radius (O1 of the MAC oracle).
 *  N4  Boundaries.  WALL: natural condition -- boundary nodes are unknowns, sums run over the cells that exist,
 *      the boundary integral vanishes for U.n = 0.  OUTFLOW: phi = 0 on the nodes of that side; they are not
 *      unknowns (their rhs, residual and phi are 0).  PERIODIC: node n is node 0; arrays keep n+1 entries per
 *      axis, entry n is ignored on input and written equal to entry 0 on output.
 *  N5  No OUTFLOW side: the system is singular.  m = sum_a rhs_a / sum_a w_a with w_a = (cells around a)/8 (sum
 *      over the unknowns; sum_a w_a = cell count) is removed as a uniform volumetric source, rhs_a -= m w_a, and
 *      phi is returned with zero w-weighted mean.
 *  N6  Hierarchy: the MAC cell hierarchy; coarse sigma = mean of the 8 fine cells; coarse nodes are the even fine
 *      nodes.  Prolongation P = trilinear interpolation (weights 1, 1/2, 1/4, 1/8); restriction R = P^T / 8
 *      (the weak-form residuals V r are summed with P^T and divided by the coarse volume 8 V); rows and columns
 *      of OUTFLOW nodes dropped, periodic axes wrap.
 *  N7  Smoother: nu Jacobi sweeps, phi <- phi + omega (rhs - L phi)/L_aa, omega = sum_d g_d / (3 max_d g_d),
 *      g_d = 1/h_d^2 (= 1 for cubic cells: the eigenvalues of diag^-1 L of the Q1 stencil on high frequencies lie
 *      in [1/2, 3/2]; the formula keeps omega * lambda_max = 3/2 on stretched cells).  A 27-point stencil does
 *      not two-colour; Jacobi is order-free, hence reproducible on a GPU, and needs one pass per sweep.
 *  N8  Bottom level: solved exactly (dense elimination; singular case bordered, zero plain mean).
 *  N9  Stop: ||rhs - L phi||inf <= rel_tol ||rhs||inf over the unknowns after each cycle.  phi = 0 initially.
 *  N10 Correction: (G_d phi)_c = sum_b (2 sb_d - 1) phi_b / (4 h_d) over the 8 corners b of cell c;
 *      U_c,d -= (G_d phi)_c / rho_c.  D = -G^T.
 *
 * Pins (tests/test_oracle_nodal.py, "-m 'not gpu'"): dense direct solve (NP1), independent scipy Kronecker
 * finite-element assembly, symmetry, row sums, textbook stencil (NP2), manufactured-solution order (NP3),
 * D = -G^T and the rhs / correction against Kronecker matrices (NP4), Fourier closed form (NP5), transfer
 * operators against 1-D Kronecker P (NP6), convergence factors (NP7), the approximate-projection identity
 * D(beta0 U_new) - M beta0 S - m w = rhs - (D sigma G) phi and its O(h^2) size (NP8).
 * PARITY UNPINNED: the absolute scale of phi relative to the paper's pi (as for the MAC projection).
 *
 * Layout (x fastest): cells i + nx (j + ny k); nodes i + (nx+1) (j + (ny+1) k).
 */
#ifndef NODAL_ORACLE_H
#define NODAL_ORACLE_H

#include "mac_oracle.h"

#ifdef __cplusplus
extern "C" {
#endif

/* N7: the Jacobi damping for the grid's cell shape */
double nod_omega(const orc_grid *g);
/* kind[a] = 0 unknown, 1 OUTFLOW (Dirichlet) node, 2 periodic duplicate (N4) */
void nod_node_kind(const orc_grid *g, int *kind);
/* N5: w_a = (cells around node a)/8 at unknowns, 0 elsewhere */
void nod_weights(const orc_grid *g, double *wgt);
/* N3: sigma_c = beta0(r_c)/rho_c */
void nod_sigma(const orc_grid *g, const orc_base *b, const double *beta0, const double *rho, double *sigma);
/* N1/N2: out = L phi at the unknowns, 0 elsewhere.  phi is read through the node rules of N4 (OUTFLOW nodes
 * count as 0, periodic duplicates as their image) whatever the array holds there. */
void nod_apply(const orc_grid *g, const double *sigma, const double *phi, double *out);
void nod_diag(const orc_grid *g, const double *sigma, double *diag);
void nod_residual(const orc_grid *g, const double *sigma, const double *phi, const double *rhs, double *res);
/* N1: rhs = D(beta0 U) - M(beta0 S) at the unknowns, 0 elsewhere (S may be NULL).  No mean removal. */
void nod_rhs(const orc_grid *g, const orc_base *b, const double *beta0, const double *u, const double *v,
             const double *w, const double *S, double *rhs);
/* N7: one Jacobi sweep, in place */
void nod_jacobi(const orc_grid *g, const double *sigma, const double *rhs, double *phi, double omega);
/* N6 */
void nod_coarsen_sigma(const orc_grid *f, const double *sf, double *sc);
void nod_restrict(const orc_grid *f, const double *fine, double *coarse);
void nod_prolong_add(const orc_grid *f, const double *coarse, double *fine);
/* N8 */
int nod_bottom_solve(const orc_grid *g, const double *sigma, const double *f, double *e);
/* one V-cycle on (phi, rhs) of level g; mg->nu_pre/nu_post/coarsest_n are used */
int nod_vcycle(const orc_grid *g, const double *sigma, const double *rhs, double *phi, const orc_mg *mg);
/* N10: U <- U - (1/rho) G phi, in place */
void nod_correct(const orc_grid *g, const double *rho, const double *phi, double *u, double *v, double *w);
/* sum_a w_a f_a / sum_a w_a over the unknowns */
double nod_weighted_mean(const orc_grid *g, const double *f);
double nod_norm_inf(const orc_grid *g, const double *f);       /* over the unknowns */
/* D(beta0 U) - M(beta0 S) (same operators as nod_rhs): the constraint of P:49 in its nodal weak form */
void nod_constraint(const orc_grid *g, const orc_base *b, const double *beta0, const double *u, const double *v,
                    const double *w, const double *S, double *out);
/* The whole projection (N1..N10).  rho may be NULL (rho := rho0 profile at cell centres), S may be NULL,
 * phi (nodes) may be NULL.  u, v, w (cells) are corrected in place.  stats->rhs_mean_removed holds m of N5.
 * Returns 0 converged, 1 max_cycles reached, < 0 error (-2 unsupported hierarchy, -5 non-finite). */
int nod_project(const orc_grid *g, const orc_base *b, const orc_mg *mg, const double *beta0, const double *rho0,
                const double *rho, double *u, double *v, double *w, const double *S, double *phi, orc_stats *stats);

#ifdef __cplusplus
}
#endif
#endif
