/*
 * maestro_mac.h -- C ABI of the B200-native MAC projection of MAESTROeX (arXiv:1910.12979).
 *
 * The library solves, on a uniform 3-D cell-centred grid and entirely on one GPU (fp64),
 *
 *        D( (beta0/rho) G phi ) = D( beta0 U_edge ) - beta0 S                         (*)
 *        U <- U_edge - (1/rho_face) G phi
 *
 * so that the corrected face velocities satisfy the low Mach number divergence constraint
 *        div(beta0 U) = beta0 (S - (1/(Gamma1bar p0)) dp0/dt)      PAPER.md:49  (Sec. 2, Eq. 6)
 * (the dp0/dt term is folded into S by the caller, or registered as a profile with
 * maestro_mac_set_dpdt_term).  The coefficient beta0/rho is the weighting of
 * the pressure term (beta0/rho) grad(pi/beta0) of PAPER.md:35 (Sec. 2, Eq. 2); beta0, rho0 are the
 * one-dimensional base state of PAPER.md:29,39,45 (Eq. 4-5); (*) is solved by geometric multigrid
 * V-cycles ("multigrid linear solvers for the pressure projection steps", "second order projection
 * method", Sec. 3).  The paper gives no discretisation; the one used here is stated in
 * DESIGN.md ("Readings") and SURVEY.md Sec. 8(c): 7-point variable-coefficient operator, arithmetic
 * (or, desc.rho_mean = 1, harmonic) face densities, red-black Gauss-Seidel V(nu_pre,nu_post), 8-cell-mean restriction, cell-centred
 * trilinear prolongation, BiCGStab on the coarsest level, max-norm stopping test.
 *
 * LAYOUT (all arrays x-fastest, fp64, DEVICE memory unless stated otherwise)
 *   cells  rho, S, phi :  idx = i + nx*(j + ny*k)                      nx*ny*nz entries
 *   u (x-faces i-1/2)  :  idx = i + (nx+1)*(j + ny*k),  i in [0,nx]    (nx+1)*ny*nz
 *   v (y-faces j-1/2)  :  idx = i + nx*(j + (ny+1)*k),  j in [0,ny]    nx*(ny+1)*nz
 *   w (z-faces k-1/2)  :  idx = i + nx*(j + ny*k),      k in [0,nz]    nx*ny*(nz+1)
 *   beta0, rho0        :  nr samples at radius r_m = (m + 1/2) dr; planar geometry: r = z,
 *                         spherical: r = |x - center|.  Evaluated by linear interpolation, held
 *                         constant beyond the first and last sample.
 *   On a periodic axis the face array still has n+1 entries: entry n is ignored on input and
 *   written equal to entry 0 on output.
 *
 * OWNERSHIP  Every device array and the workspace belong to the caller; the library allocates no
 *   device memory.  The handle (host memory, a few pinned host words, CUDA events) belongs to the
 *   library until maestro_mac_free().  The base-state profiles are device pointers: they never
 *   round-trip through the host (the lesson of PAPER.md:111-113).
 *
 * ERRORS  Return codes only; the library never prints, throws or exits.
 */
#ifndef MAESTRO_MAC_H
#define MAESTRO_MAC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct maestro_mac_handle maestro_mac_handle; /* opaque */

enum { MAESTRO_MAC_PERIODIC = 0, MAESTRO_MAC_WALL = 1, MAESTRO_MAC_OUTFLOW = 2 }; /* bc */
enum { MAESTRO_MAC_PLANAR = 0, MAESTRO_MAC_SPHERICAL = 1 };                        /* geometry */
enum {
    MAESTRO_MAC_OK = 0,
    MAESTRO_MAC_NOT_CONVERGED = 1, /* max_cycles reached; u,v,w,phi hold the last iterate */
    MAESTRO_MAC_ERR_ARG = -1,      /* null pointer, non-positive size/spacing, periodic on one side
                                      only, unknown enum, struct_bytes mismatch */
    MAESTRO_MAC_ERR_UNSUPPORTED = -2, /* hierarchy ends above 4096 bottom unknowns */
    MAESTRO_MAC_ERR_WORKSPACE = -3,   /* workspace NULL or too small (workspace_needed is written) */
    MAESTRO_MAC_ERR_CUDA = -4,        /* a CUDA call failed */
    MAESTRO_MAC_ERR_NONFINITE = -5    /* ||rhs||inf is NaN/Inf, or some rho <= 0 / non-finite */
};

typedef struct {
    int struct_bytes;         /* = sizeof(maestro_mac_desc), for versioning */
    int nx, ny, nz;           /* cells */
    double dx[3];             /* grid spacing */
    int bc_lo[3], bc_hi[3];   /* periodic must be set on both sides of an axis */
    int geometry;             /* planar: r = z.  spherical: r = |x - center| */
    int nr;                   /* base-state samples */
    double dr;                /* sample spacing; samples at (m + 1/2) dr */
    double center[3];         /* spherical only */
    /* Defaulting rules.  maestro_mac_default_desc() fills every member with its default; a caller that builds
       the struct by hand gets the default of a member by writing the stand-in value named below.  Values are
       otherwise taken literally; anything else out of range is ERR_ARG. */
    int nu_pre, nu_post;      /* RBGS sweeps per level before / after the coarse correction, default 2, 2;
                                 either may be 0, both 0 is ERR_ARG (a V-cycle without smoothing) */
    int max_cycles;           /* default 100 (0 stands for the default); at most 128 are recorded in stats */
    double rel_tol;           /* on ||r||inf / ||rhs||inf ; < 0 stands for the default 1e-10 ; 0 = run exactly
                                 max_cycles cycles without a stop test (with max_cycles = 0 that is 100 cycles) */
    int coarsest_n;           /* default 4 (0 stands for the default) */
    int bottom_max_iter;      /* BiCGStab iterations, default 100 (0 stands for the default) */
    double bottom_rel_tol;    /* on ||r||2 / ||f||2, default 1e-8 (<= 0 stands for the default) */
    int prolongation;         /* 0 = cell-centred trilinear (default), 1 = piecewise constant */
    int host_staging;         /* 1 = reserve device staging in the workspace so that
                                 maestro_mac_project_host() can be used;
                                 2, 3 = that many staging sets of u, v, w, phi (and two copy streams):
                                 maestro_mac_project_host_seq() overlaps the transfers of neighbouring steps.
                                 With 2 sets the upload of step k+1 waits for the download of step k-1 (a step
                                 costs max(projection, download + upload)); with 3 sets it does not
                                 (max(projection, upload, download)) */
    int smoother;             /* 0 = default: fused red+black passes with planes staged by TMA where the level
                                     allows it (nx >= 60), else by cp.async; pairs of sweeps run as ONE pass
                                     over HBM (two-sweep kernel, temporal blocking) on levels of at least
                                     48 x 16 x 8 cells;
                                 4 = as 0 but always one sweep per pass (bit-identical results);
                                 1 = reference two-pass (one kernel per colour);
                                 2 = fused single pass, cp.async staging on every level;
                                 3 = fused single pass, TMA staging with the 32x16 tile.
                                 Same arithmetic, same results.  0 is the product path; 4 is its one-sweep-per-pass
                                 form; 1, 2, 3 are kept as independent cross-checks for the parity tests (three
                                 further implementations of the same sweep) and are not tuned. */
    int stop_test;            /* how ||rhs - L phi||inf is obtained after each cycle:
                                 0 = default: where the level-0 TMA smoother runs (smoother 0, nu_pre >= 1,
                                     nu_post >= 1) the test rides on the first pre-sweep of the NEXT cycle,
                                     which evaluates the residual of its input at the red cells (after a
                                     post-sweep the black residuals vanish up to rounding); the sweep writes
                                     to a second buffer and is dropped when the test passes.  Elsewhere,
                                     and after the last allowed cycle, as 1;
                                 1 = a separate residual-norm kernel over all cells after every cycle. */
    int rho_mean;             /* density on a face from the two cells it separates, in the coefficient
                                 beta0/rho_face and in the correction (1/rho_face) G phi alike:
                                 0 = arithmetic mean of rho (default), 1 = harmonic (mean of 1/rho). */
    int timing;               /* 1 = bracket every level-0 smoother launch with a CUDA event pair on the call's
                                 stream (stats.ms_smooth0 ...; bench.py's roofline); 0 (default) = no per-launch
                                 events on the hot path */
    int nodal;                /* 1 = also reserve the level arrays of the end-of-step (nodal) projection in the
                                 workspace so that maestro_mac_nodal_project() can be used (adds about 4/6 of the
                                 MAC projection's workspace); 0 (default) = MAC projection only */
} maestro_mac_desc;

typedef struct {
    int cycles, bottom_iters_total, singular, levels;
    double rhs_norm_inf;      /* after mean removal */
    double res_norm_inf;      /* ||rhs - L phi||inf after the last cycle */
    double rhs_mean_removed;  /* singular problems: mean(rhs) that was subtracted, else 0 */
    double res_history[128];  /* ||r||inf / ||rhs||inf after each cycle */
    float ms_setup_kernels;   /* coefficients, coarsening, rhs */
    float ms_vcycles;         /* all cycles including the stop tests */
    float ms_correct;         /* mean shift, velocity correction, phi copy-out */
    int gpu_launches;         /* kernels launched by this call */
    float ms_smooth0;         /* desc.timing = 1: summed device time of the level-0 smoother launches that were
                                 timed (one CUDA event pair per launch, on the call's stream); else 0 */
    int smooth0_launches;     /* level-0 smoother launches of this call */
    int smooth0_timed;        /* how many of them ms_smooth0 covers (at most 512) */
    int smooth0_sweeps_timed; /* sweeps those launches applied (a two-sweep launch counts 2) */
} maestro_mac_stats;

/* Fill *desc with defaults for an nx*ny*nz unit-spacing periodic planar problem. */
void maestro_mac_default_desc(maestro_mac_desc *desc);

/*
 * maestro_mac_setup: validate the descriptor, build the level hierarchy (level l+1 exists while
 * every dimension of level l is even and its half is >= coarsest_n), carve `workspace` into the
 * per-level arrays.  Host-only apart from creating CUDA events; no device->host traffic.
 *   workspace        device memory owned by the caller, 256-byte aligned, kept alive and untouched
 *                    by the caller until maestro_mac_free().  May be NULL to query the size.
 *   workspace_needed always written when non-NULL (also on ERR_WORKSPACE).
 *   out              receives the handle on success.
 * Errors: ERR_ARG, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA.
 */
int maestro_mac_setup(const maestro_mac_desc *desc, void *workspace, size_t workspace_bytes,
                      size_t *workspace_needed, maestro_mac_handle **out);

/*
 * maestro_mac_project: the whole hot path on `cuda_stream` (a cudaStream_t, NULL = default stream):
 *   face coefficients beta0/rho_face -> coarsening to all levels -> rhs = D(beta0 U_edge) - beta0 S
 *   (minus its mean when no side is OUTFLOW) -> V-cycles from phi = 0 until
 *   ||rhs - L phi||inf <= rel_tol ||rhs||inf -> (singular: phi -= mean phi) ->
 *   U -= (1/rho_face) G phi.
 *   beta0, rho0  device [nr].
 *   rho          device [nx*ny*nz], or NULL: then rho := rho0 evaluated at cell centres
 *                (base-state-only projection).  Otherwise rho0 is accepted and unused.
 *   u, v, w      device, in/out.  WALL faces are left unchanged.
 *   S            device [nx*ny*nz] or NULL (= 0).
 *   phi          device [nx*ny*nz], out, or NULL.
 *   stats        HOST, out, or NULL.
 * u, v, w, phi, rho, S must not overlap each other or the workspace.  One in-flight call per
 * handle.
 * SYNCHRONISATION.  With rel_tol > 0, or with stats != NULL, the call synchronises the stream: once after
 * the assembly pass (it reads ||rhs||inf and the non-finite flags), after every cycle when rel_tol > 0
 * (the stop test), and at the end.  rhs == 0 then returns OK with cycles = 0, phi = 0 and the velocities
 * untouched.  With rel_tol == 0 AND stats == NULL the call is ASYNCHRONOUS: it enqueues the assembly,
 * exactly max_cycles cycles and the correction on the stream and returns OK without synchronising; a
 * zero rhs runs its cycles on zeros (phi = 0, velocities unchanged bit for bit), and non-finite input is
 * not detected by the call itself -- maestro_mac_status() reports it.
 * Returns OK, NOT_CONVERGED, ERR_ARG, ERR_CUDA or ERR_NONFINITE.
 */
int maestro_mac_project(maestro_mac_handle *h, const double *beta0, const double *rho0,
                        const double *rho, double *u, double *v, double *w, const double *S,
                        double *phi, maestro_mac_stats *stats, void *cuda_stream);

/*
 * maestro_mac_status: completes an asynchronous maestro_mac_project() call (rel_tol == 0, stats == NULL):
 * synchronises `cuda_stream` (the stream of that call), returns ERR_NONFINITE if the assembly pass flagged
 * a non-finite rhs or a rho <= 0 (the outputs are then garbage), else OK, and fills *stats (HOST, may be
 * NULL) as the synchronous call would have (with stats != NULL it launches one residual-norm pass for
 * res_norm_inf).  After a synchronous call it returns OK and the stats of that call without touching the
 * stream.  Returns OK, ERR_ARG, ERR_CUDA or ERR_NONFINITE.
 */
int maestro_mac_status(maestro_mac_handle *h, maestro_mac_stats *stats, void *cuda_stream);

/*
 * maestro_mac_project_host: the same call with HOST buffers (pinned memory recommended): copies
 * the inputs to the staging area reserved by desc.host_staging = 1, projects, copies u, v, w
 * (and phi when non-NULL) back, and synchronises the stream.  Same layouts and NULL conventions as
 * above.  Returns ERR_ARG if the handle was set up without host_staging.
 */
int maestro_mac_project_host(maestro_mac_handle *h, const double *beta0, const double *rho0,
                             const double *rho, double *u, double *v, double *w, const double *S,
                             double *phi, maestro_mac_stats *stats, void *cuda_stream);

/*
 * maestro_mac_project_host_seq: `nsteps` consecutive projections with HOST buffers, pipelined (BASELINE.json
 * config 5: "10 consecutive projections with new U_edge each step"; the constraint of PAPER.md:49 Eq. 6 is
 * enforced once per time step with the same base state and density).  beta0, rho0, rho, S (host; NULL
 * conventions as above) are copied to the device ONCE and serve every step; for step k the face velocities are
 * read from u_in[k], v_in[k], w_in[k] (host arrays of nsteps pointers) and the projected ones are written to
 * u_out[k], v_out[k], w_out[k] (may equal the inputs), phi (when phi_out != NULL) to phi_out[k].
 * While step k is projected on `cuda_stream`, the velocities of step k+1 travel host -> device and the results
 * of step k-1 device -> host on the handle's two copy streams (staging sets used round robin, desc.host_staging = 2
 * or 3), so
 * every step's transfers happen inside the call but only the first upload and the last download are exposed.
 * Host buffers must be page-locked for the copies to overlap, and must not be touched until the call returns
 * (it returns after everything has completed).  stats: host array of nsteps entries, or NULL.
 * Returns the first negative status met (the sequence stops there), else NOT_CONVERGED if any step returned it,
 * else OK.  ERR_ARG if the handle was set up with host_staging < 2.
 */
int maestro_mac_project_host_seq(maestro_mac_handle *h, int nsteps, const double *beta0, const double *rho0,
                                 const double *rho, const double *S,
                                 const double *const *u_in, const double *const *v_in, const double *const *w_in,
                                 double *const *u_out, double *const *v_out, double *const *w_out,
                                 double *const *phi_out, maestro_mac_stats *stats, void *cuda_stream);

/*
 * maestro_mac_base_state: the 1-D base-state quantities the projection consumes, from the thermodynamic
 * base state, on the nr profile samples r_m = (m + 1/2) dr (one small kernel on `cuda_stream`):
 *   beta0[m]      PAPER.md:45 Eq. 5, beta0(r) = rho0(0) exp(int_0^r (1/(Gamma1bar p0)) dp0/dr' dr'):
 *                 beta0[0] = rho0[0],  ln beta0[m+1] = ln beta0[m] + (ln p0[m+1] - ln p0[m]) / (0.5 (G[m] + G[m+1]))
 *   dpdt_term[m]  PAPER.md:49 Eq. 6, (1/(Gamma1bar p0)) dp0/dt = dp0dt[m] / (gamma1bar[m] p0[m])
 * All pointers are DEVICE arrays of nr doubles owned by the caller; dp0dt and dpdt_term may both be NULL.
 * p0, gamma1bar, rho0[0] must be positive.  Returns OK, ERR_ARG or ERR_CUDA.
 */
int maestro_mac_base_state(int nr, const double *rho0, const double *p0, const double *gamma1bar,
                           const double *dp0dt, double *beta0, double *dpdt_term, void *cuda_stream);

/*
 * maestro_mac_lateral_average: the base-state density from the cell density ("rho0 ... represents
 * the lateral average"), with the handle's geometry and profile sampling: cell (i,j,k) with centre radius r
 * (planar: z) belongs to sample m = min(nr-1, floor(r / dr)); rho0[m] = mean of rho over the cells of sample m;
 * samples without a cell are filled by linear interpolation in m between the nearest samples that have cells
 * (constant beyond the ends).  rho: device [nx*ny*nz]; rho0: device [nr], out.  Uses the handle's scratch
 * (not during a project call).  Asynchronous on `cuda_stream`.  Returns OK, ERR_ARG, ERR_UNSUPPORTED, ERR_CUDA.
 */
int maestro_mac_lateral_average(maestro_mac_handle *h, const double *rho, double *rho0, void *cuda_stream);

/*
 * maestro_mac_lateral_average_noalloc: the same lateral average for callers that cannot allocate device
 * memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): no handle, no
 * workspace, no cudaMalloc / cudaFree or allocating library call.  `desc` supplies nx, ny, nz, dx, geometry, nr, dr,
 * center (validated like maestro_mac_setup's; the solver fields are ignored); rho: device [nx*ny*nz]; rho0: device
 * [nr], out; both caller-owned.  The scratch (per-block partial sums and counts) is a static device array inside the
 * library, sized for nr <= MAESTRO_MAC_NOALLOC_MAX_NR (3.77 MiB, held by every GPU that loads the library until the
 * process exits); a larger nr returns ERR_UNSUPPORTED and launches nothing.  Same kernels and launch shape as
 * maestro_mac_lateral_average: bit-identical results.  Asynchronous on `cuda_stream`.  All calls share the scratch:
 * calls that overlap on the GPU (other streams, unordered host threads) race -- serialise them.  The first call on a
 * device looks up the array's address (cudaGetSymbolAddress) and opts the kernel into its shared-memory size; make
 * that call outside a capture.  Returns OK, ERR_ARG, ERR_UNSUPPORTED, ERR_CUDA.
 */
#define MAESTRO_MAC_NOALLOC_MAX_NR 2048
int maestro_mac_lateral_average_noalloc(const maestro_mac_desc *desc, const double *rho, double *rho0, void *cuda_stream);

/*
 * maestro_mac_set_dpdt_term: register the profile q = (1/(Gamma1bar p0)) dp0/dt (device, [nr], caller-owned,
 * alive and unchanged during every later project call) or NULL to clear it.  With it the right-hand side is the
 * full constraint of PAPER.md:49 Eq. 6,  rhs = D(beta0 U_edge) - beta0 (S - q(r)),  q evaluated at cell centres
 * like every profile; without it the caller folds that term into S.  Returns OK or ERR_ARG.
 */
int maestro_mac_set_dpdt_term(maestro_mac_handle *h, const double *dpdt_term);

/*
 * maestro_mac_nodal_project: the OTHER projection of the "second order projection method" with "multigrid linear
 * solvers for the pressure projection steps" (Sec. 3): the end-of-step projection of the CELL-CENTRED
 * velocity.  It enforces the same constraint div(beta0 U) = beta0 (S - ...) (Eq. 6; the dp0/dt term
 * folded into S) with the same weighting sigma = beta0/rho of the pressure term (Eq. 2) on the same base
 * state, with phi on the NODES of the grid.  The paper describes neither projection; the readings (N1..N10):
 * trilinear finite-element (27-point) operator  (L phi)_a = -(1/V) sum_c sigma_c int_c grad psi_a . grad phi,
 * rhs_a = (D(beta0 U))_a - (M(beta0 S))_a with the finite-element divergence D and the lumped source M (mean over the
 * cells around the node), U <- U - (1/rho) G phi with G the cell-mean gradient (D = -G^T; an approximate projection
 * in the sense of Almgren, Bell and Szymczak); WALL sides natural, OUTFLOW sides phi = 0 on the boundary nodes,
 * periodic sides node n = node 0; no OUTFLOW side: the uniform volumetric source m = sum(rhs)/cells is removed
 * (stats.rhs_mean_removed) and phi has zero volume-weighted mean; V(nu_pre, nu_post) cycles of Jacobi sweeps
 * (omega = sum_d h_d^-2 / (3 max_d h_d^-2), 1 for cubic cells) on the MAC projection's cell hierarchy with coarse
 * sigma = mean of the 8 children, trilinear prolongation P, restriction P^T / 8, BiCGStab on the coarsest level, stop
 * on ||rhs - L phi||inf <= rel_tol ||rhs||inf over the unknowns.
 *   beta0, rho0   device [nr]; rho device [nx*ny*nz] or NULL (rho := rho0 at cell centres); S device cells or NULL.
 *   uc, vc, wc    device CELL arrays [nx*ny*nz], in/out.
 *   phi           device NODE array [(nx+1)*(ny+1)*(nz+1)], idx = i + (nx+1)*(j + (ny+1)*k), out, or NULL; OUTFLOW
 *                 nodes hold 0, on a periodic axis entry n equals entry 0.
 *   stats         HOST, out, or NULL.
 * Needs desc.nodal = 1 (else ERR_ARG).  Synchronises the stream like maestro_mac_project with stats.  Same return codes.
 */
int maestro_mac_nodal_project(maestro_mac_handle *h, const double *beta0, const double *rho0, const double *rho,
                              double *uc, double *vc, double *wc, const double *S, double *phi,
                              maestro_mac_stats *stats, void *cuda_stream);

/* Release the handle (host memory, pinned words, events).  NULL is a no-op.  Returns OK. */
int maestro_mac_free(maestro_mac_handle *h);

/* ------------------------------------------------------------------------------------------------
 * Step API: the individual kernels of the path, for per-kernel parity tests and timing.  They act
 * on the handle's internal level arrays.  `level` 0 is the finest.  All are asynchronous on
 * `cuda_stream` unless they return a scalar to the host.
 * ---------------------------------------------------------------------------------------------- */

enum { MAESTRO_MAC_ARR_PHI = 0, MAESTRO_MAC_ARR_RHS = 1, MAESTRO_MAC_ARR_BX = 2,
       MAESTRO_MAC_ARR_BY = 3, MAESTRO_MAC_ARR_BZ = 4 };

int maestro_mac_num_levels(const maestro_mac_handle *h);
/* Launch plan of the smoother on a level (host only; for tests that must know which decomposition they hit):
 *   info[0] kernel (enum below), info[1] lateral tiles, info[2] tiles that march the whole z column (two-sweep
 *   kernel: the whole waves), info[3] z-chunks per remaining tile, info[4] planes per chunk, info[5] CTAs of one
 *   launch, info[6], info[7] periodic image columns / rows per side of the level's arrays. */
enum { MAESTRO_MAC_KERNEL_COLOR = 0, MAESTRO_MAC_KERNEL_FUSED = 1, MAESTRO_MAC_KERNEL_TMA = 2,
       MAESTRO_MAC_KERNEL_T2 = 3, MAESTRO_MAC_KERNEL_TAIL = 4, MAESTRO_MAC_KERNEL_BOTTOM = 5,
       MAESTRO_MAC_KERNEL_CLUSTER = 6 };   /* CLUSTER: the level is one of those k_cluster_vcycles walks in one launch */
int maestro_mac_level_plan(const maestro_mac_handle *h, int level, int info[8]);
/* The planners behind that, as pure host arithmetic (no handle, no CUDA call; CPU-side tests of the wave / chunk
 * decomposition): the plan of one launch on a level of nx x ny x nz cells on a device with `sms` multiprocessors.
 * which = 0: the two-sweep smoother k_rbgs_t2 (tiles of 26 x 18 finished cells, one block per SM at a time);
 * which = 1: the nodal march k_nod_march ((nx+1)(ny+1)(nz+1) nodes, tiles of 32 x 8 nodes, two blocks per SM).
 * info[1..5] as in maestro_mac_level_plan (tiles, whole-column tiles, z-chunks per remaining tile, planes per chunk,
 * blocks); info[0] = tiles along x.  Returns OK or ERR_ARG. */
int maestro_mac_plan_query(int which, int nx, int ny, int nz, int sms, int info[8]);
/* n[3] cells and h[3] spacing of a level */
int maestro_mac_level_dims(const maestro_mac_handle *h, int level, int n[3], double hh[3]);
/* Copy a level array to / from a caller DEVICE buffer in the public layout (cells, or the face
 * layout of u/v/w for BX/BY/BZ).  Coefficients are returned as b = beta0/rho_face (the internal
 * pre-scaling by 1/h^2 and the folding of boundary types are undone on WALL/OUTFLOW faces only
 * as far as recoverable: WALL faces read back as 0). */
int maestro_mac_level_get(maestro_mac_handle *h, int level, int which, double *dst, void *cuda_stream);
int maestro_mac_level_set(maestro_mac_handle *h, int level, int which, const double *src, void *cuda_stream);

/* a2 + a3: face coefficients on level 0 and coarsening to every level */
int maestro_mac_step_coefficients(maestro_mac_handle *h, const double *beta0, const double *rho0,
                                  const double *rho, void *cuda_stream);
/* a4: rhs on level 0 (mean removed if singular); host outputs may be NULL; synchronises */
int maestro_mac_step_rhs(maestro_mac_handle *h, const double *beta0, const double *u,
                         const double *v, const double *w, const double *S,
                         double *rhs_norm_inf, double *mean_removed, void *cuda_stream);
/* a5: nsweeps red-black Gauss-Seidel sweeps on a level */
int maestro_mac_step_smooth(maestro_mac_handle *h, int level, int nsweeps, void *cuda_stream);
/* a6: rhs[level+1] = restrict(rhs[level] - L phi[level]);  phi[level+1] = 0 */
int maestro_mac_step_residual_restrict(maestro_mac_handle *h, int level, void *cuda_stream);
/* a7: phi[level] += P phi[level+1] */
int maestro_mac_step_prolong(maestro_mac_handle *h, int level, void *cuda_stream);
/* a8: BiCGStab on the coarsest level: phi = L^-1 rhs */
int maestro_mac_step_bottom(maestro_mac_handle *h, void *cuda_stream);
/* one V-cycle from level 0 */
int maestro_mac_step_vcycle(maestro_mac_handle *h, void *cuda_stream);
/* a9: ||rhs - L phi||inf on a level; synchronises */
int maestro_mac_step_residual_norm(maestro_mac_handle *h, int level, double *norm_inf, void *cuda_stream);
/* a10: velocity correction from the level-0 phi */
int maestro_mac_step_correct(maestro_mac_handle *h, const double *rho0, const double *rho,
                             double *u, double *v, double *w, void *cuda_stream);

/* ---- step API of the nodal projection (desc.nodal = 1): the individual kernels on the handle's nodal level arrays.
 * Node arrays hold (nx+1)(ny+1)(nz+1) values of the level; SIGMA is a cell array.  level_get(PHI) applies the node
 * rules (OUTFLOW nodes 0, periodic entry n = entry 0); the kernels never read those entries. */
enum { MAESTRO_MAC_NODAL_PHI = 0, MAESTRO_MAC_NODAL_RHS = 1, MAESTRO_MAC_NODAL_SIGMA = 2 };
int maestro_mac_nodal_level_get(maestro_mac_handle *h, int level, int which, double *dst, void *cuda_stream);
int maestro_mac_nodal_level_set(maestro_mac_handle *h, int level, int which, const double *src, void *cuda_stream);
/* sigma = beta0(r_cell)/rho on level 0 and its coarsening to every level (also stages beta0 at the cell centres for a
 * following maestro_mac_nodal_step_rhs) */
int maestro_mac_nodal_step_sigma(maestro_mac_handle *h, const double *beta0, const double *rho0, const double *rho,
                                 void *cuda_stream);
/* rhs on level 0 (uniform source removed if singular); call right after maestro_mac_nodal_step_sigma; synchronises */
int maestro_mac_nodal_step_rhs(maestro_mac_handle *h, const double *uc, const double *vc, const double *wc,
                               const double *S, double *rhs_norm_inf, double *mean_removed, void *cuda_stream);
int maestro_mac_nodal_step_smooth(maestro_mac_handle *h, int level, int nsweeps, void *cuda_stream);      /* Jacobi */
int maestro_mac_nodal_step_residual_restrict(maestro_mac_handle *h, int level, void *cuda_stream);
int maestro_mac_nodal_step_prolong(maestro_mac_handle *h, int level, void *cuda_stream);
int maestro_mac_nodal_step_bottom(maestro_mac_handle *h, void *cuda_stream);
int maestro_mac_nodal_step_vcycle(maestro_mac_handle *h, void *cuda_stream);
int maestro_mac_nodal_step_residual_norm(maestro_mac_handle *h, int level, double *norm_inf, void *cuda_stream);
int maestro_mac_nodal_step_correct(maestro_mac_handle *h, const double *rho0, const double *rho, double *uc,
                                   double *vc, double *wc, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
