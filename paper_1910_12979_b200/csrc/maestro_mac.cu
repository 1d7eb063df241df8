// maestro_mac.cu -- host side of the C ABI declared in include/maestro_mac.h.
// Validates descriptors, builds the level hierarchy, carves the caller's workspace, and drives the
// kernels on the caller's stream: mac_setup.cuh (assembly pass), mac_smoother_t2.cuh / _tma.cuh /
// mac_smoother.cuh (smoothers), mac_tail.cuh (coarse tail), mac_kernels.cuh (transfers, bottom solve,
// correction, reductions), mac_base.cuh (base state).  No device allocation here.
#include "maestro_mac.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "mac_kernels.cuh"
#include "mac_setup.cuh"
#include "mac_smoother.cuh"
#include "mac_smoother_tma.cuh"
#include "mac_smoother_t2.cuh"
#include "mac_tail.cuh"
#include "mac_cluster.cuh"
#include "mac_base.cuh"
#include "mac_nodal.cuh"

namespace {

constexpr int kMaxLevels = 32;
constexpr int kRedBlocksPerSm = 8;        // blocks per SM of the row-walking reduction kernels
constexpr int kMaxParts = 131072;         // capacity of the partial-reduction arrays
constexpr int kBottomMax = 4096;          // largest coarsest level (unknowns)
constexpr size_t kBottomSmem = 200 * 1024; // bottom-solver vectors live in shared memory up to this size
constexpr int kLateralBlocks = 160;      // blocks of the lateral-average sum (one per SM, at most this many)
constexpr size_t kLateralSmem = 200 * 1024;
constexpr int kSmoothEvents = 512;        // level-0 smoother launches timed per call

struct Level {
    int n[3];
    double h[3];
    int px;                        // x pitch of ax
    int gx, gy;                    // ghost columns / rows per side (mac_common.cuh "Ghosts")
    int cx, ry;                    // x pitch of the cell-shaped arrays, rows per plane
    size_t ncell;                  // interior cells
    size_t acell, nax, nay, naz;   // allocated entries (ghosts included)
    size_t off_c, off_ax;          // entries from an allocation's base to the interior origin
    double *phi, *phi2, *rhs, *ax, *ay, *az;   // interior origins
    double* phi_a;                 // the buffer `phi` pointed to at carve time (tensor map `phi`)
    TmaLevelMaps tma[3];           // [0] MAC_TMA_BIG tile, [1] MAC_TMA_MID tile, [2] two-sweep kernel's 32 x 24 tile
};

struct Staging {
    double *beta0, *rho0, *rho, *u, *v, *w, *S, *phi;
    double *ux[2], *vx[2], *wx[2], *phix[2];   // further sets of u, v, w, phi (desc.host_staging = 2, 3)
};

struct NodHost {                   // one level of the nodal projection (desc.nodal = 1); layout: mac_nodal.cuh
    int n[3];
    double h[3];
    size_t nnode, ncell;           // nodes (nx+1)(ny+1)(nz+1) and cells of the level
    size_t anode, acell;           // allocated entries: one ghost node / ghost cell per side
    size_t onode, ocell;           // entries from an allocation's base to the interior origin
    int NX, NY, CX, CY;            // row pitches (even: 16-byte multiples) and rows per plane of the node / cell arrays
    double *phi, *phi2, *rhs;      // node arrays (interior origins)
    double *sigma;                 // cell array (interior origin)
    double* phi_a;                 // the buffer `phi` pointed to at carve time (tensor map tm_phi; tm_phi2 is its partner)
    CUtensorMap tm_phi, tm_phi2, tm_rhs, tm_sig;   // box loads of k_nod_march: 36 x 10 nodes, 36 x 9 cells, 32 x 8 nodes
    int tma_ok;
};

}  // namespace

struct maestro_mac_handle {
    maestro_mac_desc d;
    int nlev;
    Level lev[kMaxLevels];
    int singular;
    const double* dpdt_term;       // device profile q[nr] of Eq. 6 registered by maestro_mac_set_dpdt_term, or NULL
    int tail_start;                // first level of the one-launch coarse tail (k_coarse_tail), or -1
    size_t tail_smem;
    TailArgs tail;                 // prepared by plan_tail; level pointers are filled in at launch
    size_t cl_smem;                // dynamic shared memory per block of the cluster kernel
    int cl_start;                  // first level of the cluster kernel (k_cluster_vcycles: levels of <= 32^3 cells), or -1
    clus::Args cl;                 // prepared by plan_tail; level pointers are filled in at launch
    double *lat_part;              // lateral average: kLateralBlocks x nr partial sums (doubles) and counts (unsigned), or NULL
    double *cl_scratch;            // device: the result block of a device-side solve (cycles, norm, flag, history)
    double *host_hist, *host_hist_dev;   // mapped pinned copy of the result block (4 + 128 doubles)
    // scratch carved from the workspace
    double *part_sum, *part_max;   // kMaxParts each
    double *scal;                  // device scalars: [0] sum, [1] max (k_reduce_final output) ...
    double *bottom_vecs;           // 6 * bottom unknowns
    int *flags;                    // [0] bad rho, [1] bottom iterations
    Staging st;
    bool has_staging;
    cudaStream_t cp_in, cp_out;    // copy streams of maestro_mac_project_host_seq (host_staging = 2), else NULL
    cudaEvent_t ev_in[3], ev_done[3], ev_out[3];   // per staging set: upload complete, projection complete, download complete
    NodHost nod[kMaxLevels];       // nodal projection: level arrays (valid when has_nodal)
    double* nod_vecs;              // 6 BiCGStab vectors over the nodes of the coarsest level
    bool has_nodal;
    // host side
    double *host_scal;             // pinned and mapped, 8 doubles: kernels write the scalars the host reads (k_publish)
    int *host_flags;               // pinned and mapped, 4 ints
    double *host_scal_dev;         // the same two blocks as the device sees them (cudaHostGetDevicePointer)
    int *host_flags_dev;
    cudaEvent_t ev[4];
    int launches;
    int sms;                       // multiprocessors of the device (cudaDevAttrMultiProcessorCount at setup)
    int red_blocks;                // kRedBlocksPerSm * sms
    int deferred;                  // the last project call returned without synchronising (maestro_mac_status reports it)
    maestro_mac_stats last;        // stats of the last project call as far as the host knows them
    // level-0 smoother timing: one event pair per launch, summed after the final synchronise
    cudaEvent_t* sm_ev;            // 2 * kSmoothEvents events, or NULL
    int sm_used;                   // pairs recorded by the current call
    int sm_launches;               // level-0 smoother launches of the current call (recorded or not)
    int sm_sweeps;                 // sweeps applied by the recorded launches (a two-sweep launch counts 2)
};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

bool valid_bc(int b) { return b == MAESTRO_MAC_PERIODIC || b == MAESTRO_MAC_WALL || b == MAESTRO_MAC_OUTFLOW; }

int validate_and_default(const maestro_mac_desc* in, maestro_mac_desc* d)
{
    if (!in || in->struct_bytes != (int)sizeof(maestro_mac_desc)) return MAESTRO_MAC_ERR_ARG;
    *d = *in;
    if (d->nx <= 0 || d->ny <= 0 || d->nz <= 0) return MAESTRO_MAC_ERR_ARG;
    if (d->nx > 65535 || d->ny > 65535 || d->nz > 65535) return MAESTRO_MAC_ERR_UNSUPPORTED;
    for (int a = 0; a < 3; ++a) {
        if (!(d->dx[a] > 0.0) || !std::isfinite(d->dx[a])) return MAESTRO_MAC_ERR_ARG;
        if (!valid_bc(d->bc_lo[a]) || !valid_bc(d->bc_hi[a])) return MAESTRO_MAC_ERR_ARG;
        if ((d->bc_lo[a] == MAESTRO_MAC_PERIODIC) != (d->bc_hi[a] == MAESTRO_MAC_PERIODIC)) return MAESTRO_MAC_ERR_ARG;
    }
    if (d->geometry != MAESTRO_MAC_PLANAR && d->geometry != MAESTRO_MAC_SPHERICAL) return MAESTRO_MAC_ERR_ARG;
    if (d->nr <= 0 || !(d->dr > 0.0) || !std::isfinite(d->dr)) return MAESTRO_MAC_ERR_ARG;
    if (d->nu_pre < 0 || d->nu_post < 0 || d->max_cycles < 0 || d->coarsest_n < 0 || d->bottom_max_iter < 0)
        return MAESTRO_MAC_ERR_ARG;
    if (d->nu_pre == 0 && d->nu_post == 0) return MAESTRO_MAC_ERR_ARG;   // a V-cycle without smoothing (the defaults come from maestro_mac_default_desc)
    if (d->max_cycles == 0) d->max_cycles = 100;
    if (d->rel_tol < 0.0) d->rel_tol = 1e-10;
    if (!std::isfinite(d->rel_tol)) return MAESTRO_MAC_ERR_ARG;
    if (d->coarsest_n == 0) d->coarsest_n = 4;
    if (d->bottom_max_iter == 0) d->bottom_max_iter = 100;
    if (!(d->bottom_rel_tol > 0.0)) d->bottom_rel_tol = 1e-8;
    if (d->prolongation != 0 && d->prolongation != 1) return MAESTRO_MAC_ERR_ARG;
    if (d->host_staging < 0 || d->host_staging > 3) return MAESTRO_MAC_ERR_ARG;
    if (d->smoother < 0 || d->smoother > 4) return MAESTRO_MAC_ERR_ARG;   // 4: one sweep per pass everywhere
    if (d->stop_test != 0 && d->stop_test != 1) return MAESTRO_MAC_ERR_ARG;
    if (d->rho_mean != 0 && d->rho_mean != 1) return MAESTRO_MAC_ERR_ARG;
    if (d->timing != 0 && d->timing != 1) return MAESTRO_MAC_ERR_ARG;
    if (d->nodal != 0 && d->nodal != 1) return MAESTRO_MAC_ERR_ARG;
    return MAESTRO_MAC_OK;
}

// geometry of one level; ghosts: the level runs TMA-staged kernels and carries periodic images
void set_level(const maestro_mac_desc& d, Level& L, const int n[3], const double h[3], bool ghosts)
{
    for (int a = 0; a < 3; ++a) { L.n[a] = n[a]; L.h[a] = h[a]; }
    const int gw = d.smoother == 0 ? t2::HALO : 2;         // the two-sweep kernel's halo is 4 cells
    L.gx = (ghosts && d.bc_lo[0] == MAESTRO_MAC_PERIODIC) ? gw : 0;
    L.gy = (ghosts && d.bc_lo[1] == MAESTRO_MAC_PERIODIC) ? gw : 0;
    L.cx = n[0] + 2 * L.gx;
    L.ry = n[1] + 2 * L.gy;
    L.px = (int)align_up((size_t)n[0] + 1 + 2 * L.gx, 4);
    L.ncell = (size_t)n[0] * n[1] * n[2];
    L.acell = (size_t)L.cx * L.ry * n[2];
    L.nax = (size_t)L.px * L.ry * n[2];
    L.nay = (size_t)L.cx * (L.ry + 1) * n[2];
    L.naz = (size_t)L.cx * L.ry * (n[2] + 1);
    L.off_c = (size_t)L.gx + (size_t)L.cx * L.gy;
    L.off_ax = (size_t)L.gx + (size_t)L.px * L.gy;
}

// Build level geometry; returns OK or UNSUPPORTED.
int build_levels(const maestro_mac_desc& d, Level* lev, int* nlev)
{
    int n[3] = {d.nx, d.ny, d.nz};
    double h[3] = {d.dx[0], d.dx[1], d.dx[2]};
    int l = 0;
    for (;;) {
        // levels that run the TMA-staged kernels carry periodic image columns / rows (TMA cannot wrap)
        // (a periodic axis must hold both image strips apart: n >= 2 x ghost width, else the level keeps the plain layout)
        const int gw = d.smoother == 0 ? t2::HALO : 2;
        const bool per_ok = (d.bc_lo[0] != MAESTRO_MAC_PERIODIC || n[0] >= 2 * gw) && (d.bc_lo[1] != MAESTRO_MAC_PERIODIC || n[1] >= 2 * gw);
        const bool tma_level = (d.smoother == 0 || d.smoother == 3 || d.smoother == 4) && n[0] >= 60 && (n[0] & 1) == 0 && n[1] >= 4 && per_ok;
        bool can = l + 1 < kMaxLevels;
        for (int a = 0; a < 3; ++a)
            if ((n[a] & 1) || n[a] / 2 < d.coarsest_n) can = false;
        set_level(d, lev[l], n, h, tma_level && can);      // the coarsest level is only solved, never smoothed: plain layout
        ++l;
        if (!can) break;
        for (int a = 0; a < 3; ++a) { n[a] /= 2; h[a] *= 2.0; }
    }
    *nlev = l;
    if (lev[l - 1].ncell > (size_t)kBottomMax) return MAESTRO_MAC_ERR_UNSUPPORTED;
    return MAESTRO_MAC_OK;
}

// Carve (or just size) the workspace.  base may be NULL when only sizing.
size_t carve(maestro_mac_handle* H, char* base)
{
    size_t off = 0;
    auto take = [&](size_t count, size_t elem) -> void* {
        off = align_up(off, 256);
        void* p = base ? (void*)(base + off) : nullptr;
        off += count * elem;
        return p;
    };
    for (int l = 0; l < H->nlev; ++l) {
        Level& L = H->lev[l];
        auto at = [&](void* b, size_t o) -> double* { return b ? (double*)b + o : nullptr; };
        L.phi = at(take(L.acell, 8), L.off_c);
        L.phi_a = L.phi;
        L.phi2 = at(take(L.acell, 8), L.off_c);
        L.rhs = at(take(L.acell, 8), L.off_c);
        L.ax = at(take(L.nax, 8), L.off_ax);
        L.ay = at(take(L.nay, 8), L.off_c);
        L.az = at(take(L.naz, 8), L.off_c);
    }
    H->part_sum = (double*)take(kMaxParts, 8);
    H->part_max = (double*)take(kMaxParts, 8);
    H->scal = (double*)take(16, 8);
    H->bottom_vecs = (double*)take(6 * H->lev[H->nlev - 1].ncell, 8);
    H->flags = (int*)take(16, 4);
    H->cl_scratch = (double*)take(8 + 4 + 128, 8);
    H->lat_part = (size_t)H->d.nr * 12 <= kLateralSmem ? (double*)take((size_t)kLateralBlocks * H->d.nr * 12 / 8 + 8, 8) : nullptr;
    H->has_nodal = H->d.nodal == 1;
    H->nod_vecs = nullptr;
    if (H->has_nodal) {
        for (int l = 0; l < H->nlev; ++l) {
            NodHost& N = H->nod[l];
            for (int a = 0; a < 3; ++a) { N.n[a] = H->lev[l].n[a]; N.h[a] = H->lev[l].h[a]; }
            N.nnode = (size_t)(N.n[0] + 1) * (N.n[1] + 1) * (N.n[2] + 1);
            N.ncell = H->lev[l].ncell;
            N.NX = (N.n[0] + 4 + 1) & ~1; N.NY = N.n[1] + 3;     // rows: pad, ghost, nodes 0..nx, ghost
            N.CX = (N.n[0] + 3 + 1) & ~1; N.CY = N.n[1] + 2;     // rows: pad, ghost, cells 0..nx-1, ghost
            N.anode = (size_t)N.NX * N.NY * (N.n[2] + 3);
            N.acell = (size_t)N.CX * N.CY * (N.n[2] + 2);
            N.onode = 2 + (size_t)N.NX * (1 + (size_t)N.NY);
            N.ocell = 2 + (size_t)N.CX * (1 + (size_t)N.CY);
            auto at = [&](void* b, size_t o) -> double* { return b ? (double*)b + o : nullptr; };
            N.phi = at(take(N.anode, 8), N.onode);
            N.phi_a = N.phi;
            N.phi2 = at(take(N.anode, 8), N.onode);
            N.rhs = at(take(N.anode, 8), N.onode);
            N.sigma = at(take(N.acell, 8), N.ocell);
        }
        H->nod_vecs = (double*)take(6 * H->nod[H->nlev - 1].anode, 8);
    }
    H->has_staging = H->d.host_staging >= 1;
    if (H->has_staging) {
        const maestro_mac_desc& d = H->d;
        size_t nc = (size_t)d.nx * d.ny * d.nz;
        H->st.beta0 = (double*)take(d.nr, 8);
        H->st.rho0 = (double*)take(d.nr, 8);
        H->st.rho = (double*)take(nc, 8);
        H->st.S = (double*)take(nc, 8);
        H->st.phi = (double*)take(nc, 8);
        H->st.u = (double*)take((size_t)(d.nx + 1) * d.ny * d.nz, 8);
        H->st.v = (double*)take((size_t)d.nx * (d.ny + 1) * d.nz, 8);
        H->st.w = (double*)take((size_t)d.nx * d.ny * (d.nz + 1), 8);
        for (int q = 0; q < 2; ++q) {
            H->st.ux[q] = H->st.vx[q] = H->st.wx[q] = H->st.phix[q] = nullptr;
            if (d.host_staging < q + 2) continue;
            H->st.phix[q] = (double*)take(nc, 8);
            H->st.ux[q] = (double*)take((size_t)(d.nx + 1) * d.ny * d.nz, 8);
            H->st.vx[q] = (double*)take((size_t)d.nx * (d.ny + 1) * d.nz, 8);
            H->st.wx[q] = (double*)take((size_t)d.nx * d.ny * (d.nz + 1), 8);
        }
    }
    return align_up(off, 256);
}

LevelDev dev_level(const maestro_mac_handle* H, int l)
{
    const Level& L = H->lev[l];
    LevelDev D;
    D.nx = L.n[0]; D.ny = L.n[1]; D.nz = L.n[2]; D.px = L.px;
    D.cx = L.cx; D.ry = L.ry; D.gx = L.gx; D.gy = L.gy;
    for (int a = 0; a < 3; ++a) { D.bclo[a] = H->d.bc_lo[a]; D.bchi[a] = H->d.bc_hi[a]; }
    D.phi = L.phi; D.phi2 = L.phi2; D.rhs = L.rhs; D.ax = L.ax; D.ay = L.ay; D.az = L.az;
    return D;
}

GeoDev dev_geo(const maestro_mac_handle* H)
{
    const maestro_mac_desc& d = H->d;
    GeoDev G;
    G.nx = d.nx; G.ny = d.ny; G.nz = d.nz;
    G.dx = d.dx[0]; G.dy = d.dx[1]; G.dz = d.dx[2];
    for (int a = 0; a < 3; ++a) { G.bclo[a] = d.bc_lo[a]; G.bchi[a] = d.bc_hi[a]; }
    G.geometry = d.geometry; G.nr = d.nr; G.dr = d.dr;
    G.cx = d.center[0]; G.cy = d.center[1]; G.cz = d.center[2];
    G.rho_mean = d.rho_mean;
    return G;
}

GeoInv dev_geo_inv(const maestro_mac_handle* H)
{
    const maestro_mac_desc& d = H->d;
    GeoInv I;
    I.idx = 1.0 / d.dx[0]; I.idy = 1.0 / d.dx[1]; I.idz = 1.0 / d.dx[2];
    I.idx2 = 1.0 / (d.dx[0] * d.dx[0]); I.idy2 = 1.0 / (d.dx[1] * d.dx[1]); I.idz2 = 1.0 / (d.dx[2] * d.dx[2]);
    I.idr = 1.0 / d.dr;
    return I;
}

// block (bx, by) with bx*by = 256 and grid covering (ex, ey, ez)
void dims3(int ex, int ey, int ez, dim3* grid, dim3* block)
{
    int bx = 32;
    while (bx < 128 && bx < ex) bx *= 2;
    int by = 256 / bx;
    *block = dim3(bx, by, 1);
    *grid = dim3((ex + bx - 1) / bx, (ey + by - 1) / by, ez);
}

// The scalars the host reads (norms, flags) are WRITTEN into mapped pinned memory by a one-thread kernel instead of
// being fetched by cudaMemcpyAsync: a device-to-host copy queues on the copy engine behind whatever bulk download is
// in flight (maestro_mac_project_host_seq overlaps those with the projection), and every V-cycle would wait for it.
__global__ void k_publish(double* __restrict__ dst, const double* __restrict__ src, int n)
{
    for (int q = threadIdx.x; q < n; q += blockDim.x) dst[q] = src[q];
    __threadfence_system();
}
__global__ void k_publish_int(int* __restrict__ dst, const int* __restrict__ src, int n)
{
    for (int q = threadIdx.x; q < n; q += blockDim.x) dst[q] = src[q];
    __threadfence_system();
}

#define CUDA_OK(call) do { if ((call) != cudaSuccess) return MAESTRO_MAC_ERR_CUDA; } while (0)
#define LAUNCHED(H) do { ++(H)->launches; if (cudaPeekAtLastError() != cudaSuccess) return MAESTRO_MAC_ERR_CUDA; } while (0)

// host_scal[at .. at+n) <- scal[at .. at+n) / host_flags likewise, visible to the host after the stream is synchronised
int publish_scal(maestro_mac_handle* H, int at, int n, cudaStream_t s)
{
    k_publish<<<1, 32, 0, s>>>(H->host_scal_dev + at, H->scal + at, n);
    ++H->launches;
    return cudaPeekAtLastError() == cudaSuccess ? MAESTRO_MAC_OK : MAESTRO_MAC_ERR_CUDA;
}
int publish_flags(maestro_mac_handle* H, int at, int n, cudaStream_t s)
{
    k_publish_int<<<1, 32, 0, s>>>(H->host_flags_dev + at, H->flags + at, n);
    ++H->launches;
    return cudaPeekAtLastError() == cudaSuccess ? MAESTRO_MAC_OK : MAESTRO_MAC_ERR_CUDA;
}

int red_blocks(const maestro_mac_handle* H, int rows) { return rows < H->red_blocks ? rows : H->red_blocks; }

enum { GH_PHI = 1, GH_RHS = 2, GH_AX = 4, GH_AY = 8, GH_AZ = 16 };

// periodic images of the selected arrays of a ghosted level (no-op on other levels)
int do_fill_ghosts(maestro_mac_handle* H, int l, int which, cudaStream_t s)
{
    const Level& L = H->lev[l];
    if (L.gx == 0 && L.gy == 0) return MAESTRO_MAC_OK;
    const int per_plane = 2 * L.gx * (L.n[1] + 1 + 2 * L.gy) + 2 * L.gy * (L.n[0] + 1);
    k_fill_ghosts<<<dim3((per_plane + 255) / 256, L.n[2] + 1), 256, 0, s>>>(dev_level(H, l), which);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

// ---- individual steps ------------------------------------------------------------------------

int do_coarsen(maestro_mac_handle* H, cudaStream_t s);
int do_rhs_finish(maestro_mac_handle* H, int nb, cudaStream_t s);

// grid of k_setup over the extended index space; the z-chunk grows until the block partials fit
dim3 setup_grid(const GeoDev& G, int* zchunk)
{
    int zc = 16;
    dim3 gg((G.nx + 64) / 64, (G.ny + 4) / 4, (G.nz + zc - 1) / zc);
    while ((long)gg.x * gg.y * gg.z > kMaxParts) { zc *= 2; gg.z = (G.nz + zc - 1) / zc; }
    *zchunk = zc;
    return gg;
}

int do_coefficients(maestro_mac_handle* H, const double* beta0, const double* rho0, const double* rho, cudaStream_t s)
{
    GeoDev G = dev_geo(H);
    dim3 g, b;
    CUDA_OK(cudaMemsetAsync(H->flags, 0, 16 * sizeof(int), s));
    if (H->d.smoother != 1 && rho) {
        const int zc = 16;
        dim3 gg((G.nx + 64) / 64, (G.ny + 4) / 4, (G.nz + zc - 1) / zc);
        if (H->d.rho_mean)
            k_setup<true, false, true><<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, rho, nullptr, nullptr,
                                                                  nullptr, nullptr, nullptr, zc, H->flags, nullptr, nullptr);
        else
            k_setup<true, false, false><<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, rho, nullptr, nullptr,
                                                                   nullptr, nullptr, nullptr, zc, H->flags, nullptr, nullptr);
    } else if (H->d.smoother != 1) {
        const int zc = 16;
        dim3 gg((G.nx + 64) / 64, (G.ny + 4) / 4, (G.nz + zc) / zc);
        k_face_coeff2<<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, rho, rho0, zc, H->flags);
    } else {
        dims3(G.nx + 1, G.ny + 1, G.nz + 1, &g, &b);
        k_face_coeff<<<g, b, 0, s>>>(G, dev_level(H, 0), beta0, rho, rho0, H->flags);
    }
    LAUNCHED(H);
    return do_coarsen(H, s);
}

// a3: periodic images of the level-0 coefficients, then every coarser level
int do_coarsen(maestro_mac_handle* H, cudaStream_t s)
{
    dim3 g, b;
    int rc;
    if ((rc = do_fill_ghosts(H, 0, GH_AX | GH_AY | GH_AZ, s)) != 0) return rc;
    for (int l = 0; l + 1 < H->nlev; ++l) {
        LevelDev C = dev_level(H, l + 1);
        dims3(C.nx + 1, C.ny + 1, C.nz + 1, &g, &b);
        k_coarsen_coeff<<<g, b, 0, s>>>(dev_level(H, l), C);
        LAUNCHED(H);
        if ((rc = do_fill_ghosts(H, l + 1, GH_AX | GH_AY | GH_AZ, s)) != 0) return rc;
    }
    return MAESTRO_MAC_OK;
}

// rhs on level 0; leaves sum/max of the final rhs in scal[0..1] and the removed sum in scal[2]
int do_rhs(maestro_mac_handle* H, const double* beta0, const double* u, const double* v, const double* w,
           const double* S, cudaStream_t s)
{
    GeoDev G = dev_geo(H);
    int nb;
    if (H->d.smoother != 1) {
        int zc;
        const dim3 gg = setup_grid(G, &zc);
        nb = (int)(gg.x * gg.y * gg.z);
        if (H->dpdt_term)
            k_setup<false, true, true><<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, nullptr, u, v, w, S,
                                                                  H->dpdt_term, zc, H->flags, H->part_sum, H->part_max);
        else
            k_setup<false, true, false><<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, nullptr, u, v, w, S,
                                                                   nullptr, zc, H->flags, H->part_sum, H->part_max);
    } else {
        int rows = G.ny * G.nz;
        nb = red_blocks(H, rows);
        int bt = G.nx >= 256 ? 256 : (G.nx >= 128 ? 128 : 64);
        k_rhs<<<nb, bt, 0, s>>>(G, dev_level(H, 0), beta0, u, v, w, S, H->dpdt_term, H->part_sum, H->part_max);
    }
    LAUNCHED(H);
    return do_rhs_finish(H, nb, s);
}

// a2 + a4 in one pass (k_setup<true, true>), then coarsening and the rhs reductions
int do_setup_fused(maestro_mac_handle* H, const double* beta0, const double* rho, const double* u, const double* v,
                   const double* w, const double* S, cudaStream_t s)
{
    GeoDev G = dev_geo(H);
    CUDA_OK(cudaMemsetAsync(H->flags, 0, 16 * sizeof(int), s));
    int zc;
    const dim3 gg = setup_grid(G, &zc);
    if (H->d.rho_mean || H->dpdt_term)
        k_setup<true, true, true><<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, rho, u, v, w, S,
                                                             H->dpdt_term, zc, H->flags, H->part_sum, H->part_max);
    else
        k_setup<true, true, false><<<gg, dim3(64, 4), 0, s>>>(G, dev_geo_inv(H), dev_level(H, 0), beta0, rho, u, v, w, S, nullptr,
                                                              zc, H->flags, H->part_sum, H->part_max);
    LAUNCHED(H);
    int rc;
    if ((rc = do_coarsen(H, s)) != 0) return rc;
    return do_rhs_finish(H, (int)(gg.x * gg.y * gg.z), s);
}

// folds the nb block partials of the rhs pass: sum/max of the final rhs in scal[0..1], removed sum in scal[2]
int do_rhs_finish(maestro_mac_handle* H, int nb, cudaStream_t s)
{
    Level& L0 = H->lev[0];
    k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, nb, H->scal);
    LAUNCHED(H);
    if (H->singular) {
        k_publish<<<1, 32, 0, s>>>(H->scal + 2, H->scal, 1);
        k_shift_mean<<<H->red_blocks, 256, 0, s>>>(dev_level(H, 0), L0.rhs, H->scal + 2, 1.0 / (double)L0.ncell, H->part_sum, H->part_max);
        LAUNCHED(H);
        k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, H->red_blocks, H->scal);
        LAUNCHED(H);
    } else {
        CUDA_OK(cudaMemsetAsync(H->scal + 2, 0, sizeof(double), s));
    }
    return do_fill_ghosts(H, 0, GH_RHS, s);
}

// One sweep on level l.  norm_parts != NULL (level-0 TMA path only, see fused_norm_ok): the sweep also
// writes per-CTA maxima of the red-cell residual of its INPUT to part_max and their count to *norm_parts.
// swap == false leaves the level's phi/phi2 roles untouched (the caller decides later; the result is in phi2).
int do_sweep(maestro_mac_handle* H, int l, cudaStream_t s, int* norm_parts = nullptr, bool swap = true)
{
    LevelDev L = dev_level(H, l);
    const bool timed = l == 0 && H->sm_ev && H->sm_used < kSmoothEvents;
    if (l == 0) ++H->sm_launches;
    if (timed) CUDA_OK(cudaEventRecord(H->sm_ev[2 * H->sm_used], s));
    const int sm = H->d.smoother;
    const int tv = ((sm == 0 || sm == 4) && L.nx >= 60) ? 0 : (sm == 3 ? 1 : -1);   // TMA tile variant, or -1
    if (tv >= 0 && H->lev[l].tma[tv].ok) {
        int rc = launch_tma_sweep(H->lev[l].tma[tv], H->lev[l].phi != H->lev[l].phi_a, H->lev[l].phi2, L, tv, H->sms, s,
                                  norm_parts ? H->part_max : nullptr, kMaxParts, norm_parts);
        if (rc != 0) return MAESTRO_MAC_ERR_CUDA;
        ++H->launches;
        if (swap) { double* t = H->lev[l].phi; H->lev[l].phi = H->lev[l].phi2; H->lev[l].phi2 = t; }
    } else if (norm_parts) {
        return MAESTRO_MAC_ERR_ARG;                                           // callers check fused_norm_ok first
    } else if (sm != 1 && fused_sweep_supported(L)) {
        int rc = launch_fused_sweep(H->lev[l].phi, H->lev[l].phi2, L, H->sms, s);
        if (rc != 0) return MAESTRO_MAC_ERR_CUDA;
        ++H->launches;
        // the fused sweep ping-pongs: result is in phi2; swap the level's buffers
        if (swap) { double* t = H->lev[l].phi; H->lev[l].phi = H->lev[l].phi2; H->lev[l].phi2 = t; }
    } else {
        dim3 g, b;
        dims3((L.nx + 1) / 2, L.ny, L.nz, &g, &b);
        k_rbgs_color<<<g, b, 0, s>>>(L, 0);
        LAUNCHED(H);
        k_rbgs_color<<<g, b, 0, s>>>(L, 1);
        LAUNCHED(H);
    }
    if (timed) { CUDA_OK(cudaEventRecord(H->sm_ev[2 * H->sm_used + 1], s)); ++H->sm_used; ++H->sm_sweeps; }
    return MAESTRO_MAC_OK;
}

// the two-sweep kernel runs with the default smoother on levels its tile and halo fit
bool t2_ok(const maestro_mac_handle* H, int l)
{
    return H->d.smoother == 0 && H->lev[l].tma[2].ok && t2_level_ok(dev_level(H, l));
}

// Two sweeps on level l in one pass (k_rbgs_t2).  norm_parts / swap as in do_sweep.
int do_sweep2(maestro_mac_handle* H, int l, cudaStream_t s, int* norm_parts = nullptr, bool swap = true)
{
    Level& Lv = H->lev[l];
    const bool timed = l == 0 && H->sm_ev && H->sm_used < kSmoothEvents;
    if (l == 0) ++H->sm_launches;
    if (timed) CUDA_OK(cudaEventRecord(H->sm_ev[2 * H->sm_used], s));
    const int nl = launch_t2_sweep(Lv.tma[2], Lv.phi != Lv.phi_a, Lv.phi2, dev_level(H, l), H->sms, s, norm_parts ? H->part_max : nullptr,
                                   kMaxParts, norm_parts);
    if (nl < 0) return MAESTRO_MAC_ERR_CUDA;
    H->launches += nl;
    if (swap) { double* t = Lv.phi; Lv.phi = Lv.phi2; Lv.phi2 = t; }
    if (timed) { CUDA_OK(cudaEventRecord(H->sm_ev[2 * H->sm_used + 1], s)); ++H->sm_used; H->sm_sweeps += 2; }
    return MAESTRO_MAC_OK;
}

int do_smooth(maestro_mac_handle* H, int l, int nsweeps, cudaStream_t s)
{
    if (t2_ok(H, l))
        for (; nsweeps >= 2; nsweeps -= 2) {
            int rc = do_sweep2(H, l, s);
            if (rc != 0) return rc;
        }
    for (int sw = 0; sw < nsweeps; ++sw) {
        int rc = do_sweep(H, l, s);
        if (rc != 0) return rc;
    }
    return MAESTRO_MAC_OK;
}

// TMA transfer kernels are used with the default smoother on levels the tensor maps cover
bool tma_aux(const maestro_mac_handle* H, int l)
{
    return (H->d.smoother == 0 || H->d.smoother == 4) && H->lev[l].tma[0].ok && H->lev[l].n[0] >= 60 && H->lev[l].n[2] >= 2;
}

int do_residual_restrict(maestro_mac_handle* H, int l, cudaStream_t s)
{
    if (tma_aux(H, l)) {
        Level& F = H->lev[l];
        int n = launch_tma_resid(F.tma[0], F.phi != F.phi_a, dev_level(H, l), dev_level(H, l + 1),
                                 H->part_max, kMaxParts, tma::RES_RESTRICT, H->sms, s);
        if (n < 0) return MAESTRO_MAC_ERR_CUDA;
        ++H->launches;
        return MAESTRO_MAC_OK;
    }
    LevelDev C = dev_level(H, l + 1);
    dim3 g, b;
    dims3(C.nx, C.ny, C.nz, &g, &b);
    k_residual_restrict<<<g, b, 0, s>>>(dev_level(H, l), C);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

int do_prolong(maestro_mac_handle* H, int l, cudaStream_t s)
{
    LevelDev F = dev_level(H, l);
    dim3 g, b;
    if (H->d.smoother != 1 && (F.nx & 1) == 0) {             // bandwidth form: one thread per coarse cell
        LevelDev C = dev_level(H, l + 1);
        dims3(C.nx, C.ny, C.nz, &g, &b);
#ifdef MAC_PROLONG_INPLACE
        k_prolong_add2<<<g, b, 0, s>>>(F, C, H->d.prolongation, F.phi);
        LAUNCHED(H);
#else
        k_prolong_add2<<<g, b, 0, s>>>(F, C, H->d.prolongation, F.phi2);      // phi + P e into the ping-pong partner, then swap
        LAUNCHED(H);
        { double* t = H->lev[l].phi; H->lev[l].phi = H->lev[l].phi2; H->lev[l].phi2 = t; }
#endif
        return MAESTRO_MAC_OK;
    }
    dims3(F.nx, F.ny, F.nz, &g, &b);
    k_prolong_add<<<g, b, 0, s>>>(F, dev_level(H, l + 1), H->d.prolongation);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

// The coarse tail: the first level of at most kTailMaxCells cells from which everything down to the coarsest
// level fits one thread block's shared memory.  Not with the reference (1) and cp.async-only (2) smoothers,
// which keep one launch per step on every level.
unsigned tail_magic(int d) { return d <= 1 ? 0u : (unsigned)((1ull << 32) / (unsigned)d + 1ull); }

void plan_tail(maestro_mac_handle* H, bool allow_cluster = true)
{
    H->tail_start = -1;
    H->tail_smem = 0;
    H->cl_start = -1;
    if (H->d.smoother == 1 || H->d.smoother == 2) return;
    // the cluster kernel takes every level from the first one of at most 32^3 cells (plain layout) down to the bottom,
    // if the slabs fit the blocks' shared memory and the bottom level is small enough for block 0
    for (int t0 = 0; allow_cluster && t0 + 1 < H->nlev && H->d.smoother == 0; ++t0) {
        if (H->lev[t0].ncell > (size_t)clus::kMaxCells || H->nlev - t0 > clus::kMaxLevels) continue;
        if (H->lev[t0].gx || H->lev[t0].gy) continue;
        if (H->lev[H->nlev - 1].ncell > (size_t)clus::kMaxBottom) break;
        clus::Args& A = H->cl;
        A.nlev = H->nlev - t0;
        size_t off = 0;
        for (int q = 0; q < A.nlev; ++q) {
            const Level& L = H->lev[t0 + q];
            clus::Lev& V = A.V[q];
            const bool bottom = q + 1 == A.nlev;
            V.hx = (L.n[0] + 1) / 2;
            V.mx = tail_magic(L.n[0]); V.mxy = tail_magic(L.n[0] * L.n[1]);
            V.mhx = tail_magic(V.hx); V.mhxy = tail_magic(V.hx * L.n[1]);
            V.ppc = bottom ? L.n[2] : (L.n[2] + clus::kCtas - 1) / clus::kCtas;
            V.mppc = tail_magic(V.ppc);
            const size_t pe = (size_t)L.n[0] * L.n[1];
            V.o_phi = (int)off; off += pe * V.ppc;
            V.o_rhs = (int)off; off += pe * V.ppc;
            V.o_ax = V.o_ay = V.o_az = 0;
            if (!bottom) {                                 // the bottom is solved by BiCGStab from the global coefficients
                V.o_ax = (int)off; off += (size_t)(L.n[0] + 1) * L.n[1] * V.ppc;
                V.o_ay = (int)off; off += (size_t)L.n[0] * (L.n[1] + 1) * V.ppc;
                V.o_az = (int)off; off += pe * (V.ppc + 1);
            }
        }
        A.o_vecs = (int)off;
        if (H->lev[H->nlev - 1].ncell > (size_t)clus::kWarpBottom) off += 6 * H->lev[H->nlev - 1].ncell;
        A.o_scr = (int)off;
        {
            size_t scr = 0;
            for (int q = 1; q < A.nlev; ++q) {
                const Level& L = H->lev[t0 + q];
                const size_t own = (size_t)L.n[0] * L.n[1] * A.V[q].ppc * 8;
                if (own > scr) scr = own;
            }
            off += scr;
        }
        if (off * sizeof(double) > clus::kSmemMax) continue;
        H->cl_start = t0;
        H->cl_smem = off * sizeof(double);
        return;
    }
    for (int t0 = 0; t0 + 1 < H->nlev; ++t0) {
        if (H->lev[t0].ncell > (size_t)kTailMaxCells || H->nlev - t0 > kTailMaxLevels) continue;
        if (H->lev[t0].gx || H->lev[t0].gy) continue;
        TailArgs& A = H->tail;
        size_t off = 0;
        A.nlev = H->nlev - t0;
        for (int q = 0; q < A.nlev; ++q) {
            const Level& L = H->lev[t0 + q];
            TailLevel& T = A.T[q];
            T.nx = L.n[0]; T.ny = L.n[1]; T.nz = L.n[2]; T.nc = (int)L.ncell;
            const int hx = (T.nx + 1) / 2;
            T.mx = tail_magic(T.nx); T.mxy = tail_magic(T.nx * T.ny); T.mhx = tail_magic(hx); T.mhxy = tail_magic(hx * T.ny);
            for (int a = 0; a < 3; ++a) T.per[a] = H->d.bc_lo[a] == MAESTRO_MAC_PERIODIC;
            T.o_phi = (int)off; off += (size_t)T.nc + 1;
            T.o_rhs = (int)off; off += (size_t)T.nc;
            T.o_ax = T.o_ay = T.o_az = 0;
            if (q + 1 < A.nlev) {                      // the coarsest level is solved by BiCGStab from the global coefficients
                T.o_ax = (int)off; off += (size_t)(T.nx + 1) * T.ny * T.nz;
                T.o_ay = (int)off; off += (size_t)T.nx * (T.ny + 1) * T.nz;
                T.o_az = (int)off; off += (size_t)T.nx * T.ny * (T.nz + 1);
            }
        }
        A.o_vecs = (int)off;
        off += 6 * H->lev[H->nlev - 1].ncell;
        if (off * sizeof(double) > kTailSmem) continue;
        H->tail_start = t0;
        H->tail_smem = off * sizeof(double);
        return;
    }
}

// levels tail_start .. coarsest in one launch
int do_tail(maestro_mac_handle* H, cudaStream_t s)
{
    TailArgs& A = H->tail;
    for (int q = 0; q < A.nlev; ++q) A.L[q] = dev_level(H, H->tail_start + q);
    A.nu_pre = H->d.nu_pre; A.nu_post = H->d.nu_post;
    A.maxit = H->d.bottom_max_iter; A.tol = H->d.bottom_rel_tol;
    A.singular = H->singular; A.prolongation = H->d.prolongation;
    A.load_phi = H->tail_start == 0 ? 1 : 0;
    const size_t nc = H->lev[H->tail_start].ncell;
    const int threads = nc >= 2048 ? 1024 : (nc >= 512 ? 256 : 64);
    k_coarse_tail<<<1, threads, H->tail_smem, s>>>(A, H->flags + 1);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

// levels cl_start .. coarsest in one launch of one cluster; solve: whole cycles with the stop test (cl_start == 0)
int do_cluster(maestro_mac_handle* H, cudaStream_t s, int solve, int max_cycles, double rel_tol)
{
    clus::Args& A = H->cl;
    for (int q = 0; q < A.nlev; ++q) A.V[q].L = dev_level(H, H->cl_start + q);
    A.nu_pre = H->d.nu_pre; A.nu_post = H->d.nu_post;
    A.maxit = H->d.bottom_max_iter; A.tol = H->d.bottom_rel_tol;
    A.singular = H->singular; A.prolongation = H->d.prolongation;
    A.solve = solve; A.max_cycles = max_cycles; A.rel_tol = rel_tol;
    A.rhs_norm = H->scal + 1;
    A.result = H->cl_scratch + 8;
    A.iters_accum = H->flags + 1;
    const size_t sm = H->cl_smem;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(clus::kCtas, 1, 1);
    cfg.blockDim = dim3(clus::kThreads, 1, 1);
    cfg.dynamicSmemBytes = sm;
    cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = clus::kCtas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    if (cudaLaunchKernelEx(&cfg, clus::k_cluster_vcycles, A) != cudaSuccess) return MAESTRO_MAC_ERR_CUDA;
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

int do_bottom(maestro_mac_handle* H, cudaStream_t s)
{
    int l = H->nlev - 1;
    int nb = (int)H->lev[l].ncell;
    int threads = nb >= 1024 ? 1024 : ((nb + 31) / 32) * 32;
    const size_t sm = 7 * (size_t)nb * sizeof(double);
    const int use_smem = sm <= kBottomSmem ? 1 : 0;
    k_bottom_bicgstab<<<1, threads, use_smem ? sm : 0, s>>>(dev_level(H, l), H->bottom_vecs, H->d.bottom_max_iter,
                                                            H->d.bottom_rel_tol, H->singular, H->flags + 1, use_smem);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

// The stop test can ride on the first level-0 pre-sweep of the NEXT cycle (k_rbgs_tma NORM variant): after
// a post-sweep the black residuals are zero up to rounding (the black pass has just solved those
// equations), so ||rhs - L phi||inf is the maximum over the red cells, which the red update has at hand.
// The sweep writes to the ping-pong partner, so a converged phi is still intact when the test passes.
bool fused_norm_ok(const maestro_mac_handle* H)
{
    const Level& L0 = H->lev[0];
    if (H->d.stop_test != 0 || (H->d.smoother != 0 && H->d.smoother != 4) || H->nlev < 2 || H->d.nu_pre < 1 || H->d.nu_post < 1) return false;
    if (!L0.tma[0].ok || L0.n[0] < 60) return false;
    const dim3 g = tma_sweep_grid(dev_level(H, 0), 0, H->sms, nullptr);
    if ((long)g.x * g.y * g.z > kMaxParts) return false;
    if (t2_ok(H, 0)) {
        if (t2_plan(dev_level(H, 0), H->sms).ncta > kMaxParts) return false;
    }
    return true;
}

// pre_done: level-0 pre-sweeps of this cycle that have already been applied (they carried the stop test
// of the previous cycle, see maestro_mac_project)
int do_vcycle(maestro_mac_handle* H, cudaStream_t s, int pre_done = 0)
{
    int rc;
    // with a coarse tail the levels from tail_start down are one launch (pre_done only ever concerns a level-0
    // TMA sweep, i.e. a level far above the tail)
    const int lend = H->cl_start >= 0 ? H->cl_start : (H->tail_start >= 0 ? H->tail_start : H->nlev - 1);
    for (int l = 0; l < lend; ++l) {
        if ((rc = do_smooth(H, l, H->d.nu_pre - (l == 0 ? pre_done : 0), s)) != 0) return rc;
        if ((rc = do_residual_restrict(H, l, s)) != 0) return rc;
    }
    if ((rc = H->cl_start >= 0 ? do_cluster(H, s, 0, 1, 0.0) : (H->tail_start >= 0 ? do_tail(H, s) : do_bottom(H, s))) != 0) return rc;
    for (int l = lend - 1; l >= 0; --l) {
        if ((rc = do_prolong(H, l, s)) != 0) return rc;
        if ((rc = do_smooth(H, l, H->d.nu_post, s)) != 0) return rc;
    }
    return MAESTRO_MAC_OK;
}

// max-norm of the residual of a level into scal[4]
int do_residual_norm(maestro_mac_handle* H, int l, cudaStream_t s)
{
    LevelDev L = dev_level(H, l);
    if (tma_aux(H, l)) {
        Level& F = H->lev[l];
        int n = launch_tma_resid(F.tma[0], F.phi != F.phi_a, L, L, H->part_max, kMaxParts, tma::RES_NORM, H->sms, s);
        if (n < 0) return MAESTRO_MAC_ERR_CUDA;
        ++H->launches;
        k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, n, H->scal + 3);
        LAUNCHED(H);
        return MAESTRO_MAC_OK;
    }
    int rows = L.ny * L.nz;
    int nb = red_blocks(H, rows);
    int bt = L.nx >= 256 ? 256 : (L.nx >= 128 ? 128 : 64);
    k_residual_norm<<<nb, bt, 0, s>>>(L, H->part_sum, H->part_max);
    LAUNCHED(H);
    k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, nb, H->scal + 3);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

int do_correct(maestro_mac_handle* H, const double* phi, const double* rho0, const double* rho,
               double* u, double* v, double* w, cudaStream_t s)
{
    GeoDev G = dev_geo(H);
    dim3 g, b;
    dims3(G.nx + 1, G.ny + 1, G.nz + 1, &g, &b);
    k_correct<<<g, b, 0, s>>>(G, dev_level(H, 0), phi, rho, rho0, u, v, w);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

}  // namespace

// ================================================================================================
// C ABI
// ================================================================================================

extern "C" void maestro_mac_default_desc(maestro_mac_desc* d)
{
    if (!d) return;
    std::memset(d, 0, sizeof(*d));
    d->struct_bytes = (int)sizeof(maestro_mac_desc);
    d->nx = d->ny = d->nz = 32;
    for (int a = 0; a < 3; ++a) { d->dx[a] = 1.0; d->bc_lo[a] = d->bc_hi[a] = MAESTRO_MAC_PERIODIC; }
    d->geometry = MAESTRO_MAC_PLANAR;
    d->nr = 32;
    d->dr = 1.0;
    d->nu_pre = d->nu_post = 2;
    d->max_cycles = 100;
    d->rel_tol = 1e-10;
    d->coarsest_n = 4;
    d->bottom_max_iter = 100;
    d->bottom_rel_tol = 1e-8;
}

extern "C" int maestro_mac_setup(const maestro_mac_desc* desc, void* workspace, size_t workspace_bytes,
                                 size_t* workspace_needed, maestro_mac_handle** out)
{
    if (out) *out = nullptr;
    maestro_mac_handle tmp;
    std::memset(&tmp, 0, sizeof(tmp));
    int rc = validate_and_default(desc, &tmp.d);
    if (rc != MAESTRO_MAC_OK) return rc;
    rc = build_levels(tmp.d, tmp.lev, &tmp.nlev);
    if (rc != MAESTRO_MAC_OK) return rc;
    size_t need = carve(&tmp, nullptr);
    if (workspace_needed) *workspace_needed = need;
    if (!workspace || workspace_bytes < need) return MAESTRO_MAC_ERR_WORKSPACE;
    if (!out) return MAESTRO_MAC_ERR_ARG;
    if (((uintptr_t)workspace & 255u) != 0) return MAESTRO_MAC_ERR_ARG;

    maestro_mac_handle* H = new (std::nothrow) maestro_mac_handle;
    if (!H) return MAESTRO_MAC_ERR_ARG;
    *H = tmp;
    carve(H, (char*)workspace);
    H->singular = 1;
    for (int a = 0; a < 3; ++a)
        if (H->d.bc_lo[a] == MAESTRO_MAC_OUTFLOW || H->d.bc_hi[a] == MAESTRO_MAC_OUTFLOW) H->singular = 0;
    H->host_scal = nullptr;
    H->host_flags = nullptr;
    H->host_hist = nullptr;
    for (int e = 0; e < 4; ++e) H->ev[e] = nullptr;
    bool ok = cudaHostAlloc((void**)&H->host_scal, 8 * sizeof(double), cudaHostAllocMapped) == cudaSuccess &&
              cudaHostAlloc((void**)&H->host_flags, 4 * sizeof(int), cudaHostAllocMapped) == cudaSuccess &&
              cudaHostGetDevicePointer((void**)&H->host_scal_dev, H->host_scal, 0) == cudaSuccess &&
              cudaHostGetDevicePointer((void**)&H->host_flags_dev, H->host_flags, 0) == cudaSuccess &&
              cudaHostAlloc((void**)&H->host_hist, (4 + 128) * sizeof(double), cudaHostAllocMapped) == cudaSuccess &&
              cudaHostGetDevicePointer((void**)&H->host_hist_dev, H->host_hist, 0) == cudaSuccess;
    for (int e = 0; ok && e < 4; ++e) ok = cudaEventCreate(&H->ev[e]) == cudaSuccess;
    H->sm_ev = nullptr;
    H->sm_used = H->sm_launches = H->sm_sweeps = 0;
    H->cp_in = H->cp_out = nullptr;
    for (int e = 0; e < 3; ++e) H->ev_in[e] = H->ev_done[e] = H->ev_out[e] = nullptr;
    if (ok && H->d.host_staging >= 2) {
        ok = cudaStreamCreateWithFlags(&H->cp_in, cudaStreamNonBlocking) == cudaSuccess &&
             cudaStreamCreateWithFlags(&H->cp_out, cudaStreamNonBlocking) == cudaSuccess;
        for (int e = 0; ok && e < 3; ++e)
            ok = cudaEventCreateWithFlags(&H->ev_in[e], cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&H->ev_done[e], cudaEventDisableTiming) == cudaSuccess &&
                 cudaEventCreateWithFlags(&H->ev_out[e], cudaEventDisableTiming) == cudaSuccess;
    }
    {
        int dev = 0, sms = 0;
        ok = ok && cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0;
        H->sms = ok ? sms : 1;
        H->red_blocks = kRedBlocksPerSm * H->sms;
        if (H->red_blocks > kMaxParts) H->red_blocks = kMaxParts;
    }
    H->deferred = 0;
    if (ok && H->d.timing) {                         // per-launch event pairs of the level-0 smoother: only on request
        H->sm_ev = (cudaEvent_t*)std::calloc(2 * kSmoothEvents, sizeof(cudaEvent_t));
        ok = H->sm_ev != nullptr;
        for (int e = 0; ok && e < 2 * kSmoothEvents; ++e) ok = cudaEventCreate(&H->sm_ev[e]) == cudaSuccess;
    }
    plan_tail(H);
    if (ok) ok = cudaFuncSetAttribute(k_coarse_tail, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kTailSmem) == cudaSuccess;
    if (ok) ok = cudaFuncSetAttribute(k_lateral_sum, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kLateralSmem) == cudaSuccess;
    if (ok) ok = cudaFuncSetAttribute(clus::k_cluster_vcycles, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)clus::kSmemMax) == cudaSuccess;
    if (ok) ok = cudaFuncSetAttribute(clus::k_cluster_vcycles, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
    if (ok && H->cl_start >= 0) {                    // can this device place a 16-block cluster with that much shared memory?
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(clus::kCtas, 1, 1);
        cfg.blockDim = dim3(clus::kThreads, 1, 1);
        cfg.dynamicSmemBytes = H->cl_smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = clus::kCtas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        int nclusters = 0;
        if (cudaOccupancyMaxActiveClusters(&nclusters, clus::k_cluster_vcycles, &cfg) != cudaSuccess || nclusters < 1) {
            (void)cudaGetLastError();
            plan_tail(H, false);                     // no: the one-block tail (or one launch per step) takes the small levels
        }
    }
    if (ok) ok = cudaFuncSetAttribute(k_bottom_bicgstab, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBottomSmem) == cudaSuccess;
    if (ok) ok = smoother_configure() == 0 && tma_smoother_configure() == 0 && tma_resid_configure() == 0 && t2_smoother_configure() == 0;
    if (ok)
        for (int l = 0; l < H->nlev; ++l) {          // tensor maps; a level that cannot use TMA keeps cp.async
            LevelDev D = dev_level(H, l);
            tma_build_maps(&H->lev[l].tma[0], D, 32, 16);
            tma_build_maps(&H->lev[l].tma[1], D, 16, 16);
            t2_build_maps(&H->lev[l].tma[2], D);
            // a level laid out with periodic images has no other smoother: its tensor maps must exist
            if ((D.gx || D.gy) && !H->lev[l].tma[H->d.smoother == 3 ? 1 : 0].ok) ok = false;
        }
    if (ok && H->has_nodal)
        for (int l = 0; l < H->nlev; ++l) {          // tensor maps of k_nod_march (Jacobi sweeps, residuals)
            NodHost& N = H->nod[l];
            const uint64_t nzn = (uint64_t)N.n[2] + 3, nzc = (uint64_t)N.n[2] + 2;
            N.tma_ok = tma_encode3(&N.tm_phi, N.phi - N.onode, N.NX, N.NY, nzn, N.NX, N.NY, nodm::BW, nodm::TY + 2) &&
                       tma_encode3(&N.tm_phi2, N.phi2 - N.onode, N.NX, N.NY, nzn, N.NX, N.NY, nodm::BW, nodm::TY + 2) &&
                       tma_encode3(&N.tm_rhs, N.rhs - N.onode, N.NX, N.NY, nzn, N.NX, N.NY, nodm::TX, nodm::TY) &&
                       tma_encode3(&N.tm_sig, N.sigma - N.ocell, N.CX, N.CY, nzc, N.CX, N.CY, nodm::BW, nodm::TY + 1);
            if (!N.tma_ok) ok = false;
        }
    if (!ok) {
        maestro_mac_free(H);
        return MAESTRO_MAC_ERR_CUDA;
    }
    *out = H;
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_free(maestro_mac_handle* H)
{
    if (!H) return MAESTRO_MAC_OK;
    if (H->host_scal) cudaFreeHost(H->host_scal);
    if (H->host_flags) cudaFreeHost(H->host_flags);
    if (H->host_hist) cudaFreeHost(H->host_hist);
    for (int e = 0; e < 4; ++e)
        if (H->ev[e]) cudaEventDestroy(H->ev[e]);
    if (H->cp_in) cudaStreamDestroy(H->cp_in);
    if (H->cp_out) cudaStreamDestroy(H->cp_out);
    for (int e = 0; e < 3; ++e) {
        if (H->ev_in[e]) cudaEventDestroy(H->ev_in[e]);
        if (H->ev_done[e]) cudaEventDestroy(H->ev_done[e]);
        if (H->ev_out[e]) cudaEventDestroy(H->ev_out[e]);
    }
    if (H->sm_ev) {
        for (int e = 0; e < 2 * kSmoothEvents; ++e)
            if (H->sm_ev[e]) cudaEventDestroy(H->sm_ev[e]);
        std::free(H->sm_ev);
    }
    delete H;
    return MAESTRO_MAC_OK;
}

// Fills the timing members of st after the stream has been synchronised.
static void collect_timings(maestro_mac_handle* H, maestro_mac_stats& st)
{
    st.bottom_iters_total = H->host_flags[1];
    cudaEventElapsedTime(&st.ms_setup_kernels, H->ev[0], H->ev[1]);
    cudaEventElapsedTime(&st.ms_vcycles, H->ev[1], H->ev[2]);
    cudaEventElapsedTime(&st.ms_correct, H->ev[2], H->ev[3]);
    st.smooth0_launches = H->sm_launches;
    st.smooth0_timed = H->sm_used;
    st.smooth0_sweeps_timed = H->sm_sweeps;
    double acc = 0.0;
    for (int q = 0; q < H->sm_used; ++q) {
        float ms = 0.0f;
        cudaEventElapsedTime(&ms, H->sm_ev[2 * q], H->sm_ev[2 * q + 1]);
        acc += ms;
    }
    st.ms_smooth0 = (float)acc;
}

extern "C" int maestro_mac_project(maestro_mac_handle* H, const double* beta0, const double* rho0,
                                   const double* rho, double* u, double* v, double* w, const double* S,
                                   double* phi, maestro_mac_stats* stats, void* cuda_stream)
{
    if (!H || !beta0 || !u || !v || !w) return MAESTRO_MAC_ERR_ARG;
    if (!rho && !rho0) return MAESTRO_MAC_ERR_ARG;
    if (u == v || u == w || v == w || (phi && (phi == u || phi == v || phi == w || phi == rho || phi == S)))
        return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const maestro_mac_desc& d = H->d;
    maestro_mac_stats st;
    std::memset(&st, 0, sizeof(st));
    st.singular = H->singular;
    st.levels = H->nlev;
    H->launches = 0;
    H->sm_used = H->sm_launches = H->sm_sweeps = 0;
    H->deferred = 0;
    int rc;
    int result = MAESTRO_MAC_OK;
    Level& L0 = H->lev[0];
    // rel_tol == 0 without stats: nothing the host must read.  The call enqueues everything and returns; the
    // non-finite check is deferred to maestro_mac_status() and a zero rhs simply runs its (trivial) cycles.
    const bool async = d.rel_tol == 0.0 && !stats;

    CUDA_OK(cudaEventRecord(H->ev[0], s));
    if (rho && d.smoother != 1) {
        if ((rc = do_setup_fused(H, beta0, rho, u, v, w, S, s)) != 0) return rc;
    } else {
        if ((rc = do_coefficients(H, beta0, rho0, rho, s)) != 0) return rc;
        if ((rc = do_rhs(H, beta0, u, v, w, S, s)) != 0) return rc;
    }
    if (publish_scal(H, 0, 3, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    if (publish_flags(H, 0, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    CUDA_OK(cudaMemsetAsync(L0.phi - L0.off_c, 0, L0.acell * sizeof(double), s));   // A16: phi = 0 (ghosts too)
    CUDA_OK(cudaEventRecord(H->ev[1], s));
    bool trivial = false;
    if (!async) {
        CUDA_OK(cudaStreamSynchronize(s));
        st.rhs_norm_inf = H->host_scal[1];
        st.rhs_mean_removed = H->singular ? H->host_scal[2] / (double)L0.ncell : 0.0;
        const bool bad = H->host_flags[0] != 0 || !std::isfinite(st.rhs_norm_inf) || !std::isfinite(H->host_scal[0]);
        if (bad) {
            if (stats) *stats = st;
            return MAESTRO_MAC_ERR_NONFINITE;
        }
        trivial = st.rhs_norm_inf == 0.0;
    }
    // a problem whose level 0 already fits the cluster kernel is solved by ONE launch: cycles and stop test on the
    // device, the host reads the cycle count and the residual history after the final synchronise
    const bool device_solve = H->cl_start == 0;
    if (!trivial && device_solve) {
        if ((rc = do_cluster(H, s, 1, d.max_cycles, d.rel_tol > 0.0 ? d.rel_tol : -1.0)) != 0) return rc;
        k_publish<<<1, 32, 0, s>>>(H->host_hist_dev, H->cl_scratch + 8, 4 + 128);
        LAUNCHED(H);
        if (d.rel_tol == 0.0) st.cycles = d.max_cycles;                       // (known without reading anything back)
    } else if (!trivial) {
        result = d.rel_tol > 0.0 ? MAESTRO_MAC_NOT_CONVERGED : MAESTRO_MAC_OK;
        if (d.rel_tol > 0.0) {
            const bool ride = fused_norm_ok(H);
            const bool ride2 = ride && d.nu_pre >= 2 && t2_ok(H, 0);     // the speculative launch is a two-sweep pass
            int pre_done = 0;
            while (st.cycles < d.max_cycles) {
                if ((rc = do_vcycle(H, s, pre_done)) != 0) return rc;
                pre_done = 0;
                const bool spec = ride && st.cycles + 1 < d.max_cycles;   // speculative first sweep(s) of the next cycle
                if (spec) {
                    int nparts = 0;
                    if ((rc = ride2 ? do_sweep2(H, 0, s, &nparts, false) : do_sweep(H, 0, s, &nparts, false)) != 0) return rc;
                    k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, nparts, H->scal + 3, H->host_scal_dev + 3);   // (published too)
                    LAUNCHED(H);
                } else {
                    if ((rc = do_residual_norm(H, 0, s)) != 0) return rc;
                    if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
                }
                CUDA_OK(cudaStreamSynchronize(s));
                st.res_norm_inf = H->host_scal[4];
                const double rel = st.res_norm_inf / st.rhs_norm_inf;
                if (st.cycles < 128) st.res_history[st.cycles] = rel;
                ++st.cycles;
                if (rel != rel) { result = MAESTRO_MAC_ERR_NONFINITE; break; }
                if (rel <= d.rel_tol) { result = MAESTRO_MAC_OK; break; }   // (a speculative sweep's output is dropped)
                if (spec) {                                                  // keep it: the next cycle's first pre-sweep(s)
                    double* t = L0.phi; L0.phi = L0.phi2; L0.phi2 = t;
                    pre_done = ride2 ? 2 : 1;
                }
            }
        } else {
            for (; st.cycles < d.max_cycles; ++st.cycles)
                if ((rc = do_vcycle(H, s)) != 0) return rc;
        }
    }
    CUDA_OK(cudaEventRecord(H->ev[2], s));
    // A10: the phi a singular problem returns has zero mean.  The correction takes differences of phi only (a singular
    // problem has no OUTFLOW face), so it runs on the iterate as it stands and the mean is removed while phi is written
    // to the caller's array -- one pass instead of an in-place shift plus a copy, and none at all when phi == NULL.
    const bool solved = !trivial && result != MAESTRO_MAC_ERR_NONFINITE;
    if (solved && (rc = do_correct(H, H->lev[0].phi, rho0, rho, u, v, w, s)) != 0) return rc;
    if (phi) {
        if (solved && H->singular) {
            k_sum<<<H->red_blocks, 256, 0, s>>>(dev_level(H, 0), H->lev[0].phi, H->part_sum, H->part_max);
            LAUNCHED(H);
            k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, H->red_blocks, H->scal + 6);
            LAUNCHED(H);
            k_shift_mean_out<<<H->red_blocks, 256, 0, s>>>(dev_level(H, 0), H->lev[0].phi, H->scal + 6, 1.0 / (double)L0.ncell, phi);
            LAUNCHED(H);
        } else if (L0.gx == 0 && L0.gy == 0) {
            CUDA_OK(cudaMemcpyAsync(phi, L0.phi, L0.ncell * sizeof(double), cudaMemcpyDeviceToDevice, s));
        } else {
            dim3 g, b;
            dims3(L0.n[0], L0.n[1], L0.n[2], &g, &b);
            k_copy_level<<<g, b, 0, s>>>(dev_level(H, 0), L0.phi, phi, 0, L0.n[0], L0.n[1], L0.n[2], 1);
            LAUNCHED(H);
        }
    }
    CUDA_OK(cudaEventRecord(H->ev[3], s));
    if (publish_flags(H, 1, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    st.gpu_launches = H->launches;
    if (async) {                                   // nothing was read back: maestro_mac_status() completes the picture
        H->deferred = 1;
        H->last = st;
        return MAESTRO_MAC_OK;
    }
    CUDA_OK(cudaStreamSynchronize(s));
    collect_timings(H, st);
    if (device_solve && !trivial) {
        st.cycles = (int)H->host_hist[0];
        st.res_norm_inf = H->host_hist[1];
        for (int c = 0; c < st.cycles && c < 128; ++c) st.res_history[c] = H->host_hist[4 + c];
        if (H->host_hist[2] != 0.0) result = MAESTRO_MAC_ERR_NONFINITE;       // (a NaN met during the cycles; results were written)
        else if (d.rel_tol > 0.0) result = st.res_norm_inf <= d.rel_tol * st.rhs_norm_inf ? MAESTRO_MAC_OK : MAESTRO_MAC_NOT_CONVERGED;
    } else if (d.rel_tol == 0.0 && !trivial) {   // fixed-cycle run: report the final residual too
        if ((rc = do_residual_norm(H, 0, s)) != 0) return rc;
        if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
        CUDA_OK(cudaStreamSynchronize(s));
        st.res_norm_inf = H->host_scal[4];
        st.gpu_launches = H->launches;
    }
    H->last = st;
    if (stats) *stats = st;
    return result;
}

extern "C" int maestro_mac_status(maestro_mac_handle* H, maestro_mac_stats* stats, void* cuda_stream)
{
    if (!H) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    if (!H->deferred) {
        if (stats) *stats = H->last;
        return MAESTRO_MAC_OK;
    }
    CUDA_OK(cudaStreamSynchronize(s));
    H->deferred = 0;
    maestro_mac_stats st = H->last;
    st.rhs_norm_inf = H->host_scal[1];
    st.rhs_mean_removed = H->singular ? H->host_scal[2] / (double)H->lev[0].ncell : 0.0;
    collect_timings(H, st);
    int result = MAESTRO_MAC_OK;
    if (H->host_flags[0] != 0 || !std::isfinite(st.rhs_norm_inf) || !std::isfinite(H->host_scal[0])) result = MAESTRO_MAC_ERR_NONFINITE;
    else if (stats) {                              // the final residual, as the synchronous fixed-cycle call reports it
        int rc;
        if ((rc = do_residual_norm(H, 0, s)) != 0) return rc;
        if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
        CUDA_OK(cudaStreamSynchronize(s));
        st.res_norm_inf = H->host_scal[4];
        st.gpu_launches = H->launches;
    }
    H->last = st;
    if (stats) *stats = st;
    return result;
}

extern "C" int maestro_mac_project_host(maestro_mac_handle* H, const double* beta0, const double* rho0,
                                        const double* rho, double* u, double* v, double* w, const double* S,
                                        double* phi, maestro_mac_stats* stats, void* cuda_stream)
{
    if (!H || !H->has_staging || !beta0 || !u || !v || !w || (!rho && !rho0)) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const maestro_mac_desc& d = H->d;
    const size_t nc = (size_t)d.nx * d.ny * d.nz;
    const size_t nu = (size_t)(d.nx + 1) * d.ny * d.nz, nv = (size_t)d.nx * (d.ny + 1) * d.nz, nw = (size_t)d.nx * d.ny * (d.nz + 1);
    Staging& T = H->st;
    CUDA_OK(cudaMemcpyAsync(T.beta0, beta0, d.nr * sizeof(double), cudaMemcpyHostToDevice, s));
    if (rho0) CUDA_OK(cudaMemcpyAsync(T.rho0, rho0, d.nr * sizeof(double), cudaMemcpyHostToDevice, s));
    if (rho) CUDA_OK(cudaMemcpyAsync(T.rho, rho, nc * sizeof(double), cudaMemcpyHostToDevice, s));
    if (S) CUDA_OK(cudaMemcpyAsync(T.S, S, nc * sizeof(double), cudaMemcpyHostToDevice, s));
    CUDA_OK(cudaMemcpyAsync(T.u, u, nu * sizeof(double), cudaMemcpyHostToDevice, s));
    CUDA_OK(cudaMemcpyAsync(T.v, v, nv * sizeof(double), cudaMemcpyHostToDevice, s));
    CUDA_OK(cudaMemcpyAsync(T.w, w, nw * sizeof(double), cudaMemcpyHostToDevice, s));
    int rc = maestro_mac_project(H, T.beta0, rho0 ? T.rho0 : nullptr, rho ? T.rho : nullptr, T.u, T.v, T.w,
                                 S ? T.S : nullptr, phi ? T.phi : nullptr, stats, cuda_stream);
    if (rc < 0) return rc;
    CUDA_OK(cudaMemcpyAsync(u, T.u, nu * sizeof(double), cudaMemcpyDeviceToHost, s));
    CUDA_OK(cudaMemcpyAsync(v, T.v, nv * sizeof(double), cudaMemcpyDeviceToHost, s));
    CUDA_OK(cudaMemcpyAsync(w, T.w, nw * sizeof(double), cudaMemcpyDeviceToHost, s));
    if (phi) CUDA_OK(cudaMemcpyAsync(phi, T.phi, nc * sizeof(double), cudaMemcpyDeviceToHost, s));
    CUDA_OK(cudaStreamSynchronize(s));
    return rc;
}

extern "C" int maestro_mac_project_host_seq(maestro_mac_handle* H, int nsteps, const double* beta0, const double* rho0,
                                            const double* rho, const double* S, const double* const* u_in,
                                            const double* const* v_in, const double* const* w_in, double* const* u_out,
                                            double* const* v_out, double* const* w_out, double* const* phi_out,
                                            maestro_mac_stats* stats, void* cuda_stream)
{
    if (!H || !H->cp_in || nsteps < 0 || !beta0 || (!rho && !rho0) || !u_in || !v_in || !w_in || !u_out || !v_out || !w_out)
        return MAESTRO_MAC_ERR_ARG;
    for (int k = 0; k < nsteps; ++k)
        if (!u_in[k] || !v_in[k] || !w_in[k] || !u_out[k] || !v_out[k] || !w_out[k] || (phi_out && !phi_out[k])) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const maestro_mac_desc& d = H->d;
    const size_t nc = (size_t)d.nx * d.ny * d.nz;
    const size_t nu = (size_t)(d.nx + 1) * d.ny * d.nz, nv = (size_t)d.nx * (d.ny + 1) * d.nz, nw = (size_t)d.nx * d.ny * (d.nz + 1);
    Staging& T = H->st;
    const int nset = d.host_staging;                // 2 or 3 sets of u, v, w, phi, used round robin
    double* su[3] = {T.u, T.ux[0], T.ux[1]}; double* sv[3] = {T.v, T.vx[0], T.vx[1]};
    double* sw[3] = {T.w, T.wx[0], T.wx[1]}; double* sp[3] = {T.phi, T.phix[0], T.phix[1]};
    // the step-invariant inputs go first on the upload stream; the first velocity upload queues behind them
    CUDA_OK(cudaMemcpyAsync(T.beta0, beta0, d.nr * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
    if (rho0) CUDA_OK(cudaMemcpyAsync(T.rho0, rho0, d.nr * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
    if (rho) CUDA_OK(cudaMemcpyAsync(T.rho, rho, nc * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
    if (S) CUDA_OK(cudaMemcpyAsync(T.S, S, nc * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
    auto upload = [&](int k) -> int {               // velocities of step k into set k % nset, once its last download is done
        const int b = k % nset;
        if (k >= nset) CUDA_OK(cudaStreamWaitEvent(H->cp_in, H->ev_out[b], 0));
        CUDA_OK(cudaMemcpyAsync(su[b], u_in[k], nu * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
        CUDA_OK(cudaMemcpyAsync(sv[b], v_in[k], nv * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
        CUDA_OK(cudaMemcpyAsync(sw[b], w_in[k], nw * sizeof(double), cudaMemcpyHostToDevice, H->cp_in));
        CUDA_OK(cudaEventRecord(H->ev_in[b], H->cp_in));
        return MAESTRO_MAC_OK;
    };
    int rc, worst = MAESTRO_MAC_OK;
    if (nsteps > 0 && (rc = upload(0)) != 0) return rc;
    for (int k = 0; k < nsteps; ++k) {
        const int b = k % nset;
        if (k + 1 < nsteps && (rc = upload(k + 1)) != 0) return rc;      // travels while step k is projected
        CUDA_OK(cudaStreamWaitEvent(s, H->ev_in[b], 0));
        rc = maestro_mac_project(H, T.beta0, rho0 ? T.rho0 : nullptr, rho ? T.rho : nullptr, su[b], sv[b], sw[b],
                                 S ? T.S : nullptr, phi_out ? sp[b] : nullptr, stats ? stats + k : nullptr, cuda_stream);
        if (rc < 0) { worst = rc; break; }
        if (rc == MAESTRO_MAC_NOT_CONVERGED) worst = rc;
        CUDA_OK(cudaEventRecord(H->ev_done[b], s));
        CUDA_OK(cudaStreamWaitEvent(H->cp_out, H->ev_done[b], 0));      // travels while step k+1 is projected
        CUDA_OK(cudaMemcpyAsync(u_out[k], su[b], nu * sizeof(double), cudaMemcpyDeviceToHost, H->cp_out));
        CUDA_OK(cudaMemcpyAsync(v_out[k], sv[b], nv * sizeof(double), cudaMemcpyDeviceToHost, H->cp_out));
        CUDA_OK(cudaMemcpyAsync(w_out[k], sw[b], nw * sizeof(double), cudaMemcpyDeviceToHost, H->cp_out));
        if (phi_out) CUDA_OK(cudaMemcpyAsync(phi_out[k], sp[b], nc * sizeof(double), cudaMemcpyDeviceToHost, H->cp_out));
        CUDA_OK(cudaEventRecord(H->ev_out[b], H->cp_out));
    }
    CUDA_OK(cudaStreamSynchronize(H->cp_in));
    CUDA_OK(cudaStreamSynchronize(H->cp_out));
    CUDA_OK(cudaStreamSynchronize(s));
    return worst;
}

// ---- base state ---------------------------------------------------

extern "C" int maestro_mac_base_state(int nr, const double* rho0, const double* p0, const double* gamma1bar,
                                      const double* dp0dt, double* beta0, double* dpdt_term, void* cuda_stream)
{
    if (nr <= 0 || !rho0 || !p0 || !gamma1bar || !beta0 || (dpdt_term && !dp0dt)) return MAESTRO_MAC_ERR_ARG;
    k_base_state<<<1, 32, 0, (cudaStream_t)cuda_stream>>>(nr, rho0, p0, gamma1bar, dp0dt, beta0, dpdt_term);
    return cudaPeekAtLastError() == cudaSuccess ? MAESTRO_MAC_OK : MAESTRO_MAC_ERR_CUDA;
}

extern "C" int maestro_mac_lateral_average(maestro_mac_handle* H, const double* rho, double* rho0, void* cuda_stream)
{
    if (!H || !rho || !rho0) return MAESTRO_MAC_ERR_ARG;
    if (H->d.nr > kMaxParts || !H->lat_part) return MAESTRO_MAC_ERR_UNSUPPORTED;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    unsigned long long* cnt = reinterpret_cast<unsigned long long*>(H->part_max);
    const int nr = H->d.nr, rows = H->d.ny * H->d.nz;
    // as many warps per block as private bin sets fit in shared memory; blocks: one per SM, capped by the scratch
    int nwarp = (int)(kLateralSmem / ((size_t)nr * 12));
    if (nwarp < 1) return MAESTRO_MAC_ERR_UNSUPPORTED;
    if (nwarp > 8) nwarp = 8;
    int nb = H->sms < kLateralBlocks ? H->sms : kLateralBlocks;
    if (nb > rows) nb = rows;
    double* psum = H->lat_part;
    unsigned* pcnt = reinterpret_cast<unsigned*>(H->lat_part + (size_t)kLateralBlocks * nr);
    k_lateral_sum<<<nb, 32 * nwarp, (size_t)nwarp * nr * 12, s>>>(dev_geo(H), rho, psum, pcnt);
    LAUNCHED(H);
    k_average_finish<<<1, 256, 0, s>>>(nr, nb, psum, pcnt, cnt, rho0);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_set_dpdt_term(maestro_mac_handle* H, const double* dpdt_term)
{
    if (!H) return MAESTRO_MAC_ERR_ARG;
    H->dpdt_term = dpdt_term;
    return MAESTRO_MAC_OK;
}

// ---- step API ----------------------------------------------------------------------------------

extern "C" int maestro_mac_num_levels(const maestro_mac_handle* H) { return H ? H->nlev : MAESTRO_MAC_ERR_ARG; }

extern "C" int maestro_mac_level_dims(const maestro_mac_handle* H, int level, int n[3], double hh[3])
{
    if (!H || level < 0 || level >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    for (int a = 0; a < 3; ++a) {
        if (n) n[a] = H->lev[level].n[a];
        if (hh) hh[a] = H->lev[level].h[a];
    }
    return MAESTRO_MAC_OK;
}

static int level_copy(maestro_mac_handle* H, int level, int which, double* pub, int to_public, cudaStream_t s)
{
    if (!H || !pub || level < 0 || level >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    Level& L = H->lev[level];
    double* internal = nullptr;
    int e[3] = {L.n[0], L.n[1], L.n[2]}, kind = 0, ghosts = 0;
    switch (which) {
        case MAESTRO_MAC_ARR_PHI: internal = L.phi; ghosts = GH_PHI; break;
        case MAESTRO_MAC_ARR_RHS: internal = L.rhs; ghosts = GH_RHS; break;
        case MAESTRO_MAC_ARR_BX: internal = L.ax; kind = 2; ++e[0]; ghosts = GH_AX; break;
        case MAESTRO_MAC_ARR_BY: internal = L.ay; kind = 3; ++e[1]; ghosts = GH_AY; break;
        case MAESTRO_MAC_ARR_BZ: internal = L.az; kind = 4; ++e[2]; ghosts = GH_AZ; break;
        default: return MAESTRO_MAC_ERR_ARG;
    }
    dim3 g, b;
    dims3(e[0], e[1], e[2], &g, &b);
    k_copy_level<<<g, b, 0, s>>>(dev_level(H, level), internal, pub, kind, e[0], e[1], e[2], to_public);
    LAUNCHED(H);
    return to_public ? MAESTRO_MAC_OK : do_fill_ghosts(H, level, ghosts, s);
}

extern "C" int maestro_mac_level_get(maestro_mac_handle* H, int level, int which, double* dst, void* cuda_stream)
{
    return level_copy(H, level, which, dst, 1, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_level_set(maestro_mac_handle* H, int level, int which, const double* src, void* cuda_stream)
{
    return level_copy(H, level, which, const_cast<double*>(src), 0, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_coefficients(maestro_mac_handle* H, const double* beta0, const double* rho0,
                                             const double* rho, void* cuda_stream)
{
    if (!H || !beta0 || (!rho && !rho0)) return MAESTRO_MAC_ERR_ARG;
    return do_coefficients(H, beta0, rho0, rho, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_rhs(maestro_mac_handle* H, const double* beta0, const double* u, const double* v,
                                    const double* w, const double* S, double* rhs_norm_inf, double* mean_removed,
                                    void* cuda_stream)
{
    if (!H || !beta0 || !u || !v || !w) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int rc = do_rhs(H, beta0, u, v, w, S, s);
    if (rc != 0) return rc;
    if (publish_scal(H, 0, 3, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    CUDA_OK(cudaStreamSynchronize(s));
    if (rhs_norm_inf) *rhs_norm_inf = H->host_scal[1];
    if (mean_removed) *mean_removed = H->singular ? H->host_scal[2] / (double)H->lev[0].ncell : 0.0;
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_step_smooth(maestro_mac_handle* H, int level, int nsweeps, void* cuda_stream)
{
    if (!H || level < 0 || level >= H->nlev || nsweeps < 0) return MAESTRO_MAC_ERR_ARG;
    for (int a = 0; a < 3; ++a)   // red-black needs even periodic extents (always true above the bottom)
        if (H->d.bc_lo[a] == MAESTRO_MAC_PERIODIC && (H->lev[level].n[a] & 1)) return MAESTRO_MAC_ERR_UNSUPPORTED;
    return do_smooth(H, level, nsweeps, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_residual_restrict(maestro_mac_handle* H, int level, void* cuda_stream)
{
    if (!H || level < 0 || level + 1 >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    return do_residual_restrict(H, level, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_prolong(maestro_mac_handle* H, int level, void* cuda_stream)
{
    if (!H || level < 0 || level + 1 >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    return do_prolong(H, level, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_bottom(maestro_mac_handle* H, void* cuda_stream)
{
    if (!H) return MAESTRO_MAC_ERR_ARG;
    return do_bottom(H, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_vcycle(maestro_mac_handle* H, void* cuda_stream)
{
    if (!H) return MAESTRO_MAC_ERR_ARG;
    return do_vcycle(H, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_step_residual_norm(maestro_mac_handle* H, int level, double* norm_inf, void* cuda_stream)
{
    if (!H || level < 0 || level >= H->nlev || !norm_inf) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    int rc = do_residual_norm(H, level, s);
    if (rc != 0) return rc;
    if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    CUDA_OK(cudaStreamSynchronize(s));
    *norm_inf = H->host_scal[4];
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_step_correct(maestro_mac_handle* H, const double* rho0, const double* rho, double* u,
                                        double* v, double* w, void* cuda_stream)
{
    if (!H || !u || !v || !w || (!rho && !rho0)) return MAESTRO_MAC_ERR_ARG;
    return do_correct(H, H->lev[0].phi, rho0, rho, u, v, w, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_level_plan(const maestro_mac_handle* H, int level, int info[8])
{
    if (!H || !info || level < 0 || level >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    const Level& L = H->lev[level];
    const LevelDev D = dev_level(H, level);
    for (int q = 0; q < 8; ++q) info[q] = 0;
    info[6] = L.gx; info[7] = L.gy;
    const int sm = H->d.smoother;
    if (level == H->nlev - 1 && H->nlev > 1 && H->cl_start < 0) { info[0] = MAESTRO_MAC_KERNEL_BOTTOM; return MAESTRO_MAC_OK; }
    if (H->cl_start >= 0 && level >= H->cl_start) { info[0] = MAESTRO_MAC_KERNEL_CLUSTER; return MAESTRO_MAC_OK; }
    if (H->tail_start >= 0 && level >= H->tail_start) { info[0] = MAESTRO_MAC_KERNEL_TAIL; return MAESTRO_MAC_OK; }
    if (t2_ok(H, level)) {
        const t2::T2Plan P = t2_plan(D, H->sms);
        info[0] = MAESTRO_MAC_KERNEL_T2; info[1] = P.tiles; info[2] = P.nfull; info[3] = P.nsplit; info[4] = P.zchunk; info[5] = P.ncta;
        return MAESTRO_MAC_OK;
    }
    const int tv = ((sm == 0 || sm == 4) && D.nx >= 60) ? 0 : (sm == 3 ? 1 : -1);
    if (tv >= 0 && L.tma[tv].ok) {
        int zc = 0;
        const dim3 g = tma_sweep_grid(D, tv, H->sms, &zc);
        info[0] = MAESTRO_MAC_KERNEL_TMA; info[1] = (int)(g.x * g.y); info[3] = (int)g.z; info[4] = zc; info[5] = (int)(g.x * g.y * g.z);
        return MAESTRO_MAC_OK;
    }
    info[0] = (sm != 1 && fused_sweep_supported(D)) ? MAESTRO_MAC_KERNEL_FUSED : MAESTRO_MAC_KERNEL_COLOR;
    return MAESTRO_MAC_OK;
}

#include "maestro_nodal.inl"
#include "maestro_noalloc.inl"
