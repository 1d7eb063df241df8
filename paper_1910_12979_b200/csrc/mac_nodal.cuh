// mac_nodal.cuh -- kernels of the end-of-step (nodal) projection (PAPER.md:63
// "second order projection method ... multigrid linear solvers for the pressure projection steps"; weighting
// beta0/rho of PAPER.md:35 Eq. 2, constraint of PAPER.md:49 Eq. 6).  Readings N1..N10 of DESIGN.md.
//
// phi lives on the nodes, sigma = beta0/rho on the cells; the velocities, rho and S are cell arrays in the public cell
// layout (idx = i + nx (j + ny k)).  Operator: the trilinear (Q1) finite-element form of div(sigma grad phi) divided by
// the cell volume,
//     (L phi)_a = -sum_c sigma_c sum_b (K^c_ab / V) phi_b
// over the up to 8 cells c around node a and their 8 corners b.  K^c_ab / V depends only on whether b is the same
// corner as a or the other one along each axis (8 classes): w[cls] = sum_d g_d k_d prod_{e != d} m_e, g_d = 1/h_d^2,
// k = +1 same / -1 other, m = 1/3 same / 1/6 other.  A neighbour node b at offset (dx, dy, dz) in {-1,0,1}^3 therefore
// enters with  -w[cls(dx,dy,dz)] * T(dx,dy,dz),  T = the sum of sigma over the cells that contain both a and b.
//
// Internal layout of a level (x fastest; pointers address the interior origin, index 0):
//   node arrays phi, phi2, rhs : idx = i + NX (j + NY k),  NX = nx + 4, NY = ny + 3, i in [-1, nx + 1]  (one ghost node per side)
//   sigma (cells)              : idx = i + CX (j + CY k),  CX = nx + 4, CY = ny + 2, i in [-1, nx]      (one ghost cell per side)
//   Rows start TWO entries before index 0 (one unused pad entry, then the ghost) and the row pitches are even: TMA wants
//   16-byte multiples for the pitch AND for the first entry of a box, and the boxes of k_nod_march start at the even
//   entries x0 - 2 (phi, sigma) and x0 (rhs) of a row.
// Node rules (N4) expressed in that layout, so that the operator needs no boundary branches:
//   * a cell outside a non-periodic boundary has sigma = 0 (its ghost entry): the terms of cells that do not exist vanish
//     whatever (finite) value the ghost nodes hold; on periodic axes ghost cells and ghost nodes hold periodic images;
//   * OUTFLOW nodes hold 0 and are not unknowns; on a periodic axis node n is the image of node 0 and not an unknown.
// The z-marching operator pass (k_nod_march) relies on the ghosts of its input: every kernel whose phi output a later
// pass reads writes the images as well (Jacobi output, prolongation), level_set fills them (k_nod_phi_ghosts).
// Everything else reads through the rules (nod_val, nod_operator_generic) and ignores the ghosts.
// Smoother: Jacobi (order-free: reproducible; one HBM pass per sweep, 32 B per node: sigma, phi, rhs in, phi out),
// ping-pong between phi and phi2; the sweep can emit max |rhs - L phi_in|, so the stop test of a cycle rides on the first
// pre-smoothing sweep of the next one at no extra pass.
#pragma once
#include "mac_kernels.cuh"
#include "mac_setup.cuh"
#include "mac_smoother_tma.cuh"

struct NodLevel {
    int nx, ny, nz;                 // cells
    int NX, NY, CX, CY;             // pitches: nodes per row / rows per plane, cells per row / rows per plane (ghosts and
                                    // one pad entry: row pitches are even, i.e. multiples of 16 bytes, as TMA wants)
    int bclo[3], bchi[3];
    double w[8];                    // class weights; bit 0 / 1 / 2: the other corner along x / y / z
    double omega;                   // Jacobi damping (N7)
    double *phi, *phi2, *rhs;       // node arrays (interior origin)
    double *sigma;                  // cell array (interior origin)
};

__device__ __forceinline__ long long nod_idx(const NodLevel& L, int i, int j, int k)
{
    return (long long)i + (long long)L.NX * ((long long)j + (long long)L.NY * (long long)k);
}
__device__ __forceinline__ long long nod_cidx(const NodLevel& L, int i, int j, int k)
{
    return (long long)i + (long long)L.CX * ((long long)j + (long long)L.CY * (long long)k);
}
__device__ __forceinline__ size_t pub_cidx(const NodLevel& L, int i, int j, int k)      // public cell layout
{
    return (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * (size_t)k);
}

// kind of node index t along axis d (N4): 0 unknown, 1 OUTFLOW node, 2 periodic duplicate
__device__ __forceinline__ int nod_axis_kind(const NodLevel& L, int d, int t)
{
    const int n = d == 0 ? L.nx : (d == 1 ? L.ny : L.nz);
    if (L.bclo[d] == MAC_PERIODIC) return t == n ? 2 : 0;
    if (t == 0 && L.bclo[d] == MAC_OUTFLOW) return 1;
    if (t == n && L.bchi[d] == MAC_OUTFLOW) return 1;
    return 0;
}
__device__ __forceinline__ int nod_kind(const NodLevel& L, int i, int j, int k)
{
    const int a = nod_axis_kind(L, 0, i), b = nod_axis_kind(L, 1, j), c = nod_axis_kind(L, 2, k);
    if (a == 1 || b == 1 || c == 1) return 1;
    return (a == 2 || b == 2 || c == 2) ? 2 : 0;
}
// offset (in index units along the axis) of the periodic image of unknown node t that the ghost layout stores: node 0
// is also node n, node 1 also node n + 1, node n - 1 also node -1; 0 = none.  (Levels that are smoothed have n >= 4.)
__device__ __forceinline__ int nod_image(const NodLevel& L, int d, int t)
{
    const int n = d == 0 ? L.nx : (d == 1 ? L.ny : L.nz);
    if (L.bclo[d] != MAC_PERIODIC) return 0;
    return t <= 1 ? n : (t == n - 1 ? -n : 0);
}
// store v at node q of array a and at its periodic images (ix, iy, iz: image offsets along the axes, 0 = none)
__device__ __forceinline__ void nod_store_images(const NodLevel& L, double* __restrict__ a, long long q, double v, int ix,
                                                 int iy, int iz)
{
    a[q] = v;
    if (ix | iy | iz) {
        const long long sy = L.NX, sz = sy * L.NY;
        const long long ox = ix, oy = (long long)iy * sy, oz = (long long)iz * sz;
        if (ix) a[q + ox] = v;
        if (iy) { a[q + oy] = v; if (ix) a[q + ox + oy] = v; }
        if (iz) {
            a[q + oz] = v;
            if (ix) a[q + ox + oz] = v;
            if (iy) { a[q + oy + oz] = v; if (ix) a[q + ox + oy + oz] = v; }
        }
    }
}

// value of a nodal array at node (I, J, K), 0 <= index <= n, under the node rules (OUTFLOW 0, periodic node n = node 0)
__device__ __forceinline__ double nod_val(const NodLevel& L, const double* __restrict__ a, int I, int J, int K)
{
    if (nod_kind(L, I, J, K) == 1) return 0.0;
    if (L.bclo[0] == MAC_PERIODIC && I == L.nx) I = 0;
    if (L.bclo[1] == MAC_PERIODIC && J == L.ny) J = 0;
    if (L.bclo[2] == MAC_PERIODIC && K == L.nz) K = 0;
    return a[nod_idx(L, I, J, K)];
}

// One axis of the 27-point neighbourhood of an unknown node t: stored indices of the nodes t-1, t, t+1 (-2: the value
// counts as 0: no such node, or an OUTFLOW node) and of the cells t-1, t (-2: no such cell).
struct NodAxis { int nd[3]; int cl[2]; };
__device__ __forceinline__ NodAxis nod_axis(const NodLevel& L, int d, int t)
{
    const int n = d == 0 ? L.nx : (d == 1 ? L.ny : L.nz);
    const bool per = L.bclo[d] == MAC_PERIODIC;
    NodAxis A;
    A.nd[1] = t;
    A.nd[0] = t > 0 ? t - 1 : (per ? n - 1 : -2);
    A.nd[2] = t < n ? (t + 1 == n && per ? 0 : t + 1) : -2;
    A.cl[0] = t > 0 ? t - 1 : (per ? n - 1 : -2);
    A.cl[1] = t < n ? t : -2;
    if (!per) {                                       // OUTFLOW nodes count as 0
        if (A.nd[0] == 0 && L.bclo[d] == MAC_OUTFLOW) A.nd[0] = -2;
        if (A.nd[2] == n && L.bchi[d] == MAC_OUTFLOW) A.nd[2] = -2;
    }
    return A;
}

// L phi at the unknown node (i, j, k) through the node rules, one node at a time: the form that does not rely on
// ghost entries (bottom solver).
__device__ __forceinline__ double nod_operator_generic(const NodLevel& L, const double* __restrict__ phi, int i, int j, int k,
                                                      double* tcentre = nullptr)      // tcentre: receives T(0,0,0), the sigma sum of the diagonal
{
    double p[3][3][3], s[2][2][2];
    const NodAxis X = nod_axis(L, 0, i), Y = nod_axis(L, 1, j), Z = nod_axis(L, 2, k);
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const bool ok = X.nd[a] >= 0 && Y.nd[b] >= 0 && Z.nd[c] >= 0;
                p[c][b][a] = ok ? phi[nod_idx(L, X.nd[a], Y.nd[b], Z.nd[c])] : 0.0;
            }
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                const bool ok = X.cl[a] >= 0 && Y.cl[b] >= 0 && Z.cl[c] >= 0;
                s[c][b][a] = ok ? __ldg(L.sigma + nod_cidx(L, X.cl[a], Y.cl[b], Z.cl[c])) : 0.0;
            }
    // T(dx,dy,dz): sigma summed over the cells that contain the node and its neighbour: expand x, then y, then z
    double tx[2][2][3], ty[2][3][3], t[3][3][3];
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b) { tx[c][b][0] = s[c][b][0]; tx[c][b][1] = s[c][b][0] + s[c][b][1]; tx[c][b][2] = s[c][b][1]; }
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int a = 0; a < 3; ++a) { ty[c][0][a] = tx[c][0][a]; ty[c][1][a] = tx[c][0][a] + tx[c][1][a]; ty[c][2][a] = tx[c][1][a]; }
#pragma unroll
    for (int b = 0; b < 3; ++b)
#pragma unroll
        for (int a = 0; a < 3; ++a) { t[0][b][a] = ty[0][b][a]; t[1][b][a] = ty[0][b][a] + ty[1][b][a]; t[2][b][a] = ty[1][b][a]; }
    double acc[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int b = 0; b < 3; ++b)
#pragma unroll
            for (int a = 0; a < 3; ++a) {
                const int cls = (a != 1 ? 1 : 0) | (b != 1 ? 2 : 0) | (c != 1 ? 4 : 0);
                acc[cls] = fma(t[c][b][a], p[c][b][a], acc[cls]);
            }
    double sum = 0.0;
#pragma unroll
    for (int q = 7; q >= 0; --q) sum = fma(L.w[q], acc[q], sum);
    if (tcentre) *tcentre = t[1][1][1];
    return -sum;
}

// ---- ghosts -----------------------------------------------------------------------------------------------------
// sigma ghost cells: periodic images, 0 outside a non-periodic boundary.  One thread per cell of the extended array.
__global__ void __launch_bounds__(256)
k_nod_sig_ghosts(NodLevel L)
{
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x) - 1, j = (int)(blockIdx.y * blockDim.y + threadIdx.y) - 1,
              k = (int)blockIdx.z - 1;
    if (i > L.nx || j > L.ny) return;
    const bool gi = i < 0 || i >= L.nx, gj = j < 0 || j >= L.ny, gk = k < 0 || k >= L.nz;
    if (!(gi || gj || gk)) return;
    const bool zero = (gi && L.bclo[0] != MAC_PERIODIC) || (gj && L.bclo[1] != MAC_PERIODIC) || (gk && L.bclo[2] != MAC_PERIODIC);
    const int si = gi ? (i < 0 ? i + L.nx : i - L.nx) : i, sj = gj ? (j < 0 ? j + L.ny : j - L.ny) : j,
              sk = gk ? (k < 0 ? k + L.nz : k - L.nz) : k;
    L.sigma[nod_cidx(L, i, j, k)] = zero ? 0.0 : L.sigma[nod_cidx(L, si, sj, sk)];
}

// nodal array a: OUTFLOW nodes := 0, periodic images (nodes -1, n, n+1) := their source, ghosts outside a non-periodic
// boundary := 0.  One thread per node of the extended array.
__global__ void __launch_bounds__(256)
k_nod_phi_ghosts(NodLevel L, double* __restrict__ a)
{
    const int i = (int)(blockIdx.x * blockDim.x + threadIdx.x) - 1, j = (int)(blockIdx.y * blockDim.y + threadIdx.y) - 1,
              k = (int)blockIdx.z - 1;
    if (i > L.nx + 1 || j > L.ny + 1) return;
    int id[3] = {i, j, k};
    bool zero = false, moved = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const int n = d == 0 ? L.nx : (d == 1 ? L.ny : L.nz), t = id[d];
        if (L.bclo[d] == MAC_PERIODIC) {
            if (t < 0) { id[d] = t + n; moved = true; } else if (t >= n) { id[d] = t - n; moved = true; }
        } else if (t < 0 || t > n || nod_axis_kind(L, d, t) == 1) zero = true;
    }
    if (zero) a[nod_idx(L, i, j, k)] = 0.0;
    else if (moved) a[nod_idx(L, i, j, k)] = a[nod_idx(L, id[0], id[1], id[2])];
}

// internal <-> public layout of a level array (step API).  node: (nx+1)(ny+1)(nz+1) values, else cells.  to_public
// with rules applies the node rules to a nodal array (OUTFLOW 0, periodic entry n = entry 0).
__global__ void __launch_bounds__(256)
k_nod_copy(NodLevel L, double* __restrict__ internal, double* __restrict__ pub, int node, int to_public, int rules)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    const int ex = L.nx + node, ey = L.ny + node;
    if (i >= ex || j >= ey) return;
    const size_t p = (size_t)i + (size_t)ex * ((size_t)j + (size_t)ey * (size_t)k);
    const long long q = node ? nod_idx(L, i, j, k) : nod_cidx(L, i, j, k);
    if (to_public) pub[p] = (node && rules) ? nod_val(L, internal, i, j, k) : internal[q];
    else internal[q] = pub[p];
}

// ---- N3: sigma = beta0(r_cell) / rho, beta0 at the cell centres (bcell, public cell layout, scratch for the rhs) ---
__global__ void __launch_bounds__(256)
k_nod_sigma(GeoDev G, NodLevel L, const double* __restrict__ beta0, const double* __restrict__ rho,
            const double* __restrict__ rho0, double* __restrict__ bcell, int* __restrict__ flags)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= G.nx || j >= G.ny) return;
    const size_t c = pub_cidx(L, i, j, k);
    const double r = radius(G, (i + 0.5) * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz);
    const double b = profile_eval(beta0, G.nr, G.dr, r);
    const double rh = rho ? __ldg(rho + c) : profile_eval(rho0, G.nr, G.dr, r);
    if (!(rh > 0.0) || !(rh <= 1.79769313486231570e308)) atomicOr(flags, 1);
    L.sigma[nod_cidx(L, i, j, k)] = b / rh;
    bcell[c] = b;
}

// ---- N6: coarse sigma = mean of the 8 children -----------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_nod_coarsen_sigma(NodLevel F, NodLevel C)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I >= C.nx || J >= C.ny) return;
    double s = 0.0;
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj)
#pragma unroll
            for (int di = 0; di < 2; ++di) s += F.sigma[nod_cidx(F, 2 * I + di, 2 * J + dj, 2 * K + dk)];
    C.sigma[nod_cidx(C, I, J, K)] = 0.125 * s;
}

// ---- N1: rhs = D(beta0 U) - M(beta0 S) at the unknowns, 0 elsewhere; block partials of sum and max|rhs| -------
__global__ void __launch_bounds__(256)
k_nod_rhs(NodLevel L, double i4hx, double i4hy, double i4hz, const double* __restrict__ bcell, const double* __restrict__ u,
          const double* __restrict__ v, const double* __restrict__ w, const double* __restrict__ S,
          double* __restrict__ part_sum, double* __restrict__ part_max, int zper)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    const bool in = i <= L.nx && j <= L.ny;
    double rsum = 0.0, rmax = 0.0;
    for (int k = blockIdx.z * zper; k < min((int)(blockIdx.z + 1) * zper, L.nz + 1); ++k) {
        double r = 0.0;
        if (in && nod_kind(L, i, j, k) == 0) {
            const NodAxis X = nod_axis(L, 0, i), Y = nod_axis(L, 1, j), Z = nod_axis(L, 2, k);
#pragma unroll
            for (int c = 0; c < 2; ++c)
#pragma unroll
                for (int b = 0; b < 2; ++b)
#pragma unroll
                    for (int a = 0; a < 2; ++a) {
                        if (X.cl[a] < 0 || Y.cl[b] < 0 || Z.cl[c] < 0) continue;
                        const size_t q = pub_cidx(L, X.cl[a], Y.cl[b], Z.cl[c]);
                        const double bc = bcell[q];
                        // the node is the HIGH corner of the cell at offset -1 (a == 0): -(2 s - 1) = -1
                        r -= (a == 0 ? 1.0 : -1.0) * (bc * __ldg(u + q)) * i4hx;
                        r -= (b == 0 ? 1.0 : -1.0) * (bc * __ldg(v + q)) * i4hy;
                        r -= (c == 0 ? 1.0 : -1.0) * (bc * __ldg(w + q)) * i4hz;
                        if (S) r -= 0.125 * (bc * __ldg(S + q));
                    }
        }
        if (in) L.rhs[nod_idx(L, i, j, k)] = r;
        rsum += r;
        rmax = nanmax(rmax, fabs(r));
    }
    block_reduce_store(rsum, rmax, part_sum, part_max, blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z));
}

// N5: w_a = (cells around node a) / 8 at the unknowns
__device__ __forceinline__ double nod_weight(const NodLevel& L, int i, int j, int k)
{
    const NodAxis X = nod_axis(L, 0, i), Y = nod_axis(L, 1, j), Z = nod_axis(L, 2, k);
    const int cx = (X.cl[0] >= 0) + (X.cl[1] >= 0), cy = (Y.cl[0] >= 0) + (Y.cl[1] >= 0), cz = (Z.cl[0] >= 0) + (Z.cl[1] >= 0);
    return 0.125 * (double)(cx * cy * cz);
}

// a[node] -= (scal[0] * inv_cells) * (WEIGHTED ? w_a : 1) at the unknowns; block partials of sum (of w_a a_a when
// WSUM) and max |a| afterwards.  scal == NULL: only the reductions.
template <bool WEIGHTED, bool WSUM>
__global__ void __launch_bounds__(256)
k_nod_shift(NodLevel L, double* __restrict__ a, const double* __restrict__ scal, double inv_cells,
            double* __restrict__ part_sum, double* __restrict__ part_max, int zper)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    double s = 0.0, m = 0.0;
    for (int k = blockIdx.z * zper; k < min((int)(blockIdx.z + 1) * zper, L.nz + 1); ++k)
        if (i <= L.nx && j <= L.ny && nod_kind(L, i, j, k) == 0) {
            const long long q = nod_idx(L, i, j, k);
            const double wa = (WEIGHTED || WSUM) ? nod_weight(L, i, j, k) : 1.0;
            double val = a[q];
            if (scal) {
                val -= (scal[0] * inv_cells) * (WEIGHTED ? wa : 1.0);
                a[q] = val;
            }
            s += WSUM ? wa * val : val;
            m = nanmax(m, fabs(val));
        }
    block_reduce_store(s, m, part_sum, part_max, blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z));
}

// ---- N7 / residual: the operator pass, marching in z ------------------------------------------------------------
// MODE bit 0 (NOD_JACOBI): out = pin + omega (rhs - L pin) / L_aa (one Jacobi sweep, pin -> out, distinct buffers; the
// periodic images of out are written too); bit 1 (NOD_RESID): out = rhs - L pin (out may be NULL; no images: the
// restriction reads through the rules); bit 2 (NOD_NORM): block partials of max |rhs - L pin| over the unknowns in
// part_max[linear block index].  OUTFLOW nodes receive 0.
//
// A thread owns a node column (i, j) and marches a chunk of planes.  It keeps the 3 x 3 phi values of planes k-1, k, k+1
// and the expanded sigma sums of the cell planes below and above in registers, so a plane costs 9 phi loads, 4 sigma
// loads, rhs and the store (the lateral neighbours come from L1: a block's tile re-reads a one-node ring), 5 additions
// for the new sigma sums and 54 multiply-adds:
//     L phi = -sum_{dx,dy} [ Tlo (w_o phi_{k-1} + w_s phi_k) + Tup (w_o phi_{k+1} + w_s phi_k) ],
// w_s / w_o = the class weight with the same / the other corner along z.  The ghost layout makes every node interior.
// The march is unrolled six-fold (period 3 of the phi planes x period 2 of the sigma planes) so that nothing moves
// between registers.
enum { NOD_JACOBI = 1, NOD_RESID = 2, NOD_NORM = 4 };

struct NodPlane { double v[3][3]; };               // [dy][dx]

__device__ __forceinline__ void nod_load_phi(NodPlane& P, const double* __restrict__ q, long long py)
{
#pragma unroll
    for (int b = 0; b < 3; ++b)
#pragma unroll
        for (int a = 0; a < 3; ++a) P.v[b][a] = q[(a - 1) + (b - 1) * py];
}
// the 2 x 2 sigmas of a cell plane around the node column, expanded to the 3 x 3 sums over the cells shared with each
// lateral neighbour
__device__ __forceinline__ void nod_load_sig(NodPlane& T, const double* __restrict__ sg, long long cy)
{
    const double s00 = __ldg(sg), s01 = __ldg(sg + 1), s10 = __ldg(sg + cy), s11 = __ldg(sg + cy + 1);
    T.v[0][0] = s00; T.v[0][1] = s00 + s01; T.v[0][2] = s01;
    T.v[2][0] = s10; T.v[2][1] = s10 + s11; T.v[2][2] = s11;
    T.v[1][0] = s00 + s10; T.v[1][1] = T.v[0][1] + T.v[2][1]; T.v[1][2] = s01 + s11;
}

// Staging: the planes a step consumes (phi plane k+1 of the tile plus a one-node ring, the sigma cell plane k, the
// rhs plane k) are brought into shared memory by TMA box loads (cp.async.bulk.tensor.3d, one elected thread, an
// mbarrier per stage; no per-thread address arithmetic) three steps ahead (ring of four stages, 7.25 KB each), so the
// DRAM latency is off the marching step and the step itself reads shared memory only.  The ghost layout keeps every
// box inside the arrays except beyond the last tile, where the hardware fills zeros that only threads outside the
// grid read.
namespace nodm {
constexpr int TX = 32, TY = 8, NS = 4, LA = 3;
constexpr int BW = TX + 4;                                            // box width of phi / sigma: entries x0-2 .. x0+33 of a row
constexpr int kPhi = 2944, kSig = 2688, kRhs = 2048;                  // bytes per stage (128-byte multiples)
constexpr int kStage = kPhi + kSig + kRhs;
constexpr unsigned kTx = (TY + 2) * BW * 8 + (TY + 1) * BW * 8 + TY * TX * 8;   // bytes landing per stage
static_assert((TY + 2) * BW * 8 <= kPhi && (TY + 1) * BW * 8 <= kSig, "stage layout");
}  // namespace nodm

// Work decomposition of one launch (host: nod_march_plan), as for the two-sweep smoother of the MAC solve: the first
// nfull tiles (whole waves of blocks) march every plane, the remaining tiles are cut into nsplit z-chunks each so that
// the last, partial wave spreads over every SM (257^3 nodes are 297 tiles of 32 x 8 on 296 block slots: uniform
// chunks need 8 rounds of 37 planes, the mixed plan one round of 257 plus one of 16).
struct NodPlan { int tiles_x, tiles, nfull, nsplit, zchunk, ncta; };

template <int MODE>
__global__ void __launch_bounds__(256, 2)
k_nod_march(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_sig,
            const __grid_constant__ CUtensorMap tm_rhs, NodLevel L, const double* __restrict__ pin, double* __restrict__ out,
            double* __restrict__ part_max, NodPlan plan)
{
    using namespace nodm;
    using tma::mbar_init; using tma::mbar_expect_tx; using tma::mbar_wait; using tma::tma_load_3d; using tma::smem_u32;
    __shared__ __align__(128) unsigned char ring[NS * kStage];
    __shared__ __align__(8) unsigned long long bars[NS];
    const int tx = threadIdx.x, ty = threadIdx.y, tid = tx + TX * ty;
    int tile = blockIdx.x, k0 = 0, k1 = L.nz + 1;
    if (tile >= plan.nfull) {
        const int q = tile - plan.nfull, rem = plan.tiles - plan.nfull, c = q / rem;
        tile = plan.nfull + (q - c * rem);
        k0 = c * plan.zchunk;
        k1 = min(k0 + plan.zchunk, L.nz + 1);
    }
    const int tby = tile / plan.tiles_x;
    const int x0 = (tile - tby * plan.tiles_x) * TX, y0 = tby * TY;
    const int i = x0 + tx, j = y0 + ty;
    int kxy = 3;                                                  // lateral kind: 0 unknown, 1 OUTFLOW, 2 duplicate, 3 outside
    if (i <= L.nx && j <= L.ny) {
        const int ka = nod_axis_kind(L, 0, i), kb = nod_axis_kind(L, 1, j);
        kxy = (ka == 1 || kb == 1) ? 1 : ((ka == 2 || kb == 2) ? 2 : 0);
    }
    const int ix = kxy == 0 ? nod_image(L, 0, i) : 0, iy = kxy == 0 ? nod_image(L, 1, j) : 0;
    double rmax = 0.0;
    const long long py = L.NX, pz = py * L.NY, cy = L.CX;
    const unsigned ring0 = smem_u32(ring), bar0 = smem_u32(bars);
    const bool producer = tid == 0;
    // stage of step k: phi plane k+1 (box origin: node (x0-2, y0-1)), cell plane k (cell (x0-2, y0-1)), rhs plane k (node
    // (x0, y0)); tensor-map coordinates count from the allocation origin: entry -2 of a row, row -1, plane -1
    auto issue = [&](int k) {
        if (k < k1) {
            const unsigned s = (unsigned)(k - k0) & (NS - 1), d = ring0 + s * kStage, bar = bar0 + 8 * s;
            mbar_expect_tx(bar, kTx);
            tma_load_3d(d, &tm_phi, bar, x0, y0, k + 2);
            tma_load_3d(d + kPhi, &tm_sig, bar, x0, y0, k + 1);
            tma_load_3d(d + kPhi + kSig, &tm_rhs, bar, x0 + 2, y0 + 1, k + 1);
        }
    };
    static_assert(NS == 4 && LA == 3, "ring arithmetic below");
    if (producer) {
        for (int q = 0; q < NS; ++q) mbar_init(bar0 + 8 * q, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        for (int q = 0; q < LA; ++q) issue(k0 + q);
    }
    // planes k0-1, k0 and the cell plane k0-1 directly (once per chunk)
    const int ic = min(i, L.nx), jc = min(j, L.ny);
    NodPlane P[3], T[2];
    {
        const double* q = pin + nod_idx(L, ic, jc, k0);
        nod_load_phi(P[0], q - pz, py);
        nod_load_phi(P[1], q, py);
        nod_load_sig(T[0], L.sigma + nod_cidx(L, ic - 1, jc - 1, k0 - 1), cy);
    }
    __syncthreads();                                              // barrier inits visible before anyone waits
    long long qo = nod_idx(L, ic, jc, k0);
    const unsigned char* mine = ring + (ty * BW + tx + 1) * 8;    // node (i-1, j-1) of the phi box = cell (i-1, j-1) of the sigma box
    unsigned phase = 0;
#pragma unroll 1
    for (int k = k0; k < k1; k += 6) {
#pragma unroll
        for (int u = 0; u < 6; ++u) {
            if (k + u >= k1) break;
            NodPlane& Pm = P[u % 3];                     // planes k-1, k, k+1 and the cell planes below / above
            NodPlane& Pc = P[(u + 1) % 3];
            NodPlane& Pp = P[(u + 2) % 3];
            NodPlane& Tlo = T[u % 2];
            NodPlane& Tup = T[(u + 1) % 2];
            const unsigned s = (unsigned)(k + u - k0) & (NS - 1);
            mbar_wait(bar0 + 8 * s, (phase >> s) & 1u);  // the stage of this step has landed
            phase ^= 1u << s;
            __syncthreads();                             // every thread has finished step k-1: its stage can be refilled
            if (producer) {
                asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                issue(k + u + LA);
            }
            const double* sphi = reinterpret_cast<const double*>(mine + s * kStage);
            const double* ssig = reinterpret_cast<const double*>(mine + s * kStage + kPhi);
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) Pp.v[b][a] = sphi[b * BW + a];
            {
                const double s00 = ssig[0], s01 = ssig[1], s10 = ssig[BW], s11 = ssig[BW + 1];
                Tup.v[0][0] = s00; Tup.v[0][1] = s00 + s01; Tup.v[0][2] = s01;
                Tup.v[2][0] = s10; Tup.v[2][1] = s10 + s11; Tup.v[2][2] = s11;
                Tup.v[1][0] = s00 + s10; Tup.v[1][1] = Tup.v[0][1] + Tup.v[2][1]; Tup.v[1][2] = s01 + s11;
            }
            const double rh = *reinterpret_cast<const double*>(ring + s * kStage + kPhi + kSig + tid * 8);
            double acc0 = 0.0, acc1 = 0.0;
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    const int cl = (a != 1 ? 1 : 0) | (b != 1 ? 2 : 0);
                    const double sc = L.w[cl] * Pc.v[b][a];
                    acc0 = fma(Tlo.v[b][a], fma(L.w[4 + cl], Pm.v[b][a], sc), acc0);
                    acc1 = fma(Tup.v[b][a], fma(L.w[4 + cl], Pp.v[b][a], sc), acc1);
                }
            const int kz = nod_axis_kind(L, 2, k + u);
            if (kxy == 0 && kz == 0) {
                const double r = rh + (acc0 + acc1);                          // rhs - L phi, L phi = -(acc0 + acc1)
                if (MODE & NOD_NORM) rmax = nanmax(rmax, fabs(r));
                if (MODE & NOD_JACOBI) {
                    const double ndg = L.w[0] * (Tlo.v[1][1] + Tup.v[1][1]);  // -L_aa > 0
                    nod_store_images(L, out, qo, Pc.v[1][1] - fast_div_pos(L.omega * r, ndg), ix, iy, nod_image(L, 2, k + u));
                } else if (out) out[qo] = r;
            } else if (kxy <= 1 && (kxy == 1 || kz == 1) && out) {
                out[qo] = 0.0;                                                // OUTFLOW node
            }
            qo += pz;
        }
    }
    if (MODE & NOD_NORM) {
        __shared__ double sh[8];
        rmax = warp_nanmax(rmax);
        if ((tid & 31) == 0) sh[tid >> 5] = rmax;
        __syncthreads();
        if (tid == 0) {
            double m = sh[0];
            for (int qq = 1; qq < 8; ++qq) m = nanmax(m, sh[qq]);
            part_max[blockIdx.x] = m;
        }
    }
}

// ---- the same passes with one thread per node, for the levels that are too small for the z-march (its pipeline
// prologue and a serial march over a handful of blocks cost 12 us on a 17^3 level; this form is launch-bound).
// Interior nodes (indices in [1, n - 1] on every axis) read their 27 neighbours and 8 cells at constant offsets; the
// others go through nod_operator_generic (node rules).  L phi = -sum_class w[class] sum_{n in class} T_n phi_n.
// grid over (nx + 1, ny + 1, nz + 1) nodes; NORM: one partial maximum per block (linear block index).
template <int MODE>
__global__ void __launch_bounds__(256)
k_nod_point(NodLevel L, const double* __restrict__ pin, double* __restrict__ out, double* __restrict__ part_sum,
            double* __restrict__ part_max)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    double rabs = 0.0;
    if (i <= L.nx && j <= L.ny) {
        const int kind = nod_kind(L, i, j, k);
        const long long q = nod_idx(L, i, j, k);
        if (kind == 0) {
            double lphi, ndg;
            if (i >= 1 && i < L.nx && j >= 1 && j < L.ny && k >= 1 && k < L.nz) {
                const double* __restrict__ p = pin + q;
                const double* __restrict__ sg = L.sigma + nod_cidx(L, i - 1, j - 1, k - 1);
                const long long py = L.NX, pz = py * L.NY, cy = L.CX, cz = cy * L.CY;
                double s8[2][2][2];
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int b = 0; b < 2; ++b) { s8[c][b][0] = __ldg(sg + b * cy + c * cz); s8[c][b][1] = __ldg(sg + 1 + b * cy + c * cz); }
                double tx[2][2][3], ty[2][3][3], t[3][3][3];
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int b = 0; b < 2; ++b) { tx[c][b][0] = s8[c][b][0]; tx[c][b][1] = s8[c][b][0] + s8[c][b][1]; tx[c][b][2] = s8[c][b][1]; }
#pragma unroll
                for (int c = 0; c < 2; ++c)
#pragma unroll
                    for (int a = 0; a < 3; ++a) { ty[c][0][a] = tx[c][0][a]; ty[c][1][a] = tx[c][0][a] + tx[c][1][a]; ty[c][2][a] = tx[c][1][a]; }
#pragma unroll
                for (int b = 0; b < 3; ++b)
#pragma unroll
                    for (int a = 0; a < 3; ++a) { t[0][b][a] = ty[0][b][a]; t[1][b][a] = ty[0][b][a] + ty[1][b][a]; t[2][b][a] = ty[1][b][a]; }
                double acc[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int c = 0; c < 3; ++c)
#pragma unroll
                    for (int b = 0; b < 3; ++b)
#pragma unroll
                        for (int a = 0; a < 3; ++a) {
                            const int cls = (a != 1 ? 1 : 0) | (b != 1 ? 2 : 0) | (c != 1 ? 4 : 0);
                            acc[cls] = fma(t[c][b][a], p[(a - 1) + (b - 1) * py + (c - 1) * pz], acc[cls]);
                        }
                double sum = 0.0;
#pragma unroll
                for (int w = 7; w >= 0; --w) sum = fma(L.w[w], acc[w], sum);
                lphi = -sum;
                ndg = L.w[0] * t[1][1][1];
            } else {
                double tc;
                lphi = nod_operator_generic(L, pin, i, j, k, &tc);
                ndg = L.w[0] * tc;
            }
            const double r = L.rhs[q] - lphi;
            if (MODE & NOD_NORM) rabs = fabs(r);
            if (MODE & NOD_JACOBI)
                nod_store_images(L, out, q, pin[q] - fast_div_pos(L.omega * r, ndg), nod_image(L, 0, i), nod_image(L, 1, j), nod_image(L, 2, k));
            else if (out) out[q] = r;
        } else if (kind == 1 && out) {
            out[q] = 0.0;                                                     // OUTFLOW node
        }
    }
    if (MODE & NOD_NORM) block_reduce_store(0.0, rabs, part_sum, part_max, blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z));
}

// ---- N6: coarse rhs = (1/8) P^T res (weights 1, 1/2 per axis over the 27 fine nodes); the coarse phi is zeroed by
// the host (whole array, ghosts included) -----------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_nod_restrict(NodLevel F, NodLevel C, const double* __restrict__ res)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I > C.nx || J > C.ny) return;
    double s = 0.0;
    if (I >= 1 && I < C.nx && J >= 1 && J < C.ny && K >= 1 && K < C.nz) {
        // interior coarse node (an unknown whatever the boundary types): its 27 fine nodes 2T - 1 .. 2T + 1 exist and need
        // no wrap -- constant offsets from one base pointer, the same terms in the same order as the general path below
        const double* __restrict__ p = res + nod_idx(F, 2 * I, 2 * J, 2 * K);
        const long long sy = F.NX, sz = sy * F.NY;
#pragma unroll
        for (int c = -1; c <= 1; ++c)
#pragma unroll
            for (int b = -1; b <= 1; ++b) {
                const double* __restrict__ r = p + b * sy + c * sz;
                const double wr = (b != 0 ? 0.5 : 1.0) * (c != 0 ? 0.5 : 1.0);
                s += (0.5 * wr) * r[-1];
                s += wr * r[0];
                s += (0.5 * wr) * r[1];
            }
        s *= 0.125;
    } else if (nod_kind(C, I, J, K) == 0) {
        int fi[3], fj[3], fk[3];
#pragma unroll
        for (int o = 0; o < 3; ++o) {                 // fine node 2 T + (o - 1) per axis, wrapped, or -2
            int t = 2 * I + o - 1;
            if (F.bclo[0] == MAC_PERIODIC) { if (t < 0) t += F.nx; if (t >= F.nx) t -= F.nx; } else if (t < 0 || t > F.nx) t = -2;
            fi[o] = t;
            t = 2 * J + o - 1;
            if (F.bclo[1] == MAC_PERIODIC) { if (t < 0) t += F.ny; if (t >= F.ny) t -= F.ny; } else if (t < 0 || t > F.ny) t = -2;
            fj[o] = t;
            t = 2 * K + o - 1;
            if (F.bclo[2] == MAC_PERIODIC) { if (t < 0) t += F.nz; if (t >= F.nz) t -= F.nz; } else if (t < 0 || t > F.nz) t = -2;
            fk[o] = t;
        }
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    if (fi[a] < 0 || fj[b] < 0 || fk[c] < 0) continue;
                    const double wt = (a != 1 ? 0.5 : 1.0) * (b != 1 ? 0.5 : 1.0) * (c != 1 ? 0.5 : 1.0);
                    s += wt * res[nod_idx(F, fi[a], fj[b], fk[c])];      // (0 at OUTFLOW nodes: they carry no residual)
                }
        s *= 0.125;
    }
    C.rhs[nod_idx(C, I, J, K)] = s;
}

// ---- N6: phi_f += P e_c at the fine unknowns (trilinear: weights 1, 1/2, 1/4, 1/8), images included --------------
// One thread per COARSE node (I, J, K) adds the interpolant to the up to 8 fine nodes
// (2I + a, 2J + b, 2K + c), a, b, c in {0, 1}: 8 coarse values (through the node rules) are shared by the 8 fine nodes,
// the fine values move as 16-byte x pairs.  Per fine node: wt * (sum of the coarse corners it lies between).
__global__ void __launch_bounds__(256)
k_nod_prolong_add2(NodLevel F, NodLevel C)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I > C.nx || J > C.ny) return;
    double e[2][2][2];
    // interior: the 8 coarse corners have indices in [1, n - 1] (unknowns, no wrap) and the 8 fine nodes indices in
    // [2, 2n - 3] (unknowns without periodic images): plain loads and stores, the same sums as the general path
    const bool fast = I >= 1 && I + 1 < C.nx && J >= 1 && J + 1 < C.ny && K >= 1 && K + 1 < C.nz;
    if (fast) {
        const double* __restrict__ ce = C.phi + nod_idx(C, I, J, K);
        const long long sy = C.NX, sz = sy * C.NY;
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int b = 0; b < 2; ++b) { e[c][b][0] = ce[b * sy + c * sz]; e[c][b][1] = ce[1 + b * sy + c * sz]; }
        double2* const fp = reinterpret_cast<double2*>(F.phi + nod_idx(F, 2 * I, 2 * J, 2 * K));   // node 2I sits at an even entry of its row
        const long long fy = F.NX / 2, fz = fy * F.NY;
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int b = 0; b < 2; ++b) {
                double s0 = 0.0, s1 = 0.0;
                for (int cc = 0; cc <= c; ++cc)
                    for (int bb = 0; bb <= b; ++bb) {
                        s0 += e[cc][bb][0];
                        s1 += e[cc][bb][0];
                        s1 += e[cc][bb][1];
                    }
                const double wt = (b ? 0.5 : 1.0) * (c ? 0.5 : 1.0);
                double2 v = fp[b * fy + c * fz];
                v.x += wt * s0;
                v.y += (0.5 * wt) * s1;
                fp[b * fy + c * fz] = v;
            }
        return;
    }
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int a = 0; a < 2; ++a)
                e[c][b][a] = (I + a <= C.nx && J + b <= C.ny && K + c <= C.nz) ? nod_val(C, C.phi, I + a, J + b, K + c) : 0.0;
    const int i = 2 * I, j = 2 * J, k = 2 * K;
    const bool x1 = i + 1 <= F.nx;
#pragma unroll
    for (int c = 0; c < 2; ++c) {
        if (k + c > F.nz) continue;
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            if (j + b > F.ny) continue;
            const long long q = nod_idx(F, i, j + b, k + c);
            // fine node (i + a, j + b, k + c): weight 1/2 per odd axis, corners (0..a, 0..b, 0..c)
            double s0 = 0.0, s1 = 0.0;
            for (int cc = 0; cc <= c; ++cc)
                for (int bb = 0; bb <= b; ++bb) {
                    s0 += e[cc][bb][0];
                    s1 += e[cc][bb][0];
                    s1 += e[cc][bb][1];
                }
            const double wt = (b ? 0.5 : 1.0) * (c ? 0.5 : 1.0);
            const int iy = nod_image(F, 1, j + b), iz = nod_image(F, 2, k + c);
            const int k0 = nod_kind(F, i, j + b, k + c), k1 = x1 ? nod_kind(F, i + 1, j + b, k + c) : 3;
            if (k0 == 0 && k1 == 0 && !(iy | iz) && nod_image(F, 0, i) == 0 && nod_image(F, 0, i + 1) == 0) {
                double2* p2 = reinterpret_cast<double2*>(F.phi + q);          // node 2I sits at an even entry of its row
                double2 v = *p2;
                v.x += wt * s0;
                v.y += (0.5 * wt) * s1;
                *p2 = v;
            } else {
                if (k0 == 0) nod_store_images(F, F.phi, q, F.phi[q] + wt * s0, nod_image(F, 0, i), iy, iz);
                if (k1 == 0) nod_store_images(F, F.phi, q + 1, F.phi[q + 1] + (0.5 * wt) * s1, nod_image(F, 0, i + 1), iy, iz);
            }
        }
    }
}

// ---- N10: U <- U - (1/rho) G phi, G the cell-mean gradient (mean of the 4 edge differences per axis) -----------
__global__ void __launch_bounds__(256)
k_nod_correct(NodLevel L, GeoDev G, double i4hx, double i4hy, double i4hz, const double* __restrict__ phi,
              const double* __restrict__ rho, const double* __restrict__ rho0, double* __restrict__ u,
              double* __restrict__ v, double* __restrict__ w)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= L.nx || j >= L.ny) return;
    double p[2][2][2];
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int a = 0; a < 2; ++a) p[c][b][a] = nod_val(L, phi, i + a, j + b, k + c);
    double gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
    for (int c = 0; c < 2; ++c)
#pragma unroll
        for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int a = 0; a < 2; ++a) {
                gx += (a ? 1.0 : -1.0) * p[c][b][a] * i4hx;
                gy += (b ? 1.0 : -1.0) * p[c][b][a] * i4hy;
                gz += (c ? 1.0 : -1.0) * p[c][b][a] * i4hz;
            }
    const size_t q = pub_cidx(L, i, j, k);
    const double rh = rho ? __ldg(rho + q) : profile_eval(rho0, G.nr, G.dr, radius(G, (i + 0.5) * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz));
    u[q] -= gx / rh;
    v[q] -= gy / rh;
    w[q] -= gz / rh;
}

// ---- N8: bottom solve, unpreconditioned BiCGStab on the unknowns of the coarsest level (one thread block).  The
// iterate x is the level's phi; the six work vectors are arrays in the same internal layout (interior origins vec0 +
// m * vstride), global memory -- the level is tiny and L1/L2-resident; entries of OUTFLOW nodes and periodic
// duplicates stay 0.  Same algorithm and stopping rule as the MAC bottom solver (reading A15).
struct NodBottomIdx { int i, j, k; long long q; bool active; };
__device__ __forceinline__ NodBottomIdx nod_bottom_idx(const NodLevel& L, int c)
{
    NodBottomIdx B;
    const int px = L.nx + 1, py = L.ny + 1;
    B.i = c % px; B.j = (c / px) % py; B.k = c / (px * py);
    B.q = nod_idx(L, B.i, B.j, B.k);
    B.active = nod_kind(L, B.i, B.j, B.k) == 0;
    return B;
}

// The usual bottom (5^3 = 125 nodes): ONE node per thread.  The thread keeps its row of the operator in registers -- the
// 27 products -w[class] T(dx,dy,dz) and the storage indices of the 27 neighbours (coefficient 0 and its own index where
// there is no such node or it is an OUTFLOW node) -- and every vector entry as a scalar; a matrix-vector product is 27
// shared-memory reads of the operand, not the index arithmetic and sigma loads of nod_operator_generic.  Same
// algorithm, stopping rule and exits as k_nod_bottom.  Needs nb <= 128 and a node layout of at most kNodSmallMax entries.
constexpr int kNodSmallMax = 1024;

__global__ void __launch_bounds__(128)
k_nod_bottom_small(NodLevel L, int maxit, double tol, int singular, int* __restrict__ iters_accum)
{
    __shared__ double sh[64];
    __shared__ double opd[kNodSmallMax];               // the operand of a product, in the level's node layout
    const int nb = (L.nx + 1) * (L.ny + 1) * (L.nz + 1), nt = blockDim.x, tid = threadIdx.x;
    const bool has = tid < nb;
    const NodBottomIdx B = nod_bottom_idx(L, has ? tid : 0);
    const bool active = has && B.active;
    const int q = (int)B.q;
    double cf[27];
    int ix[27];
#pragma unroll
    for (int n = 0; n < 27; ++n) { cf[n] = 0.0; ix[n] = q; }
    if (active) {
        const NodAxis X = nod_axis(L, 0, B.i), Y = nod_axis(L, 1, B.j), Z = nod_axis(L, 2, B.k);
        double sg[2][2][2];
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int a = 0; a < 2; ++a) {
                    const bool ok = X.cl[a] >= 0 && Y.cl[b] >= 0 && Z.cl[c] >= 0;
                    sg[c][b][a] = ok ? __ldg(L.sigma + nod_cidx(L, X.cl[a], Y.cl[b], Z.cl[c])) : 0.0;
                }
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) {
                    // T: sigma summed over the cells that contain the node and this neighbour (offset 0: both cells of the axis)
                    double t = 0.0;
#pragma unroll
                    for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                        for (int bb = 0; bb < 2; ++bb)
#pragma unroll
                            for (int aa = 0; aa < 2; ++aa) {
                                const bool in = (a == 1 || aa == (a >> 1)) && (b == 1 || bb == (b >> 1)) && (c == 1 || cc == (c >> 1));
                                if (in) t += sg[cc][bb][aa];
                            }
                    const int cls = (a != 1 ? 1 : 0) | (b != 1 ? 2 : 0) | (c != 1 ? 4 : 0);
                    const bool ok = X.nd[a] >= 0 && Y.nd[b] >= 0 && Z.nd[c] >= 0;
                    const int n = a + 3 * (b + 3 * c);
                    if (ok) { cf[n] = -L.w[cls] * t; ix[n] = (int)nod_idx(L, X.nd[a], Y.nd[b], Z.nd[c]); }
                }
    }
    auto matvec = [&](double y) -> double {            // (the operand entries of OUTFLOW nodes and duplicates are 0 by construction)
        group_sync(nt);
        if (has) opd[q] = y;
        group_sync(nt);
        double acc = 0.0;
#pragma unroll
        for (int n = 0; n < 27; ++n) acc = fma(cf[n], opd[ix[n]], acc);
        return active ? acc : 0.0;
    };
    const double f = active ? L.rhs[q] : 0.0;
    const Dot2 q0 = block_dot2(active ? 1.0 : 0.0, f, sh, nt);
    const double nunk = q0.a, fm = singular ? q0.b / q0.a : 0.0;
    double x = 0.0, r = active ? f - fm : 0.0, rhat = r, pv = 0.0, v = 0.0, sv = 0.0, tv = 0.0;
    double rr = block_dot2(r * r, 0.0, sh, nt).a;
    const double bnorm2 = rr;
    int it = 0;
    if (bnorm2 > 0.0 && bnorm2 == bnorm2) {
        const double stop2 = tol * tol * bnorm2;
        double rho = rr, rho_old = 1.0, alpha = 1.0, omega = 1.0;
        while (it < maxit && rr > stop2) {
            if (rho == 0.0) break;
            const double beta = it == 0 ? 0.0 : (rho / rho_old) * (alpha / omega);
            pv = r + beta * (pv - omega * v);
            v = matvec(pv);
            const double d = block_dot2(rhat * v, 0.0, sh, nt).a;
            if (d == 0.0) break;
            alpha = rho / d;
            sv = r - alpha * v;
            const double ss = block_dot2(sv * sv, 0.0, sh, nt).a;
            ++it;
            if (ss <= stop2) { x += alpha * pv; rr = ss; break; }
            tv = matvec(sv);
            Dot2 qd = block_dot2(tv * sv, tv * tv, sh, nt);
            if (qd.b == 0.0) { x += alpha * pv; break; }
            omega = qd.a / qd.b;
            x += alpha * pv + omega * sv;
            r = sv - omega * tv;
            qd = block_dot2(r * r, rhat * r, sh, nt);
            rr = qd.a;
            rho_old = rho;
            rho = qd.b;
            if (omega == 0.0) break;
        }
    }
    if (singular) {                                    // zero plain mean over the unknowns (N8)
        const double xm = block_dot2(active ? x : 0.0, 0.0, sh, nt).a / nunk;
        if (active) x -= xm;
    }
    if (has) L.phi[q] = active ? x : 0.0;
    if (tid == 0 && iters_accum) *iters_accum += it;
}

__global__ void __launch_bounds__(1024)
k_nod_bottom(NodLevel L, double* __restrict__ vec0, long long vstride, int maxit, double tol, int singular,
             int* __restrict__ iters_accum)
{
    __shared__ double sh[64];
    const int nb = (L.nx + 1) * (L.ny + 1) * (L.nz + 1), nt = blockDim.x, tid = threadIdx.x;
    double *x = L.phi, *r = vec0, *rhat = vec0 + vstride, *p = vec0 + 2 * vstride, *v = vec0 + 3 * vstride,
           *s = vec0 + 4 * vstride, *t = vec0 + 5 * vstride;
    const double* f = L.rhs;
#define NOD_FOR_NODES for (int c = tid; c < nb; c += nt)
    double cnt = 0.0, fs = 0.0;
    NOD_FOR_NODES {
        const NodBottomIdx B = nod_bottom_idx(L, c);
        if (B.active) { cnt += 1.0; fs += f[B.q]; }
    }
    const Dot2 q0 = block_dot2(cnt, fs, sh, nt);
    const double nunk = q0.a, fm = singular ? q0.b / q0.a : 0.0;
    double rr = 0.0;
    NOD_FOR_NODES {
        const NodBottomIdx B = nod_bottom_idx(L, c);
        const double fv = B.active ? f[B.q] - fm : 0.0;
        r[B.q] = fv; rhat[B.q] = fv; p[B.q] = 0.0; v[B.q] = 0.0; s[B.q] = 0.0; x[B.q] = 0.0;
        rr += fv * fv;
    }
    rr = block_dot2(rr, 0.0, sh, nt).a;
    const double bnorm2 = rr;
    int it = 0;
    if (bnorm2 > 0.0 && bnorm2 == bnorm2) {
        const double stop2 = tol * tol * bnorm2;
        double rho = rr, rho_old = 1.0, alpha = 1.0, omega = 1.0;
        while (it < maxit && rr > stop2) {
            if (rho == 0.0) break;
            const double beta = it == 0 ? 0.0 : (rho / rho_old) * (alpha / omega);
            NOD_FOR_NODES { const long long q = nod_bottom_idx(L, c).q; p[q] = r[q] + beta * (p[q] - omega * v[q]); }
            group_sync(nt);
            double d = 0.0;
            NOD_FOR_NODES {
                const NodBottomIdx B = nod_bottom_idx(L, c);
                const double y = B.active ? nod_operator_generic(L, p, B.i, B.j, B.k) : 0.0;
                v[B.q] = y;
                d += rhat[B.q] * y;
            }
            d = block_dot2(d, 0.0, sh, nt).a;
            if (d == 0.0) break;
            alpha = rho / d;
            double ss = 0.0;
            NOD_FOR_NODES { const long long q = nod_bottom_idx(L, c).q; const double y = r[q] - alpha * v[q]; s[q] = y; ss += y * y; }
            ss = block_dot2(ss, 0.0, sh, nt).a;
            ++it;
            if (ss <= stop2) {
                NOD_FOR_NODES { const long long q = nod_bottom_idx(L, c).q; x[q] += alpha * p[q]; }
                rr = ss;
                break;
            }
            double ts = 0.0, tt = 0.0;
            NOD_FOR_NODES {
                const NodBottomIdx B = nod_bottom_idx(L, c);
                const double y = B.active ? nod_operator_generic(L, s, B.i, B.j, B.k) : 0.0;
                t[B.q] = y;
                ts += y * s[B.q];
                tt += y * y;
            }
            Dot2 qd = block_dot2(ts, tt, sh, nt);
            if (qd.b == 0.0) {
                NOD_FOR_NODES { const long long q = nod_bottom_idx(L, c).q; x[q] += alpha * p[q]; }
                break;
            }
            omega = qd.a / qd.b;
            double r2 = 0.0, hr = 0.0;
            NOD_FOR_NODES {
                const long long q = nod_bottom_idx(L, c).q;
                x[q] += alpha * p[q] + omega * s[q];
                const double y = s[q] - omega * t[q];
                r[q] = y;
                r2 += y * y;
                hr += rhat[q] * y;
            }
            qd = block_dot2(r2, hr, sh, nt);
            rr = qd.a;
            rho_old = rho;
            rho = qd.b;
            if (omega == 0.0) break;
        }
    }
    if (singular) {                                // zero plain mean over the unknowns (N8)
        group_sync(nt);
        double a = 0.0;
        NOD_FOR_NODES a += x[nod_bottom_idx(L, c).q];
        const double xm = block_dot2(a, 0.0, sh, nt).a / nunk;
        NOD_FOR_NODES {
            const NodBottomIdx B = nod_bottom_idx(L, c);
            if (B.active) x[B.q] -= xm;
        }
    }
#undef NOD_FOR_NODES
    if (tid == 0 && iters_accum) *iters_accum += it;
}
