// mac_nodal.cuh -- kernels of the end-of-step (nodal) projection (PAPER.md:63
// "second order projection method ... multigrid linear solvers for the pressure projection steps"; weighting
// beta0/rho of PAPER.md:35 Eq. 2, constraint of PAPER.md:49 Eq. 6).  Readings N1..N10 of DESIGN.md.
//
// phi lives on the nodes, (nx+1)(ny+1)(nz+1) values (idx = i + (nx+1)(j + (ny+1)k)); sigma = beta0/rho, the
// velocities, rho and S are cell arrays in the public cell layout (idx = i + nx (j + ny k), no ghosts).
// Operator: the trilinear (Q1) finite-element form of div(sigma grad phi) divided by the cell volume,
//     (L phi)_a = -sum_c sigma_c sum_b (K^c_ab / V) phi_b
// over the up to 8 cells c around node a and their 8 corners b.  K^c_ab / V depends only on whether b is the
// same corner as a or the other one along each axis (8 classes): w[cls] = sum_d g_d k_d prod_{e != d} m_e,
// g_d = 1/h_d^2, k = +1 same / -1 other, m = 1/3 same / 1/6 other.  A neighbour node b at offset (dx, dy, dz)
// in {-1,0,1}^3 therefore enters with  -w[cls(dx,dy,dz)] * T(dx,dy,dz),  T = the sum of sigma over the cells
// that contain both a and b: 19 additions expand the 8 sigmas to the 27 sums, 27 + 8 fused multiply-adds form
// L phi.  Node rules (N4): OUTFLOW nodes count as 0 and are not unknowns; on a periodic axis node n is node 0
// (the arrays keep n+1 entries; the kernels never read entry n and write it only when the result is exported);
// cells outside a non-periodic boundary do not exist (sigma := 0).
// Smoother: Jacobi (order-free: reproducible, one HBM pass per sweep, 32 B per node: sigma, phi, rhs in, phi out),
// ping-pong between phi and phi2; the sweep can emit max |rhs - L phi_in|, so the stop test of a cycle rides on the
// first pre-smoothing sweep of the next one at no extra pass.
#pragma once
#include "mac_kernels.cuh"

struct NodLevel {
    int nx, ny, nz;                 // cells
    int bclo[3], bchi[3];
    double w[8];                    // class weights; bit 0 / 1 / 2: the other corner along x / y / z
    double omega;                   // Jacobi damping (N7)
    double *phi, *phi2, *rhs;       // node arrays
    double *sigma;                  // cell array
};

__device__ __forceinline__ size_t nod_idx(const NodLevel& L, int i, int j, int k)
{
    return (size_t)((long long)i + (long long)(L.nx + 1) * ((long long)j + (long long)(L.ny + 1) * (long long)k));
}
__device__ __forceinline__ size_t nod_cidx(const NodLevel& L, int i, int j, int k)
{
    return (size_t)((long long)i + (long long)L.nx * ((long long)j + (long long)L.ny * (long long)k));
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

// One axis of the 27-point neighbourhood of an unknown node t: stored indices of the nodes t-1, t, t+1 (-1: the
// value counts as 0: no such node, or an OUTFLOW node) and of the cells t-1, t (-1: no such cell).
struct NodAxis { int nd[3]; int cl[2]; };
__device__ __forceinline__ NodAxis nod_axis(const NodLevel& L, int d, int t)
{
    const int n = d == 0 ? L.nx : (d == 1 ? L.ny : L.nz);
    const bool per = L.bclo[d] == MAC_PERIODIC;
    NodAxis A;
    A.nd[1] = t;
    A.nd[0] = t > 0 ? t - 1 : (per ? n - 1 : -1);
    A.nd[2] = t < n ? (t + 1 == n && per ? 0 : t + 1) : -1;
    A.cl[0] = t > 0 ? t - 1 : (per ? n - 1 : -1);
    A.cl[1] = t < n ? t : -1;
    if (!per) {                                       // OUTFLOW nodes count as 0
        if (A.nd[0] == 0 && L.bclo[d] == MAC_OUTFLOW) A.nd[0] = -1;
        if (A.nd[2] == n && L.bchi[d] == MAC_OUTFLOW) A.nd[2] = -1;
    }
    return A;
}

// L phi and the diagonal at the unknown node (i, j, k).  FAST: every neighbour node and cell exists and none is an
// OUTFLOW node (all but a surface layer of nodes): plain strided loads.
template <bool FAST>
__device__ __forceinline__ void nod_operator(const NodLevel& L, const double* __restrict__ phi, int i, int j, int k,
                                             double& lphi, double& diag)
{
    double p[3][3][3], s[2][2][2];
    if (FAST) {
        const long long px = 1, py = L.nx + 1, pz = (long long)(L.nx + 1) * (L.ny + 1);
        const double* q = phi + nod_idx(L, i, j, k);
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int b = 0; b < 3; ++b)
#pragma unroll
                for (int a = 0; a < 3; ++a) p[c][b][a] = q[(a - 1) * px + (b - 1) * py + (c - 1) * pz];
        const long long cy = L.nx, cz = (long long)L.nx * L.ny;
        const double* sg = L.sigma + nod_cidx(L, i - 1, j - 1, k - 1);
#pragma unroll
        for (int c = 0; c < 2; ++c)
#pragma unroll
            for (int b = 0; b < 2; ++b)
#pragma unroll
                for (int a = 0; a < 2; ++a) s[c][b][a] = __ldg(sg + a + b * cy + c * cz);
    } else {
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
    lphi = -sum;
    diag = -(L.w[0] * t[1][1][1]);
}

__device__ __forceinline__ bool nod_fast(const NodLevel& L, int i, int j, int k)
{
    return i >= 2 && i <= L.nx - 2 && j >= 2 && j <= L.ny - 2 && k >= 2 && k <= L.nz - 2;
}

// ---- N3: sigma = beta0(r_cell) / rho, beta0 at the cell centres (bcell, scratch for the rhs), rho check ------
__global__ void __launch_bounds__(256)
k_nod_sigma(GeoDev G, const double* __restrict__ beta0, const double* __restrict__ rho, const double* __restrict__ rho0,
            double* __restrict__ sigma, double* __restrict__ bcell, int* __restrict__ flags)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i >= G.nx || j >= G.ny) return;
    const size_t c = (size_t)i + (size_t)G.nx * ((size_t)j + (size_t)G.ny * k);
    const double r = radius(G, (i + 0.5) * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz);
    const double b = profile_eval(beta0, G.nr, G.dr, r);
    const double rh = rho ? __ldg(rho + c) : profile_eval(rho0, G.nr, G.dr, r);
    if (!(rh > 0.0) || !(rh <= 1.79769313486231570e308)) atomicOr(flags, 1);
    sigma[c] = b / rh;
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
                    const size_t q = nod_cidx(L, X.cl[a], Y.cl[b], Z.cl[c]);
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
// WSUM) and max |a| afterwards.  shift == NULL: only the reductions.
template <bool WEIGHTED, bool WSUM>
__global__ void __launch_bounds__(256)
k_nod_shift(NodLevel L, double* __restrict__ a, const double* __restrict__ scal, double inv_cells,
            double* __restrict__ part_sum, double* __restrict__ part_max, int zper)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    double s = 0.0, m = 0.0;
    for (int k = blockIdx.z * zper; k < min((int)(blockIdx.z + 1) * zper, L.nz + 1); ++k)
    if (i <= L.nx && j <= L.ny && nod_kind(L, i, j, k) == 0) {
        const size_t q = nod_idx(L, i, j, k);
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

// ---- N7: one Jacobi sweep pin -> pout (distinct buffers); NORM: block partials of max |rhs - L phi_in| ---------
template <bool NORM>
__global__ void __launch_bounds__(256)
k_nod_jacobi(NodLevel L, const double* __restrict__ pin, double* __restrict__ pout, double* __restrict__ part_max, int zper)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    double rabs = 0.0;
    for (int k = blockIdx.z * zper; k < min((int)(blockIdx.z + 1) * zper, L.nz + 1); ++k)
    if (i <= L.nx && j <= L.ny) {
        const size_t q = nod_idx(L, i, j, k);
        double out = 0.0;
        if (nod_kind(L, i, j, k) == 0) {
            double lp, dg;
            if (nod_fast(L, i, j, k)) nod_operator<true>(L, pin, i, j, k, lp, dg);
            else nod_operator<false>(L, pin, i, j, k, lp, dg);
            const double r = L.rhs[q] - lp;
            rabs = nanmax(rabs, fabs(r));
            out = pin[q] + L.omega * r / dg;
        }
        pout[q] = out;
    }
    if (NORM) {
        __shared__ double sh[8];
        const int tid = threadIdx.x + blockDim.x * threadIdx.y;
        rabs = warp_nanmax(rabs);
        if ((tid & 31) == 0) sh[tid >> 5] = rabs;
        __syncthreads();
        if (tid == 0) {
            double m = sh[0];
            for (int q = 1; q < (int)(blockDim.x * blockDim.y + 31) / 32; ++q) m = nanmax(m, sh[q]);
            part_max[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = m;
        }
    }
}

// ---- residual r = rhs - L phi at the unknowns, 0 elsewhere (res may be NULL); block partials of max |r| ---------
__global__ void __launch_bounds__(256)
k_nod_residual(NodLevel L, const double* __restrict__ phi, double* __restrict__ res, double* __restrict__ part_sum,
               double* __restrict__ part_max, int zper)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y;
    double rmax = 0.0;
    for (int k = blockIdx.z * zper; k < min((int)(blockIdx.z + 1) * zper, L.nz + 1); ++k)
    if (i <= L.nx && j <= L.ny) {
        double r = 0.0;
        const size_t q = nod_idx(L, i, j, k);
        if (nod_kind(L, i, j, k) == 0) {
            double lp, dg;
            if (nod_fast(L, i, j, k)) nod_operator<true>(L, phi, i, j, k, lp, dg);
            else nod_operator<false>(L, phi, i, j, k, lp, dg);
            r = L.rhs[q] - lp;
        }
        if (res) res[q] = r;
        rmax = nanmax(rmax, fabs(r));
    }
    block_reduce_store(0.0, rmax, part_sum, part_max, blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z));
}

// ---- N6: coarse rhs = (1/8) P^T res (weights 1, 1/2 per axis over the 27 fine nodes), coarse phi = 0 -----------
__global__ void __launch_bounds__(256)
k_nod_restrict(NodLevel F, NodLevel C, const double* __restrict__ res)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x, J = blockIdx.y * blockDim.y + threadIdx.y, K = blockIdx.z;
    if (I > C.nx || J > C.ny) return;
    double s = 0.0;
    if (nod_kind(C, I, J, K) == 0) {
        int fi[3], fj[3], fk[3];
#pragma unroll
        for (int o = 0; o < 3; ++o) {                 // fine node 2 T + (o - 1) per axis, wrapped, or -1
            int t = 2 * I + o - 1;
            if (F.bclo[0] == MAC_PERIODIC) { if (t < 0) t += F.nx; if (t >= F.nx) t -= F.nx; } else if (t < 0 || t > F.nx) t = -1;
            fi[o] = t;
            t = 2 * J + o - 1;
            if (F.bclo[1] == MAC_PERIODIC) { if (t < 0) t += F.ny; if (t >= F.ny) t -= F.ny; } else if (t < 0 || t > F.ny) t = -1;
            fj[o] = t;
            t = 2 * K + o - 1;
            if (F.bclo[2] == MAC_PERIODIC) { if (t < 0) t += F.nz; if (t >= F.nz) t -= F.nz; } else if (t < 0 || t > F.nz) t = -1;
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
    const size_t q = nod_idx(C, I, J, K);
    C.rhs[q] = s;
    C.phi[q] = 0.0;
}

// value of a coarse nodal array at node (I, J, K) under the node rules (OUTFLOW 0, periodic node n = node 0)
__device__ __forceinline__ double nod_val(const NodLevel& L, const double* __restrict__ a, int I, int J, int K)
{
    if (nod_kind(L, I, J, K) == 1) return 0.0;
    if (L.bclo[0] == MAC_PERIODIC && I == L.nx) I = 0;
    if (L.bclo[1] == MAC_PERIODIC && J == L.ny) J = 0;
    if (L.bclo[2] == MAC_PERIODIC && K == L.nz) K = 0;
    return a[nod_idx(L, I, J, K)];
}

// ---- N6: phi_f += P e_c at the fine unknowns (trilinear: weights 1, 1/2, 1/4, 1/8) -----------------------------
__global__ void __launch_bounds__(256)
k_nod_prolong_add(NodLevel F, NodLevel C)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i > F.nx || j > F.ny || nod_kind(F, i, j, k) != 0) return;
    const int I = i >> 1, J = j >> 1, K = k >> 1, oi = i & 1, oj = j & 1, ok = k & 1;
    const double wt = (oi ? 0.5 : 1.0) * (oj ? 0.5 : 1.0) * (ok ? 0.5 : 1.0);
    double s = 0.0;
    for (int c = 0; c <= ok; ++c)
        for (int b = 0; b <= oj; ++b)
            for (int a = 0; a <= oi; ++a) s += wt * nod_val(C, C.phi, I + a, J + b, K + c);
    F.phi[nod_idx(F, i, j, k)] += s;
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
    const size_t q = nod_cidx(L, i, j, k);
    const double rh = rho ? __ldg(rho + q) : profile_eval(rho0, G.nr, G.dr, radius(G, (i + 0.5) * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz));
    u[q] -= gx / rh;
    v[q] -= gy / rh;
    w[q] -= gz / rh;
}

// export: OUTFLOW nodes 0, periodic duplicates equal their image; src and dst may be the same array
__global__ void __launch_bounds__(256)
k_nod_export(NodLevel L, const double* __restrict__ src, double* __restrict__ dst)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y * blockDim.y + threadIdx.y, k = blockIdx.z;
    if (i > L.nx || j > L.ny) return;
    dst[nod_idx(L, i, j, k)] = nod_val(L, src, i, j, k);
}

// ---- N8: bottom solve, unpreconditioned BiCGStab on the unknowns of the coarsest level (one thread block, vectors
// over ALL nodes of the level in global memory -- the level is tiny and L1/L2-resident; entries of OUTFLOW nodes and
// periodic duplicates stay 0).  Same algorithm and stopping rule as the MAC bottom solver (reading A15).
__device__ __forceinline__ double nod_matvec_at(const NodLevel& L, const double* __restrict__ x, int c, bool active)
{
    if (!active) return 0.0;
    const int px = L.nx + 1, py = L.ny + 1;
    const int i = c % px, j = (c / px) % py, k = c / (px * py);
    double lp, dg;
    nod_operator<false>(L, x, i, j, k, lp, dg);
    return lp;
}

__global__ void __launch_bounds__(1024)
k_nod_bottom(NodLevel L, double* __restrict__ vecs, int maxit, double tol, int singular, int* __restrict__ iters_accum)
{
    __shared__ double sh[64];
    const int nb = (L.nx + 1) * (L.ny + 1) * (L.nz + 1), nt = blockDim.x, tid = threadIdx.x;
    double *x = L.phi, *r = vecs, *rhat = vecs + nb, *p = vecs + 2 * (size_t)nb, *v = vecs + 3 * (size_t)nb,
           *s = vecs + 4 * (size_t)nb, *t = vecs + 5 * (size_t)nb;
    const double* f = L.rhs;
    auto active = [&](int c) {
        const int px = L.nx + 1, py = L.ny + 1;
        return nod_kind(L, c % px, (c / px) % py, c / (px * py)) == 0;
    };
    double cnt = 0.0, fs = 0.0;
    for (int c = tid; c < nb; c += nt)
        if (active(c)) { cnt += 1.0; fs += f[c]; }
    const Dot2 q0 = block_dot2(cnt, fs, sh, nt);
    const double nunk = q0.a, fm = singular ? q0.b / q0.a : 0.0;
    double rr = 0.0;
    for (int c = tid; c < nb; c += nt) {
        const double fv = active(c) ? f[c] - fm : 0.0;
        r[c] = fv; rhat[c] = fv; p[c] = 0.0; v[c] = 0.0; x[c] = 0.0;
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
            for (int c = tid; c < nb; c += nt) p[c] = r[c] + beta * (p[c] - omega * v[c]);
            group_sync(nt);
            double d = 0.0;
            for (int c = tid; c < nb; c += nt) { const double y = nod_matvec_at(L, p, c, active(c)); v[c] = y; d += rhat[c] * y; }
            d = block_dot2(d, 0.0, sh, nt).a;
            if (d == 0.0) break;
            alpha = rho / d;
            double ss = 0.0;
            for (int c = tid; c < nb; c += nt) { const double y = r[c] - alpha * v[c]; s[c] = y; ss += y * y; }
            ss = block_dot2(ss, 0.0, sh, nt).a;
            ++it;
            if (ss <= stop2) {
                for (int c = tid; c < nb; c += nt) x[c] += alpha * p[c];
                rr = ss;
                break;
            }
            double ts = 0.0, tt = 0.0;
            for (int c = tid; c < nb; c += nt) { const double y = nod_matvec_at(L, s, c, active(c)); t[c] = y; ts += y * s[c]; tt += y * y; }
            Dot2 q = block_dot2(ts, tt, sh, nt);
            if (q.b == 0.0) {
                for (int c = tid; c < nb; c += nt) x[c] += alpha * p[c];
                break;
            }
            omega = q.a / q.b;
            double r2 = 0.0, hr = 0.0;
            for (int c = tid; c < nb; c += nt) {
                x[c] += alpha * p[c] + omega * s[c];
                const double y = s[c] - omega * t[c];
                r[c] = y;
                r2 += y * y;
                hr += rhat[c] * y;
            }
            q = block_dot2(r2, hr, sh, nt);
            rr = q.a;
            rho_old = rho;
            rho = q.b;
            if (omega == 0.0) break;
        }
    }
    if (singular) {                                // zero plain mean over the unknowns (N8)
        group_sync(nt);
        double a = 0.0;
        for (int c = tid; c < nb; c += nt) a += x[c];
        const double xm = block_dot2(a, 0.0, sh, nt).a / nunk;
        for (int c = tid; c < nb; c += nt)
            if (active(c)) x[c] -= xm;
    }
    if (tid == 0 && iters_accum) *iters_accum += it;
}
