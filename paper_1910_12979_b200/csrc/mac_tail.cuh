// mac_tail.cuh -- the coarse tail of the V-cycle in ONE launch ("a single
// persistent kernel" for the small levels; Sec. 7 hard part "coarse levels are launch-latency bound").
//
// Levels of at most 16^3 cells do a few microseconds of arithmetic each, but as separate launches every
// sweep, transfer and the bottom solve costs a launch plus a drained pipeline (5-15 us apiece, ~20
// launches per cycle).  Here ONE thread block walks the whole tail
//     for l = t0 .. bottom-1:  nu_pre RBGS sweeps, residual + restriction
//     BiCGStab on the bottom level
//     for l = bottom-1 .. t0:  prolongation + correction, nu_post RBGS sweeps
// with phi, rhs and the face coefficients of every tail level and the solver's vectors in shared memory
// (compact copies; a zero slot behind phi stands for neighbours outside the domain, which the folded
// coefficients want as 0) and __syncthreads between colour passes.  One SM issues every instruction of
// the tail, so the passes are written for instruction count: magic-number index splits, no boundary
// branches, the reciprocal-Newton quotient of the fused smoothers.  Tail levels are narrower than any
// TMA level and therefore in the plain (ghost-free) layout.
#pragma once
#include "mac_kernels.cuh"
#include "mac_smoother.cuh"

constexpr int kTailMaxLevels = 6;
constexpr int kTailMaxCells = 4096;                 // a level joins the tail when it has at most this many cells
constexpr size_t kTailSmem = 220 * 1024;

struct TailLevel {                                  // compact (pitch-free) copy of one level in shared memory
    int nx, ny, nz, nc;
    unsigned mx, mxy, mhx, mhxy;                    // magic multipliers: q / nx, q / (nx ny), q / hx, q / (hx ny), hx = ceil(nx/2)
    int per[3];                                     // periodic axes
    int o_phi, o_rhs, o_ax, o_ay, o_az;             // offsets (doubles) into the dynamic segment; phi has nc + 1 entries,
};                                                  // the last one is the constant 0 read for neighbours outside the domain

struct TailArgs {
    int nlev;                                       // levels in the tail; the last one is the coarsest of the hierarchy
    LevelDev L[kTailMaxLevels];
    TailLevel T[kTailMaxLevels];
    int o_vecs;                                     // six BiCGStab vectors of the last level
    int nu_pre, nu_post, maxit, singular, prolongation;
    int load_phi;                                   // 1: the first tail level is level 0 of the solve (phi is an iterate, not 0)
    double tol;
};

// q / d for q d < 2^32 with m = floor(2^32 / d) + 1
__device__ __forceinline__ int magic_div(int q, unsigned m) { return m ? (int)__umulhi((unsigned)q, m) : q; }   // m == 0: d == 1

// index of the neighbour at offset +-1 along an axis of extent n: wrapped if periodic, else the zero slot
__device__ __forceinline__ int tail_nb(int c, int f, int n, int stride, int dir, int per, int zslot)
{
    const int g = f + dir;
    if (g >= 0 && g < n) return c + dir * stride;
    return per ? c - dir * (n - 1) * stride : zslot;
}

// sum_f a_f phi_nb and sum_f a_f at cell (i, j, k) of a tail level (same term order as stencil_sums)
struct TailStencil { double axl, axh, ayl, ayh, azl, azh, w, e, s, n, d, u; };
__device__ __forceinline__ TailStencil tail_stencil(const TailLevel& T, const double* sm, const double* phi, int i, int j, int k, int c)
{
    TailStencil S;
    const int sxy = T.nx * T.ny;
    const double* ax = sm + T.o_ax + i + (T.nx + 1) * (j + T.ny * k);
    const double* ay = sm + T.o_ay + i + T.nx * (j + (T.ny + 1) * k);
    const double* az = sm + T.o_az + c;
    S.axl = ax[0]; S.axh = ax[1]; S.ayl = ay[0]; S.ayh = ay[T.nx]; S.azl = az[0]; S.azh = az[sxy];
    S.w = phi[tail_nb(c, i, T.nx, 1, -1, T.per[0], T.nc)];
    S.e = phi[tail_nb(c, i, T.nx, 1, +1, T.per[0], T.nc)];
    S.s = phi[tail_nb(c, j, T.ny, T.nx, -1, T.per[1], T.nc)];
    S.n = phi[tail_nb(c, j, T.ny, T.nx, +1, T.per[1], T.nc)];
    S.d = phi[tail_nb(c, k, T.nz, sxy, -1, T.per[2], T.nc)];
    S.u = phi[tail_nb(c, k, T.nz, sxy, +1, T.per[2], T.nc)];
    return S;
}

// one colour of red-black Gauss-Seidel
__device__ __forceinline__ void tail_color_pass(const TailLevel& T, double* sm, int color)
{
    double* phi = sm + T.o_phi;
    const double* rhs = sm + T.o_rhs;
    const int hx = (T.nx + 1) >> 1, n = hx * T.ny * T.nz;
    for (int q = threadIdx.x; q < n; q += blockDim.x) {
        const int k = magic_div(q, T.mhxy), r = q - k * hx * T.ny;
        const int j = magic_div(r, T.mhx), p = r - j * hx;
        const int i = 2 * p + ((j + k + color) & 1);
        if (i >= T.nx) continue;
        const int c = i + T.nx * (j + T.ny * k);
        const TailStencil S = tail_stencil(T, sm, phi, i, j, k, c);
        double a, dg;
        phi[c] = fused::gs_value(S.axl, S.axh, S.ayl, S.ayh, S.azl, S.azh, rhs[c], S.w, S.e, S.s, S.n, S.d, S.u, a, dg);
    }
    __syncthreads();
}

__device__ __forceinline__ double tail_residual_at(const TailLevel& T, const double* sm, int i, int j, int k)
{
    const double* phi = sm + T.o_phi;
    const int c = i + T.nx * (j + T.ny * k);
    const TailStencil S = tail_stencil(T, sm, phi, i, j, k, c);
    const double off = S.axl * S.w + S.axh * S.e + S.ayl * S.s + S.ayh * S.n + S.azl * S.d + S.azh * S.u;
    const double dg = ((S.axl + S.axh) + (S.ayl + S.ayh)) + (S.azl + S.azh);
    return sm[T.o_rhs + c] - (off - phi[c] * dg);
}

__device__ __forceinline__ void tail_residual_restrict(const TailLevel& F, const TailLevel& C, double* sm)
{
    for (int q = threadIdx.x; q < C.nc; q += blockDim.x) {
        const int K = magic_div(q, C.mxy), r = q - K * C.nx * C.ny;
        const int J = magic_div(r, C.mx), I = r - J * C.nx;
        double s = 0.0;
#pragma unroll
        for (int dk = 0; dk < 2; ++dk)
#pragma unroll
            for (int dj = 0; dj < 2; ++dj)
#pragma unroll
                for (int di = 0; di < 2; ++di) s += tail_residual_at(F, sm, 2 * I + di, 2 * J + dj, 2 * K + dk);
        sm[C.o_rhs + q] = 0.125 * s;
        sm[C.o_phi + q] = 0.0;
    }
    __syncthreads();
}

__device__ __forceinline__ void tail_prolong_add(const TailLevel& F, const TailLevel& C, const LevelDev& CL, double* sm,
                                                 int prolongation)
{
    double* phi = sm + F.o_phi;
    const double* e = sm + C.o_phi;
    for (int q = threadIdx.x; q < F.nc; q += blockDim.x) {
        const int k = magic_div(q, F.mxy), r = q - k * F.nx * F.ny;
        const int j = magic_div(r, F.mx), i = r - j * F.nx;
        const int I = i >> 1, J = j >> 1, K = k >> 1;
        auto ce = [&](int a, int b, int c) { return e[a + C.nx * (b + C.ny * c)]; };
        double val;
        if (prolongation == 1) {
            val = ce(I, J, K);
        } else {
            double sx = 1.0, sy = 1.0, sz = 1.0;
            const int I2 = ghost_index(I + ((i & 1) ? 1 : -1), C.nx, CL.bclo[0], CL.bchi[0], sx);
            const int J2 = ghost_index(J + ((j & 1) ? 1 : -1), C.ny, CL.bclo[1], CL.bchi[1], sy);
            const int K2 = ghost_index(K + ((k & 1) ? 1 : -1), C.nz, CL.bclo[2], CL.bchi[2], sz);
            const double wx1 = 0.25 * sx, wy1 = 0.25 * sy, wz1 = 0.25 * sz;
            val = 0.75 * (0.75 * (0.75 * ce(I, J, K) + wx1 * ce(I2, J, K)) + wy1 * (0.75 * ce(I, J2, K) + wx1 * ce(I2, J2, K))) +
                  wz1 * (0.75 * (0.75 * ce(I, J, K2) + wx1 * ce(I2, J, K2)) + wy1 * (0.75 * ce(I, J2, K2) + wx1 * ce(I2, J2, K2)));
        }
        phi[q] += val;
    }
    __syncthreads();
}

// stage a level's coefficients (global, pitched) into the compact shared-memory copy
__device__ __forceinline__ void tail_load_coeffs(const TailLevel& T, const LevelDev& L, double* sm)
{
    const int nax = (T.nx + 1) * T.ny * T.nz, nay = T.nx * (T.ny + 1) * T.nz, naz = T.nx * T.ny * (T.nz + 1);
    for (int q = threadIdx.x; q < nax; q += blockDim.x) {
        const int row = q / (T.nx + 1), i = q - row * (T.nx + 1);
        sm[T.o_ax + q] = L.ax[(size_t)i + (size_t)L.px * row];              // rows (j, k): pitch px, ry == ny
    }
    for (int q = threadIdx.x; q < nay; q += blockDim.x) sm[T.o_ay + q] = L.ay[q];     // plain layout: cx == nx
    for (int q = threadIdx.x; q < naz; q += blockDim.x) sm[T.o_az + q] = L.az[q];
    if (threadIdx.x == 0) sm[T.o_phi + T.nc] = 0.0;
}

// dynamic shared memory: per tail level phi[nc + 1], rhs[nc], ax, ay, az (compact); then the BiCGStab vectors
__global__ void __launch_bounds__(1024)
k_coarse_tail(const __grid_constant__ TailArgs A, int* __restrict__ iters_accum)
{
    __shared__ double sh[64];
    extern __shared__ double tail_sm[];
    double* sm = tail_sm;
    const int last = A.nlev - 1;
    for (int q = 0; q < last; ++q) tail_load_coeffs(A.T[q], A.L[q], sm);
    {   // entry: rhs of the first tail level (and phi when it is an iterate) from global memory
        const LevelDev& L = A.L[0];
        const TailLevel& T = A.T[0];
        for (int c = threadIdx.x; c < T.nc; c += blockDim.x) {
            sm[T.o_rhs + c] = L.rhs[c];
            sm[T.o_phi + c] = A.load_phi ? L.phi[c] : 0.0;
        }
    }
    __syncthreads();
    for (int q = 0; q < last; ++q) {
        for (int sw = 0; sw < A.nu_pre; ++sw) {
            tail_color_pass(A.T[q], sm, 0);
            tail_color_pass(A.T[q], sm, 1);
        }
        tail_residual_restrict(A.T[q], A.T[q + 1], sm);
    }
    {
        const TailLevel& T = A.T[last];
        const size_t nb = (size_t)T.nc;
        double* vecs = sm + A.o_vecs;
        // the solver runs on as many warps as the coarsest level has work for; the others wait below
        const int nt = min((int)blockDim.x, ((T.nc + 31) / 32) * 32);
        if ((int)threadIdx.x < nt) {
            const int it = bicgstab_block(A.L[last], sm + T.o_phi, sm + T.o_rhs, vecs, vecs + nb, vecs + 2 * nb, vecs + 3 * nb,
                                          vecs + 4 * nb, vecs + 5 * nb, A.maxit, A.tol, A.singular, sh, nt);
            if (threadIdx.x == 0 && iters_accum) *iters_accum += it;
        }
        __syncthreads();
    }
    for (int q = last - 1; q >= 0; --q) {
        tail_prolong_add(A.T[q], A.T[q + 1], A.L[q + 1], sm, A.prolongation);
        for (int sw = 0; sw < A.nu_post; ++sw) {
            tail_color_pass(A.T[q], sm, 0);
            tail_color_pass(A.T[q], sm, 1);
        }
    }
    {   // exit: the first tail level's phi back to global memory
        const LevelDev& L = A.L[0];
        const TailLevel& T = A.T[0];
        for (int c = threadIdx.x; c < T.nc; c += blockDim.x) L.phi[c] = sm[T.o_phi + c];
    }
}
