// mac_tail.cuh -- the coarse tail of the V-cycle in ONE launch ("a single
// persistent kernel" for the small levels; Sec. 7 hard part "coarse levels are launch-latency bound").
//
// Levels of at most 16^3 cells do a few microseconds of arithmetic each, but as separate launches every
// sweep, transfer and the bottom solve costs a launch plus a drained pipeline (5-15 us apiece, ~20
// launches per cycle).  Here ONE thread block walks the whole tail
//     for l = t0 .. bottom-1:  nu_pre RBGS sweeps, residual + restriction
//     BiCGStab on the bottom level
//     for l = bottom-1 .. t0:  prolongation + correction, nu_post RBGS sweeps
// with phi and rhs of every tail level and the solver's vectors in shared memory and __syncthreads
// between colour passes.  Coefficients are read from global memory (read-only during a cycle, L1
// resident).  Arithmetic per update is that of the reference kernels (k_rbgs_color,
// k_residual_restrict, k_prolong_add, k_bottom_bicgstab); tail levels are narrower than any TMA level
// and therefore in the plain (ghost-free) layout.
#pragma once
#include "mac_kernels.cuh"

constexpr int kTailMaxLevels = 6;
constexpr int kTailMaxCells = 4096;                 // a level joins the tail when it has at most this many cells
constexpr size_t kTailSmem = 200 * 1024;

struct TailArgs {
    int nlev;                                       // levels in the tail; the last one is the coarsest of the hierarchy
    LevelDev L[kTailMaxLevels];
    int nu_pre, nu_post, maxit, singular, prolongation;
    int load_phi;                                   // 1: the first tail level is level 0 of the solve (phi is an iterate, not 0)
    double tol;
};

// one colour of red-black Gauss-Seidel on level L with phi, rhs in shared memory
__device__ __forceinline__ void tail_color_pass(const LevelDev& L, double* phi, const double* rhs, int color)
{
    const int hx = (L.nx + 1) >> 1, n = hx * L.ny * L.nz;
    for (int q = threadIdx.x; q < n; q += blockDim.x) {
        const int p = q % hx, j = (q / hx) % L.ny, k = q / (hx * L.ny);
        const int i = 2 * p + ((j + k + color) & 1);
        if (i >= L.nx) continue;
        double off, dg;
        stencil_sums(L, phi, i, j, k, off, dg);
        const size_t c = cidx(L, i, j, k);
        phi[c] = (off - rhs[c]) / dg;
    }
    __syncthreads();
}

__device__ __forceinline__ void tail_residual_restrict(const LevelDev& F, const double* phi, const double* rhs,
                                                       const LevelDev& C, double* crhs, double* cphi)
{
    const int n = C.nx * C.ny * C.nz;
    for (int q = threadIdx.x; q < n; q += blockDim.x) {
        const int I = q % C.nx, J = (q / C.nx) % C.ny, K = q / (C.nx * C.ny);
        double s = 0.0;
#pragma unroll
        for (int dk = 0; dk < 2; ++dk)
#pragma unroll
            for (int dj = 0; dj < 2; ++dj)
#pragma unroll
                for (int di = 0; di < 2; ++di) {
                    const int i = 2 * I + di, j = 2 * J + dj, k = 2 * K + dk;
                    double off, dg;
                    stencil_sums(F, phi, i, j, k, off, dg);
                    const size_t c = cidx(F, i, j, k);
                    s += rhs[c] - (off - phi[c] * dg);
                }
        crhs[q] = 0.125 * s;
        cphi[q] = 0.0;
    }
    __syncthreads();
}

__device__ __forceinline__ void tail_prolong_add(const LevelDev& F, double* phi, const LevelDev& C, const double* e,
                                                 int prolongation)
{
    const int n = F.nx * F.ny * F.nz;
    for (int q = threadIdx.x; q < n; q += blockDim.x) {
        const int i = q % F.nx, j = (q / F.nx) % F.ny, k = q / (F.nx * F.ny);
        const int I = i >> 1, J = j >> 1, K = k >> 1;
        double val;
        if (prolongation == 1) {
            val = e[cidx(C, I, J, K)];
        } else {
            double sx = 1.0, sy = 1.0, sz = 1.0;
            const int I2 = ghost_index(I + ((i & 1) ? 1 : -1), C.nx, C.bclo[0], C.bchi[0], sx);
            const int J2 = ghost_index(J + ((j & 1) ? 1 : -1), C.ny, C.bclo[1], C.bchi[1], sy);
            const int K2 = ghost_index(K + ((k & 1) ? 1 : -1), C.nz, C.bclo[2], C.bchi[2], sz);
            const double wx1 = 0.25 * sx, wy1 = 0.25 * sy, wz1 = 0.25 * sz;
            val = 0.75 * (0.75 * (0.75 * e[cidx(C, I, J, K)] + wx1 * e[cidx(C, I2, J, K)]) +
                          wy1 * (0.75 * e[cidx(C, I, J2, K)] + wx1 * e[cidx(C, I2, J2, K)])) +
                  wz1 * (0.75 * (0.75 * e[cidx(C, I, J, K2)] + wx1 * e[cidx(C, I2, J, K2)]) +
                         wy1 * (0.75 * e[cidx(C, I, J2, K2)] + wx1 * e[cidx(C, I2, J2, K2)]));
        }
        phi[q] += val;
    }
    __syncthreads();
}

// shared memory: per tail level phi[ncell], rhs[ncell]; then the six BiCGStab vectors of the last level
__global__ void __launch_bounds__(1024)
k_coarse_tail(TailArgs A, int* __restrict__ iters_accum)
{
    __shared__ double sh[64];
    extern __shared__ double tail_sm[];
    double* phi[kTailMaxLevels];
    double* rhs[kTailMaxLevels];
    size_t off = 0;
    for (int q = 0; q < A.nlev; ++q) {
        const size_t nc = (size_t)A.L[q].nx * A.L[q].ny * A.L[q].nz;
        phi[q] = tail_sm + off; rhs[q] = tail_sm + off + nc;
        off += 2 * nc;
    }
    double* vecs = tail_sm + off;
    const int last = A.nlev - 1;
    {   // entry: rhs of the first tail level (and phi when it is an iterate) from global memory
        const LevelDev& L = A.L[0];
        const int n = L.nx * L.ny * L.nz;
        for (int c = threadIdx.x; c < n; c += blockDim.x) {
            rhs[0][c] = L.rhs[c];
            phi[0][c] = A.load_phi ? L.phi[c] : 0.0;
        }
        __syncthreads();
    }
    for (int q = 0; q < last; ++q) {
        for (int sw = 0; sw < A.nu_pre; ++sw) {
            tail_color_pass(A.L[q], phi[q], rhs[q], 0);
            tail_color_pass(A.L[q], phi[q], rhs[q], 1);
        }
        tail_residual_restrict(A.L[q], phi[q], rhs[q], A.L[q + 1], rhs[q + 1], phi[q + 1]);
    }
    {
        const size_t nb = (size_t)A.L[last].nx * A.L[last].ny * A.L[last].nz;
        const int it = bicgstab_block(A.L[last], phi[last], rhs[last], vecs, vecs + nb, vecs + 2 * nb, vecs + 3 * nb,
                                      vecs + 4 * nb, vecs + 5 * nb, A.maxit, A.tol, A.singular, sh);
        if (threadIdx.x == 0 && iters_accum) *iters_accum += it;
    }
    for (int q = last - 1; q >= 0; --q) {
        tail_prolong_add(A.L[q], phi[q], A.L[q + 1], phi[q + 1], A.prolongation);
        for (int sw = 0; sw < A.nu_post; ++sw) {
            tail_color_pass(A.L[q], phi[q], rhs[q], 0);
            tail_color_pass(A.L[q], phi[q], rhs[q], 1);
        }
    }
    {   // exit: the first tail level's phi back to global memory
        const LevelDev& L = A.L[0];
        const int n = L.nx * L.ny * L.nz;
        for (int c = threadIdx.x; c < n; c += blockDim.x) L.phi[c] = phi[0][c];
    }
}
