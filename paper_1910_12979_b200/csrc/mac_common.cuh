// mac_common.cuh -- shared device-side types and helpers of the MAC projection kernels (sm_100a).
//
// Internal data layout of one multigrid level (all fp64, x fastest).  Pointers address the interior
// origin (i, j, k) = (0, 0, 0); a level may carry gx ghost columns on each side in x and gy ghost
// rows on each side in y (see below), so the pitches are not the cell counts:
//   cell arrays  phi, rhs        idx = i + cx*(j + ry*k)         cx = nx + 2 gx, ry = ny + 2 gy
//   ax (x faces)                 idx = i + px*(j + ry*k),        i in [0,nx], px = roundup(nx+1+2gx, 4)
//   ay (y faces)                 idx = i + cx*(j + (ry+1)*k),    j in [0,ny]
//   az (z faces)                 idx = i + cx*(j + ry*k),        k in [0,nz]
// The stored coefficient is  a_f = c_f * (beta0/rho_face) / h_d^2  with the boundary type folded
// in: c_f = 1 on interior and periodic faces, 0 on WALL faces, 2 on OUTFLOW faces (SURVEY.md
// Sec. 8(c) O5).  With this folding the operator is
//        (L phi)_0 = sum_f a_f phi_nb(f) - phi_0 sum_f a_f ,   phi_nb := 0 outside the domain
// (periodic: wrapped), which is algebraically the ghost-cell form of the oracle:
// WALL ghost = +phi_0 gives zero flux (a_f = 0), OUTFLOW ghost = -phi_0 gives -2 b phi_0 / h^2.
//
// Ghosts.  The TMA-staged kernels load rectangular boxes and cannot wrap, so a level that is
// periodic in x and/or y and runs those kernels stores two periodic image columns / rows of every
// array on each side (gx = 2 and/or gy = 2; 0 otherwise).  Kernels that index with wrap-around
// never read them; every kernel that writes such an array also writes the images (in-kernel
// image stores in the per-cycle kernels, k_fill_ghosts after the once-per-projection ones).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MAC_PERIODIC 0
#define MAC_WALL 1
#define MAC_OUTFLOW 2

struct LevelDev {
    int nx, ny, nz, px;        // cells, x pitch of ax
    int cx, ry;                // x pitch of the cell-shaped arrays; rows per plane (ay has ry + 1)
    int gx, gy;                // ghost columns / rows per side (0 or 2)
    int bclo[3], bchi[3];
    double *phi, *phi2, *rhs, *ax, *ay, *az;
};

struct GeoDev {                // level-0 geometry for base-state profile evaluation
    int nx, ny, nz;
    double dx, dy, dz;
    int bclo[3], bchi[3];
    int geometry, nr;
    double dr, cx, cy, cz;
    int rho_mean;              // face density: 0 arithmetic mean of rho, 1 harmonic (mean of 1/rho); reading A3
};

// density on a face from the two cells it separates (O2; `harmonic`: the variant of reading A3)
__device__ __forceinline__ double face_rho(double rl, double rr, int harmonic)
{
    return harmonic ? 2.0 / (1.0 / rl + 1.0 / rr) : 0.5 * (rl + rr);
}

__device__ __forceinline__ size_t cidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)((long long)i + (long long)L.cx * ((long long)j + (long long)L.ry * (long long)k));
}
__device__ __forceinline__ size_t axidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)((long long)i + (long long)L.px * ((long long)j + (long long)L.ry * (long long)k));
}
__device__ __forceinline__ size_t ayidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)((long long)i + (long long)L.cx * ((long long)j + (long long)(L.ry + 1) * (long long)k));
}
__device__ __forceinline__ size_t azidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)((long long)i + (long long)L.cx * ((long long)j + (long long)L.ry * (long long)k));
}

// Offsets (in elements, 0 = none) of the periodic images of interior cell (i, j) of a cell-shaped array.
__device__ __forceinline__ long long image_dx(const LevelDev& L, int i)
{
    return L.gx == 0 ? 0 : (i < L.gx ? (long long)L.nx : (i >= L.nx - L.gx ? -(long long)L.nx : 0));
}
__device__ __forceinline__ long long image_dy(const LevelDev& L, int j)
{
    return L.gy == 0 ? 0 : (j < L.gy ? (long long)L.ny * L.cx : (j >= L.ny - L.gy ? -(long long)L.ny * L.cx : 0));
}
// store v at p and at its periodic images
template <typename T>
__device__ __forceinline__ void store_images(T* p, const T& v, long long dx, long long dy)
{
    *p = v;
    if (dx) p[dx / (long long)(sizeof(T) / 8)] = v;
    if (dy) {
        p[dy / (long long)(sizeof(T) / 8)] = v;
        if (dx) p[(dx + dy) / (long long)(sizeof(T) / 8)] = v;
    }
}

// Base-state profile f sampled at (m+1/2) dr: linear between samples, constant beyond the ends.
__device__ __forceinline__ double profile_eval(const double* __restrict__ f, int nr, double dr, double r)
{
    double s = r / dr - 0.5;
    if (s <= 0.0) return __ldg(f);
    if (s >= (double)(nr - 1)) return __ldg(f + nr - 1);
    int m = (int)s;
    double t = s - (double)m;
    return (1.0 - t) * __ldg(f + m) + t * __ldg(f + m + 1);
}

__device__ __forceinline__ double radius(const GeoDev& G, double x, double y, double z)
{
    if (G.geometry == 0) return z;
    double ax = x - G.cx, ay = y - G.cy, az = z - G.cz;
    return sqrt(ax * ax + ay * ay + az * az);
}

// NaN-propagating max of non-negative values
__device__ __forceinline__ double nanmax(double m, double v) { return (v > m || v != v) ? v : m; }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double warp_nanmax(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = nanmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
