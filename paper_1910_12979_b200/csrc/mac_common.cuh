// mac_common.cuh -- shared device-side types and helpers of the MAC projection kernels (sm_100a).
//
// Internal data layout of one multigrid level (all fp64, x fastest):
//   cell arrays  phi, rhs        idx = i + nx*(j + ny*k)
//   ax (x faces)                 idx = i + px*(j + ny*k),  i in [0,nx], px = roundup(nx+1, 4)
//   ay (y faces)                 idx = i + nx*(j + (ny+1)*k), j in [0,ny]
//   az (z faces)                 idx = i + nx*(j + ny*k),  k in [0,nz]
// The stored coefficient is  a_f = c_f * (beta0/rho_face) / h_d^2  with the boundary type folded
// in: c_f = 1 on interior and periodic faces, 0 on WALL faces, 2 on OUTFLOW faces (SURVEY.md
// Sec. 8(c) O5).  With this folding the operator is
//        (L phi)_0 = sum_f a_f phi_nb(f) - phi_0 sum_f a_f ,   phi_nb := 0 outside the domain
// (periodic: wrapped), which is algebraically the ghost-cell form of the oracle:
// WALL ghost = +phi_0 gives zero flux (a_f = 0), OUTFLOW ghost = -phi_0 gives -2 b phi_0 / h^2.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MAC_PERIODIC 0
#define MAC_WALL 1
#define MAC_OUTFLOW 2

struct LevelDev {
    int nx, ny, nz, px;        // cells, x pitch of ax
    int bclo[3], bchi[3];
    double *phi, *phi2, *rhs, *ax, *ay, *az;
};

struct GeoDev {                // level-0 geometry for base-state profile evaluation
    int nx, ny, nz;
    double dx, dy, dz;
    int bclo[3], bchi[3];
    int geometry, nr;
    double dr, cx, cy, cz;
};

__device__ __forceinline__ size_t cidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * (size_t)k);
}
__device__ __forceinline__ size_t axidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)i + (size_t)L.px * ((size_t)j + (size_t)L.ny * (size_t)k);
}
__device__ __forceinline__ size_t ayidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)(L.ny + 1) * (size_t)k);
}
__device__ __forceinline__ size_t azidx(const LevelDev& L, int i, int j, int k)
{
    return (size_t)i + (size_t)L.nx * ((size_t)j + (size_t)L.ny * (size_t)k);
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
