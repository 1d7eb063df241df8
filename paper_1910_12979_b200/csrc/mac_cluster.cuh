// mac_cluster.cuh -- every level of at most 32^3 cells in ONE launch of ONE thread-block cluster, the level data
// resident in (distributed) shared memory ("a single persistent kernel for levels
// <= 32^3"; Sec. 7 "coarse levels are launch-latency bound").
//
// A level of 32^3 cells is 0.26 MB per array: its sweeps are a few microseconds of arithmetic, but as separate
// launches every colour pass, transfer and the bottom solve costs a launch and a drained GPU (5-15 us apiece), and
// when such a level is the whole problem (BASELINE.json config 1) every cycle also costs a host round trip for the
// stop test.  Here a cluster of 16 thread blocks (8192 threads on 16 SMs of one GPC) walks
//     for l = first .. bottom-1:  nu_pre red-black sweeps, residual + restriction
//     BiCGStab on the bottom level (block 0; one warp when the level has at most 64 unknowns)
//     for l = bottom-1 .. first:  prolongation + correction, nu_post sweeps
// with the hardware cluster barrier (barrier.cluster: 0.25 us measured on 16 blocks) between passes instead of kernel
// boundaries.  Data: every level is cut into z-slabs of ppc = ceil(nz / 16) planes, block r keeps planes
// [r ppc, (r+1) ppc) of phi, rhs and the three coefficient arrays in its shared memory (compact, pitch-free; 32^3:
// 2 planes = 86 KB per block); the bottom level lives in block 0.  A colour pass touches only the block's own slab
// except for the plane below / above it, which it reads from the neighbouring block through distributed shared
// memory (ld.shared::cluster via a mapped generic pointer); restriction and prolongation read the other level's
// planes wherever they live.  Nothing is WRITTEN remotely.  (Measured first: the same passes on the level arrays in
// L2 with barrier.cluster cost 2-3 us per pass -- an L2 round trip and a release of global stores per pass -- and
// lost to the one-block shared-memory tail; a remote shared-memory access under the barrier costs 0.5 us.)
//   solve = 0: one V-cycle leg from level `first` down and back (called once per cycle by the host for problems
//              whose finer levels run the streaming kernels).
//   solve = 1: `first` is level 0 of the problem: the kernel runs WHOLE cycles and takes the stop test itself
//              (||rhs - L phi||inf <= rel_tol ||rhs||inf after each cycle), leaving the cycle
//              count and the residual history for the host to read once.
// Arithmetic: the Gauss-Seidel value is fused::gs_value (as in every fused smoother), residual, restriction and
// prolongation are the expressions of k_residual_restrict / k_prolong_add.
#pragma once
#include <cooperative_groups.h>

#include "mac_kernels.cuh"
#include "mac_smoother.cuh"

namespace clus {

namespace cg = cooperative_groups;

constexpr int kCtas = 16, kThreads = 512;          // 16 blocks: a non-portable cluster size (opt-in at setup)
constexpr int kMaxLevels = 8;
constexpr int kMaxCells = 32768;                   // a level joins when it has at most this many cells
constexpr int kWarpBottom = 64;                    // bottoms of at most this many unknowns are solved by one warp
constexpr int kMaxBottom = 512;                    // largest bottom level this kernel takes (vectors in block 0's shared memory)
constexpr size_t kSmemMax = 220 * 1024;

struct Lev {
    LevelDev L;                                    // global arrays (plain layout): coefficients, and phi / rhs of the first level
    int hx;                                        // ceil(nx / 2)
    unsigned mx, mxy, mhx, mhxy;                   // magic multipliers: q / nx, q / (nx ny), q / hx, q / (hx ny)
    int ppc;                                       // planes per block (the bottom level: nz, all in block 0)
    unsigned mppc;                                 // magic multiplier: k / ppc
    int o_phi, o_rhs, o_ax, o_ay, o_az;            // offsets (doubles) of the slab arrays in every block's dynamic shared memory:
};                                                 // phi, rhs: ppc planes of nx ny; ax: ppc x (nx+1) ny; ay: ppc x nx (ny+1); az: ppc + 1 planes

struct Args {
    int nlev;                                      // levels handled; the last one is the coarsest of the hierarchy
    Lev V[kMaxLevels];
    int o_vecs;                                    // block 0: six BiCGStab vectors of a bottom with more than 64 unknowns
    int o_scr;                                     // every block: restriction scratch, 8 doubles per coarse cell of its largest coarse slab
    int nu_pre, nu_post, maxit, singular, prolongation;
    double tol;                                    // BiCGStab
    int solve, max_cycles;                         // solve = 1: whole cycles with the stop test
    double rel_tol;
    const double* rhs_norm;                        // device: ||rhs||inf of level 0 (solve = 1)
    double* result;                                // device, solve = 1: [0] cycles, [1] last residual norm, [2] status flag
                                                   // (1 = NaN met), [4 + c] relative residual after cycle c (c < 128)
    int* iters_accum;
};

__device__ __forceinline__ int mdiv(int q, unsigned m) { return m ? (int)__umulhi((unsigned)q, m) : q; }

// planes [lo, lo + np) of level V belong to block `rank`
struct Slab { int lo, np; };
__device__ __forceinline__ Slab slab_of(const Lev& V, int rank)
{
    Slab S;
    S.lo = rank * V.ppc;
    S.np = max(0, min(V.ppc, V.L.nz - S.lo));
    return S;
}

// Generic pointer to plane k (0 <= k < nz; for az: k <= nz) of the slab array at shared-memory offset `off` of level V,
// wherever it lives; pe = elements per plane.  For az the plane k = lo + np of a slab is also stored by its owner, so
// `upper` selects the copy held by the owner of plane k - 1.
__device__ __forceinline__ const double* plane_of(cg::cluster_group& cl, double* sm, const Lev& V, int off, int pe, int k, int rank,
                                                  bool upper = false)
{
    const int owner = mdiv(upper ? k - 1 : k, V.mppc);
    double* base = owner == rank ? sm : cl.map_shared_rank(sm, owner);
    return base + off + (size_t)(k - owner * V.ppc) * pe;
}

// the six face coefficients and the six neighbours (0 outside the domain) of cell (i, j) of one plane:
// pm / p0 / pp: phi planes below, own, above (NULL: outside a non-periodic domain); ax, ay, az0: coefficient planes of
// the cell's plane, az1: the z faces above it
struct Sten { double axl, axh, ayl, ayh, azl, azh, w, e, s, n, d, u; };
__device__ __forceinline__ Sten sten_planes(const LevelDev& L, const double* pm, const double* p0, const double* pp, const double* ax,
                                            const double* ay, const double* az0, const double* az1, int i, int j)
{
    Sten S;
    const int c2 = i + L.nx * j;
    S.axl = ax[i + (L.nx + 1) * j]; S.axh = ax[i + 1 + (L.nx + 1) * j];
    S.ayl = ay[c2]; S.ayh = ay[c2 + L.nx];
    S.azl = az0[c2]; S.azh = az1[c2];
    const bool px = L.bclo[0] == MAC_PERIODIC, py = L.bclo[1] == MAC_PERIODIC;
    S.w = i > 0 ? p0[c2 - 1] : (px ? p0[c2 + (L.nx - 1)] : 0.0);
    S.e = i < L.nx - 1 ? p0[c2 + 1] : (px ? p0[c2 - (L.nx - 1)] : 0.0);
    S.s = j > 0 ? p0[c2 - L.nx] : (py ? p0[c2 + (L.ny - 1) * L.nx] : 0.0);
    S.n = j < L.ny - 1 ? p0[c2 + L.nx] : (py ? p0[c2 - (L.ny - 1) * L.nx] : 0.0);
    S.d = pm ? pm[c2] : 0.0;
    S.u = pp ? pp[c2] : 0.0;
    return S;
}

// phi plane k of level V for a z neighbour: wrapped on a periodic axis, NULL outside the domain
__device__ __forceinline__ const double* phi_plane(cg::cluster_group& cl, double* sm, const Lev& V, int k, int rank)
{
    const int nz = V.L.nz, pe = V.L.nx * V.L.ny;
    if (k < 0) { if (V.L.bclo[2] != MAC_PERIODIC) return nullptr; k += nz; }
    else if (k >= nz) { if (V.L.bchi[2] != MAC_PERIODIC) return nullptr; k -= nz; }
    return plane_of(cl, sm, V, V.o_phi, pe, k, rank);
}

// one colour of red-black Gauss-Seidel on the block's own slab
__device__ __forceinline__ void color_pass(cg::cluster_group& cl, double* sm, const Lev& V, int color, int rank)
{
    const LevelDev& L = V.L;
    const Slab S = slab_of(V, rank);
    if (S.np == 0) return;
    const int pe = L.nx * L.ny, pax = (L.nx + 1) * L.ny, pay = L.nx * (L.ny + 1);
    const double* pd = phi_plane(cl, sm, V, S.lo - 1, rank);          // the planes below and above the slab (other blocks)
    const double* pu = phi_plane(cl, sm, V, S.lo + S.np, rank);
    double* phi = sm + V.o_phi;
    for (int r = threadIdx.x; r < V.hx * L.ny; r += kThreads) {       // (one x pair and row per thread on a 32 x 32 plane)
        const int j = mdiv(r, V.mhx), p = r - j * V.hx;
        const int c2e = 2 * p + L.nx * j;
        for (int kl = 0; kl < S.np; ++kl) {
            const int odd = (j + S.lo + kl + color) & 1;
            const int i = 2 * p + odd;
            if (i >= L.nx) continue;
            double* p0 = phi + kl * pe;
            const Sten T = sten_planes(L, kl > 0 ? p0 - pe : pd, p0, kl < S.np - 1 ? p0 + pe : pu, sm + V.o_ax + kl * pax,
                                       sm + V.o_ay + kl * pay, sm + V.o_az + kl * pe, sm + V.o_az + (kl + 1) * pe, i, j);
            double a, dg;
            p0[c2e + odd] = fused::gs_value(T.axl, T.axh, T.ayl, T.ayh, T.azl, T.azh, sm[V.o_rhs + kl * pe + c2e + odd], T.w, T.e, T.s,
                                            T.n, T.d, T.u, a, dg);
        }
    }
}

// the planes a residual in plane k of level V needs, wherever they live
struct Planes { const double *pm, *p0, *pp, *ax, *ay, *az0, *az1, *rhs; };
__device__ __forceinline__ Planes planes_of(cg::cluster_group& cl, double* sm, const Lev& V, int k, int rank)
{
    const LevelDev& L = V.L;
    const int pe = L.nx * L.ny;
    Planes P;
    P.p0 = plane_of(cl, sm, V, V.o_phi, pe, k, rank);
    P.pm = phi_plane(cl, sm, V, k - 1, rank);
    P.pp = phi_plane(cl, sm, V, k + 1, rank);
    P.ax = plane_of(cl, sm, V, V.o_ax, (L.nx + 1) * L.ny, k, rank);
    P.ay = plane_of(cl, sm, V, V.o_ay, L.nx * (L.ny + 1), k, rank);
    P.az0 = plane_of(cl, sm, V, V.o_az, pe, k, rank);
    P.az1 = plane_of(cl, sm, V, V.o_az, pe, k + 1, rank, true);
    P.rhs = plane_of(cl, sm, V, V.o_rhs, pe, k, rank);
    return P;
}

// rhs - L phi at cell (i, j) of the plane described by P
__device__ __forceinline__ double residual_at(const LevelDev& L, const Planes& P, int i, int j)
{
    const int c2 = i + L.nx * j;
    const Sten S = sten_planes(L, P.pm, P.p0, P.pp, P.ax, P.ay, P.az0, P.az1, i, j);
    const double off = S.axl * S.w + S.axh * S.e + S.ayl * S.s + S.ayh * S.n + S.azl * S.d + S.azh * S.u;
    const double dg = ((S.axl + S.axh) + (S.ayl + S.ayh)) + (S.azl + S.azh);
    return P.rhs[c2] - (off - P.p0[c2] * dg);
}

// Restriction in two steps, so that every residual is computed where its cell lives (a block that gathers the residuals
// of a level spread over 16 blocks pays one remote round trip after another: 18 us for 8^3 -> 4^3):
// (1) the owner of a fine cell computes rhs - L phi and STORES it into the scratch array of the block that owns the
//     parent, slot [parent][child]  (remote stores do not wait);
// (2) after a cluster barrier the parent's owner adds the eight values in the order of k_residual_restrict
//     (dk, dj, di ascending) and sets phi = 0.
__device__ __forceinline__ void residual_scatter(cg::cluster_group& cl, double* sm, const Lev& F, const Lev& C, int o_scr, int rank)
{
    const LevelDev& L = F.L;
    const Slab S = slab_of(F, rank);
    const int pe = L.nx * L.ny, pec = C.L.nx * C.L.ny;
    for (int kl = 0; kl < S.np; ++kl) {
        const int k = S.lo + kl, K = k >> 1;
        const Planes P = planes_of(cl, sm, F, k, rank);
        const int owner = mdiv(K, C.mppc);
        double* scr = (owner == rank ? sm : cl.map_shared_rank(sm, owner)) + o_scr + (size_t)(K - owner * C.ppc) * pec * 8 + 4 * (k & 1);
        for (int r = threadIdx.x; r < pe; r += kThreads) {
            const int j = mdiv(r, F.mx), i = r - j * L.nx;
            scr[((i >> 1) + C.L.nx * (j >> 1)) * 8 + 2 * (j & 1) + (i & 1)] = residual_at(L, P, i, j);
        }
    }
}

__device__ __forceinline__ void restrict_gather(double* sm, const Lev& C, int o_scr, int rank)
{
    const Slab S = slab_of(C, rank);
    const int n = C.L.nx * C.L.ny * S.np;
    for (int q = threadIdx.x; q < n; q += kThreads) {
        const double* v = sm + o_scr + (size_t)q * 8;
        double s = 0.0;
#pragma unroll
        for (int c = 0; c < 8; ++c) s += v[c];
        sm[C.o_rhs + q] = 0.125 * s;
        sm[C.o_phi + q] = 0.0;
    }
}

// phi_f += P e_c on the block's own fine slab
__device__ __forceinline__ void prolong_add(cg::cluster_group& cl, double* sm, const Lev& F, const Lev& C, int prolongation, int rank)
{
    const LevelDev& Lf = F.L;
    const LevelDev& Lc = C.L;
    const Slab S = slab_of(F, rank);
    const int pe = Lf.nx * Lf.ny, pec = Lc.nx * Lc.ny, n = pe * S.np;
    for (int q = threadIdx.x; q < n; q += kThreads) {
        const int kl = mdiv(q, F.mxy), r = q - kl * pe;
        const int j = mdiv(r, F.mx), i = r - j * Lf.nx;
        const int k = S.lo + kl;
        const int I = i >> 1, J = j >> 1, K = k >> 1;
        const double* e0 = plane_of(cl, sm, C, C.o_phi, pec, K, rank);
        double val;
        if (prolongation == 1) {
            val = e0[I + Lc.nx * J];
        } else {
            double sx = 1.0, sy = 1.0, sz = 1.0;
            const int I2 = ghost_index(I + ((i & 1) ? 1 : -1), Lc.nx, Lc.bclo[0], Lc.bchi[0], sx);
            const int J2 = ghost_index(J + ((j & 1) ? 1 : -1), Lc.ny, Lc.bclo[1], Lc.bchi[1], sy);
            const int K2 = ghost_index(K + ((k & 1) ? 1 : -1), Lc.nz, Lc.bclo[2], Lc.bchi[2], sz);
            const double* e1 = plane_of(cl, sm, C, C.o_phi, pec, K2, rank);
            const double wx1 = 0.25 * sx, wy1 = 0.25 * sy, wz1 = 0.25 * sz;
            const int a = I + Lc.nx * J, b = I2 + Lc.nx * J, c = I + Lc.nx * J2, d = I2 + Lc.nx * J2;
            val = 0.75 * (0.75 * (0.75 * e0[a] + wx1 * e0[b]) + wy1 * (0.75 * e0[c] + wx1 * e0[d])) +
                  wz1 * (0.75 * (0.75 * e1[a] + wx1 * e1[b]) + wy1 * (0.75 * e1[c] + wx1 * e1[d]));
        }
        sm[F.o_phi + q] += val;
    }
}

// own slab of a level: coefficients (global, pitched) into the compact shared-memory copy
__device__ __forceinline__ void load_coeffs(double* sm, const Lev& V, int rank)
{
    const LevelDev& L = V.L;
    const Slab S = slab_of(V, rank);
    if (S.np == 0) return;
    const int nax = (L.nx + 1) * L.ny * S.np, nay = L.nx * (L.ny + 1) * S.np, naz = L.nx * L.ny * (S.np + 1);
    for (int q = threadIdx.x; q < nax; q += kThreads) {
        const int row = q / (L.nx + 1), i = q - row * (L.nx + 1);
        sm[V.o_ax + q] = L.ax[(size_t)i + (size_t)L.px * ((size_t)row + (size_t)L.ny * S.lo)];       // rows (j, k): pitch px, ry == ny
    }
    const double* ay = L.ay + (size_t)L.nx * (L.ny + 1) * S.lo;
    for (int q = threadIdx.x; q < nay; q += kThreads) sm[V.o_ay + q] = ay[q];                         // plain layout: cx == nx
    const double* az = L.az + (size_t)L.nx * L.ny * S.lo;
    for (int q = threadIdx.x; q < naz; q += kThreads) sm[V.o_az + q] = az[q];
}

// BiCGStab on a bottom level of at most 64 unknowns by ONE warp ("warp-level bottom solver,
// warp-shuffle reductions"): lane l owns unknowns l and l + 32, its two matrix rows and every vector entry live in
// registers, a matrix-vector product exchanges the operand through 64 doubles of shared memory (__syncwarp only), the
// dot products are shuffle reductions.  The algorithm, its stopping rule and its breakdown exits are those of
// bicgstab_block (x0 = 0, rhat = r0, ||r||2 <= tol ||f||2).  Returns the iteration count.
__device__ __forceinline__ void wsum2(double& a, double& b)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
}

__device__ __forceinline__ int bicgstab_warp(const LevelDev& L, double* __restrict__ xg, const double* __restrict__ fg,
                                             double* sh, int maxit, double tol, int singular)
{
    const int lane = threadIdx.x & 31;
    const int nb = L.nx * L.ny * L.nz;
    double ra[2][6], rdg[2];
    int ri[2][6];
    bool ok[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const int c = lane + 32 * h;
        ok[h] = c < nb;
        rdg[h] = 0.0;
#pragma unroll
        for (int q = 0; q < 6; ++q) { ra[h][q] = 0.0; ri[h][q] = 0; }
        if (!ok[h]) continue;
        const int i = c % L.nx, j = (c / L.nx) % L.ny, k = c / (L.nx * L.ny);
        ra[h][0] = L.ax[axidx(L, i, j, k)]; ra[h][1] = L.ax[axidx(L, i + 1, j, k)];
        ra[h][2] = L.ay[ayidx(L, i, j, k)]; ra[h][3] = L.ay[ayidx(L, i, j + 1, k)];
        ra[h][4] = L.az[azidx(L, i, j, k)]; ra[h][5] = L.az[azidx(L, i, j, k + 1)];
        rdg[h] = ((ra[h][0] + ra[h][1]) + (ra[h][2] + ra[h][3])) + (ra[h][4] + ra[h][5]);
        const int n3[3] = {L.nx, L.ny, L.nz}, st[3] = {1, L.nx, L.nx * L.ny}, f3[3] = {i, j, k};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int sd = 0; sd < 2; ++sd) {
                const int g = f3[a] + (sd ? 1 : -1);
                int idx = c + (sd ? st[a] : -st[a]);
                if (g < 0 || g >= n3[a]) {
                    if (L.bclo[a] == MAC_PERIODIC) idx = c + (sd ? -(n3[a] - 1) * st[a] : (n3[a] - 1) * st[a]);
                    else { idx = c; ra[h][2 * a + sd] = 0.0; }         // (rdg keeps the folded boundary coefficient)
                }
                ri[h][2 * a + sd] = idx;
            }
    }
    auto matvec = [&](const double (&y)[2], double (&out)[2]) {
        __syncwarp();
#pragma unroll
        for (int h = 0; h < 2; ++h) sh[lane + 32 * h] = y[h];
        __syncwarp();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double off = ra[h][0] * sh[ri[h][0]] + ra[h][1] * sh[ri[h][1]] + ra[h][2] * sh[ri[h][2]] +
                               ra[h][3] * sh[ri[h][3]] + ra[h][4] * sh[ri[h][4]] + ra[h][5] * sh[ri[h][5]];
            out[h] = ok[h] ? off - y[h] * rdg[h] : 0.0;
        }
    };
    double f[2], x[2] = {0.0, 0.0}, r[2], rhat[2], p[2] = {0.0, 0.0}, v[2] = {0.0, 0.0}, s[2], t[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) f[h] = ok[h] ? fg[lane + 32 * h] : 0.0;
    double fm = 0.0, dummy = 0.0;
    if (singular) {
        fm = f[0] + f[1];
        wsum2(fm, dummy);
        fm /= (double)nb;
    }
    double rr = 0.0;
#pragma unroll
    for (int h = 0; h < 2; ++h) { r[h] = ok[h] ? f[h] - fm : 0.0; rhat[h] = r[h]; rr += r[h] * r[h]; }
    wsum2(rr, dummy);
    const double bnorm2 = rr;
    int it = 0;
    if (bnorm2 > 0.0 && bnorm2 == bnorm2) {
        const double stop2 = tol * tol * bnorm2;
        double rho = rr, rho_old = 1.0, alpha = 1.0, omega = 1.0;
        while (it < maxit && rr > stop2) {
            if (rho == 0.0) break;                                   // breakdown
            const double beta = it == 0 ? 0.0 : (rho / rho_old) * (alpha / omega);
#pragma unroll
            for (int h = 0; h < 2; ++h) p[h] = r[h] + beta * (p[h] - omega * v[h]);
            matvec(p, v);
            double d = rhat[0] * v[0] + rhat[1] * v[1];
            wsum2(d, dummy);
            if (d == 0.0) break;
            alpha = rho / d;
            double ss = 0.0;
#pragma unroll
            for (int h = 0; h < 2; ++h) { s[h] = r[h] - alpha * v[h]; ss += s[h] * s[h]; }
            wsum2(ss, dummy);
            ++it;
            if (ss <= stop2) {
#pragma unroll
                for (int h = 0; h < 2; ++h) x[h] += alpha * p[h];
                rr = ss;
                break;
            }
            matvec(s, t);
            double ts = t[0] * s[0] + t[1] * s[1], tt = t[0] * t[0] + t[1] * t[1];
            wsum2(ts, tt);
            if (tt == 0.0) {
#pragma unroll
                for (int h = 0; h < 2; ++h) x[h] += alpha * p[h];
                break;
            }
            omega = ts / tt;
            double r2 = 0.0, hr = 0.0;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                x[h] += alpha * p[h] + omega * s[h];
                r[h] = s[h] - omega * t[h];
                r2 += r[h] * r[h];
                hr += rhat[h] * r[h];
            }
            wsum2(r2, hr);
            rr = r2;
            rho_old = rho;
            rho = hr;
            if (omega == 0.0) break;
        }
    }
    if (singular) {                            // zero-mean x
        double xm = x[0] + x[1];
        wsum2(xm, dummy);
        xm /= (double)nb;
#pragma unroll
        for (int h = 0; h < 2; ++h) x[h] -= xm;
    }
#pragma unroll
    for (int h = 0; h < 2; ++h)
        if (ok[h]) xg[lane + 32 * h] = x[h];
    return it;
}

// maximum over the cluster of a per-thread value (NaN wins); the same value in every thread of every block.
// Every block stores its partial maximum into slot[own rank] of EVERY block (remote stores), one barrier, local reads.
__device__ __forceinline__ double cluster_nanmax(cg::cluster_group& cl, double v, double* sh, double* slots, int rank)
{
    v = warp_nanmax(v);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < kCtas) {
        double m = sh[0];
        for (int q = 1; q < kThreads / 32; ++q) m = nanmax(m, sh[q]);
        cl.map_shared_rank(slots, threadIdx.x)[rank] = m;
    }
    cl.sync();
    double m = slots[0];
    for (int q = 1; q < kCtas; ++q) m = nanmax(m, slots[q]);
    cl.sync();                                  // (the slots are rewritten by the next reduction)
    return m;
}

__global__ void __launch_bounds__(kThreads, 1)
k_cluster_vcycles(const __grid_constant__ Args A)
{
    cg::cluster_group cl = cg::this_cluster();
    __shared__ double sh[64];
    __shared__ double slots[kCtas];
    __shared__ Lev sV[kMaxLevels];              // the level table, indexed at run time
    extern __shared__ double cl_sm[];
    double* sm = cl_sm;
#pragma unroll
    for (int q = 0; q < kMaxLevels; ++q)
        if ((int)threadIdx.x == q) sV[q] = A.V[q];
    __syncthreads();
    const int rank = (int)cl.block_rank();
    const int last = A.nlev - 1;
    for (int q = 0; q < last; ++q) load_coeffs(sm, sV[q], rank);
    {   // entry: phi and rhs of the first level (its own slab) from global memory
        const Lev& V = sV[0];
        const Slab S = slab_of(V, rank);
        const int pe = V.L.nx * V.L.ny, n = pe * S.np;
        const double* gp = V.L.phi + (size_t)pe * S.lo;
        const double* gr = V.L.rhs + (size_t)pe * S.lo;
        for (int q = threadIdx.x; q < n; q += kThreads) { sm[V.o_phi + q] = gp[q]; sm[V.o_rhs + q] = gr[q]; }
    }
    cl.sync();
    const int ncyc = A.solve ? A.max_cycles : 1;
    const double rnorm = A.solve ? *A.rhs_norm : 0.0;
    int done = 0;
    double res = 0.0;
    bool bad = false;
    for (int cyc = 0; cyc < ncyc; ++cyc) {
        for (int q = 0; q < last; ++q) {
            for (int sw = 0; sw < A.nu_pre; ++sw) {
                color_pass(cl, sm, sV[q], 0, rank); cl.sync();
                color_pass(cl, sm, sV[q], 1, rank); cl.sync();
            }
            residual_scatter(cl, sm, sV[q], sV[q + 1], A.o_scr, rank);
            cl.sync();
            restrict_gather(sm, sV[q + 1], A.o_scr, rank);
            cl.sync();
        }
        if (rank == 0) {                        // the bottom level lives here
            const Lev& V = sV[last];
            const int nb = V.L.nx * V.L.ny * V.L.nz;
            if (nb <= kWarpBottom) {
                if (threadIdx.x < 32) {
                    const int it = bicgstab_warp(V.L, sm + V.o_phi, sm + V.o_rhs, sh, A.maxit, A.tol, A.singular);
                    if (threadIdx.x == 0 && A.iters_accum) *A.iters_accum += it;
                }
            } else {
                double* vecs = sm + A.o_vecs;
                const int nt = min(kThreads, ((nb + 31) / 32) * 32);
                if ((int)threadIdx.x < nt) {
                    const int it = bicgstab_block(V.L, sm + V.o_phi, sm + V.o_rhs, vecs, vecs + nb, vecs + 2 * nb, vecs + 3 * nb,
                                                  vecs + 4 * nb, vecs + 5 * nb, A.maxit, A.tol, A.singular, sh, nt);
                    if (threadIdx.x == 0 && A.iters_accum) *A.iters_accum += it;
                }
            }
        }
        cl.sync();
        for (int q = last - 1; q >= 0; --q) {
            prolong_add(cl, sm, sV[q], sV[q + 1], A.prolongation, rank);
            cl.sync();
            for (int sw = 0; sw < A.nu_post; ++sw) {
                color_pass(cl, sm, sV[q], 0, rank); cl.sync();
                color_pass(cl, sm, sV[q], 1, rank); cl.sync();
            }
        }
        if (!A.solve) break;
        // stop test on level 0 (O9): max-norm of the residual relative to ||rhs||inf
        double m = 0.0;
        {
            const Lev& V = sV[0];
            const Slab S = slab_of(V, rank);
            const int pe = V.L.nx * V.L.ny;
            for (int kl = 0; kl < S.np; ++kl) {
                const Planes P = planes_of(cl, sm, V, S.lo + kl, rank);
                for (int r = threadIdx.x; r < pe; r += kThreads) {
                    const int j = mdiv(r, V.mx), i = r - j * V.L.nx;
                    m = nanmax(m, fabs(residual_at(V.L, P, i, j)));
                }
            }
        }
        res = cluster_nanmax(cl, m, sh, slots, rank);
        const double rel = res / rnorm;
        if (rank == 0 && threadIdx.x == 0 && cyc < 128) A.result[4 + cyc] = rel;
        done = cyc + 1;
        if (rel != rel) { bad = true; break; }
        if (rel <= A.rel_tol) break;
    }
    {   // exit: the first level's phi back to global memory
        const Lev& V = sV[0];
        const Slab S = slab_of(V, rank);
        const int pe = V.L.nx * V.L.ny, n = pe * S.np;
        double* gp = V.L.phi + (size_t)pe * S.lo;
        for (int q = threadIdx.x; q < n; q += kThreads) gp[q] = sm[V.o_phi + q];
    }
    if (A.solve && rank == 0 && threadIdx.x == 0) {
        A.result[0] = (double)done;
        A.result[1] = res;
        A.result[2] = bad ? 1.0 : 0.0;
    }
    cl.sync();                                  // no block leaves while another may still read its shared memory
}

}  // namespace clus
