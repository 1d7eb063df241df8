// mac_base.cuh -- the 1-D base-state steps upstream of the projection:
//   beta0 from p0 and Gamma1bar            (Eq. 5)
//   q = (1/(Gamma1bar p0)) dp0/dt          (Eq. 6; enters the rhs as S - q(r), see k_setup)
// on the nr profile samples r_m = (m + 1/2) dr.  Readings A26-A28: beta0_0 = rho0_0; the
// integrand is integrated as d(ln p0)/Gamma1bar with Gamma1bar at the midpoint of two samples.
//
// nr is a few thousand at most: one warp does the running sum -- each lane sums a contiguous chunk of
// the increments, a shuffle scan turns the lane totals into offsets -- so the order of additions is
// fixed (deterministic) and close to the oracle's sequential one.
#pragma once
#include "mac_common.cuh"

__global__ void __launch_bounds__(32)
k_base_state(int nr, const double* __restrict__ rho0, const double* __restrict__ p0,
             const double* __restrict__ gamma1bar, const double* __restrict__ dp0dt,
             double* __restrict__ beta0, double* __restrict__ q)
{
    const int lane = threadIdx.x;
    const int ninc = nr - 1;                                   // increments m -> m + 1
    const int chunk = (ninc + 31) / 32;
    const int m0 = min(lane * chunk, ninc), m1 = min(m0 + chunk, ninc);
    auto inc = [&](int m) {
        return (log(__ldg(p0 + m + 1)) - log(__ldg(p0 + m))) / (0.5 * (__ldg(gamma1bar + m) + __ldg(gamma1bar + m + 1)));
    };
    double tot = 0.0;
    for (int m = m0; m < m1; ++m) tot += inc(m);
    double run = tot;                                          // inclusive scan of the lane totals
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double t = __shfl_up_sync(0xffffffffu, run, o);
        if (lane >= o) run += t;
    }
    double lnb = log(__ldg(rho0)) + (run - tot);               // ln beta0 at sample m0
    if (lane == 0) beta0[0] = __ldg(rho0);
    for (int m = m0; m < m1; ++m) {
        lnb += inc(m);
        beta0[m + 1] = exp(lnb);
    }
    if (q && dp0dt)
        for (int m = lane; m < nr; m += 32) q[m] = __ldg(dp0dt + m) / (__ldg(gamma1bar + m) * __ldg(p0 + m));
}

// ------------------------------------------------------------------------------------------------
// Lateral average rho -> rho0(r)  ("rho0 ... represents the lateral average"; SURVEY.md
// Sec. 8(f) rank 4).  Cell (i,j,k) belongs to sample m = min(nr-1, floor(r / dr)), r the radius of its
// centre (planar: z).  The decision is an integer taken from floating point, so r and r / dr are formed
// with exactly the oracle's operations (no FMA contraction, IEEE sqrt and division): both sides bin
// every cell alike.  k_average_finish divides and fills samples without cells by linear interpolation
// in m (constant beyond the ends).
// ------------------------------------------------------------------------------------------------
// The sums are taken in a FIXED order, so the result is bit-reproducible from run to run (fp64 atomics are not): a block
// walks a fixed set of rows; every warp owns a private set of bins in shared memory (no two warps ever add to the same
// word); within a warp step the lanes that share a sample are found with __match_any_sync and their values are added
// in lane order by the lowest lane; at the end the block folds its warps' bins in warp order into partial[block][m],
// and k_average_finish folds the blocks in block order.  Shared memory: nwarp x nr x (8 + 4) bytes (dynamic); the host
// picks nwarp so that it fits.
__global__ void __launch_bounds__(256)
k_lateral_sum(GeoDev G, const double* __restrict__ rho, double* __restrict__ part_sum, unsigned* __restrict__ part_cnt)
{
    extern __shared__ double lat_sm[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    double* bsum = lat_sm + (size_t)warp * G.nr;                                  // this warp's bins
    unsigned* cnt0 = reinterpret_cast<unsigned*>(lat_sm + (size_t)nwarp * G.nr);
    unsigned* bcnt = cnt0 + (size_t)warp * G.nr;
    for (int m = lane; m < G.nr; m += 32) { bsum[m] = 0.0; bcnt[m] = 0u; }
    __syncwarp();
    const int nrows = G.ny * G.nz;
    // rows in contiguous chunks per block: the assignment depends only on the launch shape
    const int per_block = (nrows + gridDim.x - 1) / gridDim.x;
    const int r0 = blockIdx.x * per_block, r1 = min(nrows, r0 + per_block);
    for (int row = r0 + warp; row < r1; row += nwarp) {
        const int j = row % G.ny, k = row / G.ny;
        const double ay = __dsub_rn(__dmul_rn((double)j + 0.5, G.dy), G.cy), az = __dsub_rn(__dmul_rn((double)k + 0.5, G.dz), G.cz);
        const double zc = __dmul_rn((double)k + 0.5, G.dz);
        const double* __restrict__ p = rho + (size_t)G.nx * ((size_t)j + (size_t)G.ny * k);
        double vq[4];
        for (int i0 = 0; i0 < G.nx; i0 += 32) {
            const int i = i0 + lane;
            const bool on = i < G.nx;
            if ((i0 & 127) == 0) {                                    // request the next four warp-rows of values at once
#pragma unroll
                for (int q = 0; q < 4; ++q) vq[q] = i + 32 * q < G.nx ? __ldg(p + i + 32 * q) : 0.0;
            }
            double r = zc;
            if (G.geometry != 0) {
                const double ax = __dsub_rn(__dmul_rn((double)i + 0.5, G.dx), G.cx);
                r = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(ax, ax), __dmul_rn(ay, ay)), __dmul_rn(az, az)));
            }
            int m = (int)floor(__ddiv_rn(r, G.dr));
            m = max(0, min(m, G.nr - 1));
            const int qs = (i0 >> 5) & 3;
            const double v = qs == 0 ? vq[0] : (qs == 1 ? vq[1] : (qs == 2 ? vq[2] : vq[3]));
            const unsigned same = __match_any_sync(0xffffffffu, on ? m : -1 - lane);   // lanes of the same sample (idle lanes: alone)
            if (same == 0xffffffffu) {                                // one sample for the whole warp (always, in planar geometry)
                const double s = warp_sum(v);                         // fixed shuffle tree
                if (lane == 0) { bsum[m] += s; bcnt[m] += 32u; }
            } else {                                                  // the lowest lane of each group adds its values in lane order
                double s = 0.0;
                unsigned rest = same;
                while (__any_sync(0xffffffffu, rest != 0u)) {
                    const int src = rest ? __ffs(rest) - 1 : 0;
                    const double t = __shfl_sync(0xffffffffu, v, src);
                    if (rest) { s += t; rest &= rest - 1u; }
                }
                if (on && lane == __ffs(same) - 1) { bsum[m] += s; bcnt[m] += (unsigned)__popc(same); }
            }
            __syncwarp();
        }
    }
    __syncthreads();
    for (int m = threadIdx.x; m < G.nr; m += blockDim.x) {            // fold the warps in warp order
        double s = 0.0;
        unsigned c = 0u;
        for (int w = 0; w < nwarp; ++w) { s += lat_sm[(size_t)w * G.nr + m]; c += cnt0[(size_t)w * G.nr + m]; }
        part_sum[(size_t)blockIdx.x * G.nr + m] = s;
        part_cnt[(size_t)blockIdx.x * G.nr + m] = c;
    }
}

__global__ void __launch_bounds__(256)
k_average_finish(int nr, int nblocks, const double* __restrict__ part_sum, const unsigned* __restrict__ part_cnt,
                 unsigned long long* __restrict__ cnt, double* __restrict__ rho0)
{
    for (int m = threadIdx.x; m < nr; m += blockDim.x) {              // fold the blocks in block order
        double s = 0.0;
        unsigned long long c = 0ull;
        for (int b = 0; b < nblocks; ++b) { s += part_sum[(size_t)b * nr + m]; c += part_cnt[(size_t)b * nr + m]; }
        cnt[m] = c;
        if (c > 0) rho0[m] = s / (double)c;
    }
    __syncthreads();
    if (threadIdx.x == 0) {                                          // samples without cells
        int prev = -1;
        for (int m = 0; m < nr; ++m) {
            if (cnt[m] == 0) continue;
            if (prev < 0) for (int q = 0; q < m; ++q) rho0[q] = rho0[m];
            else
                for (int q = prev + 1; q < m; ++q) {
                    const double t = (double)(q - prev) / (double)(m - prev);
                    rho0[q] = (1.0 - t) * rho0[prev] + t * rho0[m];
                }
            prev = m;
        }
        if (prev >= 0) for (int q = prev + 1; q < nr; ++q) rho0[q] = rho0[prev];
    }
}
