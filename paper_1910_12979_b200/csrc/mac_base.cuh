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
// every cell alike.  Sums and counts are accumulated with atomics (a warp whose cells share one sample
// -- every warp in planar geometry -- reduces first and issues one), so the sums are exact up to the
// order of additions; k_average_finish divides and fills samples without cells by linear interpolation
// in m (constant beyond the ends).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
k_lateral_sum(GeoDev G, const double* __restrict__ rho, double* __restrict__ sum, unsigned long long* __restrict__ cnt)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int nrows = G.ny * G.nz;
    for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
        const int j = row % G.ny, k = row / G.ny;
        const double ay = __dsub_rn(__dmul_rn((double)j + 0.5, G.dy), G.cy), az = __dsub_rn(__dmul_rn((double)k + 0.5, G.dz), G.cz);
        const double zc = __dmul_rn((double)k + 0.5, G.dz);
        const double* __restrict__ p = rho + (size_t)G.nx * ((size_t)j + (size_t)G.ny * k);
        for (int i0 = warp * 32; i0 < G.nx; i0 += nwarp * 32) {
            const int i = i0 + lane;
            const bool on = i < G.nx;
            double r = zc;
            if (G.geometry != 0) {
                const double ax = __dsub_rn(__dmul_rn((double)i + 0.5, G.dx), G.cx);
                r = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(ax, ax), __dmul_rn(ay, ay)), __dmul_rn(az, az)));
            }
            int m = (int)floor(__ddiv_rn(r, G.dr));
            m = max(0, min(m, G.nr - 1));
            const double v = on ? __ldg(p + i) : 0.0;
            const unsigned act = __ballot_sync(0xffffffffu, on);
            const int m0 = __shfl_sync(0xffffffffu, m, 0);
            if (__all_sync(0xffffffffu, !on || m == m0)) {           // one sample for the whole warp
                const double s = warp_sum(v);
                if (lane == 0) { atomicAdd(sum + m0, s); atomicAdd(cnt + m0, (unsigned long long)__popc(act)); }
            } else if (on) {
                atomicAdd(sum + m, v);
                atomicAdd(cnt + m, 1ull);
            }
        }
    }
}

__global__ void __launch_bounds__(256)
k_average_finish(int nr, const double* __restrict__ sum, const unsigned long long* __restrict__ cnt, double* __restrict__ rho0)
{
    for (int m = threadIdx.x; m < nr; m += blockDim.x)
        if (cnt[m] > 0) rho0[m] = sum[m] / (double)cnt[m];
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
