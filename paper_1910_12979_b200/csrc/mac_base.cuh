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
