// mac_smoother.cuh -- the hot kernel: one red-black Gauss-Seidel sweep with red and black fused
// into ONE pass over HBM (north_star bullet 3).
//
// Algorithmic traffic: read phi, rhs, ax, ay, az once, write phi once = 48 B/cell/sweep (a
// kernel-per-colour smoother moves 96).  The result equals the two-pass red-then-black sweep:
//     new_red   = R(old black neighbours),     new_black = R(new red neighbours)
// and within a colour the update order is irrelevant, so only rounding-order differs.
//
// Scheme (2.5-D blocking with a one-plane lag, z-plane staging in shared memory).  A CTA owns a
// lateral tile of 60 x TY cells and a chunk [k0,k1) of z-planes and marches upward in z.  It reads
// phi_in (old) and writes phi_out (ping-pong, so neighbouring CTAs never see half-updated data).
// Planes are staged by cp.async (16-byte, L2-only) into a ring of NS = 5 shared-memory stages:
// while step k computes on planes k-1, k, k+1, planes k+2 and k+3 are in flight (two planes of
// lookahead per SM hide the HBM latency without spending registers).  At step k the CTA
//   (1) updates the red cells of plane k      (old black neighbours: planes k-1, k, k+1),
//   (2) updates the black cells of plane k-1  (new red neighbours:   planes k-2, k-1, k),
//   (3) stores plane k-1.
// A thread owns a PAIR of x-adjacent columns (one is red and one is black in every plane) and keeps
// their z-neighbours in registers; lateral neighbours come from the staged planes (new red values
// are written back into the stage in place).  Red cells in a one-cell ring around the tile are
// recomputed redundantly (halo: 2 cells of old phi on each side).  Every cell is updated exactly
// once per sweep, so each coefficient and rhs value is used once; a staged 16-byte pair is read
// once and the half that belongs to the other colour is carried in registers to the next step
// (two register sets alternate; the loop is unrolled by two so nothing is moved).
// One __syncthreads per plane.
//
// phi outside the domain is 0 on non-periodic sides (the boundary type is folded into the
// coefficients, mac_common.cuh) and wrapped on periodic sides; cp.async zero-fill provides the 0s.
#pragma once
#include "mac_common.cuh"

namespace fused {

constexpr int kStages = 5;
enum { A_PHI = 0, A_AX = 1, A_AY = 2, A_AZ = 3, A_RHS = 4, A_COUNT = 5 };

__device__ __forceinline__ int wrap(int f, int n)
{
    f %= n;
    return f < 0 ? f + n : f;
}

__device__ __forceinline__ void cp_async16(unsigned smem_dst, const void* gsrc, int bytes)
{
    // bytes = 16, or 0 => nothing is read and the 16 bytes are zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(smem_dst), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// The division by the diagonal: dg is a sum of positive, well-scaled face coefficients, so the guarded IEEE
// division (range checks + slow-path call) is replaced by a reciprocal seed and two Newton steps (1/dg to ~1 ulp)
// times the numerator: within ~1.5 ulp of the quotient.  -DMAC_GS_FAITHFUL adds one correction of the quotient
// (<= 1 ulp), -DMAC_IEEE_DIV restores the plain division.
// The Gauss-Seidel value  (sum_f a_f phi_f - rhs) / sum_f a_f  arranged for a short dependent chain.  In the
// marching kernels the upper neighbour u_ is the value the previous half-sweep of the SAME step has just
// produced, so it enters last: the reciprocal of the diagonal and the other five products are off the chain,
// which is then fma, mul (fp64 latency, not throughput, bounds these kernels).  *a_out = sum - rhs.
__device__ __forceinline__ double gs_value(double axw, double axe, double ays, double ayn, double azd, double azu,
                                           double rhs, double w_, double e_, double s_, double n_, double d_, double u_,
                                           double& a_out, double& dg_out)
{
    const double dg = ((axw + axe) + (ays + ayn)) + (azd + azu);
    const double t = (fma(axe, e_, axw * w_) + fma(ayn, n_, ays * s_)) + fma(azd, d_, -rhs);
    const double a = fma(azu, u_, t);
    a_out = a;
    dg_out = dg;
#ifdef MAC_IEEE_DIV
    return a / dg;
#else
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(dg));
    r = fma(fma(-dg, r, 1.0), r, r);
    r = fma(fma(-dg, r, 1.0), r, r);
    const double q = a * r;
#ifdef MAC_GS_FAITHFUL
    return fma(fma(-dg, q, a), r, q);           // one correction of the quotient: faithful (<= 1 ulp)
#else
    return q;                                   // r is 1/dg to ~1 ulp, so the quotient is within ~1.5 ulp: the correction
                                                // would put two more dependent fp64 operations on the chain of every
                                                // half-sweep (two-sweep kernel: 1.75 -> 1.64 ms without it)
#endif
#endif
}

struct Coef {                       // coefficients of one plane for a column pair, in registers
    double2 ax; double ax2; double2 ays, ayn, az, rhs;
};

template <bool X> __device__ __forceinline__ double pick(const double2& v) { return X ? v.x : v.y; }
template <bool X> __device__ __forceinline__ void put(double2& v, double s) { if (X) v.x = s; else v.y = s; }

template <int LN, int TYE>
struct Ctx {
    static constexpr int kArr = TYE * LN * 16;        // bytes of one array in a stage
    static constexpr int kStage = A_COUNT * kArr;         // bytes of one stage
    static constexpr int kRow = LN * 16;
    // per-thread constants
    const unsigned char* g_phi; const unsigned char* g_rhs; const unsigned char* g_ax;
    const unsigned char* g_ay; const unsigned char* g_az;  // global pointers at plane 0, own lateral slot
    unsigned long long s_c, s_ax, s_ay;                    // plane strides in bytes
    int b_phi, b_co, b_ax, b_ay;                           // 16 if the lateral slot is loaded, else 0
    int nz, perz;
    long long img_x, img_y;                                // offsets (doubles) of the periodic images of the own pair, 0 = none
    bool own;                                              // the pair is one this CTA stores (NORM counts only those: ring
                                                           // cells are duplicates, and outermost ghost reds are not valid)
    unsigned smem_u32;                                     // shared address of stage 0 + own slot
    unsigned char* smem_gen;                               // generic address of stage 0 + own slot
};

// issue the cp.async loads of plane p (unwrapped index) into stage `stg`
template <int LN, int TYE>
__device__ __forceinline__ void issue(const Ctx<LN, TYE>& C, int p, int stg)
{
    const bool real = C.perz || (p >= 0 && p < C.nz);
    const bool face = real || p == C.nz;                   // low z face of plane p exists (non-periodic top)
    int wp = p;
    if (C.perz) { if (wp < 0) wp += C.nz; else if (wp >= C.nz) wp -= C.nz; }
    const unsigned long long q = (real || face) ? (unsigned long long)(unsigned)wp : 0ull;
    const unsigned d = C.smem_u32 + stg * Ctx<LN, TYE>::kStage;
    cp_async16(d + A_PHI * Ctx<LN, TYE>::kArr, C.g_phi + q * C.s_c, real ? C.b_phi : 0);
    cp_async16(d + A_RHS * Ctx<LN, TYE>::kArr, C.g_rhs + q * C.s_c, real ? C.b_co : 0);
    cp_async16(d + A_AX * Ctx<LN, TYE>::kArr, C.g_ax + q * C.s_ax, real ? C.b_ax : 0);
    cp_async16(d + A_AY * Ctx<LN, TYE>::kArr, C.g_ay + q * C.s_ay, real ? C.b_ay : 0);
    cp_async16(d + A_AZ * Ctx<LN, TYE>::kArr, C.g_az + q * C.s_c, face ? C.b_co : 0);
    cp_async_commit();
}

template <int LN, int TYE> __device__ __forceinline__ double2 ld2(const unsigned char* stage_slot, int arr, int dy, int dl)
{
    return *reinterpret_cast<const double2*>(stage_slot + arr * Ctx<LN, TYE>::kArr + dy * Ctx<LN, TYE>::kRow + dl * 16);
}
template <int LN, int TYE, bool X> __device__ __forceinline__ double ld1(const unsigned char* stage_slot, int arr, int dy, int dl)
{
    return *reinterpret_cast<const double*>(stage_slot + arr * Ctx<LN, TYE>::kArr + dy * Ctx<LN, TYE>::kRow + dl * 16 + (X ? 0 : 8));
}

// One marching step at plane k.  REDX: the x-column of the pair is red in plane k.
// CUR receives the coefficients of plane k, PRV holds those of plane k-1.
// NORM: also fold |rhs - L phi_in| of the red cells it updates into *vmax (the residual of the sweep's
// INPUT at red cells costs two extra operations because `off` and `dg` are at hand).
template <int LN, int TYE, bool REDX, bool NORM = false>
__device__ __forceinline__ void step(const Ctx<LN, TYE>& C, unsigned char* s0, const unsigned char* sm,
                                     const unsigned char* sp, bool do_red, bool do_black,
                                     double* __restrict__ out_km1, double2& qm2, double2& qm1,
                                     double2& qn, double2& azn, Coef& CUR, const Coef& PRV, double* vmax = nullptr)
{
    double2 q0 = qn;                                   // old phi of plane k (staged read of the last step)
    CUR.az = azn;
    qn = ld2<LN, TYE>(sp, A_PHI, 0, 0);                // old phi and low z faces of plane k+1
    azn = ld2<LN, TYE>(sp, A_AZ, 0, 0);
    CUR.ax = ld2<LN, TYE>(s0, A_AX, 0, 0);
    CUR.ax2 = ld1<LN, TYE, true>(s0, A_AX, 0, 1);
    CUR.ays = ld2<LN, TYE>(s0, A_AY, 0, 0);
    CUR.ayn = ld2<LN, TYE>(s0, A_AY, 1, 0);
    CUR.rhs = ld2<LN, TYE>(s0, A_RHS, 0, 0);
    if (do_red) {
        const double w_ = REDX ? ld1<LN, TYE, false>(s0, A_PHI, 0, -1) : q0.x;
        const double e_ = REDX ? q0.y : ld1<LN, TYE, true>(s0, A_PHI, 0, 1);
        const double s_ = ld1<LN, TYE, REDX>(s0, A_PHI, -1, 0);
        const double n_ = ld1<LN, TYE, REDX>(s0, A_PHI, 1, 0);
        const double d_ = pick<REDX>(qm1);
        const double u_ = pick<REDX>(qn);
        const double azu = pick<REDX>(azn);
        const double axw = REDX ? CUR.ax.x : CUR.ax.y, axe = REDX ? CUR.ax.y : CUR.ax2;
        const double ays = pick<REDX>(CUR.ays), ayn = pick<REDX>(CUR.ayn);
        const double azd = pick<REDX>(CUR.az);
        double a, dg;
        const double nv = gs_value(axw, axe, ays, ayn, azd, azu, pick<REDX>(CUR.rhs), w_, e_, s_, n_, d_, u_, a, dg);
        if (NORM && C.own) *vmax = nanmax(*vmax, fabs(fma(pick<REDX>(q0), dg, -a)));   // |rhs - (sum - phi_0 dg)|
        put<REDX>(q0, nv);
        *reinterpret_cast<double*>(s0 + A_PHI * Ctx<LN, TYE>::kArr + (REDX ? 0 : 8)) = nv;
    }
    if (do_black) {
        const double w_ = REDX ? ld1<LN, TYE, false>(sm, A_PHI, 0, -1) : qm1.x;
        const double e_ = REDX ? qm1.y : ld1<LN, TYE, true>(sm, A_PHI, 0, 1);
        const double s_ = ld1<LN, TYE, REDX>(sm, A_PHI, -1, 0);
        const double n_ = ld1<LN, TYE, REDX>(sm, A_PHI, 1, 0);
        const double d_ = pick<REDX>(qm2), u_ = pick<REDX>(q0);
        const double axw = REDX ? PRV.ax.x : PRV.ax.y, axe = REDX ? PRV.ax.y : PRV.ax2;
        const double ays = pick<REDX>(PRV.ays), ayn = pick<REDX>(PRV.ayn);
        const double azd = pick<REDX>(PRV.az), azu = pick<REDX>(CUR.az);
        double a, dg;
        put<REDX>(qm1, gs_value(axw, axe, ays, ayn, azd, azu, pick<REDX>(PRV.rhs), w_, e_, s_, n_, d_, u_, a, dg));
        store_images(reinterpret_cast<double2*>(out_km1), qm1, C.img_x, C.img_y);
    }
    qm2 = qm1;
    qm1 = q0;
}

template <int LN, int TYE, bool REDX0>
__device__ __forceinline__ void march(const Ctx<LN, TYE>& C, int ks, int k0, int k1, bool red_x_ok, bool red_y_ok,
                                      bool own, double* __restrict__ out, unsigned long long out_stride)
{
    double2 qm2 = make_double2(0.0, 0.0), qm1;
    Coef cA, cB;
    cB.ax = cB.ays = cB.ayn = cB.az = cB.rhs = qm2; cB.ax2 = 0.0;
    int sI = wrap(ks, kStages);                               // stage of plane k
    qm1 = ld2<LN, TYE>(C.smem_gen + wrap(ks - 1, kStages) * Ctx<LN, TYE>::kStage, A_PHI, 0, 0);
    double2 qn = ld2<LN, TYE>(C.smem_gen + sI * Ctx<LN, TYE>::kStage, A_PHI, 0, 0);
    double2 azn = ld2<LN, TYE>(C.smem_gen + sI * Ctx<LN, TYE>::kStage, A_AZ, 0, 0);
    // out points at plane ks-1 of the thread's own pair; advanced by one plane per step
#pragma unroll 1
    for (int k = ks; k <= k1; k += 2) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int kk = k + h;
            if (kk > k1) break;
            if (kk > ks) {
                cp_async_wait<1>();                               // plane kk+1 has landed (kk+2 may be in flight)
                __syncthreads();                                  // ... for every thread; step kk-1 is finished
            }
            int sM = sI - 1; if (sM < 0) sM += kStages;
            int sP = sI + 1; if (sP >= kStages) sP -= kStages;
            int sN = sI + 3; if (sN >= kStages) sN -= kStages;    // stage that plane kk-2 just vacated
            issue<LN, TYE>(C, kk + 3, sN);
            unsigned char* s0 = C.smem_gen + sI * Ctx<LN, TYE>::kStage;
            const unsigned char* sm = C.smem_gen + sM * Ctx<LN, TYE>::kStage;
            const unsigned char* sp = C.smem_gen + sP * Ctx<LN, TYE>::kStage;
            const bool k_real = C.perz || (kk >= 0 && kk < C.nz);
            const bool do_black = own && kk - 1 >= k0 && kk - 1 < k1;
            if (h == 0)
                step<LN, TYE, REDX0>(C, s0, sm, sp, k_real && (REDX0 ? red_x_ok : red_y_ok), do_black, out, qm2, qm1, qn, azn, cA, cB);
            else
                step<LN, TYE, !REDX0>(C, s0, sm, sp, k_real && (REDX0 ? red_y_ok : red_x_ok), do_black, out, qm2, qm1, qn, azn, cB, cA);
            out += out_stride;
            sI = sP;
        }
    }
}

template <int LN, int TYE, int MINB>
__global__ void __launch_bounds__(LN * TYE, MINB)
k_rbgs_fused(LevelDev L, const double* __restrict__ pin, double* __restrict__ pout, int zchunk)
{
    constexpr int TY = TYE - 4;
    constexpr int kLanes = LN, kTX = 2 * LN - 4;
    extern __shared__ __align__(128) unsigned char smem_raw[];

    // Logical row of this thread.  With LN = 16 a warp holds two rows; they must have the same
    // parity because the red/black role (and with it the code path around __syncthreads) depends on
    // the row parity and has to be warp-uniform: warp w of a group of 4 rows takes rows {w, w+2}.
    const int lane = threadIdx.x;
    const int ty = (LN == 32) ? (int)threadIdx.y
                              : 4 * ((int)threadIdx.y >> 2) + (((int)threadIdx.y >> 1) & 1) + 2 * ((int)threadIdx.y & 1);
    static_assert(LN == 32 || (LN == 16 && TYE % 4 == 0), "row mapping needs TYE % 4 == 0 for 16-lane rows");
    const int x0 = blockIdx.x * kTX, y0 = blockIdx.y * TY;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, L.nz);
    const int gi = x0 - 2 + 2 * lane, gj = y0 - 2 + ty;            // unwrapped pair origin / row
    const bool perx = L.bclo[0] == MAC_PERIODIC, pery = L.bclo[1] == MAC_PERIODIC;
    const int wi = perx ? wrap(gi, L.nx) : gi;
    const int wj = pery ? wrap(gj, L.ny) : gj;
    const bool x_ok = perx || (gi >= 0 && gi < L.nx), xf_ok = perx || (gi >= 0 && gi <= L.nx);
    const bool y_ok = pery || (gj >= 0 && gj < L.ny), yf_ok = pery || (gj >= 0 && gj <= L.ny);
    const bool col_ok = x_ok && y_ok;
    const bool row_red = ty >= 1 && ty <= TYE - 2;                  // rows where reds are (re)computed
    const bool own = col_ok && lane >= 1 && lane <= kLanes - 2 && ty >= 2 && ty <= TYE - 3 &&
                     gi >= 0 && gi < L.nx && gi < x0 + kTX && gj >= 0 && gj < L.ny && gj < y0 + TY;

    Ctx<LN, TYE> C;
    // (this kernel wraps by index and runs on levels without ghost columns / rows: cx == nx, ry == ny)
    const size_t lat = col_ok ? (size_t)wi + (size_t)L.nx * wj : 0;
    C.g_phi = reinterpret_cast<const unsigned char*>(pin + lat);
    C.g_rhs = reinterpret_cast<const unsigned char*>(L.rhs + lat);
    C.g_az = reinterpret_cast<const unsigned char*>(L.az + lat);
    // ax: faces gi, gi+1 of row gj; the pair at gi == nx (non-periodic) holds the high boundary face
    const bool ax_ok = xf_ok && y_ok && row_red;
    C.g_ax = reinterpret_cast<const unsigned char*>(L.ax + (ax_ok ? (size_t)wi + (size_t)L.px * wj : 0));
    // ay: low y faces of row gj (also the high faces of row gj-1); row gj == ny holds the boundary face
    const bool ay_ok = x_ok && yf_ok && ty >= 1;
    C.g_ay = reinterpret_cast<const unsigned char*>(L.ay + (ay_ok ? (size_t)wi + (size_t)L.nx * wj : 0));
    C.s_c = (unsigned long long)L.nx * L.ny * 8ull;
    C.s_ax = (unsigned long long)L.px * L.ny * 8ull;
    C.s_ay = (unsigned long long)L.nx * (L.ny + 1) * 8ull;
    C.b_phi = col_ok ? 16 : 0;
    C.b_co = (col_ok && row_red) ? 16 : 0;
    C.b_ay = ay_ok ? 16 : 0;
    C.b_ax = ax_ok ? 16 : 0;
    C.nz = L.nz;
    C.perz = L.bclo[2] == MAC_PERIODIC;
    C.img_x = C.img_y = 0;
    C.own = own;
    const unsigned slot = (ty * kLanes + lane) * 16;
    C.smem_gen = smem_raw + slot;
    C.smem_u32 = (unsigned)__cvta_generic_to_shared(smem_raw) + slot;

    const int ks = k0 - 1;                                          // first step: red plane k0-1
    for (int p = ks - 1; p <= ks + 2; ++p) issue<LN, TYE>(C, p, wrap(p, kStages));
    cp_async_wait<1>();                                             // planes ks-1, ks, ks+1 have landed
    __syncthreads();

    const bool red_x_ok = col_ok && row_red && lane >= 1;           // x column is in the red region
    const bool red_y_ok = col_ok && row_red && lane <= kLanes - 2;
    double* out = pout + ((size_t)wi + (size_t)L.nx * (own ? wj : 0)) + (long long)(ks - 1) * (long long)((size_t)L.nx * L.ny);
    const unsigned long long ostride = (unsigned long long)L.nx * L.ny;
    if (((gj + ks) & 1) == 0)
        march<LN, TYE, true>(C, ks, k0, k1, red_x_ok, red_y_ok, own, out, ostride);
    else
        march<LN, TYE, false>(C, ks, k0, k1, red_x_ok, red_y_ok, own, out, ostride);
    cp_async_wait<0>();
}

template <int LN, int TYE> constexpr size_t smem_bytes() { return (size_t)Ctx<LN, TYE>::kStage * kStages; }

}  // namespace fused

static inline bool fused_sweep_supported(const LevelDev& L)
{
    return (L.nx % 2) == 0 && L.nx >= 2 && L.gx == 0 && L.gy == 0;
}

// Tile configurations: <pairs per row, rows incl. halo, min CTAs per SM>.
//   big  : 32 columns x 16 rows (28 x 12 interior), 256 threads, 100 KB of stages -> 2 CTAs per SM,
//          whose barrier phases interleave (one CTA loads shared memory while the other divides).
//   small: for levels with ny <= 8.
#define MAC_FUSED_BIG   16, 16, 2
#define MAC_FUSED_SMALL 16, 8, 2

static inline int smoother_configure()
{
    using namespace fused;
    if (cudaFuncSetAttribute(k_rbgs_fused<MAC_FUSED_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<16, 16>()) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_rbgs_fused<MAC_FUSED_SMALL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<16, 8>()) != cudaSuccess) return -1;
    return 0;
}

// One fused sweep: reads phi_in, writes phi_out (distinct buffers).
static inline int launch_fused_sweep(const double* phi_in, double* phi_out, const LevelDev& L, int sms, cudaStream_t s)
{
    using namespace fused;
    constexpr int LN = 16, kTX = 2 * LN - 4;
    const int tiles_x = (L.nx + kTX - 1) / kTX;
    const bool small = L.ny <= 8;
    const int TY = small ? 4 : 12;
    const int tiles_y = (L.ny + TY - 1) / TY;
    // enough z-chunks for a few CTAs per SM, but chunks of at least 16 planes (each chunk recomputes
    // 2 red planes and restages 4)
    const int tiles = tiles_x * tiles_y;
    int nchunk = (8 * sms + tiles - 1) / tiles;
    int maxchunk = (L.nz + 15) / 16;
    if (nchunk > maxchunk) nchunk = maxchunk;
    if (nchunk < 1) nchunk = 1;
    const int zchunk = (L.nz + nchunk - 1) / nchunk;
    nchunk = (L.nz + zchunk - 1) / zchunk;
    dim3 grid(tiles_x, tiles_y, nchunk);
    if (small)
        k_rbgs_fused<MAC_FUSED_SMALL><<<grid, dim3(LN, 8), smem_bytes<16, 8>(), s>>>(L, phi_in, phi_out, zchunk);
    else
        k_rbgs_fused<MAC_FUSED_BIG><<<grid, dim3(LN, 16), smem_bytes<16, 16>(), s>>>(L, phi_in, phi_out, zchunk);
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}
