// mac_smoother_t2.cuh -- TWO red-black Gauss-Seidel sweeps in ONE pass over HBM (temporal blocking
// of the smoother).
//
// One launch reads phi, rhs, ax, ay, az once and writes phi once (48 B/cell) and applies
//      red, black, red, black
// i.e. exactly the nu = 2 sweeps of a V(2,2) cycle.  The result is bit-identical to two launches of
// tma::k_rbgs_tma (same expressions, same order within an update).
//
// Scheme.  The single-sweep kernel marches upward in z with a one-plane lag (red of plane k, black of
// plane k-1).  Here the march carries FOUR half-sweeps with a three-plane lag: at step k a thread
// updates, on its own pair of columns,
//      (1) sweep 1 red   of plane k      (old black neighbours:         planes k-1, k,   k+1)
//      (2) sweep 1 black of plane k-1    (sweep-1 red neighbours:       planes k-2, k-1, k  )
//      (3) sweep 2 red   of plane k-2    (sweep-1 black neighbours:     planes k-3, k-2, k-1)
//      (4) sweep 2 black of plane k-3    (sweep-2 red neighbours:       planes k-4, k-3, k-2)
// and stores plane k-3.  All four updates hit the SAME column of the pair (the colour of a column
// alternates from plane to plane), vertical neighbours are the thread's own registers, lateral
// neighbours are values other threads produced ONE STEP EARLIER (exchange buffers, see "Memory"):
// the only cross-thread dependences are lateral and one step old, hence one __syncthreads per plane.
//
// Lateral halo: every half-sweep consumes one ring of cells, so a tile of 32 x 24 staged cells yields
// 24 x 16 finished ones (halo 4); the halo cells are recomputed redundantly by the neighbouring CTA
// (their HBM reads hit L2).  In z a chunk [k0, k1) redoes 6 planes.
//
// Memory.  Shared memory holds two TMA-fed rings (cp.async.bulk.tensor.3d + mbarrier, as in
// mac_smoother_tma.cuh) of 4 stages each -- phi (6 KB per plane: the OLD values, read by half-sweep (1)
// and for the plane above) and coefficients (24 KB per plane, consumed into registers, where the four
// coefficient sets of planes k .. k-3 rotate) -- and six small EXCHANGE buffers: the values a half-sweep
// produces are what the next half-sweep of the neighbouring threads reads one step later, so each thread
// writes its new value into a compact, colour-split plane (one double per pair: in a given row and plane
// all updated cells are the same column of their pairs) that is double-buffered by step parity.  Those
// reads and writes are 8-byte accesses at an 8-byte pitch (conflict-free), whereas the staged phi planes
// interleave the two colours at a 16-byte pitch (two-way bank conflicts).  The march is unrolled four-fold
// so that every shared-memory offset is a compile-time constant and nothing is moved between registers.
// All updates are computed unconditionally and selected by masks (no divergent branches around the
// dependent chain of four updates); every shared-memory read of a step precedes its writes.
#pragma once
#include <climits>

#include "mac_smoother_tma.cuh"

namespace t2 {

using fused::pick; using fused::put;
using tma::mbar_init; using tma::mbar_expect_tx; using tma::mbar_wait; using tma::tma_load_3d; using tma::smem_u32;

#ifndef MAC_T2_TYE
#define MAC_T2_TYE 24                                // thread rows of a tile (a multiple of 4)
#endif
constexpr int LN = 16, TYE = MAC_T2_TYE, NT = LN * TYE;   // 16 pairs x 24 rows = 384 threads: the COMPUTED cells (32 x 24)
constexpr int HALO = 4;                              // cells a finished cell depends on laterally (periodic image width)
// Only three of the four rings around a finished cell are COMPUTED (sweep-1 red / black, sweep-2 red); the fourth is
// the old black value that sweep-1 red reads.  So the staged phi box is one cell wider than the computed tile on every
// side (two in x, to keep box origins even: 16-byte aligned rows) and has no threads of its own, and a tile finishes
// the computed cells that are >= 3 cells inside: 26 columns (x0-1 .. x0+24 for computed x0-4 .. x0+27) x 18 rows.
constexpr int CH = 3;                                // computed rings
constexpr int kTX = 2 * LN - 2 * CH;                 // 26 finished columns per tile: [x0 - 1, x0 + 25)
constexpr int kTY = TYE - 2 * CH;                    // 18 finished rows per tile:    [y0, y0 + 18), thread row ty is row y0 - 3 + ty
constexpr int SX = 2 * LN + 4, SY = TYE + 2;         // staged phi box: columns x0-6 .. x0+29, rows y0-4 .. y0+21
constexpr int AXW = 2 * LN + 2;                      // staged ax box: faces x0-4 .. x0+29 (x0+28 is the last one read)
constexpr int kRowP = SX * 8;                        // bytes of one staged phi row
constexpr int kPlP = ((SY * kRowP + 127) / 128) * 128;   // bytes of one phi stage (128-byte multiple: TMA destinations)
constexpr int kRow = LN * 16;                        // bytes of one staged row of ay, az, rhs (the computed columns)
constexpr int kRowA = AXW * 8;                       // bytes of one staged row of ax
constexpr int kPad = 512;                            // readable slack below the phi ring
// one coefficient stage: ax (TYE rows), ay (TYE + 1 face rows), az, rhs (TYE rows); every array starts 128-byte aligned
constexpr int O_AX = 0, O_AY = O_AX + TYE * kRowA, O_AZ = O_AY + (TYE + 1) * kRow, O_RHS = O_AZ + TYE * kRow;
constexpr int kCoefStage = O_RHS + TYE * kRow;
static_assert(O_AY % 128 == 0 && O_AZ % 128 == 0 && O_RHS % 128 == 0 && kCoefStage % 128 == 0, "TMA destinations are 128-byte aligned");
constexpr int kExRow = LN * 8;                       // exchange plane: one double per pair, TYE + 2 rows (a pad row each side)
constexpr int kEx = (TYE + 2) * kExRow;
enum { EX_RA = 0, EX_BA = 2, EX_RB = 4 };            // sweep-1 red, sweep-1 black, sweep-2 red; two buffers each

template <int LA>
struct Cfg {
    static constexpr int NP = LA + 2, NC = LA + 2;   // planes k, k+1 resident + LA in flight
    static constexpr int kCoef = kCoefStage;
    static constexpr unsigned kTx = (unsigned)(SY * kRowP + kCoefStage);   // bytes landing per plane
    static constexpr size_t kSmem = (size_t)kPad + (size_t)NP * kPlP + (size_t)NC * kCoef + 6 * kEx + 8 * NP + 128;
};

__device__ __forceinline__ double2 ldp(const unsigned char* p) { return *reinterpret_cast<const double2*>(p); }
template <bool X> __device__ __forceinline__ double ldc(const unsigned char* p, int dy, int dl)
{
    return *reinterpret_cast<const double*>(p + dy * kRowP + dl * 16 + (X ? 0 : 8));
}

// 24-row tiles keep the reciprocal diagonals of sweep 1 for sweep 2 (16 registers); taller tiles (more threads, fewer
// registers each) form them again
constexpr bool kKeepRdg = TYE <= 24;

struct Coef {                                // coefficients of one plane for a column pair, in registers, and the
    double2 ax; double ax2; double2 ays, ayn, az, rhs;   // reciprocals of the two diagonals, which sweep 1 computes
    double2 rdg;                             // and sweep 2 reuses (same coefficients, two steps later)
};

// One bit per lateral condition, kept in ONE register that the compiler cannot rematerialise from (lane, row): each
// update is then selected by a single bit test (the flags as separate bools were recomputed every step as chains of
// five dependent selects on the critical path).
enum { F_RA = 1, F_BA_X = 2, F_BA_Y = 4, F_RB = 8, F_OWN_X = 16, F_OWN_Y = 32, F_IMG = 64 };

struct Th {                                  // per-thread constants
    unsigned char* base;                     // start of the phi ring (CTA-uniform); the own slots are 32-bit offsets from it,
    unsigned o_phi, o_cf, o_ax, o_ex;        // opaque to the compiler (else it recomputes them from (lane, row) every step):
                                             // phi stage 0, coefficient stage 0 (32-column arrays: add O_AY, O_AZ, O_RHS),
                                             // coefficient stage 0 array ax, exchange buffer 0
    __device__ __forceinline__ unsigned char* phi0() const { return base + o_phi; }
    __device__ __forceinline__ const unsigned char* coef0() const { return base + o_cf; }
    __device__ __forceinline__ const unsigned char* cax0() const { return base + o_ax; }
    __device__ __forceinline__ unsigned char* ex0() const { return base + o_ex; }
    unsigned fl;                             // lateral validity of the four half-sweeps (F_* bits; x / y cell of the pair)
    int img_x, img_y;                        // periodic images of the own pair (0 = none; F_IMG set iff one is not)
    // half-sweep h is applied at step kk iff (unsigned)(kk - lo[h]) <= span[h]: the planes it is wanted on
    // (sweep-1 red [k0-3, k1+2], black [k0-2, k1+1], sweep-2 red [k0-1, k1], black [k0, k1-1]) that exist
    int lo[4];
    unsigned span[4];
    int nlo; unsigned nspan;                 // NORM: planes [k0, k1)
};

// the three lateral neighbours of column X of the pair that other threads own, from a plane's phi stage
struct Lat { double we, s, n; };
template <bool X> __device__ __forceinline__ Lat lat_load(const unsigned char* ph)
{
    Lat l;
    l.we = X ? ldc<false>(ph, 0, -1) : ldc<true>(ph, 0, 1);     // west of the x cell / east of the y cell
    l.s = ldc<X>(ph, -1, 0);
    l.n = ldc<X>(ph, 1, 0);
    return l;
}

// the same three neighbours from an exchange plane (own element pointer): one double per pair
template <bool X> __device__ __forceinline__ Lat lat_ex(const unsigned char* pe)
{
    Lat l;
    l.we = *reinterpret_cast<const double*>(pe + (X ? -8 : 8));
    l.s = *reinterpret_cast<const double*>(pe - kExRow);
    l.n = *reinterpret_cast<const double*>(pe + kExRow);
    return l;
}

// Gauss-Seidel update of column X of the pair in one plane.  l: lateral neighbours, other: the pair's other cell,
// C: the plane's coefficients, az_up: low z faces of the plane above, d_ / u_: vertical neighbours (u_ is on the
// dependent chain, see fused::gs_value, whose arithmetic this is).  FIRST: sweep 1 forms the reciprocal of the
// diagonal (seed + 2 Newton steps) and leaves it in C.rdg; sweep 2 meets the same diagonal and reuses it.
template <bool X, bool FIRST>
__device__ __forceinline__ double gs_cell(const Lat& l, double other, Coef& C, const double2& az_up,
                                          double d_, double u_, double& a, double& dg)
{
    const double axw = X ? C.ax.x : C.ax.y, axe = X ? C.ax.y : C.ax2;
    const double ays = pick<X>(C.ays), ayn = pick<X>(C.ayn), azd = pick<X>(C.az), azu = pick<X>(az_up);
    const double w_ = X ? l.we : other, e_ = X ? other : l.we;
    const double t = (fma(axe, e_, axw * w_) + fma(ayn, l.n, ays * l.s)) + fma(azd, d_, -pick<X>(C.rhs));
    a = fma(azu, u_, t);
    double r;
    if (FIRST) {
        dg = ((axw + axe) + (ays + ayn)) + (azd + azu);
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(dg));
        r = fma(fma(-dg, r, 1.0), r, r);
        r = fma(fma(-dg, r, 1.0), r, r);
        if (kKeepRdg) put<X>(C.rdg, r);
    } else {
        r = pick<X>(C.rdg);
    }
    return a * r;
}

// issue the five box loads of plane p (unwrapped) into the phi stage at byte offset op / coefficient stage at oc
template <int LA>
__device__ __forceinline__ void issue_plane(const CUtensorMap* tm_phi, const CUtensorMap* tm_rhs, const CUtensorMap* tm_ax,
                                            const CUtensorMap* tm_ay, const CUtensorMap* tm_az, unsigned phi_ring,
                                            unsigned coef_ring, unsigned bar0, unsigned op, unsigned oc, int p, int nz,
                                            bool perz, int cx, int cy)
{
    using G = Cfg<LA>;
    if (perz) { if (p < 0) p += nz; else if (p >= nz) p -= nz; }
    const unsigned dp = phi_ring + op;
    const unsigned dc = coef_ring + oc;
    const unsigned bar = bar0 + op / (kPlP / 8);                               // barrier of phi stage op / kPlP
    mbar_expect_tx(bar, G::kTx);
    tma_load_3d(dp, tm_phi, bar, cx - 2, cy - 1, p);                           // SX x SY: one more ring (two columns in x)
    tma_load_3d(dc + O_RHS, tm_rhs, bar, cx, cy, p);                           // the computed cells
    tma_load_3d(dc + O_AX, tm_ax, bar, cx, cy, p);                             // AXW faces a row
    tma_load_3d(dc + O_AZ, tm_az, bar, cx, cy, p);
    tma_load_3d(dc + O_AY, tm_ay, bar, cx, cy, p);                             // TYE + 1 face rows
}

// One marching step at plane kk; X: the x column of the pair is red in plane kk; W: exchange buffers written by this
// step (the other ones, written by the previous step, are read).
// CUR receives the coefficients of plane kk; S1, S2, S3 hold those of planes kk-1, kk-2, kk-3.
template <bool X, int W, bool NORM>
__device__ __forceinline__ void step(const Th& T, int kk, const unsigned char* s0, const unsigned char* sP,
                                     const unsigned char* cI, const unsigned char* cP, const unsigned char* aI,
                                     double* __restrict__ out,
                                     double2& Pn, double2& Pm1, double2& Pm2, double2& Pm3, double2& Pm4, double2& azn,
                                     Coef& CUR, Coef& S1, Coef& S2, Coef& S3, double& vmax, bool& vnan)
{
    constexpr int R = 1 - W;
    unsigned fl = T.fl;
    asm volatile("" : "+r"(fl));                      // (keeps the bit tests from being hoisted into one register each)
    const bool v0 = (unsigned)(kk - T.lo[0]) <= T.span[0], v1 = (unsigned)(kk - T.lo[1]) <= T.span[1];
    const bool v2 = (unsigned)(kk - T.lo[2]) <= T.span[2], v3 = (unsigned)(kk - T.lo[3]) <= T.span[3];
    double2 P0 = Pn;                                  // old phi of plane kk (staged read of the last step)
    CUR.az = azn;
    Pn = ldp(sP);                                     // old phi and low z faces of plane kk+1
    azn = ldp(cP + O_AZ);
    CUR.ax = ldp(aI);
    CUR.ax2 = *reinterpret_cast<const double*>(aI + 16);
    CUR.ays = ldp(cI + O_AY);
    CUR.ayn = ldp(cI + O_AY + kRow);
    CUR.rhs = ldp(cI + O_RHS);
    const Lat l0 = lat_load<X>(s0);                                   // old black neighbours in plane kk
    const Lat l1 = lat_ex<X>(T.ex0() + (EX_RA + R) * kEx);              // sweep-1 red neighbours in plane kk-1
    const Lat l2 = lat_ex<X>(T.ex0() + (EX_BA + R) * kEx);              // sweep-1 black neighbours in plane kk-2
    const Lat l3 = lat_ex<X>(T.ex0() + (EX_RB + R) * kEx);              // sweep-2 red neighbours in plane kk-3
    double a, dg;
    // (1) sweep 1, red cells of plane kk
    const double n0 = gs_cell<X, true>(l0, pick<!X>(P0), CUR, azn, pick<X>(Pm1), pick<X>(Pn), a, dg);
    if (NORM) {                                       // |rhs - (sum - phi_0 dg)| of the input; a NaN sets the sign of vmax
        const double rr = fabs(fma(pick<X>(P0), dg, -a));
        const bool on = (fl & (X ? F_OWN_X : F_OWN_Y)) && (unsigned)(kk - T.nlo) <= T.nspan;
        vmax = fmax(vmax, on ? rr : 0.0);             // (fmax drops NaNs: they are recorded separately)
        vnan = vnan || (on && rr != rr);
    }
    put<X>(P0, ((fl & F_RA) && v0) ? n0 : pick<X>(P0));
    // (2) sweep 1, black cells of plane kk-1
    const double n1 = gs_cell<X, true>(l1, pick<!X>(Pm1), S1, CUR.az, pick<X>(Pm2), pick<X>(P0), a, dg);
    put<X>(Pm1, ((fl & (X ? F_BA_X : F_BA_Y)) && v1) ? n1 : pick<X>(Pm1));
    // (3) sweep 2, red cells of plane kk-2
    const double n2 = gs_cell<X, !kKeepRdg>(l2, pick<!X>(Pm2), S2, S1.az, pick<X>(Pm3), pick<X>(Pm1), a, dg);
    put<X>(Pm2, ((fl & F_RB) && v2) ? n2 : pick<X>(Pm2));
    // (4) sweep 2, black cells of plane kk-3; the plane is finished
    const double n3 = gs_cell<X, !kKeepRdg>(l3, pick<!X>(Pm3), S3, S2.az, pick<X>(Pm4), pick<X>(Pm2), a, dg);
    *reinterpret_cast<double*>(T.ex0() + (EX_RA + W) * kEx) = pick<X>(P0);
    *reinterpret_cast<double*>(T.ex0() + (EX_BA + W) * kEx) = pick<X>(Pm1);
    *reinterpret_cast<double*>(T.ex0() + (EX_RB + W) * kEx) = pick<X>(Pm2);
    put<X>(Pm3, ((fl & (X ? F_OWN_X : F_OWN_Y)) && v3) ? n3 : pick<X>(Pm3));
    if (v3) {                                         // plane kk-3 leaves: the owned cells of the pair (predicated stores)
        if (fl & F_OWN_X) out[0] = Pm3.x;
        if (fl & F_OWN_Y) out[1] = Pm3.y;
        if (fl & F_IMG) {                           // periodic levels, tiles at the domain edge
            const long long dx = T.img_x, dy = T.img_y;
            if (fl & F_OWN_X) { if (dx) out[dx] = Pm3.x; if (dy) { out[dy] = Pm3.x; if (dx) out[dx + dy] = Pm3.x; } }
            if (fl & F_OWN_Y) { if (dx) out[dx + 1] = Pm3.y; if (dy) { out[dy + 1] = Pm3.y; if (dx) out[dx + dy + 1] = Pm3.y; } }
        }
    }
    Pm4 = Pm3; Pm3 = Pm2; Pm2 = Pm1; Pm1 = P0;
}

// Step J (0 .. 3) of the four-fold unrolled march (the unrolling keeps the four rotating coefficient sets in fixed
// registers).  Plane kk sits in stage s0 of both rings, plane kk+1 in the next one; the rings have NS = LA + 2 stages, so
// their period is independent of the unrolling and the stage offsets are runtime values (two integer operations a step).
template <int LA, int J, bool X, bool NORM>
__device__ __forceinline__ void stage(const Th& T, int kk, int ke, unsigned& s0, unsigned& phase, const CUtensorMap* tm_phi,
                                      const CUtensorMap* tm_rhs, const CUtensorMap* tm_ax, const CUtensorMap* tm_ay,
                                      const CUtensorMap* tm_az, unsigned phi_ring, unsigned coef_ring, unsigned bar0,
                                      bool producer, int cx, int cy, int nz, bool perz, double* __restrict__ out,
                                      double2& Pn, double2& Pm1, double2& Pm2, double2& Pm3, double2& Pm4, double2& azn,
                                      Coef& CUR, Coef& S1, Coef& S2, Coef& S3, double& vmax, bool& vnan)
{
    using G = Cfg<LA>;
    constexpr unsigned NS = G::NP;
    static_assert(G::NP == G::NC, "both rings have the same depth");
    const unsigned sP = s0 + 1 == NS ? 0u : s0 + 1;            // stage of plane kk+1
    const unsigned sN = s0 == 0 ? NS - 1 : s0 - 1;             // stage plane kk-1 vacated: receives plane kk+1+LA
    // plane kk+1 has landed: a barrier is reused every NS steps, its parity flips with every reuse
    mbar_wait(bar0 + 8 * sP, (phase >> sP) & 1u);
    phase ^= 1u << sP;
    __syncthreads();                                           // every thread has finished step kk-1
    if (producer && kk + 1 + LA <= ke + 1) {                   // never leave a load in flight at exit
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        issue_plane<LA>(tm_phi, tm_rhs, tm_ax, tm_ay, tm_az, phi_ring, coef_ring, bar0, sN * kPlP, sN * G::kCoef,
                        kk + 1 + LA, nz, perz, cx, cy);
    }
    step<X, J & 1, NORM>(T, kk, T.phi0() + s0 * kPlP, T.phi0() + sP * kPlP, T.coef0() + s0 * G::kCoef, T.coef0() + sP * G::kCoef,
                         T.cax0() + s0 * G::kCoef, out, Pn, Pm1, Pm2, Pm3, Pm4, azn, CUR, S1, S2, S3, vmax, vnan);
    s0 = sP;
}

template <int LA, bool REDX0, bool NORM>
__device__ __forceinline__ void march(const Th& T, int ks, int ke, const CUtensorMap* tm_phi, const CUtensorMap* tm_rhs,
                                      const CUtensorMap* tm_ax, const CUtensorMap* tm_ay, const CUtensorMap* tm_az,
                                      unsigned phi_ring, unsigned coef_ring, unsigned bar0, bool producer, int cx, int cy,
                                      int nz, bool perz, double* __restrict__ out, unsigned long long out_stride, double& vmax, bool& vnan)
{
    using G = Cfg<LA>;
    const double2 z2 = make_double2(0.0, 0.0);
    double2 Pm1, Pm2 = z2, Pm3 = z2, Pm4 = z2;
    Coef cA, cB, cC, cD;
    cB.ax = cB.ays = cB.ayn = cB.az = cB.rhs = cB.rdg = z2; cB.ax2 = 0.0;
    cC = cB; cD = cB;
    // the prologue issued planes ks-1 .. ks+LA into stages 0 .. LA+1 of both rings (phase 0 of their barriers)
    mbar_wait(bar0 + 0, 0);
    mbar_wait(bar0 + 8, 0);
    Pm1 = ldp(T.phi0());
    double2 Pn = ldp(T.phi0() + kPlP);
    double2 azn = ldp(T.coef0() + G::kCoef + O_AZ);
    unsigned s0 = 1, phase = 3u;                               // plane ks sits in stage 1; stages 0 and 1 have completed phase 0
#define MAC_T2_STAGE(J, XX, CUR, S1, S2, S3)                                                                          \
    if (kk > ke) break;                                                                                               \
    stage<LA, J, XX, NORM>(T, kk, ke, s0, phase, tm_phi, tm_rhs, tm_ax, tm_ay, tm_az, phi_ring, coef_ring, bar0, producer,  \
                           cx, cy, nz, perz, out, Pn, Pm1, Pm2, Pm3, Pm4, azn, CUR, S1, S2, S3, vmax, vnan);                \
    out += out_stride; ++kk;
#pragma unroll 1
    for (int kk = ks; kk <= ke;) {
        MAC_T2_STAGE(0, REDX0, cA, cD, cC, cB)
        MAC_T2_STAGE(1, !REDX0, cB, cA, cD, cC)
        MAC_T2_STAGE(2, REDX0, cC, cB, cA, cD)
        MAC_T2_STAGE(3, !REDX0, cD, cC, cB, cA)
    }
#undef MAC_T2_STAGE
}

// Work decomposition of one launch (host: t2_plan).  704 tiles on 148 SMs are 4.76 waves of whole columns: the
// first nfull tiles (whole waves) march all of z, the remaining tiles are cut into nsplit z-chunks each so that the
// last, partial wave is spread over every SM.  nfull = 0: every tile is cut into nsplit chunks.
struct T2Plan { int tiles_x, tiles, nfull, nsplit, zchunk, ncta, images; };   // images: the kernel stores the periodic images of phi itself

// NORM: additionally writes, per CTA, max |rhs - L phi_in| over the red cells to part_max[linear CTA index]
template <int LA, bool NORM>
__global__ void __launch_bounds__(NT, 1)
k_rbgs_t2(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_rhs,
          const __grid_constant__ CUtensorMap tm_ax, const __grid_constant__ CUtensorMap tm_ay,
          const __grid_constant__ CUtensorMap tm_az, LevelDev L, double* __restrict__ pout, T2Plan plan,
          double* __restrict__ part_max)
{
    using G = Cfg<LA>;
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    unsigned char* smem_raw = smem_dyn + ((128u - (smem_u32(smem_dyn) & 127u)) & 127u);
    unsigned char* phi_gen = smem_raw + kPad;
    const unsigned phi_ring = smem_u32(phi_gen);
    const unsigned coef_ring = phi_ring + G::NP * kPlP;
    const unsigned bar0 = coef_ring + G::NC * G::kCoef + 6 * kEx;     // (the exchange buffers sit between the rings and the barriers)

    const int lane = threadIdx.x;
    // a warp holds two rows; they must share their parity (the colour role is warp-uniform)
    const int ty = 4 * ((int)threadIdx.y >> 2) + (((int)threadIdx.y >> 1) & 1) + 2 * ((int)threadIdx.y & 1);
    // linear CTA index -> (tile, z range): the first plan.nfull tiles march the whole column, the others a chunk each
    int tile = blockIdx.x, k0 = 0, k1 = L.nz;
    if (tile >= plan.nfull) {
        const int q = tile - plan.nfull, rem = plan.tiles - plan.nfull, c = q / rem;
        tile = plan.nfull + (q - c * rem);
        k0 = c * plan.zchunk;
        k1 = min(k0 + plan.zchunk, L.nz);
    }
    const int tyi = tile / plan.tiles_x;
    const int x0 = (tile - tyi * plan.tiles_x) * kTX, y0 = tyi * kTY;   // finished cells: [x0 - 1, x0 + 25) x [y0, y0 + 18)
    const int gi = x0 - HALO + 2 * lane, gj = y0 - CH + ty;             // x cell of the own pair (gi is even), own row
    // ghost columns / rows of a periodic level hold valid images: they are recomputed like any halo cell
    const bool col_ok = gi >= -L.gx && gi < L.nx + L.gx && gj >= -L.gy && gj < L.ny + L.gy;
    const bool producer = threadIdx.x == 0 && threadIdx.y == 0;

    // validity by distance from the edge of the computed tile: sweep-1 red everywhere (it reads the staged ring), then
    // one ring less per half-sweep; columns x0-4 (x cell of lane 0) and x0+27 (y cell of lane 15) are the outermost
    Th T;
    const bool in_y = ty >= 1 && ty <= TYE - 2, own_row = ty >= CH && ty <= TYE - 1 - CH && gj < L.ny && gi >= 0 && gi < L.nx;
    T.img_x = own_row ? (int)image_dx(L, gi) : 0;     // (a pair lies inside or outside the domain as a whole; one plane of a
    T.img_y = own_row ? (int)image_dy(L, gj) : 0;     // level has fewer than 2^31 cells: t2_level_ok)
    unsigned fl = 0;
    if (col_ok) {
        fl = F_RA | (in_y && lane >= 1 ? F_BA_X : 0) | (in_y && lane <= LN - 2 ? F_BA_Y : 0) |
             (ty >= 2 && ty <= TYE - 3 && lane >= 1 && lane <= LN - 2 ? F_RB : 0) |
             (own_row && lane >= 2 && lane <= LN - 2 ? F_OWN_X : 0) | (own_row && lane >= 1 && lane <= LN - 3 ? F_OWN_Y : 0);
        if (plan.images && (fl & (F_OWN_X | F_OWN_Y)) && (T.img_x | T.img_y)) fl |= F_IMG;
    }
    asm volatile("" : "+r"(fl));                      // opaque: keep the bits, do not recompute the conditions per step
    T.fl = fl;
    const bool perz = L.bclo[2] == MAC_PERIODIC;
    {
        const int wl[4] = {k0 - 3, k0 - 2, k0 - 1, k0}, wh[4] = {k1 + 2, k1 + 1, k1, k1 - 1};
        for (int h = 0; h < 4; ++h) {                  // half-sweep h acts on plane kk - h
            const int lo = perz ? wl[h] : max(wl[h], 0), hi = perz ? wh[h] : min(wh[h], L.nz - 1);
            T.lo[h] = lo + h;
            T.span[h] = hi >= lo ? (unsigned)(hi - lo) : 0u;
            if (hi < lo) T.lo[h] = INT_MIN / 2;        // never
        }
        T.nlo = k0;
        T.nspan = (unsigned)(k1 - 1 - k0);
    }
    T.base = phi_gen;
    T.o_phi = (ty + 1) * kRowP + 16 + lane * 16;                  // the box starts one row and two columns before the computed tile
    T.o_cf = G::NP * kPlP + ty * kRow + lane * 16;
    T.o_ax = G::NP * kPlP + O_AX + ty * kRowA + lane * 16;
    T.o_ex = G::NP * kPlP + G::NC * G::kCoef + ((ty + 1) * LN + lane) * 8;
    asm volatile("" : "+r"(T.o_phi), "+r"(T.o_cf), "+r"(T.o_ax), "+r"(T.o_ex));
    const int cx0 = x0 - HALO + L.gx, cy0 = y0 - CH + L.gy;       // tensor-map coordinates of the computed tile's origin

    const int ks = k0 - 3;
    if (producer) {
        for (int s = 0; s < G::NP; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        for (int q = 0; q < LA + 2 && ks - 1 + q <= k1 + 3; ++q)
            issue_plane<LA>(&tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, phi_ring, coef_ring, bar0, q * kPlP, q * G::kCoef, ks - 1 + q, L.nz,
                            perz, cx0, cy0);
    }
    __syncthreads();                                             // barrier inits visible before anyone waits

    const unsigned long long ostride = (unsigned long long)L.cx * L.ry;
    double* out = pout + (own_row ? (long long)gi + (long long)L.cx * gj : 0) + (long long)(ks - 3) * (long long)ostride;
    double vmax = 0.0;
    bool vnan = false;
    if (((gj + ks) & 1) == 0)
        march<LA, true, NORM>(T, ks, k1 + 2, &tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, phi_ring, coef_ring, bar0, producer, cx0, cy0, L.nz, perz, out, ostride, vmax, vnan);
    else
        march<LA, false, NORM>(T, ks, k1 + 2, &tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, phi_ring, coef_ring, bar0, producer, cx0, cy0, L.nz, perz, out, ostride, vmax, vnan);
    // every plane that was issued (<= k1 + 3) has been waited for by the last step: nothing is in flight
    if (NORM) {
        __shared__ double sh_max[32];
        const int tid = threadIdx.x + LN * threadIdx.y;
        if (vnan) vmax = __longlong_as_double(0x7ff8000000000000ll);
        vmax = warp_nanmax(vmax);
        if ((tid & 31) == 0) sh_max[tid >> 5] = vmax;
        __syncthreads();
        if (tid == 0) {
            double m = sh_max[0];
            for (int q = 1; q < NT / 32; ++q) m = nanmax(m, sh_max[q]);
            part_max[blockIdx.x] = m;
        }
    }
}

}  // namespace t2

// ---- host side ---------------------------------------------------------------------------------

#ifndef MAC_T2_IMAGES_BELOW
#define MAC_T2_IMAGES_BELOW (1ll << 18)   // cells of a level below which the two-sweep kernel stores the periodic images itself
#endif
#ifndef MAC_T2_LA
#define MAC_T2_LA 2                   // planes of TMA lookahead (4 stages per ring)
#endif

static inline int t2_smoother_configure()
{
    using namespace t2;
    const int sm = (int)Cfg<MAC_T2_LA>::kSmem;
    if (cudaFuncSetAttribute(k_rbgs_t2<MAC_T2_LA, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_rbgs_t2<MAC_T2_LA, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
    return 0;
}

// Tensor maps of the two-sweep kernel (Level::tma[2]): phi boxes carry the read-only ring (SX x SY), the coefficient
// boxes cover the computed 32 x 24 cells (ax: AXW faces a row, ay: TYE + 1 face rows).  Coordinates as in tma_build_maps.
static inline int t2_build_maps(TmaLevelMaps* T, const LevelDev& L)
{
    using namespace t2;
    T->ok = 0;
    if ((L.bclo[0] == MAC_PERIODIC && L.gx == 0) || (L.bclo[1] == MAC_PERIODIC && L.gy == 0)) return 0;   // cannot wrap
    if ((L.nx & 1) || L.nx < 2 || (L.px & 1) || (L.cx & 1)) return 0;
    const uint64_t ex = (uint64_t)L.nx + 2 * L.gx, ey = (uint64_t)L.ny + 2 * L.gy;
    const long long oc = (long long)L.gx + (long long)L.cx * L.gy, oa = (long long)L.gx + (long long)L.px * L.gy;
    bool ok = tma_encode3(&T->phi, L.phi - oc, ex, ey, L.nz, L.cx, L.ry, SX, SY) &&
              tma_encode3(&T->phi2, L.phi2 - oc, ex, ey, L.nz, L.cx, L.ry, SX, SY) &&
              tma_encode3(&T->rhs, L.rhs - oc, ex, ey, L.nz, L.cx, L.ry, 2 * LN, TYE) &&
              tma_encode3(&T->ax, L.ax - oa, ex + 1, ey, L.nz, L.px, L.ry, AXW, TYE) &&
              tma_encode3(&T->az, L.az - oc, ex, ey, (uint64_t)L.nz + 1, L.cx, L.ry, 2 * LN, TYE) &&
              tma_encode3(&T->ay, L.ay - oc, ex, ey + 1, L.nz, L.cx, (uint64_t)L.ry + 1, 2 * LN, TYE + 1);
    T->ok = ok ? 1 : 0;
    return T->ok;
}

// the two-sweep kernel needs its 4-cell halo inside the periodic images and a few planes to march through
static inline bool t2_level_ok(const LevelDev& L)
{
    if (L.nx < 48 || L.ny < 16 || L.nz < 8 || (L.nx & 1)) return false;
    if ((long long)L.cx * L.ry >= (1ll << 31)) return false;         // image offsets are ints
    if (L.bclo[0] == MAC_PERIODIC && L.gx < t2::HALO) return false;
    if (L.bclo[1] == MAC_PERIODIC && L.gy < t2::HALO) return false;
    return true;
}

static inline t2::T2Plan t2_plan(const LevelDev& L, int sms)
{
    t2::T2Plan P;
    P.tiles_x = (L.nx + 1 + t2::kTX - 1) / t2::kTX;                   // tile t finishes columns [26 t - 1, 26 t + 25)
    P.tiles = P.tiles_x * ((L.ny + t2::kTY - 1) / t2::kTY);
    const int S = sms, maxchunk = L.nz >= 8 ? L.nz / 4 : 1;                 // chunks of at least 4 planes
    // cost in marching steps of the slowest SM: rounds x (planes per chunk + the 6 redone planes + pipeline fill)
    long best = -1;
    P.nfull = 0; P.nsplit = 1;
    for (int full = 0; full <= (P.tiles / S) * S; full += S) {          // whole waves of whole columns, then chunks
        const int rem = P.tiles - full;
        for (int n = 1; n <= maxchunk; ++n) {
            const int zc = (L.nz + n - 1) / n, nn = (L.nz + zc - 1) / zc;
            const long cost = (long)(full / S) * (L.nz + 10) + (((long)rem * nn + S - 1) / S) * (zc + 10);
            if (best < 0 || cost < best) { best = cost; P.nfull = full; P.nsplit = rem > 0 ? nn : 1; }
            if (rem == 0) break;
        }
    }
    P.zchunk = (L.nz + P.nsplit - 1) / P.nsplit;
    P.ncta = P.nfull + (P.tiles - P.nfull) * P.nsplit;
    // Periodic images of the output: written by the owning threads inside the kernel on small levels (no extra launch);
    // on large ones by k_fill_ghosts after it -- measured at 512^3, the few divergent image stores of the edge tiles
    // cost the launch 10 % (y) / 4 % (x), a separate pass over the image strips 1 %
    P.images = (L.gx || L.gy) && (long long)L.nx * L.ny * L.nz < MAC_T2_IMAGES_BELOW ? 1 : 0;
    return P;
}

// Two fused sweeps: reads `in_is_phi2 ? phi2 : phi` through T (maps built for the 32 x 24 tile), writes phi_out.
// part_max != NULL: also per-CTA maxima of the input's red-cell residual; *nparts receives their count.
// Returns the number of kernels launched (2 when the images of the output are a pass of their own), or -1.
static inline int launch_t2_sweep(const TmaLevelMaps& T, bool in_is_phi2, double* phi_out, const LevelDev& L, int sms, cudaStream_t s,
                                  double* part_max = nullptr, int max_parts = 0, int* nparts = nullptr)
{
    using namespace t2;
    const T2Plan plan = t2_plan(L, sms);
    const dim3 grid(plan.ncta, 1, 1);
    const CUtensorMap& tin = in_is_phi2 ? T.phi2 : T.phi;
    const size_t sm = Cfg<MAC_T2_LA>::kSmem;
    if (part_max) {
        if ((long)grid.x * grid.y * grid.z > max_parts) return -1;
        *nparts = (int)(grid.x * grid.y * grid.z);
        k_rbgs_t2<MAC_T2_LA, true><<<grid, dim3(LN, TYE), sm, s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, phi_out, plan, part_max);
    } else
        k_rbgs_t2<MAC_T2_LA, false><<<grid, dim3(LN, TYE), sm, s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, phi_out, plan, nullptr);
    int launches = 1;
    if (!plan.images && (L.gx || L.gy)) {                   // the images of the output, as a pass of their own
        LevelDev O = L;
        O.phi = phi_out;
        const int per_plane = 2 * L.gx * (L.ny + 1 + 2 * L.gy) + 2 * L.gy * (L.nx + 1);
        k_fill_ghosts<<<dim3((per_plane + 255) / 256, L.nz + 1), 256, 0, s>>>(O, 1);
        ++launches;
    }
    return cudaPeekAtLastError() == cudaSuccess ? launches : -1;
}
