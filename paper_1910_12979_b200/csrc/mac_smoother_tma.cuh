// mac_smoother_tma.cuh -- the fused red+black Gauss-Seidel sweep of mac_smoother.cuh with the z-plane
// staging done by the Tensor Memory Accelerator (cp.async.bulk.tensor, SASS UTMALDG) instead of
// per-thread cp.async (north_star bullet 3 "shared-memory or TMA z-plane
// staging").
//
// Why: the cp.async version spends 5 LDGSTS + their address arithmetic per thread per plane and is
// bound by the MIO instruction queue (profiles/r1a_smoother_512_ncu.txt).  Here ONE thread per CTA
// issues five 3-D box loads per plane (phi, rhs, ax, ay, az) that land in the same shared-memory
// stage layout and signal an mbarrier with their byte count; out-of-range box elements (the halo
// outside the domain, planes below 0 / above nz) are zero-filled by the hardware, which is exactly
// the "phi = 0 and a_f = 0 outside the domain" convention of the folded coefficients
// (mac_common.cuh).  Arithmetic, marching order and results are those of fused::step.
//
// TMA cannot wrap: a level that is periodic in x and / or y carries periodic image columns / rows of
// every array (mac_common.cuh "Ghosts"), which the box loads read like any halo; z may be periodic
// (the plane coordinate is wrapped by the issuing thread).  One sweep per launch: the default path runs
// pairs of sweeps through mac_smoother_t2.cuh and uses this kernel for a remaining single sweep.
#pragma once
#include <cuda.h>

#include "mac_smoother.cuh"

namespace tma {

using fused::A_AX; using fused::A_AY; using fused::A_AZ; using fused::A_COUNT; using fused::A_PHI; using fused::A_RHS;
using fused::Coef; using fused::Ctx;

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, unsigned bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];\n"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

template <int LN, int TYE, int NS>
struct Cfg {
    static constexpr int kRow = LN * 16;                       // bytes of one staged row (2*LN doubles)
    static constexpr int kArr = TYE * kRow;                    // one array of a stage
    static constexpr int kStage = A_COUNT * kArr;
    static constexpr unsigned kTx = (unsigned)kRow * (TYE + (TYE - 1) + 3 * (TYE - 2));   // bytes landing per plane
    static constexpr size_t kSmem = (size_t)kStage * NS + 8 * NS + 128;
    static_assert(Ctx<LN, TYE>::kStage == kStage, "stage layout must match fused::step");
};

// issue the five box loads of plane p (unwrapped) into stage `stg`
template <int LN, int TYE, int NS>
__device__ __forceinline__ void issue_plane(const CUtensorMap* tm_phi, const CUtensorMap* tm_rhs, const CUtensorMap* tm_ax,
                                            const CUtensorMap* tm_ay, const CUtensorMap* tm_az, unsigned stage0, unsigned bar0,
                                            int stg, int p, int nz, bool perz, int cx, int cy)
{
    using C = Cfg<LN, TYE, NS>;
    if (perz) { if (p < 0) p += nz; else if (p >= nz) p -= nz; }
    const unsigned d = stage0 + stg * C::kStage;
    const unsigned bar = bar0 + 8 * stg;
    mbar_expect_tx(bar, C::kTx);
    tma_load_3d(d + A_PHI * C::kArr, tm_phi, bar, cx, cy, p);                    // rows 0 .. TYE-1
    tma_load_3d(d + A_RHS * C::kArr + C::kRow, tm_rhs, bar, cx, cy + 1, p);      // rows 1 .. TYE-2
    tma_load_3d(d + A_AX * C::kArr + C::kRow, tm_ax, bar, cx, cy + 1, p);
    tma_load_3d(d + A_AZ * C::kArr + C::kRow, tm_az, bar, cx, cy + 1, p);
    tma_load_3d(d + A_AY * C::kArr + C::kRow, tm_ay, bar, cx, cy + 1, p);        // rows 1 .. TYE-1 (faces)
}

template <int LN, int TYE, int NS, bool REDX0, bool NORM>
__device__ __forceinline__ void march(const Ctx<LN, TYE>& C, const CUtensorMap* tm_phi, const CUtensorMap* tm_rhs,
                                      const CUtensorMap* tm_ax, const CUtensorMap* tm_ay, const CUtensorMap* tm_az,
                                      unsigned stage0, unsigned bar0, bool producer, int cx, int cy, int ks, int k0, int k1,
                                      bool red_x_ok, bool red_y_ok, bool own, double* __restrict__ out,
                                      unsigned long long out_stride, double* vmax)
{
    using G = Cfg<LN, TYE, NS>;
    double2 qm2 = make_double2(0.0, 0.0), qm1;
    Coef cA, cB;
    cB.ax = cB.ays = cB.ayn = cB.az = cB.rhs = qm2; cB.ax2 = 0.0;
    // planes ks-1 .. ks+NS-3 were issued by the prologue into stages 0 .. NS-2 (plane ks-1+q -> stage q);
    // the first NS-1 waits are on phase 0 of their barriers
    mbar_wait(bar0 + 0, 0);
    mbar_wait(bar0 + 8, 0);
    int sI = 1;                                                // stage of plane k
    unsigned phase_bits = 0;                                   // bit s: parity to wait for on stage s next
    phase_bits |= 3u;                                          // stages 0 and 1 have completed phase 0
    qm1 = fused::ld2<LN, TYE>(C.smem_gen + 0 * G::kStage, A_PHI, 0, 0);
    double2 qn = fused::ld2<LN, TYE>(C.smem_gen + 1 * G::kStage, A_PHI, 0, 0);
    double2 azn = fused::ld2<LN, TYE>(C.smem_gen + 1 * G::kStage, A_AZ, 0, 0);
#pragma unroll 1
    for (int k = ks; k <= k1; k += 2) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int kk = k + h;
            if (kk > k1) break;
            int sM = sI - 1; if (sM < 0) sM += NS;
            int sP = sI + 1; if (sP >= NS) sP -= NS;
            int sN = sI + (NS - 2); if (sN >= NS) sN -= NS;       // stage that plane kk-2 vacated at the end of step kk-1
            // plane kk+1 must have landed; every thread must have finished step kk-1
            mbar_wait(bar0 + 8 * sP, (phase_bits >> sP) & 1u);
            phase_bits ^= 1u << sP;
            __syncthreads();
            if (producer && kk + NS - 2 <= k1 + 1) {           // never leave a load in flight at exit
                asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                issue_plane<LN, TYE, NS>(tm_phi, tm_rhs, tm_ax, tm_ay, tm_az, stage0, bar0, sN, kk + NS - 2, C.nz, C.perz, cx, cy);
            }
            unsigned char* s0 = C.smem_gen + sI * G::kStage;
            const unsigned char* sm = C.smem_gen + sM * G::kStage;
            const unsigned char* sp = C.smem_gen + sP * G::kStage;
            const bool k_real = C.perz || (kk >= 0 && kk < C.nz);
            const bool do_black = own && kk - 1 >= k0 && kk - 1 < k1;
            if (h == 0)
                fused::step<LN, TYE, REDX0, NORM>(C, s0, sm, sp, k_real && (REDX0 ? red_x_ok : red_y_ok), do_black, out, qm2, qm1, qn, azn, cA, cB, vmax);
            else
                fused::step<LN, TYE, !REDX0, NORM>(C, s0, sm, sp, k_real && (REDX0 ? red_y_ok : red_x_ok), do_black, out, qm2, qm1, qn, azn, cB, cA, vmax);
            out += out_stride;
            sI = sP;
        }
    }
}

// NORM: additionally writes, per CTA, max |rhs - L phi_in| over the red cells to part_max[linear CTA index]
// (the stop test of the previous cycle rides on the first sweep of the next one; see maestro_mac.cu).
template <int LN, int TYE, int NS, int MINB, bool NORM>
__global__ void __launch_bounds__(LN * TYE, MINB)
k_rbgs_tma(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_rhs,
           const __grid_constant__ CUtensorMap tm_ax, const __grid_constant__ CUtensorMap tm_ay,
           const __grid_constant__ CUtensorMap tm_az, LevelDev L, double* __restrict__ pout, int zchunk,
           double* __restrict__ part_max)
{
    using G = Cfg<LN, TYE, NS>;
    constexpr int TY = TYE - 4, kTX = 2 * LN - 4;
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    // stages need 128-byte alignment for TMA; the dynamic segment is at least 16-byte aligned.  (Pointer
    // arithmetic on the __shared__ array, not an integer round trip: the accesses must stay LDS/STS.)
    unsigned char* smem_raw = smem_dyn + ((128u - (smem_u32(smem_dyn) & 127u)) & 127u);
    const unsigned stage0 = smem_u32(smem_raw);
    const unsigned bar0 = stage0 + NS * G::kStage;

    const int lane = threadIdx.x;
    // a warp holds 32/LN rows; they must share their parity (the colour role is warp-uniform)
    const int ty = (LN == 32) ? (int)threadIdx.y
                              : 4 * ((int)threadIdx.y >> 2) + (((int)threadIdx.y >> 1) & 1) + 2 * ((int)threadIdx.y & 1);
    static_assert(LN == 32 || (LN == 16 && TYE % 4 == 0), "row mapping");
    const int x0 = blockIdx.x * kTX, y0 = blockIdx.y * TY;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, L.nz);
    const int gi = x0 - 2 + 2 * lane, gj = y0 - 2 + ty;
    // ghost columns / rows of a periodic level hold valid images: their reds are recomputed like any halo
    const bool x_ok = gi >= -L.gx && gi < L.nx + L.gx, y_ok = gj >= -L.gy && gj < L.ny + L.gy;
    const bool col_ok = x_ok && y_ok;
    const bool row_red = ty >= 1 && ty <= TYE - 2;
    const bool own = lane >= 1 && lane <= LN - 2 && ty >= 2 && ty <= TYE - 3 && gi < x0 + kTX && gj < y0 + TY &&
                     gi < L.nx && gj < L.ny;                           // (gi >= x0 >= 0, gj >= y0 >= 0 for these threads)
    const bool producer = threadIdx.x == 0 && threadIdx.y == 0;

    Ctx<LN, TYE> C;
    C.nz = L.nz;
    C.perz = L.bclo[2] == MAC_PERIODIC;
    C.own = own;
    C.img_x = own ? image_dx(L, gi) : 0;
    C.img_y = own ? image_dy(L, gj) : 0;
    const unsigned slot = (ty * LN + lane) * 16;
    C.smem_gen = smem_raw + slot;
    C.smem_u32 = stage0 + slot;
    const int cx0 = x0 - 2 + L.gx, cy0 = y0 - 2 + L.gy;          // tensor-map coordinates of the tile origin

    const int ks = k0 - 1;
    if (producer) {
        for (int s = 0; s < NS; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        for (int q = 0; q < NS - 1 && ks - 1 + q <= k1 + 1; ++q)
            issue_plane<LN, TYE, NS>(&tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, stage0, bar0, q, ks - 1 + q, L.nz, C.perz, cx0, cy0);
    }
    __syncthreads();                                             // barrier inits visible before anyone waits

    const bool red_x_ok = col_ok && row_red && lane >= 1;
    const bool red_y_ok = col_ok && row_red && lane <= LN - 2;
    const unsigned long long ostride = (unsigned long long)L.cx * L.ry;
    double* out = pout + (own ? (long long)gi + (long long)L.cx * gj : 0) + (long long)(ks - 1) * (long long)ostride;
    double vmax = 0.0;
    if (((gj + ks) & 1) == 0)
        march<LN, TYE, NS, true, NORM>(C, &tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, stage0, bar0, producer, cx0, cy0, ks, k0, k1, red_x_ok, red_y_ok, own, out, ostride, &vmax);
    else
        march<LN, TYE, NS, false, NORM>(C, &tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, stage0, bar0, producer, cx0, cy0, ks, k0, k1, red_x_ok, red_y_ok, own, out, ostride, &vmax);
    // every plane that was issued (<= k1 + 1) has been waited for by the last step: nothing is in flight
    if (NORM) {
        __shared__ double sh_max[32];
        const int tid = threadIdx.x + LN * threadIdx.y;
        vmax = warp_nanmax(vmax);
        if ((tid & 31) == 0) sh_max[tid >> 5] = vmax;
        __syncthreads();
        if (tid == 0) {
            double m = sh_max[0];
            for (int q = 1; q < (LN * TYE) / 32; ++q) m = nanmax(m, sh_max[q]);
            part_max[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = m;
        }
    }
}

template <int LN, int TYE, int NS> constexpr size_t smem_bytes() { return Cfg<LN, TYE, NS>::kSmem; }

}  // namespace tma

// ---- host side ---------------------------------------------------------------------------------

struct TmaLevelMaps {                 // tensor maps of one level for one tile configuration
    CUtensorMap phi, phi2, rhs, ax, ay, az;
    int ok;                           // 0: level not eligible (periodic x/y, odd nx, encode failed)
};

#define MAC_TMA_BIG   32, 16, 5, 1, false    // 64 x 16 staged tile (60 x 12 interior), 512 threads, 1 CTA/SM
#define MAC_TMA_BIGN  32, 16, 5, 1, true     // same, with the red-cell residual norm of the input
#define MAC_TMA_MID   16, 16, 5, 2, false    // 32 x 16 staged tile (28 x 12 interior), 256 threads, 2 CTAs/SM

typedef CUresult (*mac_encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                        const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                        CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static inline mac_encode_tiled_fn tma_encode_fn()
{
    static mac_encode_tiled_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (mac_encode_tiled_fn)p;
    }
    return fn;
}

// 3-D map over an array whose allocation starts at `base` (ghost origin): d0 x d1 x d2 entries, row pitch
// pitch0 (elements), rows_per_plane rows between planes
static inline bool tma_encode3(CUtensorMap* m, const double* base, uint64_t d0, uint64_t d1, uint64_t d2,
                               uint64_t pitch0_elems, uint64_t rows_per_plane, uint32_t b0, uint32_t b1)
{
    mac_encode_tiled_fn fn = tma_encode_fn();
    if (!fn) return false;
    cuuint64_t dims[3] = {d0, d1, d2};
    cuuint64_t strides[2] = {pitch0_elems * 8ull, pitch0_elems * rows_per_plane * 8ull};
    cuuint32_t box[3] = {b0, b1, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void*)base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Build the maps of a level for a staged tile of 2*LN x TYE cells.  Returns ok.  Coordinate (0, 0) of every
// map is the ghost origin (-gx, -gy); kernels add (gx, gy) to their tile origins.  Out-of-range box elements
// are zero-filled, which is the "phi = 0, a_f = 0 outside the domain" convention on non-periodic sides.
static inline int tma_build_maps(TmaLevelMaps* T, const LevelDev& L, int LN, int TYE)
{
    T->ok = 0;
    if ((L.bclo[0] == MAC_PERIODIC && L.gx == 0) || (L.bclo[1] == MAC_PERIODIC && L.gy == 0)) return 0;   // cannot wrap
    if ((L.nx & 1) || L.nx < 2 || (L.px & 1)) return 0;
    const uint32_t bx = 2u * LN;
    const uint64_t ex = (uint64_t)L.nx + 2 * L.gx, ey = (uint64_t)L.ny + 2 * L.gy;
    const long long oc = (long long)L.gx + (long long)L.cx * L.gy, oa = (long long)L.gx + (long long)L.px * L.gy;
    bool ok = tma_encode3(&T->phi, L.phi - oc, ex, ey, L.nz, L.cx, L.ry, bx, TYE) &&
              tma_encode3(&T->phi2, L.phi2 - oc, ex, ey, L.nz, L.cx, L.ry, bx, TYE) &&
              tma_encode3(&T->rhs, L.rhs - oc, ex, ey, L.nz, L.cx, L.ry, bx, TYE - 2) &&
              tma_encode3(&T->ax, L.ax - oa, ex + 1, ey, L.nz, L.px, L.ry, bx, TYE - 2) &&
              tma_encode3(&T->az, L.az - oc, ex, ey, (uint64_t)L.nz + 1, L.cx, L.ry, bx, TYE - 2) &&
              tma_encode3(&T->ay, L.ay - oc, ex, ey + 1, L.nz, L.cx, (uint64_t)L.ry + 1, bx, TYE - 1);
    T->ok = ok ? 1 : 0;
    return T->ok;
}

static inline int tma_smoother_configure()
{
    using namespace tma;
    if (cudaFuncSetAttribute(k_rbgs_tma<MAC_TMA_BIG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<32, 16, 5>()) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_rbgs_tma<MAC_TMA_BIGN>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<32, 16, 5>()) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_rbgs_tma<MAC_TMA_MID>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes<16, 16, 5>()) != cudaSuccess) return -1;
    return 0;
}

// z-chunking: pick the chunk count that minimises waves x (planes per chunk + restaged planes)
static inline void tma_pick_chunks(int tiles, int nz, int slots, int* nchunk_out, int* zchunk_out)
{
    long best = -1; int bn = 1;
    const int maxchunk = nz >= 16 ? nz / 8 : 1;
    for (int n = 1; n <= maxchunk; ++n) {
        const int zc = (nz + n - 1) / n;
        const int nn = (nz + zc - 1) / zc;
        const long waves = ((long)tiles * nn + slots - 1) / slots;
        const long cost = waves * (zc + 4);
        if (best < 0 || cost < best) { best = cost; bn = nn; }
    }
    *nchunk_out = bn;
    *zchunk_out = (nz + bn - 1) / bn;
}

// grid of one TMA sweep of level L (variant 0: 64x16 tile, 1: 32x16 tile)
static inline dim3 tma_sweep_grid(const LevelDev& L, int variant, int sms, int* zchunk_out)
{
    const int LN = variant == 0 ? 32 : 16;
    const int kTX = 2 * LN - 4, TY = 12;
    const int tiles_x = (L.nx + kTX - 1) / kTX, tiles_y = (L.ny + TY - 1) / TY;
    int nchunk, zchunk;
    tma_pick_chunks(tiles_x * tiles_y, L.nz, variant == 0 ? sms : 2 * sms, &nchunk, &zchunk);
    if (zchunk_out) *zchunk_out = zchunk;
    return dim3(tiles_x, tiles_y, nchunk);
}

// One fused sweep through the TMA kernel: reads `in_is_phi2 ? phi2 : phi`, writes the other buffer.
// part_max != NULL (variant 0 only): also write per-CTA maxima of the input's red-cell residual; *nparts
// receives their count.
static inline int launch_tma_sweep(const TmaLevelMaps& T, bool in_is_phi2, double* phi_out, const LevelDev& L, int variant,
                                   int sms, cudaStream_t s, double* part_max = nullptr, int max_parts = 0, int* nparts = nullptr)
{
    using namespace tma;
    int zchunk;
    const dim3 grid = tma_sweep_grid(L, variant, sms, &zchunk);
    const CUtensorMap& tin = in_is_phi2 ? T.phi2 : T.phi;
    if (part_max) {
        if (variant != 0 || (long)grid.x * grid.y * grid.z > max_parts) return -1;
        *nparts = (int)(grid.x * grid.y * grid.z);
        k_rbgs_tma<MAC_TMA_BIGN><<<grid, dim3(32, 16), smem_bytes<32, 16, 5>(), s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, phi_out, zchunk, part_max);
    } else if (variant == 0)
        k_rbgs_tma<MAC_TMA_BIG><<<grid, dim3(32, 16), smem_bytes<32, 16, 5>(), s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, phi_out, zchunk, nullptr);
    else
        k_rbgs_tma<MAC_TMA_MID><<<grid, dim3(16, 16), smem_bytes<16, 16, 5>(), s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, phi_out, zchunk, nullptr);
    return cudaPeekAtLastError() == cudaSuccess ? 0 : -1;
}

// ================================================================================================
// a6 / a9 on the same TMA plane ring:  r = rhs - L phi,  then (RESTRICT) coarse rhs = mean of the 8
// children and coarse phi = 0, and/or (NORM) per-CTA partial of ||r||inf.
//
// Same staged tile as the smoother (64 x 16 cells: x halo 2, kept for 16-byte pair alignment; y halo
// 1), same tensor maps.  A thread owns a 2 x 2 block of columns (an x pair in two adjacent rows), i.e.
// the lateral footprint of ONE coarse cell; the two planes of the coarse cell are accumulated over
// two consecutive marching steps, so the restriction needs no cross-thread reduction.  z-neighbours
// of phi are carried in registers, lateral neighbours come from the staged plane.  Nothing is
// written to shared memory, so a plane's stage is recycled as soon as every thread has passed it.
// Algorithmic traffic: 40 B/cell read + 2 B/cell written (41 B/cell).
// ================================================================================================
namespace tma {

enum { RES_RESTRICT = 1, RES_NORM = 2 };

template <int NS, int MODE>
__global__ void __launch_bounds__(32 * 7, 1)
k_resid_tma(const __grid_constant__ CUtensorMap tm_phi, const __grid_constant__ CUtensorMap tm_rhs,
            const __grid_constant__ CUtensorMap tm_ax, const __grid_constant__ CUtensorMap tm_ay,
            const __grid_constant__ CUtensorMap tm_az, LevelDev L, LevelDev Cc, double* __restrict__ part_max, int zchunk)
{
    constexpr int LN = 32, TYE = 16;
    using G = Cfg<LN, TYE, NS>;
    constexpr int kTX = 60, kTY = 14;
    extern __shared__ __align__(128) unsigned char smem_dyn[];
    unsigned char* smem_raw = smem_dyn + ((128u - (smem_u32(smem_dyn) & 127u)) & 127u);
    const unsigned stage0 = smem_u32(smem_raw);
    const unsigned bar0 = stage0 + NS * G::kStage;
    __shared__ double sh_max[8];

    const int lane = threadIdx.x, tr = threadIdx.y;
    const int x0 = blockIdx.x * kTX, y0 = blockIdx.y * kTY;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, L.nz);
    const int gi = x0 - 2 + 2 * lane;                       // even
    const int gja = y0 + 2 * tr;                            // even; rows gja, gja+1 = stage rows 2tr+1, 2tr+2
    const bool own = lane >= 1 && lane <= LN - 2 && gi < L.nx && gja < L.ny;   // nx, ny even: the 2x2 block is all in or all out
    const bool producer = threadIdx.x == 0 && threadIdx.y == 0;
    const bool perz = L.bclo[2] == MAC_PERIODIC;
    const unsigned char* base = smem_raw + ((2 * tr + 1) * LN + lane) * 16;   // row a of stage 0

    if (producer) {
        for (int s = 0; s < NS; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
        for (int q = 0; q < NS && k0 - 1 + q <= k1; ++q)         // planes k0-1 .. ; plane p -> stage (p - (k0-1)) % NS
            issue_plane<LN, TYE, NS>(&tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, stage0, bar0, q, k0 - 1 + q, L.nz, perz, x0 - 2 + L.gx, y0 - 1 + L.gy);
    }
    __syncthreads();

    unsigned phase_bits = 0;
    mbar_wait(bar0 + 0, 0);
    mbar_wait(bar0 + 8, 0);
    phase_bits = 3u;
    // own-column phi of planes k-1 (m), k (c); rows a, b
    double2 pma = fused::ld2<LN, TYE>(base, A_PHI, 0, 0), pmb = fused::ld2<LN, TYE>(base, A_PHI, 1, 0);
    double2 pca = fused::ld2<LN, TYE>(base + G::kStage, A_PHI, 0, 0), pcb = fused::ld2<LN, TYE>(base + G::kStage, A_PHI, 1, 0);
    double2 aza = fused::ld2<LN, TYE>(base + G::kStage, A_AZ, 0, 0), azb = fused::ld2<LN, TYE>(base + G::kStage, A_AZ, 1, 0);
    int sI = 1;
    double acc = 0.0, vmax = 0.0;
    // coarse outputs (RES_RESTRICT): cell (gi/2, gja/2) of the coarse level, with its periodic images
    const long long cplane = (long long)Cc.cx * Cc.ry;
    const size_t c0 = (MODE & RES_RESTRICT) && own ? cidx(Cc, gi >> 1, gja >> 1, k0 >> 1) : 0;
    double* co = (MODE & RES_RESTRICT) ? Cc.rhs + c0 : nullptr;
    double* cz = (MODE & RES_RESTRICT) ? Cc.phi + c0 : nullptr;
    const long long cix = (MODE & RES_RESTRICT) && own ? image_dx(Cc, gi >> 1) : 0;
    const long long ciy = (MODE & RES_RESTRICT) && own ? image_dy(Cc, gja >> 1) : 0;

#pragma unroll 1
    for (int kk = k0; kk < k1; ++kk) {
        int sP = sI + 1; if (sP >= NS) sP -= NS;
        int sN = sI - 1; if (sN < 0) sN += NS;                    // stage of plane kk-1: last read during step kk-1
        mbar_wait(bar0 + 8 * sP, (phase_bits >> sP) & 1u);
        phase_bits ^= 1u << sP;
        __syncthreads();
        if (producer && kk + NS - 1 <= k1) {                      // (plane k0-1 was consumed into registers by the prologue)
            asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
            issue_plane<LN, TYE, NS>(&tm_phi, &tm_rhs, &tm_ax, &tm_ay, &tm_az, stage0, bar0, sN, kk + NS - 1, L.nz, perz, x0 - 2 + L.gx, y0 - 1 + L.gy);
        }
        const unsigned char* s0 = base + sI * G::kStage;
        const unsigned char* sp = base + sP * G::kStage;
        const double2 pna = fused::ld2<LN, TYE>(sp, A_PHI, 0, 0), pnb = fused::ld2<LN, TYE>(sp, A_PHI, 1, 0);
        const double2 azna = fused::ld2<LN, TYE>(sp, A_AZ, 0, 0), aznb = fused::ld2<LN, TYE>(sp, A_AZ, 1, 0);
        if (own) {
            const double2 axa = fused::ld2<LN, TYE>(s0, A_AX, 0, 0), axb = fused::ld2<LN, TYE>(s0, A_AX, 1, 0);
            const double axa2 = fused::ld1<LN, TYE, true>(s0, A_AX, 0, 1), axb2 = fused::ld1<LN, TYE, true>(s0, A_AX, 1, 1);
            const double2 ay0 = fused::ld2<LN, TYE>(s0, A_AY, 0, 0), ay1 = fused::ld2<LN, TYE>(s0, A_AY, 1, 0), ay2 = fused::ld2<LN, TYE>(s0, A_AY, 2, 0);
            const double2 ra = fused::ld2<LN, TYE>(s0, A_RHS, 0, 0), rb = fused::ld2<LN, TYE>(s0, A_RHS, 1, 0);
            const double2 ps = fused::ld2<LN, TYE>(s0, A_PHI, -1, 0), pn = fused::ld2<LN, TYE>(s0, A_PHI, 2, 0);
            const double wa = fused::ld1<LN, TYE, false>(s0, A_PHI, 0, -1), ea = fused::ld1<LN, TYE, true>(s0, A_PHI, 0, 1);
            const double wb = fused::ld1<LN, TYE, false>(s0, A_PHI, 1, -1), eb = fused::ld1<LN, TYE, true>(s0, A_PHI, 1, 1);
            // residual r = rhs - (sum_f a_f phi_nb - phi_0 sum_f a_f) of the four cells
            auto res = [](double rhs, double p0, double axw, double axe, double ays, double ayn, double azd, double azu,
                          double w, double e, double s, double n, double d, double u) {
                const double off = axw * w + axe * e + ays * s + ayn * n + azd * d + azu * u;
                const double dg = ((axw + axe) + (ays + ayn)) + (azd + azu);
                return rhs - (off - p0 * dg);
            };
            const double r00 = res(ra.x, pca.x, axa.x, axa.y, ay0.x, ay1.x, aza.x, azna.x, wa, pca.y, ps.x, pcb.x, pma.x, pna.x);
            const double r10 = res(ra.y, pca.y, axa.y, axa2, ay0.y, ay1.y, aza.y, azna.y, pca.x, ea, ps.y, pcb.y, pma.y, pna.y);
            const double r01 = res(rb.x, pcb.x, axb.x, axb.y, ay1.x, ay2.x, azb.x, aznb.x, wb, pcb.y, pca.x, pn.x, pmb.x, pnb.x);
            const double r11 = res(rb.y, pcb.y, axb.y, axb2, ay1.y, ay2.y, azb.y, aznb.y, pcb.x, eb, pca.y, pn.y, pmb.y, pnb.y);
            if (MODE & RES_NORM) {
                vmax = nanmax(vmax, fabs(r00)); vmax = nanmax(vmax, fabs(r10));
                vmax = nanmax(vmax, fabs(r01)); vmax = nanmax(vmax, fabs(r11));
            }
            if (MODE & RES_RESTRICT) {
                const double s4 = (r00 + r10) + (r01 + r11);
                if ((kk & 1) == 0) {
                    acc = s4;
                } else {
                    store_images(co, 0.125 * (acc + s4), cix, ciy);
                    store_images(cz, 0.0, cix, ciy);
                    co += cplane;
                    cz += cplane;
                }
            }
        }
        pma = pca; pmb = pcb; pca = pna; pcb = pnb; aza = azna; azb = aznb;
        sI = sP;
    }
    if (MODE & RES_NORM) {
        vmax = warp_nanmax(vmax);
        if (lane == 0) sh_max[tr] = vmax;
        __syncthreads();
        if (tr == 0 && lane == 0) {
            double m = sh_max[0];
            for (int q = 1; q < 7; ++q) m = nanmax(m, sh_max[q]);
            part_max[blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z)] = m;
        }
    }
}

}  // namespace tma

static inline int tma_resid_configure()
{
    using namespace tma;
    const int sm = (int)smem_bytes<32, 16, 5>();
    if (cudaFuncSetAttribute(k_resid_tma<5, RES_RESTRICT>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_resid_tma<5, RES_NORM>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(k_resid_tma<5, RES_RESTRICT | RES_NORM>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm) != cudaSuccess) return -1;
    return 0;
}

// mode: tma::RES_RESTRICT and/or tma::RES_NORM.  Returns the number of CTAs (= partial maxima written), or -1.
static inline int launch_tma_resid(const TmaLevelMaps& T, bool in_is_phi2, const LevelDev& L, const LevelDev& Cc,
                                   double* part_max, int max_parts, int mode, int sms, cudaStream_t s)
{
    using namespace tma;
    const int tiles_x = (L.nx + 59) / 60, tiles_y = (L.ny + 13) / 14;
    int nchunk, zchunk;
    tma_pick_chunks(tiles_x * tiles_y, L.nz, sms, &nchunk, &zchunk);
    zchunk = (zchunk + 1) & ~1;                               // chunks start on even planes (coarse cells are not split)
    nchunk = (L.nz + zchunk - 1) / zchunk;
    while ((long)tiles_x * tiles_y * nchunk > max_parts && nchunk > 1) {
        zchunk *= 2;
        nchunk = (L.nz + zchunk - 1) / zchunk;
    }
    if ((long)tiles_x * tiles_y * nchunk > max_parts) return -1;
    dim3 grid(tiles_x, tiles_y, nchunk), block(32, 7);
    const CUtensorMap& tin = in_is_phi2 ? T.phi2 : T.phi;
    const size_t sm = smem_bytes<32, 16, 5>();
    if (mode == RES_RESTRICT)
        k_resid_tma<5, RES_RESTRICT><<<grid, block, sm, s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, Cc, part_max, zchunk);
    else if (mode == RES_NORM)
        k_resid_tma<5, RES_NORM><<<grid, block, sm, s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, Cc, part_max, zchunk);
    else
        k_resid_tma<5, RES_RESTRICT | RES_NORM><<<grid, block, sm, s>>>(tin, T.rhs, T.ax, T.ay, T.az, L, Cc, part_max, zchunk);
    return cudaPeekAtLastError() == cudaSuccess ? tiles_x * tiles_y * nchunk : -1;
}
