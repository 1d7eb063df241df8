// mac_kernels.cuh -- the pointwise / transfer / bottom kernels of the MAC projection (sm_100a).
// Hot smoother kernels live in mac_smoother.cuh.  Step names (a2..a11) follow SURVEY.md Sec. 8(a).
#pragma once
#include "mac_common.cuh"

// ------------------------------------------------------------------------------------------------
// a1/a2  face coefficients  a_f = c_f * beta0(face centre) / (0.5 (rho_L + rho_R)) / h^2
// (Eq. 2: the factor beta0/rho of the pressure term.)  One thread per index of the
// extended (nx+1, ny+1, nz+1) space writes the low x, y and z face of that index.
// ------------------------------------------------------------------------------------------------

__device__ __forceinline__ double rho_cell(const GeoDev& G, const double* __restrict__ rho,
                                           const double* __restrict__ rho0, int i, int j, int k)
{
    if (rho) return __ldg(rho + ((size_t)i + (size_t)G.nx * ((size_t)j + (size_t)G.ny * (size_t)k)));
    return profile_eval(rho0, G.nr, G.dr, radius(G, (i + 0.5) * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz));
}

// density on face f of axis d through cell (i,j,k)'s row (O2), and the folding weight c_f (O5)
template <int D>
__device__ __forceinline__ void face_rho_weight(const GeoDev& G, const double* __restrict__ rho,
                                                const double* __restrict__ rho0, int i, int j, int k,
                                                double& rf, double& cf, int& fpos)
{
    const int n = D == 0 ? G.nx : (D == 1 ? G.ny : G.nz);
    const int f = D == 0 ? i : (D == 1 ? j : k);
    const bool per = G.bclo[D] == MAC_PERIODIC;
    int lo, hi;
    cf = 1.0;
    fpos = f;
    if (f == 0 || f == n) {
        if (per) {
            lo = n - 1; hi = 0; fpos = 0;              // face n is face 0 (reading A18)
        } else if (f == 0) {
            lo = hi = 0; cf = G.bclo[D] == MAC_WALL ? 0.0 : 2.0;
        } else {
            lo = hi = n - 1; cf = G.bchi[D] == MAC_WALL ? 0.0 : 2.0;
        }
    } else {
        lo = f - 1; hi = f;
    }
    double rl = rho_cell(G, rho, rho0, D == 0 ? lo : i, D == 1 ? lo : j, D == 2 ? lo : k);
    double rr = rho_cell(G, rho, rho0, D == 0 ? hi : i, D == 1 ? hi : j, D == 2 ? hi : k);
    rf = face_rho(rl, rr, G.rho_mean);
}

__global__ void __launch_bounds__(256)
k_face_coeff(GeoDev G, LevelDev L, const double* __restrict__ beta0, const double* __restrict__ rho,
             const double* __restrict__ rho0, int* __restrict__ flags)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y * blockDim.y + threadIdx.y;
    int k = blockIdx.z;
    if (i > G.nx || j > G.ny) return;
    const bool ci = i < G.nx, cj = j < G.ny, ck = k < G.nz;
    if (ci && cj && ck) {
        double r = rho_cell(G, rho, rho0, i, j, k);
        if (!(r > 0.0) || !(r <= 1.79769313486231570e308)) atomicOr(flags, 1);
    }
    double rf, cf;
    int fp;
    if (cj && ck) {
        face_rho_weight<0>(G, rho, rho0, i, j, k, rf, cf, fp);
        double b = profile_eval(beta0, G.nr, G.dr, radius(G, fp * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz));
        L.ax[axidx(L, i, j, k)] = cf * (b / rf) / (G.dx * G.dx);
    }
    if (ci && ck) {
        face_rho_weight<1>(G, rho, rho0, i, j, k, rf, cf, fp);
        double b = profile_eval(beta0, G.nr, G.dr, radius(G, (i + 0.5) * G.dx, fp * G.dy, (k + 0.5) * G.dz));
        L.ay[ayidx(L, i, j, k)] = cf * (b / rf) / (G.dy * G.dy);
    }
    if (ci && cj) {
        face_rho_weight<2>(G, rho, rho0, i, j, k, rf, cf, fp);
        double b = profile_eval(beta0, G.nr, G.dr, radius(G, (i + 0.5) * G.dx, (j + 0.5) * G.dy, fp * G.dz));
        L.az[azidx(L, i, j, k)] = cf * (b / rf) / (G.dz * G.dz);
    }
}

// ------------------------------------------------------------------------------------------------
// a3  coefficient coarsening: coarse face = mean of the 4 fine faces that tile it (reading A11);
// with the 1/h^2 pre-scaling that is  a_c = (1/16) * sum of the 4 fine a_f.
// ------------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(256)
k_coarsen_coeff(LevelDev F, LevelDev C)
{
    int I = blockIdx.x * blockDim.x + threadIdx.x;
    int J = blockIdx.y * blockDim.y + threadIdx.y;
    int K = blockIdx.z;
    if (I > C.nx || J > C.ny) return;
    const bool ci = I < C.nx, cj = J < C.ny, ck = K < C.nz;
    if (cj && ck) {
        double s = F.ax[axidx(F, 2 * I, 2 * J, 2 * K)] + F.ax[axidx(F, 2 * I, 2 * J + 1, 2 * K)] +
                   F.ax[axidx(F, 2 * I, 2 * J, 2 * K + 1)] + F.ax[axidx(F, 2 * I, 2 * J + 1, 2 * K + 1)];
        C.ax[axidx(C, I, J, K)] = 0.0625 * s;
    }
    if (ci && ck) {
        double s = F.ay[ayidx(F, 2 * I, 2 * J, 2 * K)] + F.ay[ayidx(F, 2 * I + 1, 2 * J, 2 * K)] +
                   F.ay[ayidx(F, 2 * I, 2 * J, 2 * K + 1)] + F.ay[ayidx(F, 2 * I + 1, 2 * J, 2 * K + 1)];
        C.ay[ayidx(C, I, J, K)] = 0.0625 * s;
    }
    if (ci && cj) {
        double s = F.az[azidx(F, 2 * I, 2 * J, 2 * K)] + F.az[azidx(F, 2 * I + 1, 2 * J, 2 * K)] +
                   F.az[azidx(F, 2 * I, 2 * J + 1, 2 * K)] + F.az[azidx(F, 2 * I + 1, 2 * J + 1, 2 * K)];
        C.az[azidx(C, I, J, K)] = 0.0625 * s;
    }
}

// ------------------------------------------------------------------------------------------------
// block-level deterministic reductions: every block writes one partial (sum, nanmax) pair; a
// single-block kernel folds the partials in a fixed order.
// ------------------------------------------------------------------------------------------------

__device__ __forceinline__ void block_reduce_store(double s, double m, double* __restrict__ part_sum,
                                                   double* __restrict__ part_max, int slot)
{
    __shared__ double sh_s[32], sh_m[32];
    const int tid = threadIdx.x + blockDim.x * threadIdx.y;
    const int nthr = blockDim.x * blockDim.y;
    s = warp_sum(s);
    m = warp_nanmax(m);
    if ((tid & 31) == 0) { sh_s[tid >> 5] = s; sh_m[tid >> 5] = m; }
    __syncthreads();
    if (tid < 32) {
        int nw = (nthr + 31) >> 5;
        s = tid < nw ? sh_s[tid] : 0.0;
        m = tid < nw ? sh_m[tid] : 0.0;
        s = warp_sum(s);
        m = warp_nanmax(m);
        if (tid == 0) { part_sum[slot] = s; part_max[slot] = m; }
    }
}

// out[0] = sum of part_sum, out[1] = nanmax of part_max
__global__ void __launch_bounds__(1024)
k_reduce_final(const double* __restrict__ part_sum, const double* __restrict__ part_max, int n,
               double* __restrict__ out, double* __restrict__ host_out = nullptr)
{   // host_out: mapped pinned memory that receives the two values as well (what the host reads after its synchronise)
    double s = 0.0, m = 0.0;
    for (int q = threadIdx.x; q < n; q += blockDim.x) { s += part_sum[q]; m = nanmax(m, part_max[q]); }
    __shared__ double sh_s[32], sh_m[32];
    s = warp_sum(s);
    m = warp_nanmax(m);
    if ((threadIdx.x & 31) == 0) { sh_s[threadIdx.x >> 5] = s; sh_m[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x < 32) {
        s = sh_s[threadIdx.x];
        m = sh_m[threadIdx.x];
        s = warp_sum(s);
        m = warp_nanmax(m);
        if (threadIdx.x == 0) {
            out[0] = s; out[1] = m;
            if (host_out) { host_out[0] = s; host_out[1] = m; __threadfence_system(); }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a4  rhs = D(beta0_face U_edge) - beta0_cell S    (Eq. 6), partial sum and max|rhs|.
// Blocks walk rows (j,k) grid-stride; threads walk i.
// ------------------------------------------------------------------------------------------------

__device__ __forceinline__ double beta_at(const GeoDev& G, const double* __restrict__ beta0,
                                          double x, double y, double z)
{
    return profile_eval(beta0, G.nr, G.dr, radius(G, x, y, z));
}

__global__ void __launch_bounds__(256)
k_rhs(GeoDev G, LevelDev L, const double* __restrict__ beta0, const double* __restrict__ u,
      const double* __restrict__ v, const double* __restrict__ w, const double* __restrict__ S,
      const double* __restrict__ qprof, double* __restrict__ part_sum, double* __restrict__ part_max)
{
    const int nrows = G.ny * G.nz;
    const bool px = G.bclo[0] == MAC_PERIODIC, py = G.bclo[1] == MAC_PERIODIC, pz = G.bclo[2] == MAC_PERIODIC;
    double s = 0.0, m = 0.0;
    for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
        const int j = row % G.ny, k = row / G.ny;
        const double yc = (j + 0.5) * G.dy, zc = (k + 0.5) * G.dz;
        const int jh = (py && j + 1 == G.ny) ? 0 : j + 1;     // periodic: face n reads entry 0
        const int kh = (pz && k + 1 == G.nz) ? 0 : k + 1;
        for (int i = threadIdx.x; i < G.nx; i += blockDim.x) {
            const double xc = (i + 0.5) * G.dx;
            const int ih = (px && i + 1 == G.nx) ? 0 : i + 1;
            const size_t ub = (size_t)(G.nx + 1) * ((size_t)j + (size_t)G.ny * k);
            double fxl = beta_at(G, beta0, i * G.dx, yc, zc) * u[ub + i];
            double fxh = beta_at(G, beta0, ih * G.dx, yc, zc) * u[ub + ih];
            double fyl = beta_at(G, beta0, xc, j * G.dy, zc) * v[(size_t)i + (size_t)G.nx * ((size_t)j + (size_t)(G.ny + 1) * k)];
            double fyh = beta_at(G, beta0, xc, jh * G.dy, zc) * v[(size_t)i + (size_t)G.nx * ((size_t)jh + (size_t)(G.ny + 1) * k)];
            double fzl = beta_at(G, beta0, xc, yc, k * G.dz) * w[(size_t)i + (size_t)G.nx * ((size_t)j + (size_t)G.ny * k)];
            double fzh = beta_at(G, beta0, xc, yc, kh * G.dz) * w[(size_t)i + (size_t)G.nx * ((size_t)j + (size_t)G.ny * kh)];
            double r = (fxh - fxl) / G.dx + (fyh - fyl) / G.dy + (fzh - fzl) / G.dz;
            const size_t c = (size_t)i + (size_t)G.nx * ((size_t)j + (size_t)G.ny * k);
            if (S || qprof) {             // source S - q(r): the dp0/dt term of PAPER.md:49 Eq. 6 rides on the profile q
                double se = S ? S[c] : 0.0;
                if (qprof) se -= profile_eval(qprof, G.nr, G.dr, radius(G, xc, yc, zc));
                r -= beta_at(G, beta0, xc, yc, zc) * se;
            }
            L.rhs[cidx(L, i, j, k)] = r;
            s += r;
            m = nanmax(m, fabs(r));
        }
    }
    block_reduce_store(s, m, part_sum, part_max, blockIdx.x);
}

// a -= scal[0]/count  (mean removal) over the interior of a cell array of level L, with partial sum / max of
// the shifted values.  Blocks walk rows (j,k) grid-stride; threads walk i.
__global__ void __launch_bounds__(256)
k_shift_mean(LevelDev L, double* __restrict__ a, const double* __restrict__ scal, double inv_count,
             double* __restrict__ part_sum, double* __restrict__ part_max)
{
    const double c = scal[0] * inv_count;
    const int nrows = L.ny * L.nz;
    double s = 0.0, m = 0.0;
    for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
        double* __restrict__ p = a + cidx(L, 0, row % L.ny, row / L.ny);
        for (int i = threadIdx.x; i < L.nx; i += blockDim.x) {
            double v = p[i] - c;
            p[i] = v;
            s += v;
            m = nanmax(m, fabs(v));
        }
    }
    block_reduce_store(s, m, part_sum, part_max, blockIdx.x);
}

// pub = a - scal[0]/count: the mean removal of k_shift_mean written straight into the caller's array (public cell
// layout idx = i + nx (j + ny k)) instead of in place -- the zero-mean phi the call returns, in one pass
__global__ void __launch_bounds__(256)
k_shift_mean_out(LevelDev L, const double* __restrict__ a, const double* __restrict__ scal, double inv_count, double* __restrict__ pub)
{
    const double c = scal[0] * inv_count;
    const int nrows = L.ny * L.nz;
    for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
        const double* __restrict__ p = a + cidx(L, 0, row % L.ny, row / L.ny);
        double* __restrict__ o = pub + (size_t)L.nx * row;
        for (int i = threadIdx.x; i < L.nx; i += blockDim.x) o[i] = p[i] - c;
    }
}

__global__ void __launch_bounds__(256)
k_sum(LevelDev L, const double* __restrict__ a, double* __restrict__ part_sum, double* __restrict__ part_max)
{
    const int nrows = L.ny * L.nz;
    double s = 0.0, m = 0.0;
    for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
        const double* __restrict__ p = a + cidx(L, 0, row % L.ny, row / L.ny);
        for (int i = threadIdx.x; i < L.nx; i += blockDim.x) {
            double v = p[i];
            s += v;
            m = nanmax(m, fabs(v));
        }
    }
    block_reduce_store(s, m, part_sum, part_max, blockIdx.x);
}

// Periodic images of a ghosted level (mac_common.cuh "Ghosts"): every ghost element of the selected arrays
// := its interior image.  One thread per ghost element of a plane; blockIdx.y = plane.
//   which bit 0: phi, 1: rhs, 2: ax, 3: ay, 4: az
__device__ __forceinline__ void fill_one(double* __restrict__ a, int pitch, int rows, int nxe, int nye, int nx, int ny,
                                         int gx, int gy, int k, int t)
{
    // the array holds nxe x nye own entries per plane (cells: nx x ny; ax: nx+1; ay: ny+1) plus ghosts
    const int ncol = 2 * gx, wrows = nye + 2 * gy;
    int i, j;
    if (t < ncol * wrows) {                       // ghost columns, all rows (corners included)
        const int c = t % ncol;
        j = t / ncol - gy;
        i = c < gx ? c - gx : nxe + (c - gx);
    } else {                                      // ghost rows, own columns
        t -= ncol * wrows;
        if (t >= 2 * gy * nxe) return;
        const int r = t / nxe;
        i = t % nxe;
        j = r < gy ? r - gy : nye + (r - gy);
    }
    int si = i, sj = j;
    if (si < 0) si += nx; else if (si >= nxe) si -= nx;
    if (sj < 0) sj += ny; else if (sj >= nye) sj -= ny;
    const long long plane = (long long)pitch * rows * k;
    a[plane + (long long)j * pitch + i] = a[plane + (long long)sj * pitch + si];
}

__global__ void __launch_bounds__(256)
k_fill_ghosts(LevelDev L, int which)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int k = blockIdx.y;
    if (k < L.nz) {
        if (which & 1) fill_one(L.phi, L.cx, L.ry, L.nx, L.ny, L.nx, L.ny, L.gx, L.gy, k, t);
        if (which & 2) fill_one(L.rhs, L.cx, L.ry, L.nx, L.ny, L.nx, L.ny, L.gx, L.gy, k, t);
        if (which & 4) fill_one(L.ax, L.px, L.ry, L.nx + 1, L.ny, L.nx, L.ny, L.gx, L.gy, k, t);
        if (which & 8) fill_one(L.ay, L.cx, L.ry + 1, L.nx, L.ny + 1, L.nx, L.ny, L.gx, L.gy, k, t);
    }
    if (which & 16) fill_one(L.az, L.cx, L.ry, L.nx, L.ny, L.nx, L.ny, L.gx, L.gy, k, t);   // nz + 1 planes
}

// ------------------------------------------------------------------------------------------------
// operator pieces shared by the reference smoother, residual and bottom solver
// ------------------------------------------------------------------------------------------------

// phi at a neighbour index that may be one outside along axis D: wrapped if periodic, else 0
template <int D>
__device__ __forceinline__ double nb_val(const LevelDev& L, const double* __restrict__ p, int i, int j, int k)
{
    const int n = D == 0 ? L.nx : (D == 1 ? L.ny : L.nz);
    int f = D == 0 ? i : (D == 1 ? j : k);
    if (f < 0) {
        if (L.bclo[D] != MAC_PERIODIC) return 0.0;
        f += n;
    } else if (f >= n) {
        if (L.bchi[D] != MAC_PERIODIC) return 0.0;
        f -= n;
    }
    return p[cidx(L, D == 0 ? f : i, D == 1 ? f : j, D == 2 ? f : k)];
}

// off = sum_f a_f phi_nb, dg = sum_f a_f
__device__ __forceinline__ void stencil_sums(const LevelDev& L, const double* __restrict__ p, int i, int j,
                                             int k, double& off, double& dg)
{
    const double axl = L.ax[axidx(L, i, j, k)], axh = L.ax[axidx(L, i + 1, j, k)];
    const double ayl = L.ay[ayidx(L, i, j, k)], ayh = L.ay[ayidx(L, i, j + 1, k)];
    const double azl = L.az[azidx(L, i, j, k)], azh = L.az[azidx(L, i, j, k + 1)];
    off = axl * nb_val<0>(L, p, i - 1, j, k) + axh * nb_val<0>(L, p, i + 1, j, k) +
          ayl * nb_val<1>(L, p, i, j - 1, k) + ayh * nb_val<1>(L, p, i, j + 1, k) +
          azl * nb_val<2>(L, p, i, j, k - 1) + azh * nb_val<2>(L, p, i, j, k + 1);
    dg = ((axl + axh) + (ayl + ayh)) + (azl + azh);
}

// ------------------------------------------------------------------------------------------------
// a5 (reference form)  one colour of red-black Gauss-Seidel, in place:
//   phi_0 <- phi_0 + (rhs_0 - (L phi)_0)/L_diag  ==  (sum_f a_f phi_nb - rhs_0) / sum_f a_f
// One thread per cell pair along x; the pair holds exactly one cell of each colour.
// ------------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(256)
k_rbgs_color(LevelDev L, int color)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (j >= L.ny) return;
    const int i = 2 * p + ((j + k + color) & 1);
    if (i >= L.nx) return;
    double off, dg;
    stencil_sums(L, L.phi, i, j, k, off, dg);
    const size_t c = cidx(L, i, j, k);
    L.phi[c] = (off - L.rhs[c]) / dg;
}

// ------------------------------------------------------------------------------------------------
// a6 (reference form)  coarse rhs = mean over the 8 children of (rhs - L phi); coarse phi = 0
// ------------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(256)
k_residual_restrict(LevelDev F, LevelDev C)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int K = blockIdx.z;
    if (I >= C.nx || J >= C.ny) return;
    double s = 0.0;
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj)
#pragma unroll
            for (int di = 0; di < 2; ++di) {
                const int i = 2 * I + di, j = 2 * J + dj, k = 2 * K + dk;
                double off, dg;
                stencil_sums(F, F.phi, i, j, k, off, dg);
                const size_t c = cidx(F, i, j, k);
                s += F.rhs[c] - (off - F.phi[c] * dg);
            }
    const size_t cc = cidx(C, I, J, K);
    const long long ix = image_dx(C, I), iy = image_dy(C, J);
    store_images(C.rhs + cc, 0.125 * s, ix, iy);
    store_images(C.phi + cc, 0.0, ix, iy);
}

// ------------------------------------------------------------------------------------------------
// a7  phi_f += P e_c : cell-centred trilinear (3/4 parent, 1/4 neighbour on the child's side per
// axis); coarse neighbours outside the grid follow the ghost rule (periodic wrap, WALL +e_0,
// OUTFLOW -e_0).  prolongation == 1: piecewise constant.
// ------------------------------------------------------------------------------------------------

__device__ __forceinline__ int ghost_index(int f, int n, int lo, int hi, double& sign)
{
    if (f < 0) {
        if (lo == MAC_PERIODIC) return f + n;
        if (lo == MAC_OUTFLOW) sign = -sign;
        return -1 - f;
    }
    if (f >= n) {
        if (hi == MAC_PERIODIC) return f - n;
        if (hi == MAC_OUTFLOW) sign = -sign;
        return 2 * n - 1 - f;
    }
    return f;
}

__global__ void __launch_bounds__(256)
k_prolong_add(LevelDev F, LevelDev C, int prolongation)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k = blockIdx.z;
    if (i >= F.nx || j >= F.ny) return;
    const int I = i >> 1, J = j >> 1, K = k >> 1;
    double val;
    if (prolongation == 1) {
        val = C.phi[cidx(C, I, J, K)];
    } else {
        double sx = 1.0, sy = 1.0, sz = 1.0;
        const int I2 = ghost_index(I + ((i & 1) ? 1 : -1), C.nx, C.bclo[0], C.bchi[0], sx);
        const int J2 = ghost_index(J + ((j & 1) ? 1 : -1), C.ny, C.bclo[1], C.bchi[1], sy);
        const int K2 = ghost_index(K + ((k & 1) ? 1 : -1), C.nz, C.bclo[2], C.bchi[2], sz);
        const double* __restrict__ e = C.phi;
        const double wx0 = 0.75, wx1 = 0.25 * sx, wy0 = 0.75, wy1 = 0.25 * sy, wz0 = 0.75, wz1 = 0.25 * sz;
        val = wz0 * (wy0 * (wx0 * e[cidx(C, I, J, K)] + wx1 * e[cidx(C, I2, J, K)]) +
                     wy1 * (wx0 * e[cidx(C, I, J2, K)] + wx1 * e[cidx(C, I2, J2, K)])) +
              wz1 * (wy0 * (wx0 * e[cidx(C, I, J, K2)] + wx1 * e[cidx(C, I2, J, K2)]) +
                     wy1 * (wx0 * e[cidx(C, I, J2, K2)] + wx1 * e[cidx(C, I2, J2, K2)]));
    }
    double* p = F.phi + cidx(F, i, j, k);
    store_images(p, *p + val, image_dx(F, i), image_dy(F, j));
}

// a7, bandwidth form: one thread per COARSE cell adds the interpolant to its 8 children.  The 27
// coarse values come from L1/L2 (the coarse array is 1/8 of the fine one); the children are read and
// written as four 16-byte x pairs, so a warp moves 512 contiguous bytes per row.  Interpolation is
// done axis by axis in the order x, y, z, i.e. the expression tree of k_prolong_add.
__global__ void __launch_bounds__(256, 4)
k_prolong_add2(LevelDev F, LevelDev C, int prolongation, double* fout)
{
    const int I = blockIdx.x * blockDim.x + threadIdx.x;
    const int J = blockIdx.y * blockDim.y + threadIdx.y;
    const int K = blockIdx.z;
    if (I >= C.nx || J >= C.ny) return;
    // the eight children, requested first: their HBM latency overlaps the (cache-resident) coarse reads below
    // fout: the array that receives phi + P e (same layout as F.phi; F.phi itself for the in-place form).  Out of place
    // (the level's ping-pong partner) the pass is two plain streams instead of a read-modify-write of the same lines.
    const size_t fo = cidx(F, 2 * I, 2 * J, 2 * K);
    const double2* const fp = reinterpret_cast<const double2*>(F.phi + fo);
    double2* const fq = reinterpret_cast<double2*>(fout + fo);
    const long long frow = F.cx / 2, fpl = (long long)F.cx * F.ry / 2;      // strides in double2 (cx is even here)
    double2 fv[2][2];
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj) fv[dk][dj] = fp[dk * fpl + dj * frow];
    double out[2][2][2];                      // [dk][dj][di]
    const double* __restrict__ e = C.phi;
    if (prolongation == 1) {
        const double v = e[cidx(C, I, J, K)];
#pragma unroll
        for (int q = 0; q < 8; ++q) out[q >> 2][(q >> 1) & 1][q & 1] = v;
    } else {
        int ix[3], jy[3], kz[3];
        double wx[3], wy[3], wz[3];           // weight of the neighbour on side 0 (low) / 2 (high)
        ix[1] = I; jy[1] = J; kz[1] = K;
#pragma unroll
        for (int sd = 0; sd < 3; sd += 2) {
            double sg = 1.0;
            ix[sd] = ghost_index(I + sd - 1, C.nx, C.bclo[0], C.bchi[0], sg); wx[sd] = 0.25 * sg;
            sg = 1.0;
            jy[sd] = ghost_index(J + sd - 1, C.ny, C.bclo[1], C.bchi[1], sg); wy[sd] = 0.25 * sg;
            sg = 1.0;
            kz[sd] = ghost_index(K + sd - 1, C.nz, C.bclo[2], C.bchi[2], sg); wz[sd] = 0.25 * sg;
        }
        long long jo[3], ko[3];
#pragma unroll
        for (int q = 0; q < 3; ++q) { jo[q] = (long long)C.cx * jy[q]; ko[q] = (long long)C.cx * C.ry * kz[q]; }
        double xi[3][3][2];                   // [dz][dy][child di] after x interpolation
#pragma unroll
        for (int dz = 0; dz < 3; ++dz)
#pragma unroll
            for (int dy = 0; dy < 3; ++dy) {
                const long long row = jo[dy] + ko[dz];
                const double c0 = e[row + ix[1]], cm = e[row + ix[0]], cp = e[row + ix[2]];
                xi[dz][dy][0] = 0.75 * c0 + wx[0] * cm;
                xi[dz][dy][1] = 0.75 * c0 + wx[2] * cp;
            }
#pragma unroll
        for (int di = 0; di < 2; ++di) {
            double yi[3][2];                  // [dz][child dj]
#pragma unroll
            for (int dz = 0; dz < 3; ++dz) {
                yi[dz][0] = 0.75 * xi[dz][1][di] + wy[0] * xi[dz][0][di];
                yi[dz][1] = 0.75 * xi[dz][1][di] + wy[2] * xi[dz][2][di];
            }
#pragma unroll
            for (int dj = 0; dj < 2; ++dj) {
                out[0][dj][di] = 0.75 * yi[1][dj] + wz[0] * yi[0][dj];
                out[1][dj][di] = 0.75 * yi[1][dj] + wz[2] * yi[2][dj];
            }
        }
    }
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj) {
            double2* p = fq + dk * fpl + dj * frow;
            double2 v = fv[dk][dj];
            v.x += out[dk][dj][0];
            v.y += out[dk][dj][1];
            store_images(p, v, image_dx(F, 2 * I), image_dy(F, 2 * J + dj));
        }
}

// ------------------------------------------------------------------------------------------------
// a9  ||rhs - L phi||inf  (block partial maxima; folded by k_reduce_final)
// ------------------------------------------------------------------------------------------------

__global__ void __launch_bounds__(256)
k_residual_norm(LevelDev L, double* __restrict__ part_sum, double* __restrict__ part_max)
{
    const int nrows = L.ny * L.nz;
    double m = 0.0;
    for (int row = blockIdx.x; row < nrows; row += gridDim.x) {
        const int j = row % L.ny, k = row / L.ny;
        for (int i = threadIdx.x; i < L.nx; i += blockDim.x) {
            double off, dg;
            stencil_sums(L, L.phi, i, j, k, off, dg);
            const size_t c = cidx(L, i, j, k);
            m = nanmax(m, fabs(L.rhs[c] - (off - L.phi[c] * dg)));
        }
    }
    block_reduce_store(0.0, m, part_sum, part_max, blockIdx.x);
}

// ------------------------------------------------------------------------------------------------
// a8  bottom solve: unpreconditioned BiCGStab, x0 = 0, rhat = r0, one thread block; dot products
// by warp shuffles + one shared-memory stage (deterministic).  Stops at ||r||2 <= tol ||f||2,
// maxit iterations, or breakdown (the current iterate is kept) -- reading A15.
// Singular problems: f is projected to zero mean first and x to zero mean last.
// Vectors r, rhat, p, v, s, t and the iterate x live in shared memory when 7 * nb doubles fit
// (use_smem; every vector operation is then an on-chip round trip instead of an L2 one: a value
// written by one thread and read by another does not stay in L1), else in `vecs` / L.phi.
// ------------------------------------------------------------------------------------------------

struct Dot2 { double a, b; };

// barrier among the first nt threads of the block (nt a multiple of 32): the solver runs on as many warps as
// the coarsest level has work for, also inside a larger block (k_coarse_tail)
__device__ __forceinline__ void group_sync(int nt) { asm volatile("bar.sync 1, %0;" ::"r"(nt) : "memory"); }

__device__ __forceinline__ Dot2 block_dot2(double a, double b, double* sh, int nt)
{
    a = warp_sum(a);
    b = warp_sum(b);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (nt + 31) >> 5;
    group_sync(nt);                      // protect sh from the previous use
    if (l == 0) { sh[2 * w] = a; sh[2 * w + 1] = b; }
    group_sync(nt);
    a = l < nw ? sh[2 * l] : 0.0;
    b = l < nw ? sh[2 * l + 1] : 0.0;
    Dot2 r;
    r.a = warp_sum(a);
    r.b = warp_sum(b);
    return r;
}

__device__ __forceinline__ double bottom_matvec_at(const LevelDev& L, const double* __restrict__ x, int c)
{
    const int i = c % L.nx, j = (c / L.nx) % L.ny, k = c / (L.nx * L.ny);
    double off, dg;
    stencil_sums(L, x, i, j, k, off, dg);
    return off - x[c] * dg;
}

// The solver proper, run by the first nt threads of one thread block: solves L x = f (x, f and the six work vectors may live in shared or
// global memory; x and f in the level's plain layout).  Returns the iteration count (same in every thread).
__device__ __forceinline__ int bicgstab_block(const LevelDev& L, double* x, const double* f, double* r, double* rhat,
                                              double* p, double* v, double* s, double* t, int maxit, double tol,
                                              int singular, double* sh, int nt)
{
    const int nb = L.nx * L.ny * L.nz;
    const int tid = threadIdx.x;                   // < nt: only the first nt threads of the block call this
    // one unknown per thread (the usual 4^3 bottom): the thread keeps its row of the matrix in registers
    // (coefficient 0 and the own index where the neighbour is outside the domain), so a matrix-vector product is
    // six shared-memory reads instead of index arithmetic, boundary branches and global coefficient loads
    const bool row_regs = nb <= nt;
    double ra[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, rdg = 0.0;
    int ri[6] = {0, 0, 0, 0, 0, 0};
    if (row_regs && tid < nb) {
        const int i = tid % L.nx, j = (tid / L.nx) % L.ny, k = tid / (L.nx * L.ny);
        ra[0] = L.ax[axidx(L, i, j, k)]; ra[1] = L.ax[axidx(L, i + 1, j, k)];
        ra[2] = L.ay[ayidx(L, i, j, k)]; ra[3] = L.ay[ayidx(L, i, j + 1, k)];
        ra[4] = L.az[azidx(L, i, j, k)]; ra[5] = L.az[azidx(L, i, j, k + 1)];
        rdg = ((ra[0] + ra[1]) + (ra[2] + ra[3])) + (ra[4] + ra[5]);
        const int n3[3] = {L.nx, L.ny, L.nz}, st[3] = {1, L.nx, L.nx * L.ny}, f3[3] = {i, j, k};
#pragma unroll
        for (int a = 0; a < 3; ++a)
#pragma unroll
            for (int sd = 0; sd < 2; ++sd) {
                const int g = f3[a] + (sd ? 1 : -1);
                int idx = tid + (sd ? st[a] : -st[a]);
                if (g < 0 || g >= n3[a]) {
                    if (L.bclo[a] == MAC_PERIODIC) idx = tid + (sd ? -(n3[a] - 1) * st[a] : (n3[a] - 1) * st[a]);
                    else { idx = tid; ra[2 * a + sd] = 0.0; }          // (rdg keeps the folded boundary coefficient)
                }
                ri[2 * a + sd] = idx;
            }
    }
    auto matvec = [&](const double* x, int c) -> double {
        if (!row_regs) return bottom_matvec_at(L, x, c);
        const double off = ra[0] * x[ri[0]] + ra[1] * x[ri[1]] + ra[2] * x[ri[2]] + ra[3] * x[ri[3]] + ra[4] * x[ri[4]] + ra[5] * x[ri[5]];
        return off - x[c] * rdg;
    };
    double fm = 0.0;
    if (singular) {
        double a = 0.0;
        for (int c = tid; c < nb; c += nt) a += f[c];
        fm = block_dot2(a, 0.0, sh, nt).a / (double)nb;
    }
    double rr = 0.0;
    for (int c = tid; c < nb; c += nt) {
        double fv = f[c] - fm;
        r[c] = fv; rhat[c] = fv; p[c] = 0.0; v[c] = 0.0; x[c] = 0.0;
        rr += fv * fv;
    }
    rr = block_dot2(rr, 0.0, sh, nt).a;            // (r,r) = (rhat,r)
    const double bnorm2 = rr;
    int it = 0;
    if (bnorm2 > 0.0 && bnorm2 == bnorm2) {
        const double stop2 = tol * tol * bnorm2;
        double rho = rr, rho_old = 1.0, alpha = 1.0, omega = 1.0;
        while (it < maxit && rr > stop2) {
            if (rho == 0.0) break;                                   // breakdown
            const double beta = it == 0 ? 0.0 : (rho / rho_old) * (alpha / omega);
            for (int c = tid; c < nb; c += nt) p[c] = r[c] + beta * (p[c] - omega * v[c]);
            group_sync(nt);
            double d = 0.0;
            for (int c = tid; c < nb; c += nt) { double y = matvec(p, c); v[c] = y; d += rhat[c] * y; }
            d = block_dot2(d, 0.0, sh, nt).a;
            if (d == 0.0) break;
            alpha = rho / d;
            double ss = 0.0;
            for (int c = tid; c < nb; c += nt) { double y = r[c] - alpha * v[c]; s[c] = y; ss += y * y; }
            ss = block_dot2(ss, 0.0, sh, nt).a;                          // also makes s visible
            ++it;
            if (ss <= stop2) {
                for (int c = tid; c < nb; c += nt) x[c] += alpha * p[c];
                rr = ss;
                break;
            }
            double ts = 0.0, tt = 0.0;
            for (int c = tid; c < nb; c += nt) { double y = matvec(s, c); t[c] = y; ts += y * s[c]; tt += y * y; }
            Dot2 q = block_dot2(ts, tt, sh, nt);
            if (q.b == 0.0) {
                for (int c = tid; c < nb; c += nt) x[c] += alpha * p[c];
                break;
            }
            omega = q.a / q.b;
            double r2 = 0.0, hr = 0.0;
            for (int c = tid; c < nb; c += nt) {
                x[c] += alpha * p[c] + omega * s[c];
                double y = s[c] - omega * t[c];
                r[c] = y;
                r2 += y * y;
                hr += rhat[c] * y;
            }
            q = block_dot2(r2, hr, sh, nt);
            rr = q.a;
            rho_old = rho;
            rho = q.b;
            if (omega == 0.0) break;
        }
    }
    if (singular) {                            // zero-mean x
        group_sync(nt);
        double a = 0.0;
        for (int c = tid; c < nb; c += nt) a += x[c];
        const double xm = block_dot2(a, 0.0, sh, nt).a / (double)nb;
        for (int c = tid; c < nb; c += nt) x[c] -= xm;
    }
    group_sync(nt);
    return it;
}

__global__ void __launch_bounds__(1024)
k_bottom_bicgstab(LevelDev L, double* vecs, int maxit, double tol, int singular,
                  int* __restrict__ iters_accum, int use_smem)
{
    __shared__ double sh[64];
    extern __shared__ double bottom_sm[];
    const int nb = L.nx * L.ny * L.nz;
    double* base = use_smem ? bottom_sm : vecs;
    double* x = use_smem ? base + 6 * (size_t)nb : L.phi;
    const int it = bicgstab_block(L, x, L.rhs, base, base + nb, base + 2 * (size_t)nb, base + 3 * (size_t)nb,
                                  base + 4 * (size_t)nb, base + 5 * (size_t)nb, maxit, tol, singular, sh, blockDim.x);
    if (use_smem)
        for (int c = threadIdx.x; c < nb; c += blockDim.x) L.phi[c] = x[c];
    if (threadIdx.x == 0 && iters_accum) *iters_accum += it;
}

// ------------------------------------------------------------------------------------------------
// a10  U <- U_edge - (1/rho_face) G phi  (Eq. 2).  WALL faces unchanged; OUTFLOW faces
// use the ghost -phi_0; periodic: entry n written equal to entry 0.
// ------------------------------------------------------------------------------------------------

template <int D>
__device__ __forceinline__ void correct_face(const GeoDev& G, const LevelDev& L, const double* __restrict__ phi,
                                             const double* __restrict__ rho, const double* __restrict__ rho0,
                                             double* __restrict__ vel, int i, int j, int k)
{
    const int n = D == 0 ? G.nx : (D == 1 ? G.ny : G.nz);
    const double h = D == 0 ? G.dx : (D == 1 ? G.dy : G.dz);
    const int f = D == 0 ? i : (D == 1 ? j : k);
    const bool per = G.bclo[D] == MAC_PERIODIC;
    const size_t sx = G.nx + (D == 0), sy = G.ny + (D == 1);
    const size_t fi = (size_t)i + sx * ((size_t)j + sy * (size_t)k);
    if (f == n && per) return;                       // written by the thread of face 0
    int lo = f - 1, hi = f;
    double glo = 1.0, ghi = 1.0;                     // multipliers of phi[lo], phi[hi]
    if (f == 0) {
        if (per) lo = n - 1;
        else { if (G.bclo[D] == MAC_WALL) return; lo = 0; glo = -1.0; }     // ghost = -phi_0
    } else if (f == n) {
        if (G.bchi[D] == MAC_WALL) return;
        hi = n - 1; ghi = -1.0;
    }
    auto cell = [&](int q) -> size_t { return cidx(L, D == 0 ? q : i, D == 1 ? q : j, D == 2 ? q : k); };
    const double grad = (ghi * phi[cell(hi)] - glo * phi[cell(lo)]) * (1.0 / h);
    const double rf = face_rho(rho_cell(G, rho, rho0, D == 0 ? lo : i, D == 1 ? lo : j, D == 2 ? lo : k),
                               rho_cell(G, rho, rho0, D == 0 ? hi : i, D == 1 ? hi : j, D == 2 ? hi : k), G.rho_mean);
    double rr;                                       // grad / rf, rf > 0 (validated by the coefficient pass)
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rr) : "d"(rf));
    rr = fma(fma(-rf, rr, 1.0), rr, rr);
    rr = fma(fma(-rf, rr, 1.0), rr, rr);
    const double qq = grad * rr;
    const double nv = vel[fi] - fma(fma(-rf, qq, grad), rr, qq);
    vel[fi] = nv;
    if (f == 0 && per) {
        const size_t fn = (size_t)(D == 0 ? n : i) + sx * ((size_t)(D == 1 ? n : j) + sy * (size_t)(D == 2 ? n : k));
        vel[fn] = nv;
    }
}

__global__ void __launch_bounds__(256)
k_correct(GeoDev G, LevelDev L, const double* __restrict__ phi, const double* __restrict__ rho,
          const double* __restrict__ rho0, double* __restrict__ u, double* __restrict__ v,
          double* __restrict__ w)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y * blockDim.y + threadIdx.y;
    int k = blockIdx.z;
    if (i > G.nx || j > G.ny) return;
    if (rho && i > 0 && i < G.nx && j > 0 && j < G.ny && k > 0 && k < G.nz) {
        // all three low faces are interior (all but a surface layer of threads): no boundary logic, one index each
        const size_t sx = (size_t)G.nx, sxy = sx * G.ny;
        const size_t c = (size_t)i + sx * ((size_t)j + (size_t)G.ny * k);
        const size_t cp = cidx(L, i, j, k), px = (size_t)L.cx, pxy = px * L.ry;
        double* pu = u + c + (size_t)j + (size_t)G.ny * k;            // (nx+1)-pitched rows
        double* pv = v + c + sx * k;                                   // (ny+1) rows per plane
        double* pw = w + c;
        const double p0 = phi[cp], r0 = __ldg(rho + c);
        const double pxm = phi[cp - 1], pym = phi[cp - px], pzm = phi[cp - pxy];
        const double rxm = __ldg(rho + c - 1), rym = __ldg(rho + c - sx), rzm = __ldg(rho + c - sxy);
        const double u0 = *pu, v0 = *pv, w0 = *pw;
        auto quot = [](double g, double rf) {                          // g / rf, rf > 0
            double rr;
            asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rr) : "d"(rf));
            rr = fma(fma(-rf, rr, 1.0), rr, rr);
            rr = fma(fma(-rf, rr, 1.0), rr, rr);
            const double qq = g * rr;
            return fma(fma(-rf, qq, g), rr, qq);
        };
        *pu = u0 - quot((p0 - pxm) * (1.0 / G.dx), face_rho(rxm, r0, G.rho_mean));
        *pv = v0 - quot((p0 - pym) * (1.0 / G.dy), face_rho(rym, r0, G.rho_mean));
        *pw = w0 - quot((p0 - pzm) * (1.0 / G.dz), face_rho(rzm, r0, G.rho_mean));
        return;
    }
    const bool ci = i < G.nx, cj = j < G.ny, ck = k < G.nz;
    if (cj && ck) correct_face<0>(G, L, phi, rho, rho0, u, i, j, k);
    if (ci && ck) correct_face<1>(G, L, phi, rho, rho0, v, i, j, k);
    if (ci && cj) correct_face<2>(G, L, phi, rho, rho0, w, i, j, k);
}

// ------------------------------------------------------------------------------------------------
// layout conversion for the step API: public face layout <-> internal (pitched) ax
// ------------------------------------------------------------------------------------------------

// which: 0 cell array `a` (phi or rhs), 2 ax, 3 ay, 4 az;  extents of the public array (ex, ey, ez)
__global__ void k_copy_level(LevelDev L, double* a, double* pub, int which, int ex, int ey, int ez, int to_public)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    int j = blockIdx.y * blockDim.y + threadIdx.y;
    int k = blockIdx.z;
    if (i >= ex || j >= ey || k >= ez) return;
    const size_t q = which == 2 ? axidx(L, i, j, k) : (which == 3 ? ayidx(L, i, j, k) : cidx(L, i, j, k));
    const size_t b = (size_t)i + (size_t)ex * ((size_t)j + (size_t)ey * k);
    if (to_public) pub[b] = a[q];
    else a[q] = pub[b];
}

// ================================================================================================
// Bandwidth forms of the once-per-projection kernels (a2, a4, a10).  One thread per (i, j) column
// marches a chunk of z-planes; x-neighbours come from the adjacent lane (warp shuffle), the plane
// below from registers.  Divisions by the grid spacing are multiplications by precomputed
// reciprocals; the base-state profile is evaluated once per face instead of once per cell side.
// ================================================================================================

struct GeoInv { double idx, idy, idz, idx2, idy2, idz2, idr; };

__device__ __forceinline__ double profile_eval_inv(const double* __restrict__ f, int nr, double idr, double r)
{
    double s = r * idr - 0.5;
    if (s <= 0.0) return __ldg(f);
    if (s >= (double)(nr - 1)) return __ldg(f + nr - 1);
    int m = (int)s;
    double t = s - (double)m;
    return (1.0 - t) * __ldg(f + m) + t * __ldg(f + m + 1);
}
__device__ __forceinline__ double beta_inv(const GeoDev& G, const GeoInv& I, const double* __restrict__ f, double x, double y, double z)
{
    return profile_eval_inv(f, G.nr, I.idr, radius(G, x, y, z));
}

// a2: face coefficients.  Threads cover the extended index space i in [0,nx], j in [0,ny]; planes k in [k0,k1]
// (the plane k == nz writes only the top z faces).  grid (ceil((nx+1)/64), ceil((ny+1)/4), chunks), block (64, 4)
__global__ void __launch_bounds__(256)
k_face_coeff2(GeoDev G, GeoInv I, LevelDev L, const double* __restrict__ beta0, const double* __restrict__ rho,
              const double* __restrict__ rho0, int zchunk, int* __restrict__ flags)
{
    const int i = blockIdx.x * 64 + threadIdx.x, j = blockIdx.y * 4 + threadIdx.y;
    const int k0 = blockIdx.z * zchunk, k1 = min(k0 + zchunk, G.nz + 1);
    if (i > G.nx || j > G.ny) return;
    const bool ci = i < G.nx, cj = j < G.ny;
#pragma unroll 4
    for (int k = k0; k < k1; ++k) {
        const bool ck = k < G.nz;
        double rf, cf;
        int fp;
        if (ci && cj && ck) {
            const double r = rho_cell(G, rho, rho0, i, j, k);
            if (!(r > 0.0) || !(r <= 1.79769313486231570e308)) atomicOr(flags, 1);
        }
        if (cj && ck) {
            face_rho_weight<0>(G, rho, rho0, i, j, k, rf, cf, fp);
            const double b = beta_inv(G, I, beta0, fp * G.dx, (j + 0.5) * G.dy, (k + 0.5) * G.dz);
            L.ax[axidx(L, i, j, k)] = cf * (b / rf) * I.idx2;
        }
        if (ci && ck) {
            face_rho_weight<1>(G, rho, rho0, i, j, k, rf, cf, fp);
            const double b = beta_inv(G, I, beta0, (i + 0.5) * G.dx, fp * G.dy, (k + 0.5) * G.dz);
            L.ay[ayidx(L, i, j, k)] = cf * (b / rf) * I.idy2;
        }
        if (ci && cj) {
            face_rho_weight<2>(G, rho, rho0, i, j, k, rf, cf, fp);
            const double b = beta_inv(G, I, beta0, (i + 0.5) * G.dx, (j + 0.5) * G.dy, fp * G.dz);
            L.az[azidx(L, i, j, k)] = cf * (b / rf) * I.idz2;
        }
    }
}
