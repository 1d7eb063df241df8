// maestro_nodal.inl -- host side of the nodal (end-of-step) projection entry points of include/maestro_mac.h.
// Included at the end of maestro_mac.cu (it uses the handle, the reduction helpers and the launch macros there).
// Kernels: mac_nodal.cuh.  Readings N1..N10: DESIGN.md.

namespace {

NodLevel dev_nod(const maestro_mac_handle* H, int l)
{
    const NodHost& N = H->nod[l];
    NodLevel D;
    D.nx = N.n[0]; D.ny = N.n[1]; D.nz = N.n[2];
    D.NX = N.NX; D.NY = N.NY; D.CX = N.CX; D.CY = N.CY;
    double g[3], gsum = 0.0, gmax = 0.0;
    for (int a = 0; a < 3; ++a) {
        D.bclo[a] = H->d.bc_lo[a]; D.bchi[a] = H->d.bc_hi[a];
        g[a] = 1.0 / (N.h[a] * N.h[a]);
        gsum += g[a];
        if (g[a] > gmax) gmax = g[a];
    }
    for (int cls = 0; cls < 8; ++cls) {            // N2: K_ab / V for the 8 same / other-corner classes
        double w = 0.0;
        for (int d = 0; d < 3; ++d) {
            double t = ((cls >> d) & 1 ? -1.0 : 1.0) * g[d];
            for (int e = 0; e < 3; ++e)
                if (e != d) t *= ((cls >> e) & 1) ? (1.0 / 6.0) : (1.0 / 3.0);
            w += t;
        }
        D.w[cls] = w;
    }
    D.omega = gsum / (3.0 * gmax);                 // N7
    D.phi = N.phi; D.phi2 = N.phi2; D.rhs = N.rhs; D.sigma = N.sigma;
    return D;
}

void nod_dims(int ex, int ey, int ez, dim3* grid, dim3* block) { dims3(ex, ey, ez, grid, block); }

// grid of a node kernel that also leaves one partial per block: planes per block chosen so that the partials fit
void nod_dims_red(int ex, int ey, int ez, dim3* grid, dim3* block, int* zper)
{
    dims3(ex, ey, ez, grid, block);
    int zp = 1;
    while ((long)grid->x * grid->y * ((ez + zp - 1) / zp) > kMaxParts) zp *= 2;
    grid->z = (ez + zp - 1) / zp;
    *zper = zp;
}

#ifndef MAC_NOD_POINT_MAX
#define MAC_NOD_POINT_MAX 40000           // levels of at most this many nodes run the one-thread-per-node passes (k_nod_point)
#endif
bool nod_point_level(const maestro_mac_handle* H, int l) { return H->nod[l].nnode <= (size_t)MAC_NOD_POINT_MAX; }

// plan of the z-marching operator pass (k_nod_march, 32 x 8 node tiles, two blocks per SM): whole waves of tiles march
// every plane, the tiles of the last partial wave are cut into z-chunks (of at least 16 planes); the combination that
// minimises rounds x (planes per chunk + the planes a chunk loads directly); at most kMaxParts blocks
NodPlan nod_march_plan_sms(int sms, const NodLevel& L);
NodPlan nod_march_plan(const maestro_mac_handle* H, const NodLevel& L) { return nod_march_plan_sms(H->sms, L); }
NodPlan nod_march_plan_sms(int sms, const NodLevel& L)
{
    NodPlan P;
    P.tiles_x = (L.nx + 1 + 31) / 32;
    P.tiles = P.tiles_x * ((L.ny + 1 + 7) / 8);
    const int nzn = L.nz + 1, S = 2 * sms, maxchunk = nzn >= 16 ? nzn / 8 : 1;
    long best = -1;
    P.nfull = 0; P.nsplit = 1;
    for (int full = 0; full <= (P.tiles / S) * S; full += S) {
        const int rem = P.tiles - full;
        for (int n = 1; n <= maxchunk; ++n) {
            const int zc = (nzn + n - 1) / n, nn = (nzn + zc - 1) / zc;
            if ((long)full + (long)rem * nn > kMaxParts) break;
            const long cost = (long)(full / S) * (nzn + 4) + (((long)rem * nn + S - 1) / S) * (zc + 4);
            if (best < 0 || cost < best) { best = cost; P.nfull = full; P.nsplit = rem > 0 ? nn : 1; }
            if (rem == 0) break;
        }
    }
    P.zchunk = (nzn + P.nsplit - 1) / P.nsplit;
    P.ncta = P.nfull + (P.tiles - P.nfull) * P.nsplit;
    return P;
}

// folds nb block partials into scal[off] (sum) and scal[off + 1] (max)
int nod_fold(maestro_mac_handle* H, int nb, int off, cudaStream_t s)
{
    k_reduce_final<<<1, 1024, 0, s>>>(H->part_sum, H->part_max, nb, H->scal + off);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

// beta0 at the cell centres of level 0 in the public cell layout: staged in level 0's second phi buffer (allocation
// base; (nx+3)(ny+3)(nz+3) >= nx ny nz entries), which is free between nod_do_sigma and the first sweep
double* nod_bcell(const maestro_mac_handle* H) { return H->nod[0].phi2 - H->nod[0].onode; }

int nod_sig_ghosts(maestro_mac_handle* H, int l, cudaStream_t s)
{
    const NodLevel L = dev_nod(H, l);
    dim3 g, b;
    nod_dims(L.nx + 2, L.ny + 2, L.nz + 2, &g, &b);
    k_nod_sig_ghosts<<<g, b, 0, s>>>(L);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

int nod_phi_ghosts(maestro_mac_handle* H, int l, double* a, cudaStream_t s)
{
    const NodLevel L = dev_nod(H, l);
    dim3 g, b;
    nod_dims(L.nx + 3, L.ny + 3, L.nz + 3, &g, &b);
    k_nod_phi_ghosts<<<g, b, 0, s>>>(L, a);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

// every nodal phi buffer := 0, ghosts included (they must hold finite values: the operator multiplies them by sigma = 0)
int nod_zero_phi(maestro_mac_handle* H, cudaStream_t s)
{
    for (int l = 0; l < H->nlev; ++l) {
        const NodHost& N = H->nod[l];
        CUDA_OK(cudaMemsetAsync(N.phi - N.onode, 0, N.anode * sizeof(double), s));
        CUDA_OK(cudaMemsetAsync(N.phi2 - N.onode, 0, N.anode * sizeof(double), s));
    }
    return MAESTRO_MAC_OK;
}

int nod_do_sigma(maestro_mac_handle* H, const double* beta0, const double* rho0, const double* rho, cudaStream_t s)
{
    dim3 g, b;
    const GeoDev G = dev_geo(H);
    CUDA_OK(cudaMemsetAsync(H->flags, 0, 16 * sizeof(int), s));
    nod_dims(G.nx, G.ny, G.nz, &g, &b);
    k_nod_sigma<<<g, b, 0, s>>>(G, dev_nod(H, 0), beta0, rho, rho0, nod_bcell(H), H->flags);
    LAUNCHED(H);
    int rc;
    if ((rc = nod_sig_ghosts(H, 0, s)) != 0) return rc;
    for (int l = 0; l + 1 < H->nlev; ++l) {
        const NodLevel C = dev_nod(H, l + 1);
        nod_dims(C.nx, C.ny, C.nz, &g, &b);
        k_nod_coarsen_sigma<<<g, b, 0, s>>>(dev_nod(H, l), C);
        LAUNCHED(H);
        if ((rc = nod_sig_ghosts(H, l + 1, s)) != 0) return rc;
    }
    return MAESTRO_MAC_OK;
}

// rhs on level 0 (after nod_do_sigma of the same call); scal[0..1] = sum, max of the final rhs, scal[2] = removed sum
int nod_do_rhs(maestro_mac_handle* H, const double* u, const double* v, const double* w, const double* S, cudaStream_t s)
{
    const NodLevel L = dev_nod(H, 0);
    dim3 g, b;
    int zper;
    nod_dims_red(L.nx + 1, L.ny + 1, L.nz + 1, &g, &b, &zper);
    const int nb = (int)(g.x * g.y * g.z);
    const double* hh = H->nod[0].h;
    k_nod_rhs<<<g, b, 0, s>>>(L, 1.0 / (4.0 * hh[0]), 1.0 / (4.0 * hh[1]), 1.0 / (4.0 * hh[2]), nod_bcell(H), u, v, w, S,
                              H->part_sum, H->part_max, zper);
    LAUNCHED(H);
    int rc;
    if ((rc = nod_fold(H, nb, 0, s)) != 0) return rc;
    if (H->singular) {                             // N5: remove the uniform volumetric source m = sum / cells
        k_publish<<<1, 32, 0, s>>>(H->scal + 2, H->scal, 1);
        k_nod_shift<true, false><<<g, b, 0, s>>>(L, L.rhs, H->scal + 2, 1.0 / (double)H->nod[0].ncell, H->part_sum, H->part_max, zper);
        LAUNCHED(H);
        if ((rc = nod_fold(H, nb, 0, s)) != 0) return rc;
    } else {
        CUDA_OK(cudaMemsetAsync(H->scal + 2, 0, sizeof(double), s));
    }
    return MAESTRO_MAC_OK;
}

// One Jacobi sweep on level l (phi -> phi2, then the roles swap unless swap == false).  norm_parts != NULL: the sweep
// also leaves block maxima of |rhs - L phi_in| in part_max and their count in *norm_parts.
int nod_do_jacobi(maestro_mac_handle* H, int l, cudaStream_t s, int* norm_parts = nullptr, bool swap = true)
{
    const NodLevel L = dev_nod(H, l);
    if (nod_point_level(H, l)) {
        dim3 g, b;
        nod_dims(L.nx + 1, L.ny + 1, L.nz + 1, &g, &b);
        if (norm_parts) {
            if ((long)g.x * g.y * g.z > kMaxParts) return MAESTRO_MAC_ERR_UNSUPPORTED;
            *norm_parts = (int)(g.x * g.y * g.z);
            k_nod_point<NOD_JACOBI | NOD_NORM><<<g, b, 0, s>>>(L, L.phi, L.phi2, H->part_sum, H->part_max);
        } else
            k_nod_point<NOD_JACOBI><<<g, b, 0, s>>>(L, L.phi, L.phi2, nullptr, nullptr);
        LAUNCHED(H);
        if (swap) { double* t = H->nod[l].phi; H->nod[l].phi = H->nod[l].phi2; H->nod[l].phi2 = t; }
        return MAESTRO_MAC_OK;
    }
    const NodPlan plan = nod_march_plan(H, L);
    const dim3 g(plan.ncta, 1, 1);
    const NodHost& N = H->nod[l];
    const CUtensorMap& tin = N.phi == N.phi_a ? N.tm_phi : N.tm_phi2;
    if (norm_parts) {
        *norm_parts = plan.ncta;
        k_nod_march<NOD_JACOBI | NOD_NORM><<<g, dim3(32, 8), 0, s>>>(tin, N.tm_sig, N.tm_rhs, L, L.phi, L.phi2, H->part_max, plan);
    } else
        k_nod_march<NOD_JACOBI><<<g, dim3(32, 8), 0, s>>>(tin, N.tm_sig, N.tm_rhs, L, L.phi, L.phi2, nullptr, plan);
    LAUNCHED(H);
    if (swap) { double* t = H->nod[l].phi; H->nod[l].phi = H->nod[l].phi2; H->nod[l].phi2 = t; }
    return MAESTRO_MAC_OK;
}

int nod_do_smooth(maestro_mac_handle* H, int l, int nsweeps, cudaStream_t s)
{
    for (int q = 0; q < nsweeps; ++q) {
        const int rc = nod_do_jacobi(H, l, s);
        if (rc != 0) return rc;
    }
    return MAESTRO_MAC_OK;
}

// rhs[l+1] = (1/8) P^T (rhs[l] - L phi[l]), phi[l+1] = 0; the residual passes through phi2[l]
int nod_do_residual_restrict(maestro_mac_handle* H, int l, cudaStream_t s)
{
    const NodLevel F = dev_nod(H, l), C = dev_nod(H, l + 1);
    dim3 g, b;
    if (nod_point_level(H, l)) {
        nod_dims(F.nx + 1, F.ny + 1, F.nz + 1, &g, &b);
        k_nod_point<NOD_RESID><<<g, b, 0, s>>>(F, F.phi, F.phi2, nullptr, nullptr);
    } else {
        const NodPlan plan = nod_march_plan(H, F);
        const NodHost& N = H->nod[l];
        k_nod_march<NOD_RESID><<<dim3(plan.ncta, 1, 1), dim3(32, 8), 0, s>>>(N.phi == N.phi_a ? N.tm_phi : N.tm_phi2, N.tm_sig, N.tm_rhs, F, F.phi, F.phi2, nullptr, plan);
    }
    LAUNCHED(H);
    nod_dims(C.nx + 1, C.ny + 1, C.nz + 1, &g, &b);
    k_nod_restrict<<<g, b, 0, s>>>(F, C, F.phi2);
    LAUNCHED(H);
    CUDA_OK(cudaMemsetAsync(H->nod[l + 1].phi - H->nod[l + 1].onode, 0, H->nod[l + 1].anode * sizeof(double), s));   // coarse phi = 0
    return MAESTRO_MAC_OK;
}

int nod_do_prolong(maestro_mac_handle* H, int l, cudaStream_t s)
{
    const NodLevel F = dev_nod(H, l), C = dev_nod(H, l + 1);
    dim3 g, b;
    nod_dims(C.nx + 1, C.ny + 1, C.nz + 1, &g, &b);
    k_nod_prolong_add2<<<g, b, 0, s>>>(F, C);                       // one thread per coarse node
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

int nod_do_bottom(maestro_mac_handle* H, cudaStream_t s)
{
    const int l = H->nlev - 1;
    const int nb = (int)H->nod[l].nnode;
    const int threads = nb >= 1024 ? 1024 : ((nb + 31) / 32) * 32;
    if (nb <= 128 && H->nod[l].anode <= (size_t)kNodSmallMax) {      // one node per thread, its operator row in registers
        k_nod_bottom_small<<<1, threads, 0, s>>>(dev_nod(H, l), H->d.bottom_max_iter, H->d.bottom_rel_tol, H->singular, H->flags + 1);
        LAUNCHED(H);
        return MAESTRO_MAC_OK;
    }
    k_nod_bottom<<<1, threads, 0, s>>>(dev_nod(H, l), H->nod_vecs + H->nod[l].onode, (long long)H->nod[l].anode, H->d.bottom_max_iter,
                                      H->d.bottom_rel_tol, H->singular, H->flags + 1);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

int nod_do_vcycle(maestro_mac_handle* H, cudaStream_t s, int pre_done = 0)
{
    int rc;
    const int last = H->nlev - 1;
    for (int l = 0; l < last; ++l) {
        if ((rc = nod_do_smooth(H, l, H->d.nu_pre - (l == 0 ? pre_done : 0), s)) != 0) return rc;
        if ((rc = nod_do_residual_restrict(H, l, s)) != 0) return rc;
    }
    if ((rc = nod_do_bottom(H, s)) != 0) return rc;
    for (int l = last - 1; l >= 0; --l) {
        if ((rc = nod_do_prolong(H, l, s)) != 0) return rc;
        if ((rc = nod_do_smooth(H, l, H->d.nu_post, s)) != 0) return rc;
    }
    return MAESTRO_MAC_OK;
}

// max |rhs - L phi| over the unknowns of level l into scal[4]
int nod_do_residual_norm(maestro_mac_handle* H, int l, cudaStream_t s)
{
    const NodLevel L = dev_nod(H, l);
    if (nod_point_level(H, l)) {
        dim3 g, b;
        nod_dims(L.nx + 1, L.ny + 1, L.nz + 1, &g, &b);
        if ((long)g.x * g.y * g.z > kMaxParts) return MAESTRO_MAC_ERR_UNSUPPORTED;
        k_nod_point<NOD_RESID | NOD_NORM><<<g, b, 0, s>>>(L, L.phi, nullptr, H->part_sum, H->part_max);
        LAUNCHED(H);
        return nod_fold(H, (int)(g.x * g.y * g.z), 3, s);
    }
    const NodPlan plan = nod_march_plan(H, L);
    const NodHost& N = H->nod[l];
    k_nod_march<NOD_RESID | NOD_NORM><<<dim3(plan.ncta, 1, 1), dim3(32, 8), 0, s>>>(N.phi == N.phi_a ? N.tm_phi : N.tm_phi2, N.tm_sig, N.tm_rhs, L,
                                                                                    L.phi, nullptr, H->part_max, plan);
    LAUNCHED(H);
    return nod_fold(H, plan.ncta, 3, s);
}

int nod_do_correct(maestro_mac_handle* H, const double* phi, const double* rho0, const double* rho, double* u, double* v,
                   double* w, cudaStream_t s)
{
    const NodLevel L = dev_nod(H, 0);
    dim3 g, b;
    nod_dims(L.nx, L.ny, L.nz, &g, &b);
    const double* hh = H->nod[0].h;
    k_nod_correct<<<g, b, 0, s>>>(L, dev_geo(H), 1.0 / (4.0 * hh[0]), 1.0 / (4.0 * hh[1]), 1.0 / (4.0 * hh[2]), phi, rho, rho0, u, v, w);
    LAUNCHED(H);
    return MAESTRO_MAC_OK;
}

}  // namespace

extern "C" int maestro_mac_nodal_project(maestro_mac_handle* H, const double* beta0, const double* rho0, const double* rho,
                                         double* uc, double* vc, double* wc, const double* S, double* phi,
                                         maestro_mac_stats* stats, void* cuda_stream)
{
    if (!H || !H->has_nodal || !beta0 || !uc || !vc || !wc || (!rho && !rho0)) return MAESTRO_MAC_ERR_ARG;
    if (uc == vc || uc == wc || vc == wc || (phi && (phi == uc || phi == vc || phi == wc || phi == rho || phi == S)))
        return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const maestro_mac_desc& d = H->d;
    maestro_mac_stats st;
    std::memset(&st, 0, sizeof(st));
    st.singular = H->singular;
    st.levels = H->nlev;
    H->launches = 0;
    H->sm_used = H->sm_launches = H->sm_sweeps = 0;
    H->deferred = 0;
    int rc, result = MAESTRO_MAC_OK;
    NodHost& N0 = H->nod[0];

    CUDA_OK(cudaEventRecord(H->ev[0], s));
    if ((rc = nod_do_sigma(H, beta0, rho0, rho, s)) != 0) return rc;
    if ((rc = nod_do_rhs(H, uc, vc, wc, S, s)) != 0) return rc;
    if (publish_scal(H, 0, 3, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    if (publish_flags(H, 0, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    if ((rc = nod_zero_phi(H, s)) != 0) return rc;                          // N9: phi = 0 (and finite ghosts everywhere)
    CUDA_OK(cudaEventRecord(H->ev[1], s));
    CUDA_OK(cudaStreamSynchronize(s));
    st.rhs_norm_inf = H->host_scal[1];
    st.rhs_mean_removed = H->singular ? H->host_scal[2] / (double)N0.ncell : 0.0;
    if (H->host_flags[0] != 0 || !std::isfinite(st.rhs_norm_inf) || !std::isfinite(H->host_scal[0])) {
        if (stats) *stats = st;
        return MAESTRO_MAC_ERR_NONFINITE;
    }
    const bool trivial = st.rhs_norm_inf == 0.0;
    if (!trivial) {
        result = d.rel_tol > 0.0 ? MAESTRO_MAC_NOT_CONVERGED : MAESTRO_MAC_OK;
        if (d.rel_tol > 0.0) {
            // the Jacobi sweep forms rhs - L phi of its input: the stop test rides on the first pre-sweep of the next cycle
            const bool ride = d.stop_test == 0 && d.nu_pre >= 1 && H->nlev >= 2;
            int pre_done = 0;
            while (st.cycles < d.max_cycles) {
                if ((rc = nod_do_vcycle(H, s, pre_done)) != 0) return rc;
                pre_done = 0;
                const bool spec = ride && st.cycles + 1 < d.max_cycles;
                if (spec) {
                    int nparts = 0;
                    if ((rc = nod_do_jacobi(H, 0, s, &nparts, false)) != 0) return rc;
                    if ((rc = nod_fold(H, nparts, 3, s)) != 0) return rc;
                } else if ((rc = nod_do_residual_norm(H, 0, s)) != 0) return rc;
                if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
                CUDA_OK(cudaStreamSynchronize(s));
                st.res_norm_inf = H->host_scal[4];
                const double rel = st.res_norm_inf / st.rhs_norm_inf;
                if (st.cycles < 128) st.res_history[st.cycles] = rel;
                ++st.cycles;
                if (rel != rel) { result = MAESTRO_MAC_ERR_NONFINITE; break; }
                if (rel <= d.rel_tol) { result = MAESTRO_MAC_OK; break; }
                if (spec) {
                    double* t = N0.phi; N0.phi = N0.phi2; N0.phi2 = t;
                    pre_done = 1;
                }
            }
        } else {
            for (; st.cycles < d.max_cycles; ++st.cycles)
                if ((rc = nod_do_vcycle(H, s)) != 0) return rc;
        }
    }
    CUDA_OK(cudaEventRecord(H->ev[2], s));
    const NodLevel L0 = dev_nod(H, 0);
    dim3 g, b;
    if (!trivial && result != MAESTRO_MAC_ERR_NONFINITE) {
        if (H->singular) {                         // N5: zero w-weighted mean
            int zper;
            nod_dims_red(L0.nx + 1, L0.ny + 1, L0.nz + 1, &g, &b, &zper);
            const int nb = (int)(g.x * g.y * g.z);
            k_nod_shift<false, true><<<g, b, 0, s>>>(L0, L0.phi, nullptr, 0.0, H->part_sum, H->part_max, zper);
            LAUNCHED(H);
            if ((rc = nod_fold(H, nb, 6, s)) != 0) return rc;
            k_nod_shift<false, false><<<g, b, 0, s>>>(L0, L0.phi, H->scal + 6, 1.0 / (double)N0.ncell, H->part_sum, H->part_max, zper);
            LAUNCHED(H);
        }
        if ((rc = nod_do_correct(H, L0.phi, rho0, rho, uc, vc, wc, s)) != 0) return rc;
    }
    nod_dims(L0.nx + 1, L0.ny + 1, L0.nz + 1, &g, &b);
    if (phi) {
        k_nod_copy<<<g, b, 0, s>>>(L0, L0.phi, phi, 1, 1, 1);
        LAUNCHED(H);
    }
    CUDA_OK(cudaEventRecord(H->ev[3], s));
    if (publish_flags(H, 1, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    CUDA_OK(cudaStreamSynchronize(s));
    collect_timings(H, st);
    if (d.rel_tol == 0.0 && !trivial) {
        if (H->singular && (rc = nod_phi_ghosts(H, 0, H->nod[0].phi, s)) != 0) return rc;   // the mean shift left the images stale
        if ((rc = nod_do_residual_norm(H, 0, s)) != 0) return rc;
        if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
        CUDA_OK(cudaStreamSynchronize(s));
        st.res_norm_inf = H->host_scal[4];
    }
    st.gpu_launches = H->launches;
    H->last = st;
    if (stats) *stats = st;
    return result;
}

// ---- step API of the nodal projection ---------------------------------------------------------------------------

static int nod_level_copy(maestro_mac_handle* H, int level, int which, double* pub, int to_public, cudaStream_t s)
{
    if (!H || !H->has_nodal || !pub || level < 0 || level >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    const NodLevel L = dev_nod(H, level);
    double* internal = which == MAESTRO_MAC_NODAL_PHI ? L.phi : (which == MAESTRO_MAC_NODAL_RHS ? L.rhs : (which == MAESTRO_MAC_NODAL_SIGMA ? L.sigma : nullptr));
    if (!internal) return MAESTRO_MAC_ERR_ARG;
    const int node = which == MAESTRO_MAC_NODAL_SIGMA ? 0 : 1;
    dim3 g, b;
    nod_dims(L.nx + node, L.ny + node, L.nz + node, &g, &b);
    k_nod_copy<<<g, b, 0, s>>>(L, internal, pub, node, to_public, which == MAESTRO_MAC_NODAL_PHI ? 1 : 0);
    LAUNCHED(H);
    if (to_public) return MAESTRO_MAC_OK;
    if (which == MAESTRO_MAC_NODAL_SIGMA) return nod_sig_ghosts(H, level, s);
    if (which == MAESTRO_MAC_NODAL_PHI) {          // the second buffer must hold finite ghosts too (see nod_zero_phi)
        const NodHost& N = H->nod[level];
        CUDA_OK(cudaMemsetAsync(N.phi2 - N.onode, 0, N.anode * sizeof(double), s));
        return nod_phi_ghosts(H, level, internal, s);
    }
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_nodal_level_get(maestro_mac_handle* H, int level, int which, double* dst, void* cuda_stream)
{
    return nod_level_copy(H, level, which, dst, 1, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_level_set(maestro_mac_handle* H, int level, int which, const double* src, void* cuda_stream)
{
    return nod_level_copy(H, level, which, const_cast<double*>(src), 0, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_sigma(maestro_mac_handle* H, const double* beta0, const double* rho0, const double* rho,
                                            void* cuda_stream)
{
    if (!H || !H->has_nodal || !beta0 || (!rho && !rho0)) return MAESTRO_MAC_ERR_ARG;
    return nod_do_sigma(H, beta0, rho0, rho, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_rhs(maestro_mac_handle* H, const double* uc, const double* vc, const double* wc,
                                          const double* S, double* rhs_norm_inf, double* mean_removed, void* cuda_stream)
{
    if (!H || !H->has_nodal || !uc || !vc || !wc) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int rc = nod_do_rhs(H, uc, vc, wc, S, s);
    if (rc != 0) return rc;
    if (publish_scal(H, 0, 3, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    CUDA_OK(cudaStreamSynchronize(s));
    if (rhs_norm_inf) *rhs_norm_inf = H->host_scal[1];
    if (mean_removed) *mean_removed = H->singular ? H->host_scal[2] / (double)H->nod[0].ncell : 0.0;
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_nodal_step_smooth(maestro_mac_handle* H, int level, int nsweeps, void* cuda_stream)
{
    if (!H || !H->has_nodal || level < 0 || level >= H->nlev || nsweeps < 0) return MAESTRO_MAC_ERR_ARG;
    return nod_do_smooth(H, level, nsweeps, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_residual_restrict(maestro_mac_handle* H, int level, void* cuda_stream)
{
    if (!H || !H->has_nodal || level < 0 || level + 1 >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    return nod_do_residual_restrict(H, level, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_prolong(maestro_mac_handle* H, int level, void* cuda_stream)
{
    if (!H || !H->has_nodal || level < 0 || level + 1 >= H->nlev) return MAESTRO_MAC_ERR_ARG;
    return nod_do_prolong(H, level, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_bottom(maestro_mac_handle* H, void* cuda_stream)
{
    if (!H || !H->has_nodal) return MAESTRO_MAC_ERR_ARG;
    return nod_do_bottom(H, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_vcycle(maestro_mac_handle* H, void* cuda_stream)
{
    if (!H || !H->has_nodal) return MAESTRO_MAC_ERR_ARG;
    return nod_do_vcycle(H, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_nodal_step_residual_norm(maestro_mac_handle* H, int level, double* norm_inf, void* cuda_stream)
{
    if (!H || !H->has_nodal || level < 0 || level >= H->nlev || !norm_inf) return MAESTRO_MAC_ERR_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int rc = nod_do_residual_norm(H, level, s);
    if (rc != 0) return rc;
    if (publish_scal(H, 4, 1, s) != 0) return MAESTRO_MAC_ERR_CUDA;
    CUDA_OK(cudaStreamSynchronize(s));
    *norm_inf = H->host_scal[4];
    return MAESTRO_MAC_OK;
}

extern "C" int maestro_mac_nodal_step_correct(maestro_mac_handle* H, const double* rho0, const double* rho, double* uc,
                                              double* vc, double* wc, void* cuda_stream)
{
    if (!H || !H->has_nodal || !uc || !vc || !wc || (!rho && !rho0)) return MAESTRO_MAC_ERR_ARG;
    return nod_do_correct(H, H->nod[0].phi, rho0, rho, uc, vc, wc, (cudaStream_t)cuda_stream);
}

extern "C" int maestro_mac_plan_query(int which, int nx, int ny, int nz, int sms, int info[8])
{
    if (!info || nx < 1 || ny < 1 || nz < 1 || sms < 1 || (which != 0 && which != 1)) return MAESTRO_MAC_ERR_ARG;
    for (int q = 0; q < 8; ++q) info[q] = 0;
    if (which == 0) {
        LevelDev L;
        std::memset(&L, 0, sizeof(L));
        L.nx = nx; L.ny = ny; L.nz = nz;
        const t2::T2Plan P = t2_plan(L, sms);
        info[0] = P.tiles_x; info[1] = P.tiles; info[2] = P.nfull; info[3] = P.nsplit; info[4] = P.zchunk; info[5] = P.ncta;
    } else {
        NodLevel L;
        std::memset(&L, 0, sizeof(L));
        L.nx = nx; L.ny = ny; L.nz = nz;
        const NodPlan P = nod_march_plan_sms(sms, L);
        info[0] = P.tiles_x; info[1] = P.tiles; info[2] = P.nfull; info[3] = P.nsplit; info[4] = P.zchunk; info[5] = P.ncta;
    }
    return MAESTRO_MAC_OK;
}
