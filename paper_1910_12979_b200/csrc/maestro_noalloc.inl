// maestro_noalloc.inl -- ONE entry point that allocates nothing, for callers that cannot call cudaMalloc (code under
// CUDA graph capture, tight serving loops, harnesses that forbid it): the lateral average rho -> rho0(r) of
// PAPER.md:39 (maestro_mac_lateral_average) without a handle and without a workspace.  Included at the end of
// maestro_mac.cu (same translation unit as the kernels it launches and as the scratch array below).
//
// The scratch of that operation -- per-block partial sums and counts of every sample, and the folded counts -- lives in
// a file-scope device array of a fixed, modest size: kNoAllocBytes = 3.77 MiB for profiles of up to
// MAESTRO_MAC_NOALLOC_MAX_NR = 2048 samples (spherical 1024^3 with dr = dx/2 needs 1775).  Every GPU that loads the
// library holds it until the process exits.  The kernels are the ones of the handle path (k_lateral_sum,
// k_average_finish: fixed-order sums, same launch shape), given the address of this array instead of workspace
// pointers, so the result is bit-identical to maestro_mac_lateral_average on the same device.
//
// In host code the array's NAME is a host-side stand-in, not a device address: the address is taken once per device,
// with that device current, by cudaGetSymbolAddress (checked), and only that pointer is passed to kernels.
// All calls share the array.  It keeps the last call's contents; nothing in it has to start at zero: every word a call
// reads (the partials of the nb blocks it launches, the nr folded counts) is written earlier by the same call, so stale
// data of a larger previous call is never read.  Calls that overlap on the GPU (different streams, or different host
// threads without ordering) race on it: serialise them.
namespace {

constexpr int kNoAllocMaxNr = MAESTRO_MAC_NOALLOC_MAX_NR;
constexpr size_t kNoAllocSumBytes = (size_t)kLateralBlocks * kNoAllocMaxNr * sizeof(double);      // partial sums
constexpr size_t kNoAllocCntBytes = (size_t)kLateralBlocks * kNoAllocMaxNr * sizeof(unsigned);    // partial counts
constexpr size_t kNoAllocBytes = kNoAllocSumBytes + kNoAllocCntBytes + (size_t)kNoAllocMaxNr * sizeof(unsigned long long);
static_assert(kNoAllocSumBytes % 256 == 0 && kNoAllocCntBytes % 256 == 0, "sub-arrays stay 256-byte aligned");
static_assert((size_t)kNoAllocMaxNr * 12 <= kLateralSmem, "one warp's private bins fit the kernel's shared memory");

constexpr int kNoAllocMaxDevices = 64;
struct NoAllocDevice { unsigned char* scratch; int sms; int ready; };
NoAllocDevice g_noalloc_dev[kNoAllocMaxDevices];       // zero-initialised; filled once per device under the mutex below
std::mutex g_noalloc_mutex;

}  // namespace

static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

namespace {

// set-up of the current device (once): the scratch array's device address, the SM count, the kernel's shared-memory
// opt-in.  No allocation: cudaGetSymbolAddress returns the address of memory that came with the module.
int noalloc_device(NoAllocDevice** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return MAESTRO_MAC_ERR_CUDA;
    if (dev < 0 || dev >= kNoAllocMaxDevices) return MAESTRO_MAC_ERR_UNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    NoAllocDevice& D = g_noalloc_dev[dev];
    if (!D.ready) {
        unsigned char* ptr = nullptr;
        if (cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch) != cudaSuccess || !ptr) return MAESTRO_MAC_ERR_CUDA;
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return MAESTRO_MAC_ERR_CUDA;
        if (cudaFuncSetAttribute(k_lateral_sum, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kLateralSmem) != cudaSuccess)
            return MAESTRO_MAC_ERR_CUDA;
        D.scratch = ptr;
        D.sms = sms;
        D.ready = 1;
    }
    *out = &D;
    return MAESTRO_MAC_OK;
}

}  // namespace

extern "C" int maestro_mac_lateral_average_noalloc(const maestro_mac_desc* desc, const double* rho, double* rho0,
                                                   void* cuda_stream)
{
    if (!desc || !rho || !rho0) return MAESTRO_MAC_ERR_ARG;
    maestro_mac_desc d;
    int rc = validate_and_default(desc, &d);
    if (rc != MAESTRO_MAC_OK) return rc;
    if (d.nr > kNoAllocMaxNr) return MAESTRO_MAC_ERR_UNSUPPORTED;       // the static scratch holds MAESTRO_MAC_NOALLOC_MAX_NR samples
    NoAllocDevice* D = nullptr;
    if ((rc = noalloc_device(&D)) != MAESTRO_MAC_OK) return rc;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    GeoDev G;
    G.nx = d.nx; G.ny = d.ny; G.nz = d.nz;
    G.dx = d.dx[0]; G.dy = d.dx[1]; G.dz = d.dx[2];
    for (int a = 0; a < 3; ++a) { G.bclo[a] = d.bc_lo[a]; G.bchi[a] = d.bc_hi[a]; }
    G.geometry = d.geometry; G.nr = d.nr; G.dr = d.dr;
    G.cx = d.center[0]; G.cy = d.center[1]; G.cz = d.center[2];
    G.rho_mean = d.rho_mean;
    // the launch shape of maestro_mac_lateral_average: as many warps per block as private bin sets fit in shared
    // memory, one block per SM (at most kLateralBlocks, at most one per row)
    const int nr = d.nr, rows = d.ny * d.nz;
    int nwarp = (int)(kLateralSmem / ((size_t)nr * 12));
    if (nwarp > 8) nwarp = 8;
    int nb = D->sms < kLateralBlocks ? D->sms : kLateralBlocks;
    if (nb > rows) nb = rows;
    double* psum = reinterpret_cast<double*>(D->scratch);
    unsigned* pcnt = reinterpret_cast<unsigned*>(D->scratch + kNoAllocSumBytes);
    unsigned long long* cnt = reinterpret_cast<unsigned long long*>(D->scratch + kNoAllocSumBytes + kNoAllocCntBytes);
    k_lateral_sum<<<nb, 32 * nwarp, (size_t)nwarp * nr * 12, s>>>(G, rho, psum, pcnt);
    if (cudaPeekAtLastError() != cudaSuccess) return MAESTRO_MAC_ERR_CUDA;
    k_average_finish<<<1, 256, 0, s>>>(nr, nb, psum, pcnt, cnt, rho0);
    return cudaPeekAtLastError() == cudaSuccess ? MAESTRO_MAC_OK : MAESTRO_MAC_ERR_CUDA;
}
