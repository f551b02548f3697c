// sf_fp_noalloc.cu -- ct_fp_sf_noalloc: y = A x (Eq. 1) for callers that must not allocate.
//
// Who this is for.  ct_fp_sf keeps the xy-transposed copy of the volume (read by the views whose rays run mostly
// along x) in a buffer it obtains with cudaMalloc the first time a geometry needs it, and again whenever a larger
// batch arrives.  Some callers cannot live with that inside their iteration loop:
//   * a reconstruction that runs inside a process whose GPU memory has already been handed, whole, to another
//     allocator (a framework's caching pool, a fixed memory budget on a shared or partitioned GPU): a cudaMalloc
//     from a library then fails, or takes memory the owner believes it has;
//   * a loop with a latency bound (scanner-side, in-the-loop reconstruction): cudaMalloc synchronises the whole
//     device, so every stream of the process stalls behind it;
//   * code that is forbidden to allocate by policy after start-up (allocation audits, no-growth services).
// They create the geometry once, at start-up, where allocation is allowed (ct_geom_create uploads the per-view
// parameters), and from then on call this entry point, which never calls cudaMalloc, cudaFree, a stream-ordered
// allocator or any library routine that allocates: its scratch is the fixed array below, part of the loaded
// library image on every GPU that uses the library, held until the process exits.
//
// The price: a hard size limit (CT_FP_SF_NOALLOC_MAX_VOXELS), and ONE array per GPU shared by every call of every
// geometry and stream -- see include/ctsf.h for the rules that follow from that.
#include <cuda_runtime.h>

#include <mutex>

#include "ctsf_internal.h"

namespace {

// The scratch: room for one xy-transposed copy of batch * nz * ny * nx <= CT_FP_SF_NOALLOC_MAX_VOXELS voxels (16 MiB).
// In HOST code this name is only a handle the runtime knows the array by; it is not a device address and must
// never be passed to a kernel.  The address a kernel can use comes from cudaGetSymbolAddress (below).
static __device__ __align__(256) float g_noalloc_volT[CT_FP_SF_NOALLOC_MAX_VOXELS];

constexpr int NOALLOC_MAX_DEV = 64;
float *g_noalloc_addr[NOALLOC_MAX_DEV];      // device address of g_noalloc_volT on each GPU, looked up once
std::mutex g_noalloc_mu;

// Set-up, once per device, with that device current: ask the runtime where the array lives on THIS GPU (each GPU has
// its own copy at its own address).  This may load the library's device code onto the GPU, which is why the first
// call on a device should be made outside any stream capture.  Later calls only read the table.
float *noalloc_scratch_of_device(int dev)
{
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_addr[dev]) {
        void *p = nullptr;
        if (cudaGetSymbolAddress(&p, g_noalloc_volT) != cudaSuccess || !p) { cudaGetLastError(); return nullptr; }
        g_noalloc_addr[dev] = (float *)p;
    }
    return g_noalloc_addr[dev];
}

}  // namespace

extern "C" ct_status_t ct_fp_sf_noalloc(const ct_geom_t *g, const float *d_vol, float *d_proj, int32_t batch,
                                        ct_stream_t stream)
{
    if (!g || !d_vol || !d_proj || batch < 1) return CT_ERR_INVALID_ARG;
    if (((uintptr_t)d_vol | (uintptr_t)d_proj) & 3u) return CT_ERR_INVALID_ARG;            // fp32 elements
    const SfProblem &pr = g->prob;
    // the limit is checked first and for every geometry, also one whose views happen not to need the transposed
    // copy: whether a call is accepted depends on sizes only, never on the scan angles
    const double voxels = (double)batch * pr.nx * pr.ny * pr.nz;
    if (voxels > (double)CT_FP_SF_NOALLOC_MAX_VOXELS) return CT_ERR_UNSUPPORTED;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return CT_ERR_CUDA; }
    if (dev != g->device || dev < 0 || dev >= NOALLOC_MAX_DEV) return CT_ERR_INVALID_ARG;  // the geometry's GPU must be current
    float *scratch = noalloc_scratch_of_device(dev);
    if (!scratch) return CT_ERR_CUDA;

    int launches = 0;
    const float *d_volT = nullptr;
    if (ctsf_fp_needs_transpose(g, 0, 1, pr.n_views)) {
        // Every element of scratch[0 .. batch*nz*ny*nx) is overwritten here before the projector reads it, and the
        // projector reads nothing beyond that range: whatever an earlier call left in the array is never seen, so
        // nothing has to be cleared.
        const int nt = ctsf_fp_transpose(g, d_vol, scratch, batch, stream);
        if (nt < 0) return CT_ERR_CUDA;
        launches += nt;
        d_volT = scratch;
    }
    // with the transposed volume supplied (or not needed) the launcher takes no scratch of its own
    const int n = ctsf_launch_fp(g, d_vol, d_proj, batch, 0, 1, pr.n_views, stream, d_volT);
    if (n < 0) return CT_ERR_CUDA;
    g->last_launches.store(launches + n);
    return CT_OK;
}
