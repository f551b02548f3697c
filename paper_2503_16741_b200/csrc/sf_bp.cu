// sf_bp.cu -- ct_bp_sf: voxel-driven SF-TR backprojector x = A^T y (Eq. 2).
//
// One thread owns one voxel (all NB batch images of it), loops over the views, accumulates in
// registers and stores each voxel exactly once.  Per-view parameters are staged through shared
// memory in chunks.  Detector cells are read through the read-only path (L1/L2).
#include <cuda_runtime.h>

#include "ctsf_internal.h"
#include "sf_footprint.cuh"

namespace {

constexpr int BP_VC = 16;     // views staged per chunk

template <int DIM, int ARC, int NB>
__global__ void __launch_bounds__(128)
bp_voxel_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ proj,
                float *__restrict__ vol, int view_begin, int view_stride, int view_count,
                size_t proj_bstride, size_t vol_bstride, int nzb)
{
    __shared__ SfView sv[BP_VC];
    const int ix = blockIdx.x * blockDim.x + threadIdx.x;
    const int iy = blockIdx.y * blockDim.y + threadIdx.y;
    int iz = 0, b0 = blockIdx.z * NB;
    if (DIM == 3) {
        int zb = blockIdx.z % nzb;
        b0 = (blockIdx.z / nzb) * NB;
        iz = zb * blockDim.z + threadIdx.z;
    }
    const bool inside = ix < pr.nx && iy < pr.ny && iz < pr.nz;
    const int tid = (threadIdx.z * blockDim.y + threadIdx.y) * blockDim.x + threadIdx.x;
    const int nthr = blockDim.x * blockDim.y * blockDim.z;
    const float p = (float)ix, q = (float)iy, z = (float)iz;
    const size_t view_cells = (size_t)pr.nu * pr.nv;
    proj += (size_t)b0 * proj_bstride;

    float acc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) acc[b] = 0.0f;

    for (int v0 = 0; v0 < view_count; v0 += BP_VC) {
        const int nvc = min(BP_VC, view_count - v0);
        __syncthreads();
        {   // stage the chunk's view parameters
            const int words = nvc * (int)(sizeof(SfView) / 4);
            uint32_t *dst = reinterpret_cast<uint32_t *>(sv);
            for (int w = tid; w < words; w += nthr) {
                int j = w / (int)(sizeof(SfView) / 4), o = w - j * (int)(sizeof(SfView) / 4);
                dst[w] = reinterpret_cast<const uint32_t *>(views + view_begin + (size_t)(v0 + j) * view_stride)[o];
            }
        }
        __syncthreads();
        if (!inside) continue;
        for (int j = 0; j < nvc; ++j) {
            const SfView &v = sv[j];
            const float a = fmaf(z, v.az, fmaf(q, v.aq, fmaf(p, v.ap, v.a0)));
            const float b = fmaf(z, v.bz, fmaf(q, v.bq, fmaf(p, v.bp, v.b0)));
            const float c = DIM == 3 ? fmaf(z, v.cz, fmaf(q, v.cq, fmaf(p, v.cp, v.c0))) : 0.0f;
            const float inv_a = rcp_nr(a);
            SfTrans T;
            sf_transaxial<ARC>(v, a, b, inv_a, T);
            const int k_lo = max(0, (int)floorf(T.kc + T.t0));
            const int k_hi = min(pr.nu - 1, (int)floorf(T.kc + T.t3));
            if (k_lo > k_hi) continue;
            SfAxial A;
            int l_lo = 0, l_hi = 0;
            if (DIM == 3) {
                sf_axial<ARC>(v, a, b, c, inv_a, A);
                l_lo = max(0, (int)floorf(A.lc + A.tlo));
                l_hi = min(pr.nv - 1, (int)floorf(A.lc + A.thi));
                if (l_lo > l_hi) continue;
            }
            const float amp = sf_amplitude(v, a, b, c, p, q);
            const float *y = proj + (size_t)(v0 + j) * view_cells;
            float sum[NB];
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) sum[bb] = 0.0f;
            float g0 = sf_G(T, (float)k_lo - T.kc);
            for (int k = k_lo; k <= k_hi; ++k) {
                const float g1 = sf_G(T, (float)(k + 1) - T.kc);
                const float f1 = g1 - g0;
                g0 = g1;
                if (DIM == 3) {
                    float col[NB];
#pragma unroll
                    for (int bb = 0; bb < NB; ++bb) col[bb] = 0.0f;
                    for (int l = l_lo; l <= l_hi; ++l) {
                        const float f2 = sf_F2(A, (float)l);
                        const float *yy = y + (size_t)l * pr.nu + k;
#pragma unroll
                        for (int bb = 0; bb < NB; ++bb) col[bb] = fmaf(f2, __ldg(yy + bb * proj_bstride), col[bb]);
                    }
#pragma unroll
                    for (int bb = 0; bb < NB; ++bb) sum[bb] = fmaf(f1, col[bb], sum[bb]);
                } else {
#pragma unroll
                    for (int bb = 0; bb < NB; ++bb) sum[bb] = fmaf(f1, __ldg(y + k + bb * proj_bstride), sum[bb]);
                }
            }
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) acc[bb] = fmaf(amp, sum[bb], acc[bb]);
        }
    }
    if (inside) {
        float *o = vol + (size_t)b0 * vol_bstride + ((size_t)iz * pr.ny + iy) * pr.nx + ix;
#pragma unroll
        for (int bb = 0; bb < NB; ++bb) o[bb * vol_bstride] = acc[bb];
    }
}

template <int DIM, int ARC, int NB>
void launch_one(const ct_geom *g, const float *d_proj, float *d_vol, int b0, int nb_groups,
                int vb, int vs, int vc, cudaStream_t st)
{
    const SfProblem &pr = g->prob;
    const size_t pbs = (size_t)vc * pr.nv * pr.nu, vbs = (size_t)pr.nx * pr.ny * pr.nz;
    dim3 block = DIM == 3 ? dim3(8, 4, 4) : dim3(16, 8, 1);
    int nzb = DIM == 3 ? (pr.nz + block.z - 1) / block.z : 1;
    dim3 grid((pr.nx + block.x - 1) / block.x, (pr.ny + block.y - 1) / block.y, nzb * nb_groups);
    bp_voxel_kernel<DIM, ARC, NB><<<grid, block, 0, st>>>(pr, g->d_bp, d_proj + (size_t)b0 * pbs,
                                                          d_vol + (size_t)b0 * vbs, vb, vs, vc, pbs, vbs, nzb);
}

template <int DIM, int ARC>
int launch_batches(const ct_geom *g, const float *d_proj, float *d_vol, int batch, int vb, int vs, int vc,
                   cudaStream_t st)
{
    // batch images share the weights (S6): groups of 8, 4, 2, 1 images per thread
    int launches = 0, b0 = 0;
    const int sizes[4] = {8, 4, 2, 1};
    for (int s = 0; s < 4; ++s) {
        int nb = sizes[s], groups = (batch - b0) / nb;
        if (groups <= 0) continue;
        // grid.z limit 65535
        while (groups > 0) {
            int gnow = groups;
            int nzb = DIM == 3 ? (g->prob.nz + 3) / 4 : 1;
            if ((long)gnow * nzb > 65535) gnow = 65535 / nzb > 0 ? 65535 / nzb : 1;
            switch (nb) {
                case 8: launch_one<DIM, ARC, 8>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st); break;
                case 4: launch_one<DIM, ARC, 4>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st); break;
                case 2: launch_one<DIM, ARC, 2>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st); break;
                default: launch_one<DIM, ARC, 1>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st); break;
            }
            ++launches;
            b0 += gnow * nb;
            groups -= gnow;
        }
    }
    return launches;
}

}  // namespace

int ctsf_launch_bp(const ct_geom *g, const float *d_proj, float *d_vol, int batch,
                   int view_begin, int view_stride, int view_count, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const int arc = g->prob.det_type, dim = g->prob.dim;
    int n;
    if (dim == 2) n = arc ? launch_batches<2, 1>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st)
                          : launch_batches<2, 0>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st);
    else          n = arc ? launch_batches<3, 1>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st)
                          : launch_batches<3, 0>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st);
    return cudaGetLastError() == cudaSuccess ? n : -1;
}
