// sf_fp.cu -- ct_fp_sf: SF-TR forward projector y = A x (Eq. 1).
//
// Output-exclusive design, no atomics of any kind.  One CTA owns one detector tile (TK x TL cells)
// of one view and keeps it in shared memory for the whole pass.  It walks the voxel slabs
// perpendicular to the view's dominant ray axis; per slab it inverse-projects the (expanded) tile
// onto the slab to find the voxels that can touch it, and adds their footprints into the tile in
// "colour" phases: voxels of one phase lie on a lattice (col_p, col_z) coarse enough that their
// footprints are pairwise disjoint (bounds derived in geom.cpp), so the plain read-modify-writes
// of a phase never collide and the summation order is fixed.  Each detector cell is stored once.
//
// Views whose rays run mostly along x read the volume through an xy-transposed copy so that the
// in-slab index p is always the memory-fastest one.
#include <cuda_runtime.h>

#include "ctsf_internal.h"
#include "sf_footprint.cuh"

namespace {

constexpr int FP_THREADS = 256;

__global__ void transpose_xy_kernel(const float *__restrict__ src, float *__restrict__ dst, int nx, int ny)
{
    __shared__ float t[32][33];
    const size_t slice = (size_t)blockIdx.z * nx * ny;
    int x = blockIdx.x * 32 + threadIdx.x, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y)
        if (x < nx && y0 + j < ny) t[j][threadIdx.x] = src[slice + (size_t)(y0 + j) * nx + x];
    __syncthreads();
    int y = y0 + threadIdx.x, x0 = blockIdx.x * 32;
    for (int j = threadIdx.y; j < 32; j += blockDim.y)
        if (y < ny && x0 + j < nx) dst[slice + (size_t)(x0 + j) * ny + y] = t[threadIdx.x][j];
}

struct Ray { float dp, dq, dz; };

template <int ARC>
__device__ __forceinline__ Ray tile_ray(const SfView &v, float kf, float lf)
{
    Ray r;
    const float t = lf - v.lv0c;
    if (ARC == 0) {
        const float s = kf - v.ku0c;
        r.dp = fmaf(s, v.Up, fmaf(t, v.Vp, v.Dp));
        r.dq = fmaf(s, v.Uq, fmaf(t, v.Vq, v.Dq));
        r.dz = fmaf(s, v.Uz, fmaf(t, v.Vz, v.Dz));
    } else {
        float sg, cg;
        sincosf((kf - v.ku0c) / v.Ru, &sg, &cg);
        r.dp = fmaf(sg, v.Up, fmaf(cg, v.Dp, t * v.Vp));
        r.dq = fmaf(sg, v.Uq, fmaf(cg, v.Dq, t * v.Vq));
        r.dz = fmaf(sg, v.Uz, fmaf(cg, v.Dz, t * v.Vz));
    }
    return r;
}

// tile: [NB][TL][TK] floats in dynamic shared memory
template <int DIM, int ARC, int NB>
__global__ void __launch_bounds__(FP_THREADS)
fp_tile_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ vol,
               const float *__restrict__ volT, float *__restrict__ proj, int view_begin, int view_stride,
               int TK, int TL, int tiles_k, size_t vol_bstride, size_t proj_bstride)
{
    extern __shared__ float tile[];
    __shared__ SfView sview;
    __shared__ Ray rays[6];
    const int tid = threadIdx.x;
    const int jview = blockIdx.y;
    const int tk = blockIdx.x % tiles_k, tl = blockIdx.x / tiles_k;
    const int k0 = tk * TK, l0 = tl * TL;
    const int tkw = min(TK, pr.nu - k0), tlh = min(TL, pr.nv - l0);
    const int b0 = blockIdx.z * NB;

    for (int w = tid; w < (int)(sizeof(SfView) / 4); w += FP_THREADS)
        reinterpret_cast<uint32_t *>(&sview)[w] =
            reinterpret_cast<const uint32_t *>(views + view_begin + (size_t)jview * view_stride)[w];
    for (int i = tid; i < NB * TL * TK; i += FP_THREADS) tile[i] = 0.0f;
    __syncthreads();
    const SfView &v = sview;
    if (tid < 6) {
        // expanded tile: corners (and, for the arc, the mid column: the slab image of an arc tile bulges)
        const float kA = (float)k0 - v.ek, kB = (float)(k0 + tkw) + v.ek;
        const float lA = (float)l0 - v.el, lB = (float)(l0 + tlh) + v.el;
        const float kk = (tid % 3 == 0) ? kA : (tid % 3 == 1 ? kB : 0.5f * (kA + kB));
        rays[tid] = tile_ray<ARC>(v, kk, tid < 3 ? lA : lB);
    }
    __syncthreads();

    const int np = v.swap_xy ? pr.ny : pr.nx, nq = v.swap_xy ? pr.nx : pr.ny, nz = pr.nz;
    const float *src = (v.swap_xy ? volT : vol) + (size_t)b0 * vol_bstride;
    const int col_p = v.col_p, col_z = DIM == 3 ? v.col_z : 1;

    for (int iq = 0; iq < nq; ++iq) {
        // ---- voxel region of this slab that can touch the tile (identical in every thread) -------
        float pmin = 1e30f, pmax = -1e30f, zmin = 1e30f, zmax = -1e30f;
        bool whole = false;
        const float dqc = (float)iq - v.Sq;
#pragma unroll
        for (int r = 0; r < 6; ++r) {
            if (DIM == 2 && r >= 3) break;
            const Ray ry = rays[r];
            if (!(ry.dq * dqc > 0.0f) || fabsf(ry.dq) < 1e-3f * (fabsf(ry.dp) + fabsf(ry.dz))) whole = true;
            const float lam = dqc / ry.dq;
            const float pp = fmaf(lam, ry.dp, v.Sp), zz = fmaf(lam, ry.dz, v.Sz);
            pmin = fminf(pmin, pp); pmax = fmaxf(pmax, pp);
            zmin = fminf(zmin, zz); zmax = fmaxf(zmax, zz);
        }
        int p_lo = 0, p_hi = np - 1, z_lo = 0, z_hi = nz - 1;
        if (!whole) {
            p_lo = max(0, (int)ceilf(pmin - 0.3f)); p_hi = min(np - 1, (int)floorf(pmax + 0.3f));
            if (DIM == 3) { z_lo = max(0, (int)ceilf(zmin - 0.3f)); z_hi = min(nz - 1, (int)floorf(zmax + 0.3f)); }
        }
        if (p_lo > p_hi || z_lo > z_hi) continue;
        const int npr = p_hi - p_lo + 1, nzr = z_hi - z_lo + 1;
        const float q = (float)iq;
        const float aq0 = fmaf(q, v.aq, v.a0), bq0 = fmaf(q, v.bq, v.b0), cq0 = fmaf(q, v.cq, v.c0);
        const float *slab = src + (size_t)iq * np;

        for (int cz_i = 0; cz_i < col_z; ++cz_i) {
            if (cz_i >= nzr) break;
            const int cnt_z = (nzr - cz_i + col_z - 1) / col_z;
            for (int cp_i = 0; cp_i < col_p; ++cp_i) {
                if (cp_i >= npr) break;
                const int cnt_p = (npr - cp_i + col_p - 1) / col_p;
                const int cnt = cnt_p * cnt_z;
                for (int t = tid; t < cnt; t += FP_THREADS) {
                    const int zi = t / cnt_p, pi = t - zi * cnt_p;
                    const int ip = p_lo + cp_i + pi * col_p, iz = z_lo + cz_i + zi * col_z;
                    const float p = (float)ip, z = (float)iz;
                    const float a = fmaf(z, v.az, fmaf(p, v.ap, aq0));
                    const float b = fmaf(z, v.bz, fmaf(p, v.bp, bq0));
                    const float c = DIM == 3 ? fmaf(z, v.cz, fmaf(p, v.cp, cq0)) : 0.0f;
                    const float inv_a = rcp_nr(a);
                    SfTrans T;
                    sf_transaxial<ARC>(v, a, b, inv_a, T);
                    const int k_lo = max(k0, (int)floorf(T.kc + T.t0));
                    const int k_hi = min(k0 + tkw - 1, (int)floorf(T.kc + T.t3));
                    if (k_lo > k_hi) continue;
                    SfAxial A;
                    int l_lo = 0, l_hi = 0;
                    if (DIM == 3) {
                        sf_axial<ARC>(v, a, b, c, inv_a, A);
                        l_lo = max(l0, (int)floorf(A.lc + A.tlo));
                        l_hi = min(l0 + tlh - 1, (int)floorf(A.lc + A.thi));
                        if (l_lo > l_hi) continue;
                    }
                    const float amp = sf_amplitude(v, a, b, c, p, q);
                    float xv[NB];
                    const float *xp = slab + (size_t)iz * np * nq + ip;
#pragma unroll
                    for (int bb = 0; bb < NB; ++bb) xv[bb] = amp * __ldg(xp + bb * vol_bstride);
                    float g0 = sf_G(T, (float)k_lo - T.kc);
                    for (int k = k_lo; k <= k_hi; ++k) {
                        const float g1 = sf_G(T, (float)(k + 1) - T.kc);
                        const float f1 = g1 - g0;
                        g0 = g1;
                        float *tc = tile + (k - k0);
                        if (DIM == 3) {
                            for (int l = l_lo; l <= l_hi; ++l) {
                                const float w = f1 * sf_F2(A, (float)l);
#pragma unroll
                                for (int bb = 0; bb < NB; ++bb) {
                                    float *c2 = tc + (bb * TL + (l - l0)) * TK;
                                    *c2 = fmaf(w, xv[bb], *c2);
                                }
                            }
                        } else {
#pragma unroll
                            for (int bb = 0; bb < NB; ++bb) {
                                float *c2 = tc + bb * TL * TK;
                                *c2 = fmaf(f1, xv[bb], *c2);
                            }
                        }
                    }
                }
                __syncthreads();
            }
        }
    }
    __syncthreads();
    // every cell of the tile is stored exactly once
    for (int i = tid; i < NB * tlh * tkw; i += FP_THREADS) {
        const int k = i % tkw, r = i / tkw, l = r % tlh, bb = r / tlh;
        proj[(size_t)(b0 + bb) * proj_bstride + ((size_t)jview * pr.nv + (l0 + l)) * pr.nu + (k0 + k)] =
            tile[(bb * TL + l) * TK + k];
    }
}

template <int DIM, int ARC, int NB>
void launch_fp(const ct_geom *g, const float *d_vol, const float *d_volT, float *d_proj, int b0, int groups,
               int vb, int vs, int vc, cudaStream_t st)
{
    const SfProblem &pr = g->prob;
    const int TK = DIM == 3 ? 128 : 256, TL = DIM == 3 ? (pr.nv >= 64 ? 64 : (pr.nv >= 32 ? 32 : 16)) : 1;
    const int tiles_k = (pr.nu + TK - 1) / TK, tiles_l = (pr.nv + TL - 1) / TL;
    const size_t vbs = (size_t)pr.nx * pr.ny * pr.nz, pbs = (size_t)vc * pr.nv * pr.nu;
    const size_t smem = (size_t)NB * TK * TL * sizeof(float);
    auto kern = fp_tile_kernel<DIM, ARC, NB>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    dim3 grid(tiles_k * tiles_l, vc, groups);
    kern<<<grid, FP_THREADS, smem, st>>>(pr, g->d_fp, d_vol + (size_t)b0 * vbs,
                                         d_volT ? d_volT + (size_t)b0 * vbs : nullptr,
                                         d_proj + (size_t)b0 * pbs, vb, vs, TK, TL, tiles_k, vbs, pbs);
}

template <int DIM, int ARC>
int launch_fp_batches(const ct_geom *g, const float *d_vol, const float *d_volT, float *d_proj, int batch,
                      int vb, int vs, int vc, cudaStream_t st)
{
    int launches = 0, b0 = 0;
    if (vc <= 0) return 0;
    if (DIM == 2) {
        const int sizes[5] = {16, 8, 4, 2, 1};
        for (int s = 0; s < 5; ++s) {
            int nb = sizes[s], groups = (batch - b0) / nb;
            while (groups > 0) {
                int gnow = groups > 65535 ? 65535 : groups;
                switch (nb) {
                    case 16: launch_fp<2, ARC, 16>(g, d_vol, d_volT, d_proj, b0, gnow, vb, vs, vc, st); break;
                    case 8: launch_fp<2, ARC, 8>(g, d_vol, d_volT, d_proj, b0, gnow, vb, vs, vc, st); break;
                    case 4: launch_fp<2, ARC, 4>(g, d_vol, d_volT, d_proj, b0, gnow, vb, vs, vc, st); break;
                    case 2: launch_fp<2, ARC, 2>(g, d_vol, d_volT, d_proj, b0, gnow, vb, vs, vc, st); break;
                    default: launch_fp<2, ARC, 1>(g, d_vol, d_volT, d_proj, b0, gnow, vb, vs, vc, st); break;
                }
                ++launches; b0 += gnow * nb; groups -= gnow;
            }
        }
    } else {
        int groups = batch;
        while (groups > 0) {
            int gnow = groups > 65535 ? 65535 : groups;
            launch_fp<3, ARC, 1>(g, d_vol, d_volT, d_proj, b0, gnow, vb, vs, vc, st);
            ++launches; b0 += gnow; groups -= gnow;
        }
    }
    return launches;
}

}  // namespace

int ctsf_launch_fp(const ct_geom *g, const float *d_vol, float *d_proj, int batch,
                   int view_begin, int view_stride, int view_count, void *stream)
{
    cudaStream_t st = (cudaStream_t)stream;
    const SfProblem &pr = g->prob;
    int launches = 0;
    float *d_volT = nullptr;
    bool need_T = false;
    for (int j = 0; j < view_count && !need_T; ++j) need_T = g->h_fp[view_begin + (size_t)j * view_stride].swap_xy != 0;
    if (need_T) {
        const size_t n = (size_t)batch * pr.nx * pr.ny * pr.nz;
        if (cudaMallocAsync((void **)&d_volT, n * sizeof(float), st) != cudaSuccess) return -1;
        dim3 grid((pr.nx + 31) / 32, (pr.ny + 31) / 32, 1), block(32, 8);
        // one launch per chunk of <= 65535 slices
        const long slices = (long)batch * pr.nz;
        for (long s0 = 0; s0 < slices; s0 += 65535) {
            grid.z = (unsigned)((slices - s0) < 65535 ? (slices - s0) : 65535);
            transpose_xy_kernel<<<grid, block, 0, st>>>(d_vol + (size_t)s0 * pr.nx * pr.ny,
                                                        d_volT + (size_t)s0 * pr.nx * pr.ny, pr.nx, pr.ny);
            ++launches;
        }
    }
    const int arc = pr.det_type;
    if (pr.dim == 2) launches += arc ? launch_fp_batches<2, 1>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st)
                                     : launch_fp_batches<2, 0>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st);
    else             launches += arc ? launch_fp_batches<3, 1>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st)
                                     : launch_fp_batches<3, 0>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st);
    if (d_volT) cudaFreeAsync(d_volT, st);
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}
