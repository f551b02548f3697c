// sf_bp.cu -- ct_bp_sf: voxel-driven SF-TR backprojector x = A^T y (Eq. 2).
//
// 3-D: one CTA owns a brick of BX x BY x BZ voxels and loops over the views.  Per view, eight lanes
// project the brick's corners, a warp-shuffle min/max gives the brick's shadow on the detector, and
// one elected thread pulls that detector tile into shared memory with a TMA tensor copy
// (cp.async.bulk.tensor, out-of-range cells zero-filled by hardware = detector-edge clipping for
// free), double-buffered against the computation of the current view.  Every thread then walks its
// (x, y) column's z-run, evaluates the footprint and gathers its K x L cells from the shared tile.
// Bricks whose shadow misses the detector skip the view.  Accumulators live in shared memory
// (conflict-free, one read-modify-write per voxel x view) and each voxel is stored exactly once.
// When the projection row pitch is not a multiple of 16 bytes (TMA requirement) the tile is staged
// with 4-byte cp.async instead.
//
// 2-D: one thread per pixel and NB batch images, views looped, cells read through L1 (no z to
// amortise a tile over).
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdlib>
#include <cstring>

#include "ctsf_internal.h"
#include "sf_footprint.cuh"

namespace {

// ---------------------------------------------------------------------------------------------------
// 2-D: thread per pixel
// ---------------------------------------------------------------------------------------------------
constexpr int BP_VC = 16;     // views staged per chunk

template <int ARC, int NB, int RECON, int MODEL>
__global__ void __launch_bounds__(128)
bp_pixel_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ proj,
                float *__restrict__ vol, int view_begin, int view_stride, int view_count,
                unsigned proj_bstride, unsigned vol_bstride)
{
    __shared__ SfView sv[BP_VC];
    const int ix = blockIdx.x * blockDim.x + threadIdx.x;
    const int iy = blockIdx.y * blockDim.y + threadIdx.y;
    const int b0 = blockIdx.z * NB;
    const bool inside = ix < pr.nx && iy < pr.ny;
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;
    const int nthr = blockDim.x * blockDim.y;
    const float p = (float)ix, q = (float)iy;
    proj += (size_t)b0 * proj_bstride;

    float acc[NB];
#pragma unroll
    for (int b = 0; b < NB; ++b) acc[b] = 0.0f;

    for (int v0 = 0; v0 < view_count; v0 += BP_VC) {
        const int nvc = min(BP_VC, view_count - v0);
        __syncthreads();
        {
            constexpr int W = (int)(sizeof(SfView) / 4);
            uint32_t *dst = reinterpret_cast<uint32_t *>(sv);
            for (int w = tid; w < nvc * W; w += nthr) {
                int j = w / W, o = w - j * W;
                dst[w] = reinterpret_cast<const uint32_t *>(views + view_begin + (size_t)(v0 + j) * view_stride)[o];
            }
        }
        __syncthreads();
        if (!inside) continue;
        for (int j = 0; j < nvc; ++j) {
            const SfView &v = sv[j];
            const float a = fmaf(q, v.aq, fmaf(p, v.ap, v.a0));
            const float b = fmaf(q, v.bq, fmaf(p, v.bp, v.b0));
            const float inv_a = rcp_nr(a);
            SfTrans T;
            sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T, p, q);
            const int k_lo = max(0, (int)floorf(T.kc + T.t0));
            const int k_hi = min(pr.nu - 1, (int)floorf(T.kc + T.t3));
            if (k_lo > k_hi) continue;
            const float amp = RECON ? sf_recon_weight<ARC>(v, T, 1.0f, a, b) : sf_amplitude(v, a, b, 0.0f, p, q);
            const float *y = proj + (size_t)(v0 + j) * pr.nu;
            float sum[NB];
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) sum[bb] = 0.0f;
            float g0 = sf_G<MODEL>(T, (float)k_lo - T.kc);
            for (int k = k_lo; k <= k_hi; ++k) {
                const float g1 = sf_G<MODEL>(T, (float)(k + 1) - T.kc);
                const float f1 = g1 - g0;
                g0 = g1;
#pragma unroll
                for (int bb = 0; bb < NB; ++bb) sum[bb] = fmaf(f1, __ldg(y + (unsigned)k + bb * proj_bstride), sum[bb]);
            }
#pragma unroll
            for (int bb = 0; bb < NB; ++bb) acc[bb] = fmaf(amp, sum[bb], acc[bb]);
        }
    }
    if (inside) {
        float *o = vol + (size_t)b0 * vol_bstride + (size_t)iy * pr.nx + ix;
#pragma unroll
        for (int bb = 0; bb < NB; ++bb) o[(size_t)bb * vol_bstride] = acc[bb];
    }
}

// ---------------------------------------------------------------------------------------------------
// 3-D: brick per CTA, detector tile in shared memory (TMA)
// ---------------------------------------------------------------------------------------------------
constexpr int BX = 16, BY = 16, BZ = 16;         // brick (voxels); 256 threads, one (x, y) column each
constexpr int TW = 96, TH = 64;                  // detector tile (cells x rows) = one TMA box
constexpr int LM = 4;                            // rows gathered per pass (registers f2[LM])
constexpr int BRICK_THREADS = BX * BY;
#ifndef BP2_MINB
#define BP2_MINB 2                               // CTAs per SM the packed kernel's register budget is sized for
#endif
constexpr int TILE_FLOATS = TW * (TH + LM);      // + LM zero rows so row chunks never read outside

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1, int c2)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

struct TileInfo { int k0, l0, nbk, nbl, live; };   // origin of the shadow, number of boxes, live flag

// Shadow of the brick [p0-.5, p1+.5] x [q0-.5, q1+.5] x [z0-.5, z1+.5] on the detector, by lanes 0..7 of
// a full warp; result valid in every lane.
template <int ARC>
__device__ __forceinline__ TileInfo brick_shadow(const SfView &v, const SfProblem &pr, float p0, float p1,
                                                 float q0, float q1, float z0, float z1, int lane)
{
    const float p = (lane & 1) ? p1 + 0.5f : p0 - 0.5f;
    const float q = (lane & 2) ? q1 + 0.5f : q0 - 0.5f;
    const float z = (lane & 4) ? z1 + 0.5f : z0 - 0.5f;
    const float a = fmaf(z, v.az, fmaf(q, v.aq, fmaf(p, v.ap, v.a0)));
    const float b = fmaf(z, v.bz, fmaf(q, v.bq, fmaf(p, v.bp, v.b0)));
    const float c = fmaf(z, v.cz, fmaf(q, v.cq, fmaf(p, v.cp, v.c0)));
    float kf, lf;
    if (ARC == 0) {
        const float ia = rcp_nr(a);
        kf = fmaf(v.Ru, b * ia, v.ku0);
        lf = fmaf(v.Rv, c * ia, v.lv0);
    } else {
        kf = fmaf(v.Ru, atan2f(b, a), v.ku0);
        lf = fmaf(v.Rv * c, rsqrt_nr(fmaf(a, a, b * b)), v.lv0);
    }
    float kmin = kf, kmax = kf, lmin = lf, lmax = lf;
#pragma unroll
    for (int s = 1; s < 8; s <<= 1) {            // warp-shuffle footprint-extent reduction
        kmin = fminf(kmin, __shfl_xor_sync(0xffffffffu, kmin, s));
        kmax = fmaxf(kmax, __shfl_xor_sync(0xffffffffu, kmax, s));
        lmin = fminf(lmin, __shfl_xor_sync(0xffffffffu, lmin, s));
        lmax = fmaxf(lmax, __shfl_xor_sync(0xffffffffu, lmax, s));
    }
    kmin = __shfl_sync(0xffffffffu, kmin, 0); kmax = __shfl_sync(0xffffffffu, kmax, 0);
    lmin = __shfl_sync(0xffffffffu, lmin, 0); lmax = __shfl_sync(0xffffffffu, lmax, 0);
    // margins: fp32 rounding of the corner projections, and (arc) the bulge of rows between corners
    const float mk = 0.75f, ml = (ARC ? 1.5f : 0.75f) + v.lpad;
    TileInfo t;
    // TMA: the innermost box coordinate must be 16-byte aligned (measured on B200: an odd start
    // coordinate raises 'illegal instruction'), so the tile origin is rounded down to 4 cells
    const int ka = max(0, (int)floorf(kmin - mk)) & ~3, kb = min(pr.nu - 1, (int)floorf(kmax + mk));
    const int la = max(0, (int)floorf(lmin - ml)), lb = min(pr.nv - 1, (int)floorf(lmax + ml));
    t.live = (ka <= kb && la <= lb) ? 1 : 0;
    t.k0 = ka; t.l0 = la;
    t.nbk = t.live ? (kb - ka + TW) / TW : 0;
    t.nbl = t.live ? (lb - la + TH) / TH : 0;
    return t;
}

__device__ __forceinline__ float lds_f32(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }

// gather one voxel's footprint from the tile (shared-memory byte address tile_a) whose origin is (tk0, tl0);
// returns sum_kl F1 F2 y.  The four row loads of a column are issued first (explicit ld.shared keeps that order),
// the trapezoid CDF is evaluated under their latency.
template <int MODEL>
__device__ __forceinline__ float gather_tile(uint32_t tile_a, const SfTrans &T, const SfAxial &A,
                                             int k_lo, int k_hi, int l_lo, int l_hi, int tk0, int tl0)
{
    float sum = 0.0f;
    for (int lb = l_lo; lb <= l_hi; lb += LM) {
        // rows past l_hi get weight 0 by themselves (x >= thi), rows past the tile read the zero pad rows
        float f2[LM];
        sf_F2_run<LM, MODEL>(A, (float)lb, f2);
        uint32_t ra = tile_a + 4u * (unsigned)((lb - tl0) * TW + (k_lo - tk0));
        float xi = (float)k_lo - T.kc;
        float g0 = sf_G<MODEL>(T, xi);
#pragma unroll 1
        for (int k = k_lo; k <= k_hi; ++k, ra += 4) {
            const float y0 = lds_f32(ra), y1 = lds_f32(ra + 4 * TW), y2 = lds_f32(ra + 8 * TW), y3 = lds_f32(ra + 12 * TW);
            xi += 1.0f;
            const float g1 = sf_G<MODEL>(T, xi);
            float s = f2[0] * y0;
            s = fmaf(f2[1], y1, s); s = fmaf(f2[2], y2, s); s = fmaf(f2[3], y3, s);
            sum = fmaf(g1 - g0, s, sum);
            g0 = g1;
        }
    }
    return sum;
}

// plain-pointer version (compiler-scheduled loads): the overflow branch of the untilted kernels
template <int MODEL>
__device__ __forceinline__ float gather_tile_ptr(const float *__restrict__ tile, const SfTrans &T, const SfAxial &A,
                                                 int k_lo, int k_hi, int l_lo, int l_hi, int tk0, int tl0)
{
    float sum = 0.0f;
    for (int lb = l_lo; lb <= l_hi; lb += LM) {
        float f2[LM];
        sf_F2_run<LM, MODEL>(A, (float)lb, f2);
        const float *row = tile + (lb - tl0) * TW + (k_lo - tk0);
        float xi = (float)k_lo - T.kc;
        float g0 = sf_G<MODEL>(T, xi);
#pragma unroll 1
        for (int k = k_lo; k <= k_hi; ++k) {
            xi += 1.0f;
            const float g1 = sf_G<MODEL>(T, xi);
            float s = 0.0f;
#pragma unroll
            for (int j = 0; j < LM; ++j) s = fmaf(f2[j], row[j * TW], s);
            sum = fmaf(g1 - g0, s, sum);
            g0 = g1;
            ++row;
        }
    }
    return sum;
}

// the same with the F1 weights of columns k_lo .. k_lo + K - 1 given (untilted frames, K <= BKR: computed once
// per (x, y) column and view and reused along the z-run)
constexpr int BKR = 6;
__device__ __forceinline__ float gather_tile_w(const float *__restrict__ tile, const float (&f1)[BKR], int K,
                                               const SfAxial &A, int k_lo, int l_lo, int l_hi, int tk0, int tl0)
{
    float sum = 0.0f;
    for (int lb = l_lo; lb <= l_hi; lb += LM) {
        float f2[LM];
        sf_F2_run<LM>(A, (float)lb, f2);
        const float *row = tile + (lb - tl0) * TW + (k_lo - tk0);
#pragma unroll
        for (int k = 0; k < BKR; ++k) {
            if (k < K) {
                float s = 0.0f;
#pragma unroll
                for (int j = 0; j < LM; ++j) s = fmaf(f2[j], row[j * TW + k], s);
                sum = fmaf(f1[k], s, sum);
            }
        }
    }
    return sum;
}

template <int ARC, int RECON, int UNT, int MODEL>
__global__ void __launch_bounds__(BRICK_THREADS, 3)
bp_brick_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ proj,
                const __grid_constant__ CUtensorMap tmap, int use_tma, float *__restrict__ vol,
                int view_begin, int view_stride, int view_count, int j_lo, int j_hi, int nbz, int accumulate)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *tile0 = reinterpret_cast<float *>(smem_raw);
    float *tile1 = tile0 + TILE_FLOATS;
    float *accs = tile1 + TILE_FLOATS;                          // [BZ][256]
    __shared__ SfView sview[2];
    __shared__ TileInfo tinfo[2];
    __shared__ __align__(8) uint64_t mbar[2];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx = tid % BX, ty = tid / BX;
    const int bzi = blockIdx.z % nbz, batch = blockIdx.z / nbz;
    const int p0 = blockIdx.x * BX, q0 = blockIdx.y * BY, z0 = bzi * BZ;
    const int p1 = min(p0 + BX, pr.nx) - 1, q1 = min(q0 + BY, pr.ny) - 1, z1 = min(z0 + BZ, pr.nz) - 1;
    const int ip = p0 + tx, iq = q0 + ty;
    const bool col_in = ip < pr.nx && iq < pr.ny;
    const float p = (float)ip, q = (float)iq;
    const int view_off = batch * view_count;                    // this image's first view in the buffer

    for (int i = tid; i < BZ * BRICK_THREADS; i += BRICK_THREADS) accs[i] = 0.0f;
    for (int i = tid; i < LM * TW; i += BRICK_THREADS) { tile0[TH * TW + i] = 0.0f; tile1[TH * TW + i] = 0.0f; }
    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // stage view j's parameters and tile into buffer s (called by warp 0 only; TMA path)
    auto prefetch = [&](int j, int s) {
        const SfView *gv = views + view_begin + (size_t)j * view_stride;
        constexpr int W = (int)(sizeof(SfView) / 4);
        for (int w = lane; w < W; w += 32)
            reinterpret_cast<uint32_t *>(&sview[s])[w] = reinterpret_cast<const uint32_t *>(gv)[w];
        __syncwarp();
        TileInfo t = brick_shadow<ARC>(sview[s], pr, (float)p0, (float)p1, (float)q0, (float)q1, (float)z0, (float)z1, lane);
        if (lane == 0) {
            tinfo[s] = t;
            if (t.live && (use_tma & 1)) {
                mbar_expect_tx(&mbar[s], TW * TH * 4);
                tma_load_3d(s ? tile1 : tile0, &tmap, &mbar[s], t.k0, t.l0, view_off + j);
            }
        }
    };
    // cooperative 4-byte cp.async load of box (bk, bl) of view j into `dst` (all threads)
    auto coop_load = [&](float *dst, int k0, int l0, int j) {
        const float *src = proj + (size_t)(view_off + j) * pr.nu * pr.nv;
        for (int i = tid; i < TW * TH; i += BRICK_THREADS) {
            const int r = i / TW, cidx = i - r * TW;
            const int k = k0 + cidx, l = l0 + r;
            const bool ok = k >= 0 && k < pr.nu && l >= 0 && l < pr.nv;
            const float *gp = ok ? src + (size_t)l * pr.nu + k : src;
            const int sz = ok ? 4 : 0;
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(smem_u32(dst + i)), "l"(gp), "r"(sz) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    };

    uint32_t phase[2] = {0u, 0u};
    if (warp == 0 && j_lo < j_hi) prefetch(j_lo, j_lo & 1);
    __syncthreads();

    for (int j = j_lo; j < j_hi; ++j) {         // this launch's chunk of the call's views
        const int s = j & 1;
        if (warp == 0 && j + 1 < j_hi) prefetch(j + 1, s ^ 1);
        const TileInfo t = tinfo[s];
        if (t.live) {
            const SfView v = sview[s];          // local copy: the fields in use stay in registers over the z-run
            float *tile = s ? tile1 : tile0;
            uint32_t tile_a = smem_u32(tile);
            if (!UNT) asm volatile("" : "+r"(tile_a));   // one register instead of a rebuild per voxel
            const float a_col = fmaf(q, v.aq, fmaf(p, v.ap, v.a0));
            const float b_col = fmaf(q, v.bq, fmaf(p, v.bp, v.b0));
            const float c_col = fmaf(q, v.cq, fmaf(p, v.cp, v.c0));
            for (int bl = 0; bl < t.nbl; ++bl)
                for (int bk = 0; bk < t.nbk; ++bk) {
                    const int tk0 = t.k0 + bk * TW, tl0 = t.l0 + bl * TH;
                    if (bk == 0 && bl == 0 && (use_tma & 2)) {
                        mbar_wait(&mbar[s], phase[s]);
                        phase[s] ^= 1u;
                    } else {                       // unaligned pitch, or a shadow larger than one box (rare)
                        __syncthreads();
                        coop_load(tile, tk0, tl0, j);
                        __syncthreads();
                    }
                    if (col_in) {
                        // untilted frames: the transaxial footprint does not depend on z -> once per column
                        const bool unt = UNT || v.untilted != 0;
                        float a = a_col, b = b_col, inv_a = 0.0f;
                        SfTrans T;
                        int k_lo = 0, k_hi = -1;
                        float f1[BKR], sumF1 = 0.0f;           // UNT: the weights themselves, once per column
                        if (unt) {
                            inv_a = rcp_nr(a);
                            sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T, p, q);
                            k_lo = max(max(0, tk0), (int)floorf(T.kc + T.t0));
                            k_hi = min(min(pr.nu - 1, tk0 + TW - 1), (int)floorf(T.kc + T.t3));
                            if (UNT) {
                                sumF1 = T.h01 + T.w12 + T.h23;
                                float xi = (float)k_lo - T.kc, g0 = sf_G<MODEL>(T, xi);
#pragma unroll
                                for (int k = 0; k < BKR; ++k) {
                                    xi += 1.0f;
                                    const float g1 = sf_G<MODEL>(T, xi);
                                    f1[k] = g1 - g0;
                                    g0 = g1;
                                }
                            }
                        }
                        for (int zi = 0; zi <= z1 - z0; ++zi) {
                            const float z = (float)(z0 + zi);
                            if (!unt) {
                                a = fmaf(z, v.az, a_col); b = fmaf(z, v.bz, b_col);
                                inv_a = rcp_nr(a);
                                sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T, p, q);
                                k_lo = max(max(0, tk0), (int)floorf(T.kc + T.t0));
                                k_hi = min(min(pr.nu - 1, tk0 + TW - 1), (int)floorf(T.kc + T.t3));
                            }
                            if (k_lo > k_hi) continue;
                            const float c = fmaf(z, v.cz, c_col);
                            SfAxial A;
                            sf_axial<ARC, MODEL>(v, a, b, c, inv_a, A, p, q);
                            const int l_lo = max(max(0, tl0), (int)floorf(A.lc + A.tlo));
                            const int l_hi = min(min(pr.nv - 1, tl0 + TH - 1), (int)floorf(A.lc + A.thi));
                            if (l_lo > l_hi) continue;
                            float amp, sum;
                            if (UNT) {
                                amp = RECON ? sf_recon_weight_s<ARC>(v, sumF1, sf_axial_sum<MODEL>(A), a, b)
                                            : sf_amplitude(v, a, b, c, p, q);
                                const int K = k_hi - k_lo + 1;
                                if (K <= BKR) {
                                    sum = gather_tile_w(tile, f1, K, A, k_lo, l_lo, l_hi, tk0, tl0);
                                } else {            // footprint wider than the host's bound (never expected)
                                    SfTrans T2;
                                    sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T2, p, q);
                                    sum = gather_tile_ptr<MODEL>(tile, T2, A, k_lo, k_hi, l_lo, l_hi, tk0, tl0);
                                }
                            } else {
                                amp = RECON ? sf_recon_weight<ARC>(v, T, sf_axial_sum<MODEL>(A), a, b)
                                            : sf_amplitude(v, a, b, c, p, q);
                                sum = gather_tile<MODEL>(tile_a, T, A, k_lo, k_hi, l_lo, l_hi, tk0, tl0);
                            }
                            float *ap = accs + zi * BRICK_THREADS + tid;
                            *ap = fmaf(amp, sum, *ap);
                        }
                    }
                }
            // This view's tile buffer may have been written by cp.async (generic proxy); the next write into it is
            // warp 0's TMA (async proxy) two views on, ordered behind these writes only by the barrier below.  Writes
            // of one proxy followed by writes of the other need a proxy fence by the writing threads.
            if ((use_tma & 1) && (t.nbk * t.nbl > 1 || !(use_tma & 2)))
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncthreads();
    }
    if (col_in) {
        float *o = vol + (size_t)batch * pr.nx * pr.ny * pr.nz + ((size_t)z0 * pr.ny + iq) * pr.nx + ip;
        for (int zi = 0; zi <= z1 - z0; ++zi) {
            float *oz = o + (size_t)zi * pr.ny * pr.nx;
            const float r = accs[zi * BRICK_THREADS + tid];
            *oz = accumulate ? *oz + r : r;          // accumulate: view-chunked host pipeline only
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// General (tilted-frame) brick kernel, two voxels per thread, barrier-free view pipeline.
// Same brick / shadow / TMA-tile scheme as bp_brick_kernel, but
//  (1) every thread walks its z-run in PAIRS (z, z + 1) and evaluates both footprints in lockstep with the packed
//      FFMA2 / FMUL2 / FADD2 instructions of sm_100 (sf_footprint.cuh, "Packed pairs"): the kernel is bound by
//      instruction issue, and the packed forms carry two voxels' multiply-adds in one issue slot.  The column and
//      row loops run over max(K_a, K_b) x max(L_a, L_b); each footprint is cut at its own last cell edges, so the
//      cells past them weigh exactly 0 and their loads stay inside the stage's own tile and zero rows (see "parked");
//  (2) the views flow through a ring of BP2_STAGES tile buffers guarded by mbarrier pairs: full[s] completes when
//      the TMA bytes of the view have landed (one warp, in rotation, stages the view's parameters and the brick's
//      shadow and arms it), empty[s] when all warps have finished reading the stage.  No __syncthreads in the view loop: warps
//      drift up to a view apart instead of waiting for the slowest one at every view (0.9 barrier stalls per
//      issued instruction in the round-1 kernel).  Shadows larger than one box (rare) fall back to block-wide
//      cp.async staging inside the view, which re-synchronises the CTA.
// Accumulators: one float2 per thread and z-pair in shared memory, thread-private and conflict-free (a register
// array indexed by the z loop would force the loop to be fully unrolled: 8 copies of the ~600-instruction body).
// Requires the TMA path (16-byte aligned pitch and base); otherwise the launcher takes bp_brick_kernel.
#ifndef BP2_STAGES_N
#define BP2_STAGES_N 3
#endif
#ifndef BP2_SERIES
#define BP2_SERIES 0
#endif
constexpr int BP2_STAGES = BP2_STAGES_N;

__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <int ARC, int RECON, int MODEL>
__global__ void __launch_bounds__(BRICK_THREADS, BP2_MINB)
bp_brick2_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ proj,
                 const __grid_constant__ CUtensorMap tmap, float *__restrict__ vol,
                 int view_begin, int view_stride, int view_count, int j_lo, int j_hi, int nbz, int accumulate, int poison)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    float *tiles = reinterpret_cast<float *>(smem_raw);                                    // [BP2_STAGES][TILE_FLOATS]
    float2 *accs = reinterpret_cast<float2 *>(tiles + BP2_STAGES * TILE_FLOATS);           // [BZ / 2][256]
    __shared__ SfView sview[BP2_STAGES];
    __shared__ TileInfo tinfo[BP2_STAGES];
    __shared__ __align__(8) uint64_t full[BP2_STAGES], empty[BP2_STAGES];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tx = tid % BX, ty = tid / BX;
    const int bzi = blockIdx.z % nbz, batch = blockIdx.z / nbz;
    const int p0 = blockIdx.x * BX, q0 = blockIdx.y * BY, z0 = bzi * BZ;
    const int p1 = min(p0 + BX, pr.nx) - 1, q1 = min(q0 + BY, pr.ny) - 1, z1 = min(z0 + BZ, pr.nz) - 1;
    const int ip = p0 + tx, iq = q0 + ty;
    const bool col_in = ip < pr.nx && iq < pr.ny;
    const float p = (float)ip, q = (float)iq;
    const int view_off = batch * view_count;
    const int nzb = z1 - z0 + 1;                                 // voxels in this brick's z-run

    for (int i = tid; i < (BZ / 2) * BRICK_THREADS; i += BRICK_THREADS) accs[i] = make_float2(0.0f, 0.0f);
    for (int i = tid; i < BP2_STAGES * LM * TW; i += BRICK_THREADS)
        tiles[(i / (LM * TW)) * TILE_FLOATS + TH * TW + i % (LM * TW)] = 0.0f;
    if (poison) {
        // testing aid (CtsfDebug::bp_poison): the data rows of every ring stage start as NaN, the worst that
        // uninitialised shared memory can hold; a stage that no view is staged into keeps them.  No load that feeds a
        // result may ever reach such a stage (a weight of exactly 0 does not help: 0 * NaN = NaN).
        for (int i = tid; i < BP2_STAGES * TH * TW; i += BRICK_THREADS)
            tiles[(i / (TH * TW)) * TILE_FLOATS + i % (TH * TW)] = __int_as_float(0x7fc00000);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // ordered before the TMA writes that follow
    }
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < BP2_STAGES; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], BRICK_THREADS / 32); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // warp 0: stage view j into ring slot s (parameters, shadow, TMA) and arm full[s]
    auto produce = [&](int j, int s) {
        const SfView *gv = views + view_begin + (size_t)j * view_stride;
        constexpr int W = (int)(sizeof(SfView) / 4);
        for (int w = lane; w < W; w += 32)
            reinterpret_cast<uint32_t *>(&sview[s])[w] = reinterpret_cast<const uint32_t *>(gv)[w];
        __syncwarp();
        TileInfo t = brick_shadow<ARC>(sview[s], pr, (float)p0, (float)p1, (float)q0, (float)q1, (float)z0, (float)z1, lane);
        if (lane == 0) {
            tinfo[s] = t;
            if (t.live) {
                mbar_expect_tx(&full[s], TW * TH * 4);              // arrive (release: the stores above) + tx count
                tma_load_3d(tiles + s * TILE_FLOATS, &tmap, &full[s], t.k0, t.l0, view_off + j);
            } else {
                mbar_arrive(&full[s]);
            }
        }
        __syncwarp();
    };
    auto coop_load = [&](float *dst, int k0, int l0, int j) {
        const float *src = proj + (size_t)(view_off + j) * pr.nu * pr.nv;
        for (int i = tid; i < TW * TH; i += BRICK_THREADS) {
            const int r = i / TW, cidx = i - r * TW;
            const int k = k0 + cidx, l = l0 + r;
            const bool ok = k >= 0 && k < pr.nu && l >= 0 && l < pr.nv;
            const float *gp = ok ? src + (size_t)l * pr.nu + k : src;
            const int sz = ok ? 4 : 0;
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" ::"r"(smem_u32(dst + i)), "l"(gp), "r"(sz) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
        asm volatile("cp.async.wait_group 0;" ::: "memory");
    };

    if (warp == 0)
        for (int d = 0; d < BP2_STAGES - 1 && j_lo + d < j_hi; ++d) produce(j_lo + d, d);

    int s = 0, sp = BP2_STAGES - 1;           // slot of view j / of view j + BP2_STAGES - 1
    uint32_t par = 0u;                        // phase parity of slot s's current use
    for (int j = j_lo; j < j_hi; ++j) {
        // the producer role rotates over the warps (view j + 2 is staged by warp (j mod 8)), so that no warp is
        // systematically behind the others by the staging work
        if (warp == ((j - j_lo) & (BRICK_THREADS / 32 - 1)) && j + BP2_STAGES - 1 < j_hi) {
            // slot sp held view j - 1: every warp must have left it (its first use needs no wait)
            if (j > j_lo) mbar_wait(&empty[sp], (uint32_t)(((j - 1 - j_lo) / BP2_STAGES) & 1));
            produce(j + BP2_STAGES - 1, sp);
        }
        mbar_wait(&full[s], par);
        const TileInfo t = tinfo[s];
        if (t.live) {
            const SfView v = sview[s];
            float *tile = tiles + s * TILE_FLOATS;
            uint32_t tile_a = smem_u32(tile);
            asm volatile("" : "+r"(tile_a));
            const float a_col = fmaf(q, v.aq, fmaf(p, v.ap, v.a0));
            const float b_col = fmaf(q, v.bq, fmaf(p, v.bp, v.b0));
            const float c_col = fmaf(q, v.cq, fmaf(p, v.cp, v.c0));
            const float m_amp = fmaxf(fabsf(p + v.ep0), fabsf(q + v.eq0));
            for (int bl = 0; bl < t.nbl; ++bl)
                for (int bk = 0; bk < t.nbk; ++bk) {
                    const int tk0 = t.k0 + bk * TW, tl0 = t.l0 + bl * TH;
                    if (bk != 0 || bl != 0) {            // a shadow larger than one box (rare): block-wide staging
                        __syncthreads();
                        coop_load(tile, tk0, tl0, j);
                        __syncthreads();
                    }
                    if (!col_in) continue;
                    const int kmin = max(0, tk0), kmax = min(pr.nu - 1, tk0 + TW - 1);
                    const int lmin = max(0, tl0), lmax = min(pr.nv - 1, tl0 + TH - 1);
                    for (int zi = 0; zi < nzb; zi += 2) {
                        const float2 z = p2((float)(z0 + zi), (float)(z0 + zi + 1));
                        const float2 a = p2fma(z, p2s(v.az), p2s(a_col)), b = p2fma(z, p2s(v.bz), p2s(b_col));
                        const float2 c = p2fma(z, p2s(v.cz), p2s(c_col));
                        const float2 inv_a = p2rcp_nr(a);
                        SfTrans2 T;
                        sf_transaxial2<ARC, MODEL, BP2_SERIES>(v, a, b, inv_a, T, p, q);
                        const float2 kf0 = p2add(T.kc, T.t0), kf3 = p2add(T.kc, T.t3);
                        int kloA = max(kmin, (int)floorf(kf0.x)), khiA = min(kmax, (int)floorf(kf3.x));
                        int kloB = max(kmin, (int)floorf(kf0.y)), khiB = min(kmax, (int)floorf(kf3.y));
                        SfAxial2 A;
                        sf_axial2<ARC, BP2_SERIES>(v, a, b, c, inv_a, A);
                        const float2 lf0 = p2add(A.lc, A.tlo), lf1 = p2add(A.lc, A.thi);
                        int lloA = max(lmin, (int)floorf(lf0.x)), lhiA = min(lmax, (int)floorf(lf1.x));
                        int lloB = max(lmin, (int)floorf(lf0.y)), lhiB = min(lmax, (int)floorf(lf1.y));
                        const bool liveA = kloA <= khiA && lloA <= lhiA;
                        const bool liveB = kloB <= khiB && lloB <= lhiB && zi + 1 < nzb;
                        if (!liveA && !liveB) continue;
                        // a dead partner rides along with zero weights on a valid address
                        if (!liveA) { kloA = kmin; khiA = kmin - 1; lloA = lmin; lhiA = lmin - 1; }
                        if (!liveB) { kloB = kmin; khiB = kmin - 1; lloB = lmin; lhiB = lmin - 1; }
                        float2 amp;
                        if (RECON) {
                            amp = p2(sf_recon_weight_s<ARC>(v, T.h01.x + T.w12.x + T.h23.x, A.thi.x - A.tlo.x, a.x, b.x),
                                     sf_recon_weight_s<ARC>(v, T.h01.y + T.w12.y + T.h23.y, A.thi.y - A.tlo.y, a.y, b.y));
                        } else {
                            amp = sf_amplitude2(a, b, c, m_amp);
                        }
                        const int Kmax = max(khiA - kloA, khiB - kloB) + 1;
                        const int Lmax = max(lhiA - lloA, lhiB - lloB) + 1;
                        // the row loop runs over max(L_a, L_b) rows too: each footprint is cut at the lower edge of its
                        // own last row, so the rows past it weigh exactly 0 (also where a box or the detector ends)
                        A.thi = p2min(A.thi, p2sub(p2((float)(lhiA + 1), (float)(lhiB + 1)), A.lc));
                        const float2 xi0 = p2sub(p2((float)kloA, (float)kloB), T.kc);
                        const float2 xe = p2sub(p2((float)(khiA + 1), (float)(khiB + 1)), T.kc);   // last edge of each voxel
                        const float2 g00 = sf_G2<MODEL>(T, xi0);
                        float2 sum = p2s(0.0f);
                        const uint32_t baseA = tile_a + 4u * (unsigned)((lloA - tl0) * TW + (kloA - tk0));
                        const uint32_t baseB = tile_a + 4u * (unsigned)((lloB - tl0) * TW + (kloB - tk0));
                        // Both voxels walk max(L_a, L_b) rows and max(K_a, K_b) columns from their own first cell.  The
                        // one whose footprint ends first (cut by the box or the detector) would run on past the LM zero
                        // rows below the tile -- into the next ring stage or the accumulators, which may hold anything,
                        // and 0 * NaN is NaN.  A row chunk that would start at or below row TH (all of its rows weigh 0
                        // for that voxel) is PARKED on the zero rows at column 0 instead: K_max <= TW columns from there
                        // stay inside them.  With 0 <= column < TW, "row >= TH" is "address >= first zero row", so one
                        // min does it.  A chunk that starts inside the tile ends at row TH + 2 at most, and its columns
                        // past TW wrap into the next row of the same tile.
                        const uint32_t zero_rows = tile_a + 4u * (unsigned)(TH * TW);
                        for (int lb = 0; lb < Lmax; lb += LM) {
                            float2 f2[LM];
                            sf_F2_run2<LM>(A, p2((float)(lloA + lb), (float)(lloB + lb)), f2);
                            uint32_t ra = min(baseA + 4u * (unsigned)(lb * TW), zero_rows);
                            uint32_t rb = min(baseB + 4u * (unsigned)(lb * TW), zero_rows);
                            float2 xi = xi0, g0 = g00;
#pragma unroll 1
                            for (int k = 0; k < Kmax; ++k, ra += 4, rb += 4) {
                                const float ya0 = lds_f32(ra), ya1 = lds_f32(ra + 4 * TW), ya2 = lds_f32(ra + 8 * TW), ya3 = lds_f32(ra + 12 * TW);
                                const float yb0 = lds_f32(rb), yb1 = lds_f32(rb + 4 * TW), yb2 = lds_f32(rb + 8 * TW), yb3 = lds_f32(rb + 12 * TW);
                                xi = p2add(xi, p2s(1.0f));
                                const float2 g1 = sf_G2<MODEL>(T, p2min(xi, xe));
                                float2 sr = p2mul(f2[0], p2(ya0, yb0));
                                sr = p2fma(f2[1], p2(ya1, yb1), sr);
                                sr = p2fma(f2[2], p2(ya2, yb2), sr);
                                sr = p2fma(f2[3], p2(ya3, yb3), sr);
                                sum = p2fma(p2sub(g1, g0), sr, sum);
                                g0 = g1;
                            }
                        }
                        float2 *ap = accs + (zi >> 1) * BRICK_THREADS + tid;
                        *ap = p2fma(amp, sum, *ap);
                    }
                }
            // extra boxes were staged into this slot by cp.async (generic proxy); the slot's next writer is a TMA (async
            // proxy) issued after empty[s] completes: every writing thread fences across the proxies before it arrives
            if (t.nbk * t.nbl > 1) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
        sp = s;
        if (++s == BP2_STAGES) { s = 0; par ^= 1u; }
    }
    if (col_in) {
        float *o = vol + (size_t)batch * pr.nx * pr.ny * pr.nz + ((size_t)z0 * pr.ny + iq) * pr.nx + ip;
        for (int zi = 0; zi < nzb; ++zi) {
            float *oz = o + (size_t)zi * pr.ny * pr.nx;
            const float2 r2 = accs[(zi >> 1) * BRICK_THREADS + tid];
            const float r = (zi & 1) ? r2.y : r2.x;
            *oz = accumulate ? *oz + r : r;
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode()
{
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        else
            cudaGetLastError();
    }
    return fn;
}

template <int ARC>
int launch_brick(const ct_geom *g, const float *d_proj, float *d_vol, int batch, int vb, int vs, int vc, cudaStream_t st,
                 int accumulate, int recon)
{
    const SfProblem &pr = g->prob;
    CUtensorMap tmap;
    memset(&tmap, 0, sizeof tmap);
    int use_tma = 0;
    EncodeTiledFn enc = get_encode();
    const int dbg_tma = g_ctsf_debug.bp_tma;            // testing aid: -1 default, 0 cp.async only, 1..3 partial TMA use
    if (enc && dbg_tma != 0 && vc > 0 && pr.nu % 4 == 0 && ((uintptr_t)d_proj & 15u) == 0) {
        cuuint64_t dims[3] = {(cuuint64_t)pr.nu, (cuuint64_t)pr.nv, (cuuint64_t)vc * batch};
        cuuint64_t strides[2] = {(cuuint64_t)pr.nu * 4, (cuuint64_t)pr.nu * pr.nv * 4};
        cuuint32_t box[3] = {TW, TH, 1}, es[3] = {1, 1, 1};
        if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)d_proj, dims, strides, box, es,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS)
            use_tma = (dbg_tma >= 1 && dbg_tma <= 3) ? dbg_tma : 3;
    }
    const size_t smem = (size_t)(2 * TILE_FLOATS + BZ * BRICK_THREADS) * sizeof(float);
    const size_t smem2 = (size_t)(BP2_STAGES * TILE_FLOATS + BZ * BRICK_THREADS) * sizeof(float);
    // untilted frames with small footprints (host bound): F1 weights live in registers along the z-run
    // (testing aids bp_nohoist / bp_forcehoist of CtsfDebug, as for the forward kernel)
    const bool hoist = !g_ctsf_debug.bp_nohoist &&
                       (g->fp_hoist_ok || (g->all_untilted && g_ctsf_debug.bp_forcehoist)) && g->model != 2;
    // general frames: the packed two-voxel kernel (needs the TMA path); the testing aid bp_scalar keeps the
    // one-voxel-per-thread kernel
    const bool packed = !hoist && use_tma == 3 && !g_ctsf_debug.bp_scalar && g->model == 0;   // DD: its rectangle footprint has no packed form worth having (measured 306 vs 289 ms)
    auto kern = g->model == 2 ? (recon ? bp_brick_kernel<ARC, 1, 0, 2> : bp_brick_kernel<ARC, 0, 0, 2>)
        : g->model == 1
        ? (hoist ? (recon ? bp_brick_kernel<ARC, 1, 1, 1> : bp_brick_kernel<ARC, 0, 1, 1>)
                 : (recon ? bp_brick_kernel<ARC, 1, 0, 1> : bp_brick_kernel<ARC, 0, 0, 1>))
        : (hoist ? (recon ? bp_brick_kernel<ARC, 1, 1, 0> : bp_brick_kernel<ARC, 0, 1, 0>)
                 : (recon ? bp_brick_kernel<ARC, 1, 0, 0> : bp_brick_kernel<ARC, 0, 0, 0>));
    auto kern2 = g->model == 1 ? (recon ? bp_brick2_kernel<ARC, 1, 1> : bp_brick2_kernel<ARC, 0, 1>)
                               : (recon ? bp_brick2_kernel<ARC, 1, 0> : bp_brick2_kernel<ARC, 0, 0>);
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (packed) cudaFuncSetAttribute(kern2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
    const int nbz = (pr.nz + BZ - 1) / BZ;
    int launches = 0;
    // The view loop is cut into chunks of ~288 MB of projections, one launch each (every launch after the first adds
    // to the volume): all bricks sweep one chunk while most of it stays in the 126 MB L2, instead of each wave of CTAs
    // streaming the whole projection set from HBM again.  Measured at config 4 (B200, per A^T; time / DRAM read + written):
    // 40 views per launch 394.8 ms / 13.4 + 8.7 GB; 80: 390.0 / 13.9 + 4.4; 120: 389.1 / 15.0 + 2.9; 240: 389.1 / 22.5 + 1.5;
    // all 720 in one launch 390.5 / 105 + 0.5.  120 views (283 MB) is the fastest and moves the fewest bytes.
    const size_t view_bytes = (size_t)pr.nu * pr.nv * sizeof(float) * batch;
    int chunk = (int)((288u << 20) / (view_bytes ? view_bytes : 1));
    if (chunk < 8) chunk = 8;
    if (g_ctsf_debug.bp_chunk > 0) chunk = g_ctsf_debug.bp_chunk;
    for (int j_lo = 0; j_lo < vc || (vc == 0 && j_lo == 0); j_lo += chunk) {
        const int j_hi = j_lo + chunk < vc ? j_lo + chunk : vc;
        for (int b0 = 0; b0 < batch;) {
            int nb = batch - b0;
            if ((long)nb * nbz > 65535) nb = 65535 / nbz > 0 ? 65535 / nbz : 1;
            dim3 grid((pr.nx + BX - 1) / BX, (pr.ny + BY - 1) / BY, nbz * nb);
            // the tensor map addresses view (batch*vc + j): pass the buffer of image b0 by offsetting batch in-kernel
            if (packed && b0 == 0)
                kern2<<<grid, BRICK_THREADS, smem2, st>>>(pr, g->d_bp, d_proj, tmap, d_vol, vb, vs, vc, j_lo, j_hi, nbz,
                                                          accumulate || j_lo > 0, g_ctsf_debug.bp_poison ? 1 : 0);
            else
                kern<<<grid, BRICK_THREADS, smem, st>>>(pr, g->d_bp, d_proj + (size_t)b0 * vc * pr.nv * pr.nu, tmap, b0 == 0 ? use_tma : 0,
                                                        d_vol + (size_t)b0 * pr.nx * pr.ny * pr.nz, vb, vs, vc, j_lo, j_hi, nbz,
                                                        accumulate || j_lo > 0);
            ++launches;
            b0 += nb;
        }
        if (vc == 0) break;
    }
    return launches;
}

template <int ARC, int NB>
void launch_pixel(const ct_geom *g, const float *d_proj, float *d_vol, int b0, int groups, int vb, int vs, int vc,
                  cudaStream_t st, int recon)
{
    const SfProblem &pr = g->prob;
    const size_t pbs = (size_t)vc * pr.nu, vbs = (size_t)pr.nx * pr.ny;
    dim3 block(16, 8, 1);
    dim3 grid((pr.nx + block.x - 1) / block.x, (pr.ny + block.y - 1) / block.y, groups);
    auto kern = g->model == 1 ? (recon ? bp_pixel_kernel<ARC, NB, 1, 1> : bp_pixel_kernel<ARC, NB, 0, 1>)     // 2-D: SF-TT == SF-TR
                              : (recon ? bp_pixel_kernel<ARC, NB, 1, 0> : bp_pixel_kernel<ARC, NB, 0, 0>);
    kern<<<grid, block, 0, st>>>(pr, g->d_bp, d_proj + (size_t)b0 * pbs, d_vol + (size_t)b0 * vbs,
                                 vb, vs, vc, (unsigned)pbs, (unsigned)vbs);
}

template <int ARC>
int launch_pixel_batches(const ct_geom *g, const float *d_proj, float *d_vol, int batch, int vb, int vs, int vc,
                         cudaStream_t st, int recon)
{
    // batch images share the weights (S6): groups of 16, 8, 4, 2, 1 images per thread
    int launches = 0, b0 = 0;
    const int sizes[5] = {16, 8, 4, 2, 1};
    for (int s = 0; s < 5; ++s) {
        const int nb = sizes[s];
        int groups = (batch - b0) / nb;
        while (groups > 0) {
            const int gnow = groups > 65535 ? 65535 : groups;
            switch (nb) {
                case 16: launch_pixel<ARC, 16>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st, recon); break;
                case 8: launch_pixel<ARC, 8>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st, recon); break;
                case 4: launch_pixel<ARC, 4>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st, recon); break;
                case 2: launch_pixel<ARC, 2>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st, recon); break;
                default: launch_pixel<ARC, 1>(g, d_proj, d_vol, b0, gnow, vb, vs, vc, st, recon); break;
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
                   int view_begin, int view_stride, int view_count, void *stream, int accumulate, int recon)
{
    cudaStream_t st = (cudaStream_t)stream;
    const int arc = g->prob.det_type, dim = g->prob.dim;
    if (accumulate && dim != 3) return -1;       // only the 3-D brick kernel can add to its output
    int n;
    if (dim == 2) n = arc ? launch_pixel_batches<1>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st, recon)
                          : launch_pixel_batches<0>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st, recon);
    else          n = arc ? launch_brick<1>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st, accumulate, recon)
                          : launch_brick<0>(g, d_proj, d_vol, batch, view_begin, view_stride, view_count, st, accumulate, recon);
    return cudaGetLastError() == cudaSuccess ? n : -1;
}
