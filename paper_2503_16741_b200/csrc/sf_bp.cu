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
    const float mk = 0.75f, ml = ARC ? 1.5f : 0.75f;
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
        sf_F2_run<LM>(A, (float)lb, f2);
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
        sf_F2_run<LM>(A, (float)lb, f2);
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
                            sf_axial<ARC>(v, a, b, c, inv_a, A);
                            const int l_lo = max(max(0, tl0), (int)floorf(A.lc + A.tlo));
                            const int l_hi = min(min(pr.nv - 1, tl0 + TH - 1), (int)floorf(A.lc + A.thi));
                            if (l_lo > l_hi) continue;
                            float amp, sum;
                            if (UNT) {
                                amp = RECON ? sf_recon_weight_s<ARC>(v, sumF1, A.thi - A.tlo, a, b)
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
                                amp = RECON ? sf_recon_weight<ARC>(v, T, A.thi - A.tlo, a, b)
                                            : sf_amplitude(v, a, b, c, p, q);
                                sum = gather_tile<MODEL>(tile_a, T, A, k_lo, k_hi, l_lo, l_hi, tk0, tl0);
                            }
                            float *ap = accs + zi * BRICK_THREADS + tid;
                            *ap = fmaf(amp, sum, *ap);
                        }
                    }
                }
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
    const char *dbg = getenv("CTSF_BP_TMA");
    if (enc && !(dbg && dbg[0] == '0') && vc > 0 && pr.nu % 4 == 0 && ((uintptr_t)d_proj & 15u) == 0) {
        cuuint64_t dims[3] = {(cuuint64_t)pr.nu, (cuuint64_t)pr.nv, (cuuint64_t)vc * batch};
        cuuint64_t strides[2] = {(cuuint64_t)pr.nu * 4, (cuuint64_t)pr.nu * pr.nv * 4};
        cuuint32_t box[3] = {TW, TH, 1}, es[3] = {1, 1, 1};
        if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)d_proj, dims, strides, box, es,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS)
            use_tma = (dbg && dbg[0] >= '1' && dbg[0] <= '3') ? dbg[0] - '0' : 3;
    }
    const size_t smem = (size_t)(2 * TILE_FLOATS + BZ * BRICK_THREADS) * sizeof(float);
    // untilted frames with small footprints (host bound): F1 weights live in registers along the z-run
    // (testing aids: CTSF_BP_NOHOIST / CTSF_BP_FORCEHOIST, as for the forward kernel)
    const bool hoist = !getenv("CTSF_BP_NOHOIST") &&
                       (g->fp_hoist_ok || (g->all_untilted && getenv("CTSF_BP_FORCEHOIST")));
    auto kern = g->model == 1
        ? (hoist ? (recon ? bp_brick_kernel<ARC, 1, 1, 1> : bp_brick_kernel<ARC, 0, 1, 1>)
                 : (recon ? bp_brick_kernel<ARC, 1, 0, 1> : bp_brick_kernel<ARC, 0, 0, 1>))
        : (hoist ? (recon ? bp_brick_kernel<ARC, 1, 1, 0> : bp_brick_kernel<ARC, 0, 1, 0>)
                 : (recon ? bp_brick_kernel<ARC, 1, 0, 0> : bp_brick_kernel<ARC, 0, 0, 0>));
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const int nbz = (pr.nz + BZ - 1) / BZ;
    int launches = 0;
    // The view loop is cut into chunks of ~96 MB of projections, one launch each (every launch after the
    // first adds to the volume): all bricks sweep one chunk while it sits in the 126 MB L2, instead of
    // each wave of CTAs streaming the whole projection set from HBM again.
    const size_t view_bytes = (size_t)pr.nu * pr.nv * sizeof(float) * batch;
    int chunk = (int)((96u << 20) / (view_bytes ? view_bytes : 1));
    if (chunk < 8) chunk = 8;
    const char *cdbg = getenv("CTSF_BP_CHUNK");
    if (cdbg && atoi(cdbg) > 0) chunk = atoi(cdbg);
    for (int j_lo = 0; j_lo < vc || (vc == 0 && j_lo == 0); j_lo += chunk) {
        const int j_hi = j_lo + chunk < vc ? j_lo + chunk : vc;
        for (int b0 = 0; b0 < batch;) {
            int nb = batch - b0;
            if ((long)nb * nbz > 65535) nb = 65535 / nbz > 0 ? 65535 / nbz : 1;
            dim3 grid((pr.nx + BX - 1) / BX, (pr.ny + BY - 1) / BY, nbz * nb);
            // the tensor map addresses view (batch*vc + j): pass the buffer of image b0 by offsetting batch in-kernel
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
    auto kern = g->model == 1 ? (recon ? bp_pixel_kernel<ARC, NB, 1, 1> : bp_pixel_kernel<ARC, NB, 0, 1>)
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
