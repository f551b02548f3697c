// sf_fp.cu -- ct_fp_sf: SF-TR forward projector y = A x (Eq. 1).
//
// Output-exclusive design, no atomics of any kind.  One WARP owns one detector tile of one view and
// keeps it in shared memory for the whole pass.  It walks the voxel slabs perpendicular to the view's
// dominant ray axis; per slab it inverse-projects the tile onto the slab to find the voxels
// that can touch it, and adds their footprints into the tile in conflict-free "rounds" (see
// fp_band_kernel).  Each detector cell is stored exactly once; the summation order is fixed.
//
// Views whose rays run mostly along x read the volume through an xy-transposed copy so that the
// in-slab index p is always the memory-fastest one.
#include <cuda_runtime.h>

#include <climits>
#include <cstdlib>

#include "ctsf_internal.h"
#include "sf_footprint.cuh"

// the untilted instantiations (UNT = 1) leave the general sweep after their `continue` unreachable by design
#pragma nv_diag_suppress 128

namespace {

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

// ---------------------------------------------------------------------------------------------------
// warp-band forward projector
// ---------------------------------------------------------------------------------------------------
// One WARP owns one detector tile of one view: FTK cells x FTL rows (3-D) or FTK cells x NB images
// (2-D), held in the warp's private slice of shared memory for the whole pass.  No block barrier is
// ever executed.  Per slab the warp inverse-projects its tile (rays through the tile corners + the exact
// half-voxel halo) to the quadrilateral of voxels that can touch it and sweeps that region in sheared,
// flattened order, 32 voxels per pass: lane i computes its voxel's footprint once, and the warp adds
// the footprints into the tile in K "rounds": in round j every lane updates column k_lo(i) + j of its
// own footprint (all its rows).  The lanes of a pass have pairwise different k_lo, or touch disjoint
// rows (the host picks a lane stride so that neighbouring voxels project >= 1 cell apart; rows of equal
// p are interleaved half a region apart; the kernel verifies both per pass with a warp match and
// serialises the pass otherwise), so within a round no two lanes touch the same cell; rounds are
// separated by __syncwarp().  Summation order is fixed => deterministic.
constexpr int FPW = 8;            // warps per CTA (slab-split 2-D kernels; unit of the item groups)
#ifndef FP_WPC
#define FP_WPC 8                     // warps per CTA of the general kernels (measured: 1 warp per CTA is 1.5-5 % slower)
#endif
constexpr int FVG = 48;           // views per item group (multiple of FPW): consecutive CTAs sweep one tile of FVG views
constexpr int FMINB = 3;          // CTAs per SM the register budget is sized for
constexpr int FTK = 64;           // cells per warp tile
constexpr int FTL = 32;           // rows per warp tile (3-D)
constexpr int FKR = 6;            // untilted fast path: F1 weights of up to FKR columns live in registers
constexpr int FLM = 4;            // pad rows: the first FLM footprint rows are updated unconditionally
constexpr unsigned FULL = 0xffffffffu;

__device__ __forceinline__ uint32_t smem_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float lds_f32(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v)); }

// one round of one lane: tile[row j][its column] += w * f2[j] for the lane's rows.  FIRST: the first FLM rows are
// updated unconditionally (weight 0 past the footprint, pad rows past the tile); EXTRA: rows FLM .. 2 FLM - 1 exist
// for some lane of the warp.  Loads first, then FMAs, then stores (the volatile asm keeps this order).
template <bool FIRST, bool EXTRA>
__device__ __forceinline__ void fp_round_rows(uint32_t ca, float w, const float *f2, int nrow)
{
    constexpr int RB = FTK * 4;
    if (FIRST) {
        const float c0 = lds_f32(ca), c1 = lds_f32(ca + RB), c2 = lds_f32(ca + 2 * RB), c3 = lds_f32(ca + 3 * RB);
        sts_f32(ca, fmaf(w, f2[0], c0)); sts_f32(ca + RB, fmaf(w, f2[1], c1));
        sts_f32(ca + 2 * RB, fmaf(w, f2[2], c2)); sts_f32(ca + 3 * RB, fmaf(w, f2[3], c3));
    } else {
#pragma unroll
        for (int j = 0; j < FLM; ++j)
            if (j < nrow) sts_f32(ca + j * RB, fmaf(w, f2[j], lds_f32(ca + j * RB)));
    }
    if (EXTRA) {
#pragma unroll
        for (int j = FLM; j < 2 * FLM; ++j)
            if (j < nrow) sts_f32(ca + j * RB, fmaf(w, f2[j], lds_f32(ca + j * RB)));
    }
}

// the same for footprints of at most three rows (untilted frames with cells larger than half a voxel's shadow:
// configs 2, 3): three unconditional rows instead of four
__device__ __forceinline__ void fp_round_rows3(uint32_t ca, float w, const float *f2)
{
    constexpr int RB = FTK * 4;
    const float c0 = lds_f32(ca), c1 = lds_f32(ca + RB), c2 = lds_f32(ca + 2 * RB);
    sts_f32(ca, fmaf(w, f2[0], c0)); sts_f32(ca + RB, fmaf(w, f2[1], c1)); sts_f32(ca + 2 * RB, fmaf(w, f2[2], c2));
}

template <int DIM, int ARC, int NB, int UNT, int MODEL, int QS = 0>
__global__ void __launch_bounds__(32 * (QS ? FPW : FP_WPC), FMINB * FPW / (QS ? FPW : FP_WPC))
fp_band_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ vol,
               const float *__restrict__ volT, float *__restrict__ proj, int view_begin, int view_stride,
               int tiles_k, int bands_l, int n_items, int n_views_sel, size_t vol_bstride, size_t proj_bstride,
               float region_pad, int force_serial)
{
    constexpr int ROWS = DIM == 3 ? FTL + FLM : NB;
    extern __shared__ float smem[];
    // Warps per CTA.  Every warp is independent (own tile, own view parameters).  With one warp per CTA `warp` is the
    // constant 0 and every per-warp shared-memory address a compile-time offset (with 8 warps ptxas, at its 80-register
    // budget, keeps re-deriving them from threadIdx: 5-7 % of the executed instructions) -- yet measured on B200 the
    // 1-warp CTAs were slower (config 4: 673.6 vs 664.2 ms; configs 2, 3, 5: +4 %, +5.5 %, +5 %), so FP_WPC stays 8.
    constexpr int WPC = QS ? FPW : FP_WPC;
    __shared__ SfView sviews[WPC];
    __shared__ Ray srays[WPC][6];
    const int lane = threadIdx.x & 31, warp = WPC == 1 ? 0 : (int)(threadIdx.x >> 5);
    // QS (2-D, small problems): the FPW warps of a CTA share ONE item and split its slabs (warp w takes slabs w, w + FPW,
    // ...); their private tiles are summed in warp order at the end.  Otherwise every warp has an item of its own.
    const int item = QS ? (int)blockIdx.x : (int)blockIdx.x * WPC + warp;
    if (item >= n_items) return;                     // warps are independent: no block barrier below (QS: CTA-uniform)
    // item order: groups of FVG consecutive views; within a group tile-major, view fastest -- the
    // warps of one CTA (and the next FVG/FPW - 1 CTAs) sweep the SAME tile of neighbouring views, whose
    // frusta nearly coincide, so the volume is pulled through L1/L2 once per group of views instead of
    // once per view
    const int per_view = tiles_k * bands_l;
    const int grp = item / (per_view * FVG), rem_g = item - grp * (per_view * FVG);
    const int rem = rem_g / FVG, jview = grp * FVG + (rem_g - rem * FVG);
    if (jview >= n_views_sel) return;
    const int bl = rem / tiles_k, tk = rem - bl * tiles_k;
    const int k0 = tk * FTK, l0 = bl * FTL;
    const int tkw = min(FTK, pr.nu - k0), tlh = DIM == 3 ? min(FTL, pr.nv - l0) : 1;
    const int b0 = blockIdx.y * NB;
    float *tile = smem + warp * (ROWS * FTK);

    for (int w = lane; w < (int)(sizeof(SfView) / 4); w += 32)
        reinterpret_cast<uint32_t *>(&sviews[warp])[w] =
            reinterpret_cast<const uint32_t *>(views + view_begin + (size_t)jview * view_stride)[w];
    for (int i = lane; i < ROWS * FTK; i += 32) tile[i] = 0.0f;
    __syncwarp();
    const SfView &v = sviews[warp];
    // Rays through the tile's corners (and, for the arc, the mid column: the slab image of an arc tile
    // bulges).  The surfaces k = const and (flat) l = const through the source are planes, so they cut a
    // slab in straight lines and the tile's pre-image in the slab is the quadrilateral spanned by the
    // rays.  A voxel touches the tile iff one of its four transaxial corners (+-1/2, +-1/2) / its two
    // axial end points (0, 0, +-1/2) cross those lines, i.e. iff its centre lies within
    // hp = 1/2 + 1/2 |dp/dq| voxels in p and 1/2 voxel in z of the quadrilateral.
    float slope = 0.0f;
    if (lane < 6) {
        const float kA = (float)k0, kB = (float)(k0 + tkw), lA = (float)l0, lB = (float)(l0 + tlh);
        const float kk = (lane % 3 == 0) ? kA : (lane % 3 == 1 ? kB : 0.5f * (kA + kB));
        const Ray ry = tile_ray<ARC>(v, kk, lane < 3 ? lA : lB);
        // stored per unit of q: (dp/dq, sign of dq, dz/dq); sign 0 marks a ray (almost) parallel to the slabs, for which
        // the whole slab is swept.  The slab loop then needs two FMAs and one compare per ray instead of a reciprocal.
        const bool flat_ray = fabsf(ry.dq) < 1e-3f * (fabsf(ry.dp) + fabsf(ry.dz));
        const float inv_dq = flat_ray ? 0.0f : rcp_nr(ry.dq);
        Ray rn;
        rn.dp = ry.dp * inv_dq; rn.dq = flat_ray ? 0.0f : (ry.dq > 0.0f ? 1.0f : -1.0f); rn.dz = ry.dz * inv_dq;
        srays[warp][lane] = rn;
        // direction of the line {k = const, z = const} in the slab plane: the ray minus its z part along v
        float dp = ry.dp, dq = ry.dq;
        if (DIM == 3 && fabsf(v.Vz) > 1e-6f) {
            const float t = ry.dz / v.Vz;
            dp = fmaf(-t, v.Vp, dp); dq = fmaf(-t, v.Vq, dq);
        }
        slope = fabsf(dp) / fmaxf(fabsf(dq), 1e-6f);
    }
#pragma unroll
    for (int s_ = 1; s_ < 8; s_ <<= 1) slope = fmaxf(slope, __shfl_xor_sync(FULL, slope, s_));
    slope = __shfl_sync(FULL, slope, 0);
    // hp = 1/2 + 1/2 |dp/dq| is exact (+ 0.1 margin).  Beyond slope 8 (tile-edge rays within 7 degrees of the slab:
    // fans wider than ~75 degrees, or very anisotropic pitches) the whole in-slab range is swept instead
    const float hp = slope > 8.0f ? 1e9f : 0.6f + 0.5f * slope + region_pad;
    const float hz = (ARC ? 1.5f : 1.1f) + region_pad + (MODEL == 2 ? v.zpad : 0.0f);            // 1/2 voxel + 1/2 (rounded shear shift) + margin (arc: bulge)
    __syncwarp();

    const int np = v.swap_xy ? pr.ny : pr.nx, nq = v.swap_xy ? pr.nx : pr.ny, nz = pr.nz;
    const float *src = (v.swap_xy ? volT : vol) + (size_t)b0 * vol_bstride;
    const int sp = max(1, v.lane_stride);
    const int k_top = k0 + tkw - 1, l_top = l0 + tlh - 1;
    const int zstride = np * nq;
    const float v_ap = v.ap, v_bp = v.bp, v_cp = v.cp, v_az = v.az, v_bz = v.bz, v_cz = v.cz;

    for (int iq = QS ? warp : 0; iq < nq; iq += QS ? FPW : 1) {
        // ---- voxel region of this slab that can touch the tile (warp-uniform) --------------------
        // The tile's frustum cuts the slab in a quadrilateral whose rows are skewed (the row coordinate
        // depends on depth, hence on p): the region is swept in sheared coordinates (p, z' = z - shift(p)).
        float pr_[6], zr_[6];
        float pmin = 1e30f, pmax = -1e30f;
        bool whole = false;
        const float dqc = (float)iq - v.Sq;
#pragma unroll
        for (int r = 0; r < 6; ++r) {
            if (DIM == 2 && r >= 3) break;
            const Ray ry = srays[warp][r];                      // (dp/dq, sign(dq) or 0, dz/dq)
            if (!(ry.dq * dqc > 0.0f)) whole = true;            // slab behind the source along this ray, or a flat ray
            pr_[r] = fmaf(dqc, ry.dp, v.Sp); zr_[r] = fmaf(dqc, ry.dz, v.Sz);
            pmin = fminf(pmin, pr_[r]); pmax = fmaxf(pmax, pr_[r]);
        }
        int p_lo = 0, p_hi = np - 1, zs_lo = 0, zs_hi = nz - 1;
        float sigma = 0.0f;
        if (!whole) {
            p_lo = max(0, (int)ceilf(pmin - hp)); p_hi = min(np - 1, (int)floorf(pmax + hp));
            if (DIM == 3) {
                // mean slope dz/dp of the two tile edges l = const (rays 0,1 and 3,4)
                const float dpp = (pr_[1] - pr_[0]) + (pr_[4] - pr_[3]);
                const float dzz = (zr_[1] - zr_[0]) + (zr_[4] - zr_[3]);
                sigma = fabsf(dpp) > 1.0f ? dzz / dpp : 0.0f;
                float zmin = 1e30f, zmax = -1e30f;
#pragma unroll
                for (int r = 0; r < 6; ++r) {
                    const float zs = fmaf(-sigma, pr_[r] - (float)p_lo, zr_[r]);
                    zmin = fminf(zmin, zs); zmax = fmaxf(zmax, zs);
                }
                const float smax = sigma * (float)(p_hi - p_lo);           // shift range over the region
                zs_lo = max((int)ceilf(zmin - hz), -(int)ceilf(fmaxf(smax, 0.0f)) - 1);
                zs_hi = min((int)floorf(zmax + hz), nz + (int)ceilf(fmaxf(-smax, 0.0f)));
            }
        }
        if (p_lo > p_hi || zs_lo > zs_hi) continue;
        const int npr = p_hi - p_lo + 1, nrows = zs_hi - zs_lo + 1;
        const float q = (float)iq;
        const float aq0 = fmaf(q, v.aq, v.a0), bq0 = fmaf(q, v.bq, v.b0), cq0 = fmaf(q, v.cq, v.c0);
        const float *slab = src + (size_t)iq * np;
        asm volatile("" : "+l"(slab));      // pin the slab pointer in registers (ptxas otherwise rebuilds it from the
                                            // kernel parameters, ~14 instructions, in every pass)

        if (UNT) {
            // ---- untilted frames with small footprints (n.z = u.z = 0; K <= FKR columns, L <= 2 FLM rows) ---
            // Lanes keep their p while the warp walks the region's rows: the whole transaxial part (trapezoid,
            // column range, conflict check, the F1 weights themselves) is computed once per (p, q) and held in
            // registers; a pass is left with the axial rectangle, the amplitude and K rounds of pure updates.
            for (int col = 0; col < sp; ++col) {
                const int nprc = (npr - col + sp - 1) / sp;
                if (nprc <= 0) break;
                for (int c0 = 0; c0 < nprc; c0 += 32) {
                    const int pi = c0 + lane;
                    const bool actp = pi < nprc;
                    const int ip = actp ? p_lo + col + sp * pi : p_lo;
                    const int sh = __float2int_rn(sigma * (float)(ip - p_lo));
                    const float p = (float)ip;
                    const float a = fmaf(p, v_ap, aq0), b = fmaf(p, v_bp, bq0), cpq = fmaf(p, v_cp, cq0);
                    const float inv_a = rcp_nr(a);
                    SfTrans T;
                    sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T, p, q);
                    const int k_lo = (int)floorf(T.kc + T.t0);
                    const int k_hi = (int)floorf(T.kc + T.t3);
                    const bool livek = actp && k_hi >= k0 && k_lo <= k_top;
                    const int j_a = livek ? max(0, k0 - k_lo) : 0;
                    const int j_b = livek ? min(k_hi, k_top) - k_lo : -1;
                    if (__reduce_max_sync(FULL, j_b + 1) == 0) continue;
                    const unsigned same = __match_any_sync(FULL, livek ? k_lo : INT_MIN + lane) & ~(1u << lane);
                    const bool ok = __all_sync(FULL, same == 0u) && !force_serial;
                    float f1[FKR];                       // weight of column k_lo + j
                    {
                        float xi = (float)k_lo - T.kc, g0 = sf_G<MODEL>(T, xi);
#pragma unroll
                        for (int j = 0; j < FKR; ++j) {
                            xi += 1.0f;
                            const float g1 = sf_G<MODEL>(T, xi);
                            f1[j] = g1 - g0;
                            g0 = g1;
                        }
                    }
                    // z-independent parts of the axial rectangle and of the amplitude
                    const float n2ab = fmaf(a, a, b * b);
                    const float Rg = ARC ? v.Rv * rsqrt_nr(n2ab) : v.Rv * inv_a;
                    const float half = fabsf(Rg * v.hcz);
                    const float m = fmaxf(fabsf(p + v.ep0), fabsf(q + v.eq0));
                    const float m2 = m * m;
                    int ca_k = (int)smem_addr(tile) + 4 * (livek ? k_lo - k0 : 0);            // row 0, column k_lo
                    asm volatile("" : "+r"(ca_k));          // keep it in a register: ptxas otherwise rebuilds it per round
                    const float *xcol = slab + ip;
                    const int n_serial = ok ? 1 : 32;       // !ok: one lane at a time (never expected)
                    for (int r = 0; r < nrows; ++r) {
                        const int izr = zs_lo + r + sh;
                        const bool act = livek && izr >= 0 && izr < nz;
                        const int iz = act ? izr : 0;
                        const float x = __ldg(xcol + (unsigned)(iz * zstride));
                        const float c = fmaf((float)iz, v_cz, cpq);
                        SfAxial A;
                        A.lc = fmaf(Rg, c, v.lv0); A.tlo = -half; A.thi = half;
                        const int l_lo = max(l0, (int)floorf(A.lc - half));
                        const int l_hi = min(l_top, (int)floorf(A.lc + half));
                        const bool live = act && l_lo <= l_hi;
                        if (!__any_sync(FULL, live)) continue;
                        const int L = live ? l_hi - l_lo + 1 : 0;
                        const int Lmax = __reduce_max_sync(FULL, L);
                        const float n2 = fmaf(c, c, n2ab);
                        const float ax = x * n2 * rsqrt_approx(n2 * m2);
                        float f2[2 * FLM];
                        if (Lmax > FLM) sf_F2_run<2 * FLM>(A, (float)l_lo, f2);
                        else            sf_F2_run<FLM>(A, (float)l_lo, f2);
                        const uint32_t ca = (uint32_t)(ca_k + 4 * FTK * (live ? l_lo - l0 : 0));
                        const int Kall = __reduce_max_sync(FULL, live ? j_b + 1 : 0);
                        for (int ser = 0; ser < n_serial; ++ser) {
                            const bool mine = live && (ok || lane == ser);
                            if (Lmax <= 3) {
#pragma unroll
                                for (int jk = 0; jk < FKR; ++jk) {
                                    if (jk >= Kall) break;               // warp-uniform
                                    if (mine && jk >= j_a && jk <= j_b) fp_round_rows3(ca + 4u * jk, f1[jk] * ax, f2);
                                    __syncwarp();
                                }
                            } else if (Lmax <= FLM) {
#pragma unroll
                                for (int jk = 0; jk < FKR; ++jk) {
                                    if (jk >= Kall) break;               // warp-uniform
                                    if (mine && jk >= j_a && jk <= j_b)
                                        fp_round_rows<true, false>(ca + 4u * jk, f1[jk] * ax, f2, L);
                                    __syncwarp();
                                }
                            } else {
#pragma unroll
                                for (int jk = 0; jk < FKR; ++jk) {
                                    if (jk >= Kall) break;               // warp-uniform
                                    if (mine && jk >= j_a && jk <= j_b)
                                        fp_round_rows<true, true>(ca + 4u * jk, f1[jk] * ax, f2, L);
                                    __syncwarp();
                                }
                            }
                            // footprints beyond the host's bound (never expected): columns >= FKR and rows >= 2 FLM
                            // with weights evaluated on the fly
                            if (Kall > FKR || Lmax > 2 * FLM) {
                                for (int lb = 0; lb < Lmax; lb += 2 * FLM) {
                                    float g2[2 * FLM];
                                    sf_F2_run<2 * FLM>(A, (float)(l_lo + lb), g2);
                                    SfTrans T2;                  // recomputed here so that T need not stay live
                                    sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T2, p, q);
                                    for (int jk = (lb == 0 ? FKR : 0); jk < Kall; ++jk) {
                                        if (mine && jk >= j_a && jk <= j_b) {
                                            const float xi = (float)(k_lo + jk) - T2.kc;
                                            const float w = (sf_G<MODEL>(T2, xi + 1.0f) - sf_G<MODEL>(T2, xi)) * ax;
                                            fp_round_rows<false, true>(ca + 4u * jk + 4u * FTK * lb, w, g2, L - lb);
                                        }
                                        __syncwarp();
                                    }
                                }
                            }
                        }
                    }
                }
            }
            continue;
        }

        for (int col = 0; col < sp; ++col) {
            const int nprc = (npr - col + sp - 1) / sp;
            if (nprc <= 0) break;
            // flattened (row, pi) sweep, 32 consecutive entries per pass.  Rows are visited in the order
            // 0, H, 1, H+1, ... so that the (at most two) voxels of equal p that can share a pass lie H
            // rows apart and touch different detector rows; the pass verifies this before its rounds.
            const bool multi = DIM == 3 && nrows >= 6;
            const int rs = multi ? max(nprc, 16) : max(nprc, 32);
            const int total = DIM == 3 ? nrows * rs : nprc;
            const int H = (nrows + 1) >> 1;
            int row = 0, pi = lane;                      // rs >= 16: a step of 32 wraps at most twice
            if (pi >= rs) { pi -= rs; ++row; }
            if (pi >= rs) { pi -= rs; ++row; }
            for (int f0 = 0; f0 < total; f0 += 32) {
                const int ipr = p_lo + col + sp * pi;
                const int sh = DIM == 3 ? __float2int_rn(sigma * (float)(ipr - p_lo)) : 0;
                const int zrow = multi ? ((row & 1) ? H + (row >> 1) : (row >> 1)) : row;
                const int izr = DIM == 3 ? zs_lo + zrow + sh : 0;
                const bool act = pi < nprc && row < nrows && izr >= 0 && izr < nz;
                const int ip = act ? ipr : p_lo, iz = act ? izr : 0;
                // advance to the next pass
                pi += 32;
                if (pi >= rs) { pi -= rs; ++row; }
                if (pi >= rs) { pi -= rs; ++row; }
                const float p = (float)ip, z = (float)iz;
                float xv[NB];
                const float *xp = slab + (unsigned)(iz * zstride + ip);      // < 2^31 voxels per image
#pragma unroll
                for (int bb = 0; bb < NB; ++bb) xv[bb] = __ldg(xp + bb * vol_bstride);
                const float a = fmaf(p, v_ap, fmaf(z, v_az, aq0)), b = fmaf(p, v_bp, fmaf(z, v_bz, bq0));
                const float c = DIM == 3 ? fmaf(p, v_cp, fmaf(z, v_cz, cq0)) : 0.0f;
                const float inv_a = rcp_nr(a);
                // rows first: a pass whose voxels all miss the band in l (the extreme rows of the sheared
                // region) is dropped before the costlier transaxial part
                SfAxial A;
                int l_lo = 0, l_hi = 0;
                if (DIM == 3) {
                    sf_axial<ARC, MODEL>(v, a, b, c, inv_a, A, p, q);
                    l_lo = max(l0, (int)floorf(A.lc + A.tlo));
                    l_hi = min(l_top, (int)floorf(A.lc + A.thi));
                    if (!__any_sync(FULL, act && l_lo <= l_hi)) continue;
                }
                SfTrans T;
                sf_transaxial<ARC, MODEL>(v, a, b, inv_a, T, p, q);
                // unclipped column range: rounds are aligned on it, columns off the tile are skipped
                const int k_lo = (int)floorf(T.kc + T.t0);
                const int k_hi = (int)floorf(T.kc + T.t3);
                const bool live = act && k_hi >= k0 && k_lo <= k_top && l_lo <= l_hi;
                // rounds j_a .. j_b of this lane update columns k_lo + j that lie on the tile
                const int j_a = live ? max(0, k0 - k_lo) : 0;
                const int j_b = live ? min(k_hi, k_top) - k_lo : -1;
                const int L = live ? l_hi - l_lo + 1 : 0;
                const int Kmax = __reduce_max_sync(FULL, j_b + 1);
                if (Kmax == 0) continue;
                const int Lmax = DIM == 3 ? __reduce_max_sync(FULL, L) : 1;
                // conflict freedom of a round: live lanes have pairwise different k_lo, or (one partner at
                // most) touch disjoint rows.  A lane touches rows l_lo .. max(l_hi, l_lo + FLM - 1).
                const unsigned same = __match_any_sync(FULL, live ? k_lo : INT_MIN + lane) & ~(1u << lane);
                bool fine = true;
                if (DIM == 3) {
                    const int partner = same ? __ffs(same) - 1 : lane;
                    const int my_hi = max(l_hi, l_lo + FLM - 1);
                    const int o_lo = __shfl_sync(FULL, l_lo, partner), o_hi = __shfl_sync(FULL, my_hi, partner);
                    fine = same == 0u || (__popc(same) == 1 && (o_lo > my_hi || o_hi < l_lo));
                } else {
                    fine = same == 0u;
                }
                const bool ok = __all_sync(FULL, fine) && !force_serial;
                const float amp = sf_amplitude(v, a, b, c, p, q);
#pragma unroll
                for (int bb = 0; bb < NB; ++bb) xv[bb] *= amp;
                float *base = tile + (live ? (DIM == 3 ? (l_lo - l0) * FTK : 0) + (k_lo - k0) : 0);
                const float xi0 = (float)(k_lo + j_a) - T.kc;
                const int n_serial = ok ? 1 : 32;       // !ok: one lane at a time (never expected)
                for (int ser = 0; ser < n_serial; ++ser) {
                    const int jb = (ok || lane == ser) ? j_b : -1;
                    for (int lb = 0; lb < Lmax; lb += 2 * FLM) {
                        float f2[2 * FLM];
                        if (DIM == 3) {
                            if (Lmax > lb + FLM) sf_F2_run<2 * FLM, MODEL>(A, (float)(l_lo + lb), f2);
                            else                 sf_F2_run<FLM, MODEL>(A, (float)(l_lo + lb), f2);
                        }
                        float xi = xi0, g0 = sf_G<MODEL>(T, xi0);
                        uint32_t ca = smem_addr(base + lb * FTK);      // this lane's cell of round 0
                        const int nrow = L - lb;
#define CTSF_ROUNDS(...)                                             \
                        for (int jk = 0; jk < Kmax; ++jk, ca += 4) {   \
                            if (jk >= j_a && jk <= jb) {               \
                                xi += 1.0f;                            \
                                const float g1 = sf_G<MODEL>(T, xi);          \
                                const float f1 = g1 - g0;              \
                                g0 = g1;                               \
                                __VA_ARGS__                            \
                            }                                          \
                            __syncwarp();                              \
                        }
                        if (DIM == 3) {
                            if (lb == 0 && Lmax <= FLM) {
                                CTSF_ROUNDS(fp_round_rows<true, false>(ca, f1 * xv[0], f2, nrow);)
                            } else if (lb == 0) {
                                CTSF_ROUNDS(fp_round_rows<true, true>(ca, f1 * xv[0], f2, nrow);)
                            } else {
                                CTSF_ROUNDS(fp_round_rows<false, true>(ca, f1 * xv[0], f2, nrow);)
                            }
                        } else {
                            CTSF_ROUNDS(_Pragma("unroll") for (int bb = 0; bb < NB; ++bb)
                                            sts_f32(ca + bb * FTK * 4, fmaf(f1, xv[bb], lds_f32(ca + bb * FTK * 4)));)
                        }
#undef CTSF_ROUNDS
#undef CTSF_ROUNDS
                    }
                }
            }
        }
    }
    __syncwarp();
    // every cell of the tile is stored exactly once
    if (DIM == 3) {
        float *o = proj + (size_t)b0 * proj_bstride + ((size_t)jview * pr.nv + l0) * pr.nu + k0;
        for (int l = 0; l < tlh; ++l)
            for (int k = lane; k < tkw; k += 32) o[(size_t)l * pr.nu + k] = tile[l * FTK + k];
    } else if (QS) {
        __syncthreads();                             // all FPW partial tiles of this item are complete
#pragma unroll
        for (int bb = 0; bb < NB; ++bb) {
            float *o = proj + (size_t)(b0 + bb) * proj_bstride + (size_t)jview * pr.nu + k0;
            for (int k = threadIdx.x; k < tkw; k += 32 * FPW) {
                float sum = 0.0f;
#pragma unroll
                for (int w = 0; w < FPW; ++w) sum += smem[w * (ROWS * FTK) + bb * FTK + k];     // fixed order
                o[k] = sum;
            }
        }
    } else {
#pragma unroll
        for (int bb = 0; bb < NB; ++bb) {
            float *o = proj + (size_t)(b0 + bb) * proj_bstride + (size_t)jview * pr.nu + k0;
            for (int k = lane; k < tkw; k += 32) o[k] = tile[bb * FTK + k];
        }
    }
}

template <int DIM, int ARC, int NB>
void launch_fp(const ct_geom *g, const float *d_vol, const float *d_volT, float *d_proj, int b0, int groups,
               int vb, int vs, int vc, cudaStream_t st)
{
    const SfProblem &pr = g->prob;
    const int tiles_k = (pr.nu + FTK - 1) / FTK, bands_l = DIM == 3 ? (pr.nv + FTL - 1) / FTL : 1;
    const size_t vbs = (size_t)pr.nx * pr.ny * pr.nz, pbs = (size_t)vc * pr.nv * pr.nu;
    constexpr int ROWS = DIM == 3 ? FTL + FLM : NB;
    const int wpc_general = FP_WPC;
    size_t smem = (size_t)wpc_general * ROWS * FTK * sizeof(float);
    // testing aids (CtsfDebug): fp_nohoist never uses the untilted fast path; fp_forcehoist uses it for every
    // untilted 3-D geometry, also when footprints exceed its register windows (exercises its overflow branch)
    const bool hoist = DIM == 3 && !g_ctsf_debug.fp_nohoist &&
                       (g->fp_hoist_ok || (g->all_untilted && g_ctsf_debug.fp_forcehoist)) && g->model != 2;
    // SF-TT (model 2) differs from SF-TR in the axial factor only: 2-D geometries run the SF-TR instantiation
    auto kern = (g->model == 2 && DIM == 3) ? fp_band_kernel<DIM, ARC, NB, 0, DIM == 3 ? 2 : 0>
        : g->model == 1
        ? (hoist ? fp_band_kernel<DIM, ARC, NB, DIM == 3 ? 1 : 0, 1> : fp_band_kernel<DIM, ARC, NB, 0, 1>)
        : (hoist ? fp_band_kernel<DIM, ARC, NB, DIM == 3 ? 1 : 0, 0> : fp_band_kernel<DIM, ARC, NB, 0, 0>);
    const long n_items = (long)tiles_k * bands_l * ((vc + FVG - 1) / FVG) * FVG;
    // 2-D problems with fewer warp items than the machine holds (148 SMs x 24 warps): split every item's slabs over
    // the warps of a CTA (config 1: 768 items -> 768 CTAs instead of 96)
    const bool qsplit = DIM == 2 && n_items * groups < 148L * FPW * FMINB;
    if (qsplit) kern = g->model == 1 ? fp_band_kernel<DIM, ARC, NB, 0, 1, DIM == 2 ? 1 : 0>
                                     : fp_band_kernel<DIM, ARC, NB, 0, 0, DIM == 2 ? 1 : 0>;
    const int wpc = qsplit ? FPW : wpc_general;
    smem = (size_t)wpc * ROWS * FTK * sizeof(float);
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    // testing aid: fp_pad = <voxels> widens the swept voxel region; the result must not change beyond
    // summation order (tests/test_gpu_fullsize.py uses it to prove that the tight region misses nothing)
    const float region_pad = g_ctsf_debug.fp_pad;
    dim3 grid((unsigned)(qsplit ? n_items : (n_items + wpc - 1) / wpc), groups, 1);
    kern<<<grid, 32 * wpc, smem, st>>>(pr, g->d_fp, d_vol + (size_t)b0 * vbs,
                                       d_volT ? d_volT + (size_t)b0 * vbs : nullptr,
                                       d_proj + (size_t)b0 * pbs, vb, vs, tiles_k, bands_l, (int)n_items, vc, vbs, pbs, region_pad,
                                       g_ctsf_debug.fp_serial ? 1 : 0);   // testing aid: take the lane-serial branch
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

long ctsf_fp_cta_count(const ct_geom *g, int view_count)
{
    const SfProblem &pr = g->prob;
    const long tiles = (long)((pr.nu + FTK - 1) / FTK) * (pr.dim == 3 ? (pr.nv + FTL - 1) / FTL : 1);
    return tiles * ((view_count + FVG - 1) / FVG) * FVG / FPW;
}

bool ctsf_fp_needs_transpose(const ct_geom *g, int view_begin, int view_stride, int view_count)
{
    for (int j = 0; j < view_count; ++j)
        if (g->h_fp[view_begin + (size_t)j * view_stride].swap_xy != 0) return true;
    return false;
}

int ctsf_fp_transpose(const ct_geom *g, const float *d_vol, float *d_volT, int batch, void *stream)
{
    const SfProblem &pr = g->prob;
    int launches = 0;
    dim3 grid((pr.nx + 31) / 32, (pr.ny + 31) / 32, 1), block(32, 8);
    const long slices = (long)batch * pr.nz;                 // one launch per chunk of <= 65535 slices
    for (long s0 = 0; s0 < slices; s0 += 65535) {
        grid.z = (unsigned)((slices - s0) < 65535 ? (slices - s0) : 65535);
        transpose_xy_kernel<<<grid, block, 0, (cudaStream_t)stream>>>(d_vol + (size_t)s0 * pr.nx * pr.ny,
                                                                      d_volT + (size_t)s0 * pr.nx * pr.ny, pr.nx, pr.ny);
        ++launches;
    }
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}

int ctsf_launch_fp(const ct_geom *g, const float *d_vol, float *d_proj, int batch,
                   int view_begin, int view_stride, int view_count, void *stream, const float *d_volT_in)
{
    cudaStream_t st = (cudaStream_t)stream;
    const SfProblem &pr = g->prob;
    int launches = 0;
    const float *d_volT = d_volT_in;
    float *scratch = nullptr;
    if (!d_volT && ctsf_fp_needs_transpose(g, view_begin, view_stride, view_count)) {
        const size_t n = (size_t)batch * pr.nx * pr.ny * pr.nz;
        scratch = (float *)ctsf_scratch_acquire(g, n * sizeof(float), stream);
        if (!scratch) return -1;
        const int nt = ctsf_fp_transpose(g, d_vol, scratch, batch, stream);
        if (nt < 0) { ctsf_scratch_release(g, scratch, stream); return -1; }
        launches += nt;
        d_volT = scratch;
    }
    const int arc = pr.det_type;
    if (pr.dim == 2) launches += arc ? launch_fp_batches<2, 1>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st)
                                     : launch_fp_batches<2, 0>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st);
    else             launches += arc ? launch_fp_batches<3, 1>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st)
                                     : launch_fp_batches<3, 0>(g, d_vol, d_volT, d_proj, batch, view_begin, view_stride, view_count, st);
    if (scratch) ctsf_scratch_release(g, scratch, stream);
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}
