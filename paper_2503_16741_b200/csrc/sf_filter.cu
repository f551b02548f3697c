// sf_filter.cu -- recon mode, step 1: cosine pre-weight + discrete ramp filter along the detector channels
// ("a discrete ramp filter"; reading R24).  The paper gives no formula; the reading is the
// textbook band-limited ramp sampled at the channel pitch, in the spatial domain:
//     q[k] = du * sum_m p'[m] h[k - m],   h[0] = 1/(4 du^2),  h[even] = 0,
//     h[odd n] = -1/(pi n du)^2 (flat)   or   -1/(pi R sin(n du / R))^2 (arc, equi-angular),
//     p' = p * R/sqrt(R^2 + s^2 + t^2) (flat; (s, t) from the foot of the source normal)
//        = p * cos(gamma) * R/sqrt(R^2 + t^2) (arc; gamma = u_k / R).
// One CTA per detector row.  The sum alternates between one large positive and many negative terms and
// cancels to a small remainder, so p', the table h and the accumulation are kept in fp64 (B200 has a full-rate
// fp64 pipe; the kernel is shared-memory bound at ~nu^2/2 fp64 loads per row); only q is rounded to fp32.
#include <cuda_runtime.h>

#include "ctsf_internal.h"

namespace {

constexpr int FLT_THREADS = 128;
__device__ __forceinline__ int HP(int n) { return n + (n >> 4); }   // padded table index
constexpr int FJ = 8;              // outputs per thread (register tile of the Toeplitz product)

template <int ARC>
__global__ void __launch_bounds__(FLT_THREADS)
fbp_filter_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ proj,
                  float *__restrict__ out, int view_begin, int view_stride, int view_count, double du, double dv, double scale)
{
    extern __shared__ double sm[];
    double *pw = sm, *h = sm + pr.nu;             // h is stored padded: entry n at HP(n) = n + n/16
    const int tid = threadIdx.x;
    const long row = (long)blockIdx.x;                   // (batch * view_count + j) * nv + l
    const int l = (int)(row % pr.nv);
    const int j = (int)((row / pr.nv) % view_count);
    const SfView &v = views[view_begin + (size_t)j * view_stride];
    const double R = (double)v.Ru * du;
    const double t = pr.dim == 3 ? ((double)l + 0.5 - (double)v.lv0) * dv : 0.0;
    const float *p = proj + (size_t)row * pr.nu;
    const double PI = 3.14159265358979323846;
    for (int k = tid; k < pr.nu; k += FLT_THREADS) {
        const double uk = ((double)k + 0.5 - (double)v.ku0) * du;              // flat: from the normal's foot; arc: arc length
        double w;
        if (ARC == 0) w = R / sqrt(R * R + uk * uk + t * t);
        else          w = cos(uk / R) * R / sqrt(R * R + t * t);
        pw[k] = (double)p[k] * w;
        double hn;
        if (k == 0) hn = 1.0 / (4.0 * du * du);
        else if ((k & 1) == 0) hn = 0.0;
        else if (ARC == 0) { const double x = PI * k * du; hn = -1.0 / (x * x); }
        else { const double x = PI * R * sin(k * du / R); hn = -1.0 / (x * x); }
        h[k + (k >> 4)] = hn;
    }
    __syncthreads();
    // Each thread owns FJ outputs of one parity, k = kb + 2 j.  Only taps of the other parity contribute
    // (h[even] = 0) besides the centre tap; for those m = m0 + 2 i the table index k - m drops by 2 per step, so
    // the FJ table values in use form a sliding window: one new p'[m] and one new h per step feed FJ fp64 FMAs.
    // The window lives in a register ring whose rotation is resolved at compile time by unrolling FJ steps.
    float *q = out + (size_t)row * pr.nu;
    const int n_groups = (pr.nu + 2 * FJ - 1) / (2 * FJ);              // groups of FJ same-parity outputs
    // lane -> (parity, group): a half-warp holds 16 consecutive groups of one parity, whose table indices differ
    // by 2 FJ = 16 -- with the table padded by one entry per 16 they fall into 16 different 8-byte banks
    const int n_slots = ((n_groups + 15) / 16) * 32;
    for (int gi = tid; gi < n_slots; gi += FLT_THREADS) {
        const int par = (gi >> 4) & 1, grp = (gi >> 5) * 16 + (gi & 15);
        if (grp >= n_groups) continue;
        const int kb = grp * (2 * FJ) + par;                          // outputs kb, kb + 2, ...
        const int m0 = 1 - par;                                        // taps m0, m0 + 2, ...
        const int n_taps = (pr.nu - m0 + 1) / 2;
        double acc[FJ], w[FJ];
#pragma unroll
        for (int j = 0; j < FJ; ++j) {
            acc[j] = 0.0;
            const int n = kb + 2 * j - m0;                             // table index of output j at step 0
            w[j] = h[HP(min(abs(n), pr.nu - 1))];
        }
        // ring: at step i the weight of output j sits in w[(j - i) mod FJ]
        int i = 0;
        for (; i + FJ <= n_taps; i += FJ) {
#pragma unroll
            for (int ii = 0; ii < FJ; ++ii) {
                const double pm = pw[m0 + 2 * (i + ii)];
#pragma unroll
                for (int j = 0; j < FJ; ++j) acc[j] = fma(pm, w[(j - ii + FJ) % FJ], acc[j]);
                // next step: output 0 needs h[|kb - m0 - 2 (i + ii + 1)|]; it replaces the slot output FJ-1 used
                const int n = kb - m0 - 2 * (i + ii + 1);
                w[(FJ - 1 - ii + FJ) % FJ] = h[HP(min(abs(n), pr.nu - 1))];
            }
        }
        for (; i < n_taps; ++i) {                                      // remainder: plain lookups
            const double pm = pw[m0 + 2 * i];
#pragma unroll
            for (int j = 0; j < FJ; ++j) acc[j] = fma(pm, h[HP(min(abs(kb + 2 * j - m0 - 2 * i), pr.nu - 1))], acc[j]);
        }
#pragma unroll
        for (int j = 0; j < FJ; ++j) {
            const int k = kb + 2 * j;
            if (k < pr.nu) q[k] = (float)(scale * du * fma(pw[k], h[0], acc[j]));      // HP(0) = 0
        }
    }
}

}  // namespace

int ctsf_launch_filter(const ct_geom *g, const float *d_proj, float *d_out, int batch,
                       int view_begin, int view_stride, int view_count, void *stream, double scale)
{
    const SfProblem &pr = g->prob;
    const long rows = (long)batch * view_count * pr.nv;
    if (rows == 0) return 0;
    const size_t smem = sizeof(double) * (2 * (size_t)pr.nu + pr.nu / 16 + 2);
    if (smem > 200 * 1024) return -1;
    auto kern = pr.det_type ? fbp_filter_kernel<1> : fbp_filter_kernel<0>;
    cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    int launches = 0;
    // rows in chunks of <= 2^31-1 blocks along x is ample; keep y = 1
    const long max_x = 2147483647L;
    for (long r0 = 0; r0 < rows; r0 += max_x) {
        const long n = rows - r0 < max_x ? rows - r0 : max_x;
        // a chunk starts at a whole number of (batch, view) rows only when r0 == 0; larger problems do not occur
        kern<<<dim3((unsigned)n, 1, 1), FLT_THREADS, smem, (cudaStream_t)stream>>>(
            pr, g->d_bp, d_proj + (size_t)r0 * pr.nu, d_out + (size_t)r0 * pr.nu, view_begin, view_stride, view_count,
            g->du, g->dv, scale);
        ++launches;
    }
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}
