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

constexpr int FLT_THREADS = 256;

template <int ARC>
__global__ void __launch_bounds__(FLT_THREADS)
fbp_filter_kernel(SfProblem pr, const SfView *__restrict__ views, const float *__restrict__ proj,
                  float *__restrict__ out, int view_begin, int view_stride, int view_count, double du, double dv)
{
    extern __shared__ double sm[];
    double *pw = sm, *h = sm + pr.nu;
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
        h[k] = hn;
    }
    __syncthreads();
    float *q = out + (size_t)row * pr.nu;
    for (int k = tid; k < pr.nu; k += FLT_THREADS) {
        double acc = pw[k] * h[0];
        for (int m = (k + 1) & 1; m < pr.nu; m += 2) acc = fma(pw[m], h[abs(k - m)], acc);   // |k - m| odd only
        q[k] = (float)(du * acc);
    }
}

}  // namespace

int ctsf_launch_filter(const ct_geom *g, const float *d_proj, float *d_out, int batch,
                       int view_begin, int view_stride, int view_count, void *stream)
{
    const SfProblem &pr = g->prob;
    const long rows = (long)batch * view_count * pr.nv;
    if (rows == 0) return 0;
    const size_t smem = 2 * sizeof(double) * (size_t)pr.nu;
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
            g->du, g->dv);
        ++launches;
    }
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}
