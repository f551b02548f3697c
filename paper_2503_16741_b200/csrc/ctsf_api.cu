// ctsf_api.cu -- the C ABI of libctsf (include/ctsf.h): argument checks, geometry lifetime,
// kernel scheduling ("C++ projector function manages kernel scheduling").
#include <cuda_runtime.h>

#include <cmath>
#include <mutex>
#include <new>
#include <string>

#include "ctsf_internal.h"

namespace {

bool finite_pos(double x) { return std::isfinite(x) && x > 0.0; }

constexpr int MAX_DEV = 64;
cudaMemPool_t g_pool[MAX_DEV];
std::mutex g_pool_mu;

cudaMemPool_t pool_of_current_device()
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) { cudaGetLastError(); return nullptr; }
    std::lock_guard<std::mutex> lock(g_pool_mu);
    if (!g_pool[dev]) {
        cudaMemPoolProps props = {};
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        cudaMemPool_t pool = nullptr;
        if (cudaMemPoolCreate(&pool, &props) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        unsigned long long keep = ~0ull;
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        g_pool[dev] = pool;
    }
    return g_pool[dev];
}

// a = input, b = output.  With an empty view subset (vc == 0) the projection-side buffer has no elements and
// may be NULL: `proj_is_a` tells which side that is.
ct_status_t check_call(const ct_geom *g, const void *a, const void *b, int batch, int vb, int vs, int vc,
                       bool proj_is_a = false, bool proj_is_b = false)
{
    if (!g || batch < 1) return CT_ERR_INVALID_ARG;
    if (vc == 0 && vs >= 1 && vb >= 0) {
        if ((!a && !proj_is_a) || (!b && !proj_is_b)) return CT_ERR_INVALID_ARG;
        return CT_OK;
    }
    if (!a || !b) return CT_ERR_INVALID_ARG;
    if (vc < 0 || vs < 1 || vb < 0) return CT_ERR_INVALID_ARG;
    if (vc > 0 && (long)vb + (long)(vc - 1) * vs >= g->prob.n_views) return CT_ERR_INVALID_ARG;
    if (((uintptr_t)a | (uintptr_t)b) & 3u) return CT_ERR_INVALID_ARG;     // fp32 elements; 16-byte alignment of the
    return CT_OK;                                                            // projections only enables the TMA path
}

ct_status_t zero_volume(const ct_geom *g, float *d_vol, int batch, ct_stream_t stream)
{
    const size_t n = (size_t)batch * g->prob.nx * g->prob.ny * g->prob.nz;
    if (cudaMemsetAsync(d_vol, 0, n * sizeof(float), (cudaStream_t)stream) != cudaSuccess) { cudaGetLastError(); return CT_ERR_CUDA; }
    g->last_launches.store(0);
    return CT_OK;
}

}  // namespace

void *ctsf_alloc_async(size_t bytes, void *stream)
{
    void *p = nullptr;
    cudaMemPool_t pool = pool_of_current_device();
    cudaError_t e = pool ? cudaMallocFromPoolAsync(&p, bytes, pool, (cudaStream_t)stream)
                         : cudaMallocAsync(&p, bytes, (cudaStream_t)stream);
    if (e != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}

void ctsf_free_async(void *p, void *stream)
{
    if (p) cudaFreeAsync(p, (cudaStream_t)stream);
}

CtsfDebug g_ctsf_debug;

void *ctsf_scratch_acquire(const ct_geom *g, size_t bytes, void *stream)
{
    std::lock_guard<std::mutex> lock(g->scratch_mu);
    // A slot between acquire and release belongs to the call that took it: host threads working on the same geometry
    // never see it as free (its event says nothing yet -- never recorded, or recorded behind an EARLIER use).
    // An idle slot is free for this call if its last use was on the same stream (stream order) or has completed.
    ct_geom::Scratch *small = nullptr;
    for (auto &sc : g->scratch) {
        if (sc.busy || !sc.ptr) continue;
        const bool idle = sc.stream == stream || (sc.done && cudaEventQuery((cudaEvent_t)sc.done) == cudaSuccess);
        if (!idle) continue;
        if (sc.bytes >= bytes) { sc.stream = stream; sc.busy = true; cudaGetLastError(); return sc.ptr; }
        if (!small) small = &sc;
    }
    cudaGetLastError();                     // cudaEventQuery's cudaErrorNotReady is not an error here
    void *ptr = nullptr;
    if (small) {
        // an idle slot that is too small (a larger batch than before) is replaced, not kept beside the new one: the
        // geometry's scratch does not grow with every batch size it has seen.  cudaFree waits for pending work on it.
        cudaFree(small->ptr);
        small->ptr = nullptr; small->bytes = 0;
        if (cudaMalloc(&ptr, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
        small->ptr = ptr; small->bytes = bytes; small->stream = stream; small->busy = true;
        return ptr;
    }
    ct_geom::Scratch sc;
    if (cudaMalloc(&ptr, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    cudaEvent_t ev = nullptr;
    if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); cudaFree(ptr); return nullptr; }
    sc.ptr = ptr; sc.bytes = bytes; sc.stream = stream; sc.done = ev; sc.busy = true;
    g->scratch.push_back(sc);
    return ptr;
}

void ctsf_scratch_release(const ct_geom *g, void *ptr, void *stream)
{
    std::lock_guard<std::mutex> lock(g->scratch_mu);
    for (auto &sc : g->scratch)
        if (sc.ptr == ptr) {
            cudaEventRecord((cudaEvent_t)sc.done, (cudaStream_t)stream);     // before the slot can be seen as idle
            sc.busy = false;
            return;
        }
}

extern "C" {

// Testing aids, deliberately NOT declared in include/ctsf.h.  ctsf_debug_set sets one switch of CtsfDebug by name (see
// ctsf_internal.h; "reset" restores every default) and returns 0, or -1 for an unknown name.  ctsf_debug_get returns
// the switch's current value, NaN for an unknown name: bench.py records with it that it timed the default paths.
// Process-wide and not thread-safe against running calls: for tests only.
static int debug_field(CtsfDebug &d, const std::string &n, float **f, int **i)
{
    *f = nullptr; *i = nullptr;
    if (n == "fp_pad") *f = &d.fp_pad;
    else if (n == "tt_pad") *f = &d.tt_pad;
    else if (n == "fp_nohoist") *i = &d.fp_nohoist;
    else if (n == "fp_forcehoist") *i = &d.fp_forcehoist;
    else if (n == "fp_serial") *i = &d.fp_serial;
    else if (n == "bp_nohoist") *i = &d.bp_nohoist;
    else if (n == "bp_forcehoist") *i = &d.bp_forcehoist;
    else if (n == "bp_tma") *i = &d.bp_tma;
    else if (n == "bp_chunk") *i = &d.bp_chunk;
    else if (n == "bp_scalar") *i = &d.bp_scalar;
    else if (n == "bp_poison") *i = &d.bp_poison;
    else if (n == "host_fp_chunks") *i = &d.host_fp_chunks;
    else if (n == "host_bp_chunks") *i = &d.host_bp_chunks;
    else return -1;
    return 0;
}

CTSF_API int ctsf_debug_set(const char *name, double value)
{
    if (!name) return -1;
    const std::string n(name);
    if (n == "reset") { g_ctsf_debug = CtsfDebug(); return 0; }
    float *f; int *i;
    if (debug_field(g_ctsf_debug, n, &f, &i) != 0) return -1;
    if (f) *f = (float)value; else *i = (int)value;
    return 0;
}

CTSF_API double ctsf_debug_get(const char *name)
{
    float *f; int *i;
    if (!name || debug_field(g_ctsf_debug, std::string(name), &f, &i) != 0) return std::nan("");
    return f ? (double)*f : (double)*i;
}

ct_status_t ct_geom_create(const ct_geom_desc_t *d, ct_geom_t **out)
{
    if (!d || !out) return CT_ERR_INVALID_ARG;
    *out = nullptr;
    if (d->dim != 2 && d->dim != 3) return CT_ERR_INVALID_ARG;
    if (d->nx < 1 || d->ny < 1 || d->nz < 1 || d->nu < 1 || d->nv < 1 || d->n_views < 1) return CT_ERR_INVALID_ARG;
    if (d->dim == 2 && (d->nz != 1 || d->nv != 1)) return CT_ERR_INVALID_ARG;
    if (!finite_pos(d->dx) || !finite_pos(d->dy) || !finite_pos(d->du)) return CT_ERR_INVALID_ARG;
    if (d->dim == 3 && (!finite_pos(d->dz) || !finite_pos(d->dv))) return CT_ERR_INVALID_ARG;
    if (!std::isfinite(d->ox) || !std::isfinite(d->oy) || (d->dim == 3 && !std::isfinite(d->oz))) return CT_ERR_INVALID_ARG;
    if (d->det_type != 0 && d->det_type != 1) return CT_ERR_INVALID_ARG;
    if (d->algo != CT_ALGO_SF && d->algo != CT_ALGO_DD && d->algo != CT_ALGO_SFTT) return CT_ERR_INVALID_ARG;
    if (!d->src || !d->det_center || !d->det_u || (d->dim == 3 && !d->det_v)) return CT_ERR_INVALID_ARG;
    if ((double)d->nx * d->ny * d->nz >= 2147483648.0 || (double)d->nu * d->nv * d->n_views >= 2147483648.0 * 4)
        return CT_ERR_UNSUPPORTED;
    for (long i = 0; i < 3L * d->n_views; ++i)
        if (!std::isfinite(d->src[i]) || !std::isfinite(d->det_center[i]) || !std::isfinite(d->det_u[i]) ||
            (d->det_v && !std::isfinite(d->det_v[i])))
            return CT_ERR_GEOMETRY;

    ct_geom *g = new (std::nothrow) ct_geom;
    if (!g) return CT_ERR_ALLOC;
    g->prob = SfProblem{d->dim, d->det_type, d->nx, d->ny, d->nz, d->nu, d->nv, d->n_views};
    g->du = d->du;
    g->model = d->algo;
    g->dv = d->dim == 3 ? d->dv : 1.0;
    ct_status_t st;
    try {
        st = ctsf_build_views(d, g);
    } catch (const std::bad_alloc &) {
        st = CT_ERR_ALLOC;
    }
    if (st != CT_OK) { delete g; return st; }

    if (cudaGetDevice(&g->device) != cudaSuccess) { cudaGetLastError(); delete g; return CT_ERR_CUDA; }
    const size_t bytes = sizeof(SfView) * (size_t)d->n_views;
    if (cudaMalloc((void **)&g->d_bp, bytes) != cudaSuccess || cudaMalloc((void **)&g->d_fp, bytes) != cudaSuccess) {
        cudaGetLastError();
        if (g->d_bp) cudaFree(g->d_bp);
        delete g;
        return CT_ERR_ALLOC;
    }
    if (cudaMemcpy(g->d_bp, g->h_bp.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(g->d_fp, g->h_fp.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(g->d_bp); cudaFree(g->d_fp);
        delete g;
        return CT_ERR_CUDA;
    }
    *out = g;
    return CT_OK;
}

ct_status_t ct_geom_destroy(ct_geom_t *g)
{
    if (!g) return CT_OK;
    if (g->d_bp) cudaFree(g->d_bp);
    if (g->d_fp) cudaFree(g->d_fp);
    for (auto &sc : g->scratch) {
        if (sc.ptr) cudaFree(sc.ptr);                                 // synchronises with pending work on it
        if (sc.done) cudaEventDestroy((cudaEvent_t)sc.done);
    }
    if (g->host_copy_stream) cudaStreamDestroy((cudaStream_t)g->host_copy_stream);
    for (void *e : g->host_events) if (e) cudaEventDestroy((cudaEvent_t)e);
    const int dev = g->device;
    delete g;
    if (dev >= 0 && dev < MAX_DEV) {
        std::lock_guard<std::mutex> lock(g_pool_mu);
        if (g_pool[dev]) cudaMemPoolTrimTo(g_pool[dev], 0);          // hand the host-buffer operators' cached buffers back
    }
    cudaGetLastError();
    return CT_OK;
}

ct_status_t ct_fp_sf_views(const ct_geom_t *g, const float *d_vol, float *d_proj, int32_t batch,
                           int32_t vb, int32_t vs, int32_t vc, ct_stream_t stream)
{
    ct_status_t st = check_call(g, d_vol, d_proj, batch, vb, vs, vc, false, true);
    if (st != CT_OK) return st;
    if (vc == 0) { g->last_launches.store(0); return CT_OK; }     // nothing to write
    int n = ctsf_launch_fp(g, d_vol, d_proj, batch, vb, vs, vc, stream);
    if (n < 0) return CT_ERR_CUDA;
    g->last_launches.store(n);
    return CT_OK;
}

ct_status_t ct_bp_sf_views(const ct_geom_t *g, const float *d_proj, float *d_vol, int32_t batch,
                           int32_t vb, int32_t vs, int32_t vc, ct_stream_t stream)
{
    ct_status_t st = check_call(g, d_proj, d_vol, batch, vb, vs, vc, true, false);
    if (st != CT_OK) return st;
    if (vc == 0) return zero_volume(g, d_vol, batch, stream);                            // empty sum
    int n = ctsf_launch_bp(g, d_proj, d_vol, batch, vb, vs, vc, stream);
    if (n < 0) return CT_ERR_CUDA;
    g->last_launches.store(n);
    return CT_OK;
}

ct_status_t ct_bp_sf_recon_views(const ct_geom_t *g, const float *d_proj, float *d_vol, int32_t batch,
                                 int32_t vb, int32_t vs, int32_t vc, ct_stream_t stream)
{
    ct_status_t st = check_call(g, d_proj, d_vol, batch, vb, vs, vc, true, false);
    if (st != CT_OK) return st;
    if (vc == 0) return zero_volume(g, d_vol, batch, stream);
    int n = ctsf_launch_bp(g, d_proj, d_vol, batch, vb, vs, vc, stream, 0, 1);
    if (n < 0) return CT_ERR_CUDA;
    g->last_launches.store(n);
    return CT_OK;
}

ct_status_t ct_bp_sf_recon(const ct_geom_t *g, const float *d_proj, float *d_vol, int32_t batch, ct_stream_t stream)
{
    if (!g) return CT_ERR_INVALID_ARG;
    return ct_bp_sf_recon_views(g, d_proj, d_vol, batch, 0, 1, g->prob.n_views, stream);
}

ct_status_t ct_fbp_filter_views(const ct_geom_t *g, const float *d_proj, float *d_out, int32_t batch,
                                int32_t vb, int32_t vs, int32_t vc, ct_stream_t stream)
{
    ct_status_t st = check_call(g, d_proj, d_out, batch, vb, vs, vc, true, true);
    if (st != CT_OK) return st;
    if (vc == 0) { g->last_launches.store(0); return CT_OK; }
    if (d_proj == d_out) return CT_ERR_INVALID_ARG;           // not in place: every output reads the whole row
    int n = ctsf_launch_filter(g, d_proj, d_out, batch, vb, vs, vc, stream);
    if (n < 0) return CT_ERR_CUDA;
    g->last_launches.store(n);
    return CT_OK;
}

ct_status_t ct_fbp_filter(const ct_geom_t *g, const float *d_proj, float *d_out, int32_t batch, ct_stream_t stream)
{
    if (!g) return CT_ERR_INVALID_ARG;
    return ct_fbp_filter_views(g, d_proj, d_out, batch, 0, 1, g->prob.n_views, stream);
}

ct_status_t ct_fbp_sf(const ct_geom_t *g, const float *d_proj, float *d_work, float *d_vol, int32_t batch, ct_stream_t stream)
{
    if (!g) return CT_ERR_INVALID_ARG;
    const int vc = g->prob.n_views;
    ct_status_t st = check_call(g, d_proj, d_work, batch, 0, 1, vc, true, true);
    if (st == CT_OK) st = check_call(g, d_work, d_vol, batch, 0, 1, vc, true, false);
    if (st != CT_OK) return st;
    if (d_proj == d_work) return CT_ERR_INVALID_ARG;
    const double PI = 3.14159265358979323846;
    const int n1 = ctsf_launch_filter(g, d_proj, d_work, batch, 0, 1, vc, stream, PI / (double)vc);     // reading R25
    if (n1 < 0) return CT_ERR_CUDA;
    const int n2 = ctsf_launch_bp(g, d_work, d_vol, batch, 0, 1, vc, stream, 0, 1);
    if (n2 < 0) return CT_ERR_CUDA;
    g->last_launches.store(n1 + n2);
    return CT_OK;
}

ct_status_t ct_fp_sf(const ct_geom_t *g, const float *d_vol, float *d_proj, int32_t batch, ct_stream_t stream)
{
    if (!g) return CT_ERR_INVALID_ARG;
    return ct_fp_sf_views(g, d_vol, d_proj, batch, 0, 1, g->prob.n_views, stream);
}

ct_status_t ct_bp_sf(const ct_geom_t *g, const float *d_proj, float *d_vol, int32_t batch, ct_stream_t stream)
{
    if (!g) return CT_ERR_INVALID_ARG;
    return ct_bp_sf_views(g, d_proj, d_vol, batch, 0, 1, g->prob.n_views, stream);
}

// Host-buffer operators.  3-D, batch 1: the views are cut into chunks and the host<->device copy of
// one chunk overlaps the kernel of its neighbour on a second stream (A: the projections of chunk c
// go home while chunk c+1 is computed; A^T: chunk c+1 arrives while chunk c is backprojected into the
// volume, every chunk after the first adding to it).  Other shapes: copy in, run, copy out.
// The copy stream and the events belong to the geometry (made on first use, reused by every call); the volume
// is transposed once per call, not once per chunk.  One host-buffer call per geometry at a time.
static ct_status_t host_op(const ct_geom_t *g, const float *h_in, float *h_out, int32_t batch, ct_stream_t stream, bool fwd)
{
    if (!g || !h_in || !h_out || batch < 1) return CT_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const SfProblem &pr = g->prob;
    const size_t cells = (size_t)pr.nv * pr.nu;
    const size_t nvol = (size_t)batch * pr.nx * pr.ny * pr.nz, nproj = (size_t)batch * pr.n_views * cells;
    std::lock_guard<std::mutex> host_lock(g->host_mu);
    float *d_vol = (float *)ctsf_alloc_async(nvol * sizeof(float), st);
    if (!d_vol) return CT_ERR_ALLOC;
    float *d_proj = (float *)ctsf_alloc_async(nproj * sizeof(float), st);
    if (!d_proj) { ctsf_free_async(d_vol, st); return CT_ERR_ALLOC; }
    ct_status_t rc = CT_OK;
    int launches = 0;
    constexpr int MAX_CHUNKS = 8;
    int n_chunks = (pr.dim == 3 && batch == 1) ? (pr.n_views >= 64 ? 6 : (pr.n_views >= 8 ? 2 : 1)) : 1;
    if (fwd && n_chunks > 1) {
        // A forward chunk must still fill the machine for several waves: the work per detector tile is very uneven
        // (edge tiles see little of the volume), and a one-wave launch runs at the pace of its slowest CTA (measured
        // at config 2: 45 of 360 views take 17.5 ms, all 360 take 72.8 ms; config 4: 8 chunks 733 ms, 3 chunks 694 ms for A).  >= 18 waves of 148 x 3 CTAs per chunk.
        const long per_chunk = 18L * 148 * 3;
        const long fit = ctsf_fp_cta_count(g, pr.n_views) / per_chunk;
        n_chunks = (int)(fit < 1 ? 1 : (fit > MAX_CHUNKS ? MAX_CHUNKS : fit));
    }
    {   // testing aids: force the number of view chunks of the 3-D batch-1 pipeline
        const int forced = fwd ? g_ctsf_debug.host_fp_chunks : g_ctsf_debug.host_bp_chunks;
        if (forced > 0 && pr.dim == 3 && batch == 1) n_chunks = forced > MAX_CHUNKS ? MAX_CHUNKS : (forced > pr.n_views ? pr.n_views : forced);
    }
    auto ok = [&](cudaError_t e) { if (e != cudaSuccess && rc == CT_OK) rc = CT_ERR_CUDA; return e == cudaSuccess; };
    if (n_chunks == 1) {
        const float *d_in = fwd ? d_vol : d_proj;
        float *d_out = fwd ? d_proj : d_vol;
        const size_t n_in = fwd ? nvol : nproj, n_out = fwd ? nproj : nvol;
        ok(cudaMemcpyAsync((void *)d_in, h_in, n_in * sizeof(float), cudaMemcpyHostToDevice, st));
        if (rc == CT_OK) {
            const int n = fwd ? ctsf_launch_fp(g, d_in, d_out, batch, 0, 1, pr.n_views, stream)
                              : ctsf_launch_bp(g, d_in, d_out, batch, 0, 1, pr.n_views, stream);
            if (n < 0) rc = CT_ERR_CUDA; else launches = n;
        }
        if (rc == CT_OK) ok(cudaMemcpyAsync(h_out, d_out, n_out * sizeof(float), cudaMemcpyDeviceToHost, st));
    } else {
        if (!g->host_copy_stream) {
            cudaStream_t cs = nullptr;
            if (ok(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking))) g->host_copy_stream = cs;
            g->host_events.assign(MAX_CHUNKS + 1, nullptr);
            for (auto &e : g->host_events) {
                cudaEvent_t ev = nullptr;
                if (ok(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming))) e = ev;
            }
        }
        cudaStream_t cs = (cudaStream_t)g->host_copy_stream;
        float *d_volT = nullptr;
        if (rc == CT_OK) {
            cudaEvent_t start = (cudaEvent_t)g->host_events[MAX_CHUNKS];
            // the copy stream may not touch the buffers before `st` has reached this call (allocation order)
            ok(cudaEventRecord(start, st));
            ok(cudaStreamWaitEvent(cs, start, 0));
            if (fwd) {
                ok(cudaMemcpyAsync(d_vol, h_in, nvol * sizeof(float), cudaMemcpyHostToDevice, st));
                if (rc == CT_OK && ctsf_fp_needs_transpose(g, 0, 1, pr.n_views)) {
                    d_volT = (float *)ctsf_scratch_acquire(g, nvol * sizeof(float), stream);
                    const int n = d_volT ? ctsf_fp_transpose(g, d_vol, d_volT, 1, stream) : -1;
                    if (n < 0) rc = d_volT ? CT_ERR_CUDA : CT_ERR_ALLOC; else launches += n;
                }
            }
        }
        for (int c = 0; c < n_chunks && rc == CT_OK; ++c) {
            const int v0 = (int)((long)pr.n_views * c / n_chunks), v1 = (int)((long)pr.n_views * (c + 1) / n_chunks);
            const size_t off = (size_t)v0 * cells, cnt = (size_t)(v1 - v0) * cells;
            cudaEvent_t ev = (cudaEvent_t)g->host_events[c];
            if (fwd) {
                const int n = ctsf_launch_fp(g, d_vol, d_proj + off, 1, v0, 1, v1 - v0, stream, d_volT);
                if (n < 0) { rc = CT_ERR_CUDA; break; }
                launches += n;
                ok(cudaEventRecord(ev, st));
                ok(cudaStreamWaitEvent(cs, ev, 0));
                ok(cudaMemcpyAsync(h_out + off, d_proj + off, cnt * sizeof(float), cudaMemcpyDeviceToHost, cs));
            } else {
                ok(cudaMemcpyAsync(d_proj + off, h_in + off, cnt * sizeof(float), cudaMemcpyHostToDevice, cs));
                ok(cudaEventRecord(ev, cs));
                ok(cudaStreamWaitEvent(st, ev, 0));
                if (rc == CT_OK) {
                    const int n = ctsf_launch_bp(g, d_proj + off, d_vol, 1, v0, 1, v1 - v0, stream, c > 0);
                    if (n < 0) rc = CT_ERR_CUDA; else launches += n;
                }
            }
        }
        if (d_volT) ctsf_scratch_release(g, d_volT, stream);
        if (!fwd && rc == CT_OK) ok(cudaMemcpyAsync(h_out, d_vol, nvol * sizeof(float), cudaMemcpyDeviceToHost, st));
        if (cs && !g->host_events.empty() && g->host_events[MAX_CHUNKS]) {
            // `st` must outlive the copies of `cs` before the buffers are freed on it
            cudaEvent_t start = (cudaEvent_t)g->host_events[MAX_CHUNKS];
            cudaEventRecord(start, cs);
            cudaStreamWaitEvent(st, start, 0);
        }
    }
    cudaFreeAsync(d_vol, st);
    cudaFreeAsync(d_proj, st);
    if (cudaStreamSynchronize(st) != cudaSuccess && rc == CT_OK) rc = CT_ERR_CUDA;
    g->last_launches.store(launches);
    if (rc != CT_OK) cudaGetLastError();
    return rc;
}

ct_status_t ct_fp_sf_host(const ct_geom_t *g, const float *h_vol, float *h_proj, int32_t batch, ct_stream_t stream)
{
    return host_op(g, h_vol, h_proj, batch, stream, true);
}

ct_status_t ct_bp_sf_host(const ct_geom_t *g, const float *h_proj, float *h_vol, int32_t batch, ct_stream_t stream)
{
    return host_op(g, h_proj, h_vol, batch, stream, false);
}

int32_t ct_last_launch_count(const ct_geom_t *g) { return g ? g->last_launches.load() : 0; }

const char *ct_status_string(ct_status_t s)
{
    switch (s) {
        case CT_OK: return "CT_OK";
        case CT_ERR_INVALID_ARG: return "CT_ERR_INVALID_ARG: null pointer, bad size, misaligned buffer or bad view range";
        case CT_ERR_GEOMETRY: return "CT_ERR_GEOMETRY: inconsistent scan geometry";
        case CT_ERR_UNSUPPORTED: return "CT_ERR_UNSUPPORTED: problem too large";
        case CT_ERR_ALLOC: return "CT_ERR_ALLOC: allocation failed";
        case CT_ERR_CUDA: return "CT_ERR_CUDA: CUDA runtime error";
    }
    return "unknown ct_status_t";
}

}  // extern "C"
