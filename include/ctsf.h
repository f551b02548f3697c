/*
 * ctsf.h -- C ABI of the B200-native separable-footprint (SF-TR) projector pair.
 *
 * The operation.  PAPER.md:93-101 (Sec. 2.3): forward projection y = A x (Eq. 1) and its exact
 * adjoint x = A^T y (Eq. 2), a "matched" pair, with the separable-footprint voxel model of
 * PAPER.md:103 ("volume-based voxel model", strict adjoint implemented), for the three scan
 * geometries of PAPER.md:72 / Table 2 (2-D fan, 3-D circular, 3-D non-circular, every parameter
 * view-specific) and flat or curved detectors.  The SF-TR arithmetic itself
 * (trapezoid transaxial x rectangle axial footprint, voxel-centre amplitude, cell-averaged
 * response) is spelled out in DESIGN.md "The method" with the readings R1-R18 it rests on.
 *
 * Conventions (all entry points):
 *  - plain C, no torch types; pointers are HOST or DEVICE as stated per argument;
 *  - volumes are dense fp32 [batch][nz][ny][nx], x fastest; projections are dense fp32
 *    [batch][n_views][nv][nu], u fastest (batch = B*C flattened);
 *  - outputs are OVERWRITTEN (y = A x, x = A^T y), never accumulated into;
 *  - device entry points are asynchronous on `stream`: no host synchronisation, no host<->device
 *    copy of image data.  Scratch memory: ct_fp_sf keeps its one scratch buffer in the geometry (a synchronising
 *    cudaMalloc the first time a geometry, a larger batch or a second concurrent stream needs it, none afterwards);
 *    ct_fp_sf_noalloc never allocates; the *_host entry points take their device buffers from the library's
 *    stream-ordered pool; no other entry point uses scratch memory;
 *  - every function returns a ct_status_t; nothing throws across the boundary;
 *  - inputs are expected to be finite: the kernels multiply cells just outside a footprint by a weight that is
 *    exactly 0 instead of skipping them, so a NaN / Inf in the input may reach outputs up to one footprint width
 *    beyond the cells and voxels it mathematically touches (finite inputs: results as documented, deterministic).
 */
#ifndef CTSF_H
#define CTSF_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define CTSF_API __attribute__((visibility("default")))
#else
#define CTSF_API
#endif

typedef struct ct_geom ct_geom_t;          /* opaque; owns the device copy of the per-view parameters */
typedef void *ct_stream_t;                 /* a cudaStream_t (0 / NULL = the legacy default stream) */

typedef enum {
    CT_OK = 0,
    CT_ERR_INVALID_ARG = 1,   /* null pointer, non-positive size, dim==2 with nz!=1 or nv!=1, batch<1 */
    CT_ERR_GEOMETRY = 2,      /* axes not unit/orthogonal, detector behind the source, arc detector not
                                 centred on the source axis, volume reaching the source plane, a 2-D
                                 geometry with out-of-plane components */
    CT_ERR_UNSUPPORTED = 3,   /* problem too large for 32-bit indexing of one image, or for the fixed scratch of
                                 ct_fp_sf_noalloc */
    CT_ERR_ALLOC = 4,         /* host or device allocation failed */
    CT_ERR_CUDA = 5           /* a CUDA runtime call or kernel launch failed (no usable device, ...) */
} ct_status_t;

/* Scan description (Table 2, in vector form: one source / detector frame per view).
 * World frame in mm.  Voxel (ix,iy,iz) is centred at (ox + (ix-(nx-1)/2) dx, oy + ..., oz + ...).
 * Detector cell (k,l) is centred at detector coordinates u_k = (k-(nu-1)/2) du, v_l = (l-(nv-1)/2) dv,
 * measured from det_center along det_u / det_v (flat), or as arc length du at radius R about the
 * line through the source parallel to det_v (arc: equi-angular channels, equi-spaced rows). */
typedef struct {
    int32_t dim;                 /* 2 or 3.  dim==2: nz==1, nv==1, no axial factor; z components must be 0 */
    int32_t nx, ny, nz;          /* voxels */
    double  dx, dy, dz;          /* voxel pitch, mm (> 0) */
    double  ox, oy, oz;          /* world position of the volume centre ("object centre") */
    int32_t nu, nv;              /* detector channels, rows */
    double  du, dv;              /* cell pitch, mm (> 0) */
    int32_t det_type;            /* 0 flat, 1 arc */
    int32_t n_views;
    const double *src;           /* HOST [n_views][3] source position */
    const double *det_center;    /* HOST [n_views][3] detector point with detector coordinates (0,0) */
    const double *det_u;         /* HOST [n_views][3] unit vector along channels */
    const double *det_v;         /* HOST [n_views][3] unit vector along rows (arc: the cylinder axis);
                                    may be NULL when dim==2 (taken as (0,0,1)) */
    int32_t algo;                /* voxel model of every operator of this geometry:
                                    CT_ALGO_SF = 0 separable footprint, trapezoid x rectangle ("volume-based");
                                    CT_ALGO_DD = 1 distance-driven ("face-based": the voxel's central face
                                    perpendicular to the ray's dominant axis, rectangle x rectangle; R26);
                                    CT_ALGO_SFTT = 2 separable footprint with a TRAPEZOID axial factor (SF-TT, for cone
                                    angles beyond ~10 degrees; R27; identical to SF in 2-D) */
} ct_geom_desc_t;

enum { CT_ALGO_SF = 0, CT_ALGO_DD = 1, CT_ALGO_SFTT = 2 };

/* Validates `desc`, derives the per-view kernel parameters in float64, rounds them to fp32 and
 * uploads them to the current CUDA device.  The host arrays are copied; the caller may free them
 * afterwards.  *out is immutable after creation and may be used from several streams at once.
 * Errors: CT_ERR_INVALID_ARG, CT_ERR_GEOMETRY, CT_ERR_UNSUPPORTED, CT_ERR_ALLOC, CT_ERR_CUDA. */
CTSF_API ct_status_t ct_geom_create(const ct_geom_desc_t *desc, ct_geom_t **out);

/* Frees the geometry and its device memory.  ct_geom_destroy(NULL) is CT_OK. */
CTSF_API ct_status_t ct_geom_destroy(ct_geom_t *geom);

/* y = A x (Eq. 1).  d_vol: DEVICE, read, [batch][nz][ny][nx].
 * d_proj: DEVICE, written (every element exactly once), [batch][n_views][nv][nu].
 * Both caller-owned, fp32-aligned, must not overlap (a 16-byte aligned projection buffer with nu % 4 == 0 lets the
 * backprojector stage its tiles by TMA; other buffers take the cp.async path -- same results).  Asynchronous on
 * `stream`; makes no allocator call once the geometry is warm (the scratch for the xy-transposed volume that views
 * along x read is owned by the geometry, grown on first use and kept until ct_geom_destroy; calls in flight on
 * different streams or from different host threads each get a buffer of their own). */
CTSF_API ct_status_t ct_fp_sf(const ct_geom_t *geom, const float *d_vol, float *d_proj,
                     int32_t batch, ct_stream_t stream);

/* y = A x like ct_fp_sf -- same arguments, layouts, kernels and results -- for callers that are not allowed to
 * allocate device memory once they are running: a reconstruction loop inside a process whose GPU memory is already
 * owned by another allocator (a framework's caching pool, a fixed budget on a shared GPU), a loop with a latency
 * bound that cannot afford the device-wide stall of a cudaMalloc, a service whose policy forbids growth after
 * start-up.  Create the geometry at start-up (ct_geom_create does allocate); this call never does: no cudaMalloc,
 * cudaFree, stream-ordered allocation or allocating library routine, on the first call or any later one.
 * Its only scratch, the xy-transposed copy of the volume that views along x read, lives in a fixed array inside the
 * library image: 16 MiB of every GPU that uses libctsf, held until the process exits.  What follows from that:
 *  - limit: batch * nz * ny * nx <= CT_FP_SF_NOALLOC_MAX_VOXELS (e.g. one 160^3 volume, sixteen 512^2 images);
 *    anything larger is refused with CT_ERR_UNSUPPORTED before any work is queued -- use ct_fp_sf for it;
 *  - the GPU the geometry was created on must be the current device (else CT_ERR_INVALID_ARG);
 *  - the first call on each GPU looks up the array's device address (cudaGetSymbolAddress, which may load the
 *    library's device code): make that first call before starting any stream capture.  Later calls do no set-up;
 *  - every call on a GPU, whatever its geometry or stream, uses the same array.  Calls queued on ONE stream are safe
 *    (each call rewrites the part of the array it reads; nothing needs clearing, stale contents are never read).
 *    Calls that may overlap on the GPU -- different streams, different host threads -- race on it and corrupt each
 *    other's results: order them yourself (one stream, or events), or use ct_fp_sf there.
 * d_vol: DEVICE, read; d_proj: DEVICE, written (every element exactly once); both caller-owned.  Asynchronous on
 * `stream`.  Errors: CT_ERR_INVALID_ARG, CT_ERR_UNSUPPORTED (over the limit), CT_ERR_CUDA. */
#define CT_FP_SF_NOALLOC_MAX_VOXELS 4194304
CTSF_API ct_status_t ct_fp_sf_noalloc(const ct_geom_t *geom, const float *d_vol, float *d_proj,
                             int32_t batch, ct_stream_t stream);

/* x = A^T y (Eq. 2): the exact transpose of the weights of ct_fp_sf.
 * d_proj: DEVICE, read; d_vol: DEVICE, written (every element exactly once).  Asynchronous. */
CTSF_API ct_status_t ct_bp_sf(const ct_geom_t *geom, const float *d_proj, float *d_vol,
                     int32_t batch, ct_stream_t stream);

/* Ordered-subset variants: the operators restricted to views
 * view_begin, view_begin + view_stride, ... (view_count of them).  The projection buffer holds
 * ONLY the selected views: [batch][view_count][nv][nu].  view_count == 0 is the empty subset: the
 * projection buffer has no elements (its pointer may be NULL), A writes nothing and A^T writes zeros. */
CTSF_API ct_status_t ct_fp_sf_views(const ct_geom_t *geom, const float *d_vol, float *d_proj, int32_t batch,
                           int32_t view_begin, int32_t view_stride, int32_t view_count, ct_stream_t stream);
CTSF_API ct_status_t ct_bp_sf_views(const ct_geom_t *geom, const float *d_proj, float *d_vol, int32_t batch,
                           int32_t view_begin, int32_t view_stride, int32_t view_count, ct_stream_t stream);

/* "recon" mode ("the backprojection used in FBP reconstruction differs slightly from the general
 * backprojection by incorporating a depth-dependent weighting ... 'recon' mode"; "discrete ramp
 * filter").  The paper prints neither formula; readings R23, R24 define them:
 *   ct_fbp_filter : q = du * (p' * h) along the channels of every row, p' the cosine-weighted projection,
 *                   h the band-limited ramp at the channel pitch (flat) / its equi-angular form (arc).
 *                   d_proj read, d_out written, both DEVICE [batch][views][nv][nu]; NOT in place.
 *   ct_bp_sf_recon: x[n] = sum_i (d_i R_i / a^2) sum_kl F1(k) F2(l) q[i,l,k] / (sum F1 sum F2): the SF footprint as
 *                   a normalised interpolation kernel times the depth weight (arc: a^2 -> a^2 + b^2);
 *                   d_i = distance from the source to the rotation centre (the world origin).
 * Filtered backprojection of N equi-angular views over 360 degrees: x = (pi / N) * ct_bp_sf_recon(ct_fbp_filter(p)).
 * Same layouts, overwrite semantics, stream behaviour and errors as ct_bp_sf; *_views take ordered subsets. */
CTSF_API ct_status_t ct_fbp_filter(const ct_geom_t *geom, const float *d_proj, float *d_out,
                          int32_t batch, ct_stream_t stream);
CTSF_API ct_status_t ct_fbp_filter_views(const ct_geom_t *geom, const float *d_proj, float *d_out, int32_t batch,
                                int32_t view_begin, int32_t view_stride, int32_t view_count, ct_stream_t stream);
CTSF_API ct_status_t ct_bp_sf_recon(const ct_geom_t *geom, const float *d_proj, float *d_vol,
                           int32_t batch, ct_stream_t stream);
CTSF_API ct_status_t ct_bp_sf_recon_views(const ct_geom_t *geom, const float *d_proj, float *d_vol, int32_t batch,
                                 int32_t view_begin, int32_t view_stride, int32_t view_count, ct_stream_t stream);

/* The whole filtered backprojection of a full 360-degree scan with equi-angular views (
 * DESIGN.md reading R25): x = (pi / n_views) * ct_bp_sf_recon(ct_fbp_filter(p)), the angular weight folded into the
 * filter.  d_proj: DEVICE, read, [batch][n_views][nv][nu]; d_work: DEVICE scratch of the same size (holds the
 * filtered projections afterwards), must not alias d_proj; d_vol: DEVICE, written.  Asynchronous on `stream`. */
CTSF_API ct_status_t ct_fbp_sf(const ct_geom_t *geom, const float *d_proj, float *d_work, float *d_vol,
                      int32_t batch, ct_stream_t stream);

/* End-to-end convenience with HOST buffers (pageable or pinned): allocates device buffers from the
 * stream-ordered pool, copies the input host->device, runs the operator, copies the result
 * device->host and synchronises `stream` before returning.  Same layouts as above; any fp32-aligned host pointers.
 * 3-D, batch 1: copies and kernels of neighbouring view chunks overlap on a second stream owned by the geometry;
 * calls on one geometry are serialised. */
CTSF_API ct_status_t ct_fp_sf_host(const ct_geom_t *geom, const float *h_vol, float *h_proj,
                          int32_t batch, ct_stream_t stream);
CTSF_API ct_status_t ct_bp_sf_host(const ct_geom_t *geom, const float *h_proj, float *h_vol,
                          int32_t batch, ct_stream_t stream);

/* Number of kernels the LAST ct_fp_sf / ct_bp_sf call on this geometry launched (for the bench's
 * gpu_launches count).  Not thread-safe against concurrent calls on the same geometry. */
CTSF_API int32_t ct_last_launch_count(const ct_geom_t *geom);

/* Measured fp32 fused-multiply-add throughput of the current device, in flop/s (2 per FMA): the peak of the
 * roofline that binds this path (it is bound by fp32 arithmetic / instruction issue, not by HBM; DESIGN.md
 * "Roofline").  Runs an FMA-only kernel (independent register chains, no memory traffic, 4 waves
 * of one 1024-thread CTA per SM), best of 3, timed with CUDA events on `stream`; SYNCHRONISES `stream`.
 * kind 0: scalar FFMA; kind 1: packed FFMA2 (two FMAs per lane and instruction, sm_100); kinds 2, 3 (design record, not
 * peaks): FFMA2 interleaved 1:1 with scalar FFMA / with an ALU-pipe FMNMX -- FMA flops of the mix.
 * *flops_per_s HOST, written; *seconds HOST, optional (duration of the timed launch).
 * Errors: CT_ERR_INVALID_ARG, CT_ERR_ALLOC, CT_ERR_CUDA. */
CTSF_API ct_status_t ct_measure_fp32_peak(int32_t kind, double *flops_per_s, double *seconds, ct_stream_t stream);

/* Static description of a status code; never NULL. */
CTSF_API const char *ct_status_string(ct_status_t status);

#ifdef __cplusplus
}
#endif
#endif /* CTSF_H */
