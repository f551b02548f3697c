// ctsf_internal.h -- private declarations shared by the translation units of libctsf.
#pragma once
#include <atomic>
#include <mutex>
#include <vector>

#include "../../include/ctsf.h"
#include "sf_params.h"

struct ct_geom {
    SfProblem prob;
    double du = 1.0, dv = 1.0;        // detector pitches, mm (ramp filter)
    int model = 0;                    // 0 separable footprint (SF-TR), 1 distance-driven (DD)
    std::vector<SfView> h_bp, h_fp;   // host copies (natural order / forward order with xy swaps)
    SfView *d_bp = nullptr, *d_fp = nullptr;
    int any_swap = 0;                 // some forward view reads the volume through its transpose
    int all_untilted = 0;             // every view: transaxial footprint independent of z
    int fp_hoist_ok = 0;              // all untilted AND every footprint spans <= 6 columns, <= 8 rows
    int device = 0;
    mutable std::atomic<int> last_launches{0};   // statistics only (ct_last_launch_count); not part of the geometry

    // Scratch of the forward projector (the xy-transposed volume), owned by the geometry so that a warmed-up
    // ct_fp_sf makes no allocator call ("any workspace is allocated in ct_geom_create" -- its size
    // depends on the batch, so it is grown on first use and kept).  A slot is reused by a later call on the same
    // stream at once (stream order), by a call on another stream only after the event recorded behind its last
    // use has completed; otherwise another slot is made.  `busy`: taken by a call that has not released it yet (its
    // event is not recorded yet, so it must not be judged by it).  An idle slot that is too small for a later, larger
    // batch is replaced by the larger buffer.  Freed by ct_geom_destroy.
    struct Scratch { void *ptr = nullptr; size_t bytes = 0; void *stream = nullptr; void *done = nullptr; bool busy = false; };
    mutable std::vector<Scratch> scratch;
    mutable std::mutex scratch_mu;
    // host-buffer entry points: copy stream and chunk events, made on first use
    mutable void *host_copy_stream = nullptr;
    mutable std::vector<void *> host_events;
    mutable std::mutex host_mu;
};

// ctsf_api.cu: a geometry-owned scratch buffer of >= bytes for work ordered on `stream` (nullptr: failed);
// ctsf_scratch_release records the end of its use on that stream.
void *ctsf_scratch_acquire(const ct_geom *g, size_t bytes, void *stream);
void ctsf_scratch_release(const ct_geom *g, void *ptr, void *stream);

// Testing aids (ctsf_debug_set; not part of the ABI of include/ctsf.h): switches that force rarely taken code paths.
// None changes a result beyond summation order.  Read by the launchers; set by tests only, never by the product.
struct CtsfDebug {
    float fp_pad = 0.0f;          // widen the forward kernel's swept voxel region by this many voxels
    int fp_nohoist = 0, fp_forcehoist = 0;   // untilted fast path of the forward kernel off / on regardless of the host bound
    int fp_serial = 0;            // forward kernel: take the lane-serial conflict branch
    int bp_nohoist = 0, bp_forcehoist = 0;   // the same for the backprojector's register-weight path
    int bp_tma = -1;              // backprojector tile staging: -1 default, 0 cp.async only, 1..3 partial TMA use
    int bp_chunk = 0;             // views per backprojector launch (0: sized for L2)
    int bp_scalar = 0;            // general frames: one voxel per thread (the round-1 kernel) instead of packed pairs
    int bp_poison = 0;            // packed backprojector: ring stages start as NaN (no load may reach an unstaged one)
    float tt_pad = 0.0f;          // SF-TT: rows / voxels added to the sampled trapezoid margins (lpad, zpad) at ct_geom_create
    int host_fp_chunks = 0;       // host-buffer A / A^T: number of view chunks of the copy/compute pipeline (0: default)
    int host_bp_chunks = 0;
};
extern CtsfDebug g_ctsf_debug;

// ctsf_api.cu: the library's own stream-ordered memory pool on the current device (scratch of the
// forward projector, device buffers of the host-buffer entry points).  Its release threshold is
// unlimited, so a buffer freed by one call is reused by the next instead of going back to the
// driver at every synchronisation; ct_geom_destroy trims it.  nullptr if pools are unavailable.
void *ctsf_alloc_async(size_t bytes, void *stream);
void ctsf_free_async(void *p, void *stream);

// geom.cpp
ct_status_t ctsf_build_views(const ct_geom_desc_t *desc, ct_geom *g);

// sf_bp.cu / sf_fp.cu: launchers.  Projection buffers hold `view_count` views; view j of the buffer
// is geometry view view_begin + j*view_stride.  Return the number of kernels launched, or -1.
// accumulate != 0 (3-D only): add to d_vol instead of overwriting it.  recon != 0: recon-mode weights (R23).
int ctsf_launch_bp(const ct_geom *g, const float *d_proj, float *d_vol, int batch,
                   int view_begin, int view_stride, int view_count, void *stream, int accumulate = 0,
                   int recon = 0);
// sf_filter.cu: cosine pre-weight + discrete ramp filter of the selected views (reading R24).
int ctsf_launch_filter(const ct_geom *g, const float *d_proj, float *d_out, int batch,
                       int view_begin, int view_stride, int view_count, void *stream, double scale = 1.0);
// d_volT: the xy-transposed volume when the caller already has it (ctsf_fp_transpose), else nullptr: made on the fly
// in the geometry's scratch when a selected view needs it.
int ctsf_launch_fp(const ct_geom *g, const float *d_vol, float *d_proj, int batch,
                   int view_begin, int view_stride, int view_count, void *stream, const float *d_volT = nullptr);
// transposes d_vol into d_volT ([batch][nz][nx][ny]); returns the number of launches, or -1
int ctsf_fp_transpose(const ct_geom *g, const float *d_vol, float *d_volT, int batch, void *stream);
bool ctsf_fp_needs_transpose(const ct_geom *g, int view_begin, int view_stride, int view_count);
// CTAs the forward kernel launches for `view_count` views of one image (the host pipeline sizes its chunks with it)
long ctsf_fp_cta_count(const ct_geom *g, int view_count);
