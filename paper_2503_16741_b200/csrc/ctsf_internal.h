// ctsf_internal.h -- private declarations shared by the translation units of libctsf.
#pragma once
#include <atomic>
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
    std::atomic<int> last_launches{0};
};

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
                       int view_begin, int view_stride, int view_count, void *stream);
int ctsf_launch_fp(const ct_geom *g, const float *d_vol, float *d_proj, int batch,
                   int view_begin, int view_stride, int view_count, void *stream);
