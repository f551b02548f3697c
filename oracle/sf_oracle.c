/*
 * sf_oracle.c -- float64 CPU oracle for the SF-TR projector pair.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code, header, table or helper with the CUDA path
 * under paper_2503_16741_b200/csrc/ and is never used as a fallback by the product.
 *
 * What it computes.  PAPER.md:93-101 (Sec. 2.3, Eq. (1) y = A x and Eq. (2) x = A^T y) with the
 * "separable footprint (SF)" voxel model of PAPER.md:103 ("volume-based voxel model", strict
 * adjoint).  The paper never prints the SF formulas; the step-by-step definition followed here
 * is the reading SURVEY.md Sec. 8(c) O1-O7 / DESIGN.md "Readings" R1-R18 (trapezoid transaxial
 * footprint x rectangular axial footprint, voxel-centre amplitude, cell-averaged response).
 * SF-TR is an approximation, so this file follows the algorithm in that order and notation; it
 * is written for legibility, not speed: no blocking, no fusion, no hoisting out of loops.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): trapezoid CDF vs quadrature; hand-worked 2-D
 * and 3-D footprints; brute-force ray/box chords; analytic disk/ellipsoid chords; mass
 * identities; parallel-beam column sums; 2-D == one-slice 3-D; dense-matrix transpose; adjoint
 * to 1e-12; symmetries; tilted frames and reversed axes against an independent ray/detector intersection model;
 * every factor of recon mode against analytic FBP/FDK; the SF-TT branch (R27) hand-worked through the same independent
 * intersection model at ~13 and ~25 degrees of polar angle, against a brute-force chord fraction, and in recon mode;
 * the DD tie rule (R26) on an exact-tie pixel; tests/test_oracle_mutations.py applies 28 one-line mutations
 * of this file and checks that a named pin fails for each.  Unpinned: model 3 ("SF-TT-A2", the row-dependent polar
 * amplitude) has the relative error table of tests/test_oracle_sftt.py only -- oracle-only, no kernel uses it.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libsf_oracle.so sf_oracle.c -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Problem description (own definition; deliberately not the product's ct_geom_desc_t header). */
typedef struct {
    int dim;                 /* 2 or 3 */
    int nx, ny, nz;
    double dx, dy, dz;       /* mm */
    double ox, oy, oz;       /* world position of the volume centre */
    int nu, nv;
    double du, dv;           /* mm; arc: du is arc length at radius R */
    int det_type;            /* 0 flat, 1 arc */
    int n_views;
    const double *src;       /* [n_views][3] */
    const double *det_center;/* [n_views][3] */
    const double *det_u;     /* [n_views][3] */
    const double *det_v;     /* [n_views][3]; dim 2: ignored, taken as (0,0,1) */
    int model;               /* 0: separable footprint SF-TR; 1: distance-driven DD (row f4, reading R26);
                                2: SF-TT, trapezoid axial footprint; 3: SF-TT with a row-dependent polar amplitude
                                (row f3, reading R27; oracle only -- measured against ray/box chords, not built on the GPU) */
} sfo_geom;

/* O1: per-view frame. */
typedef struct { double S[3], u[3], v[3], n[3], R, Du, Dv; } sfo_frame;

static double dot3(const double *a, const double *b) { return a[0]*b[0] + a[1]*b[1] + a[2]*b[2]; }

static void make_frame(const sfo_geom *g, int view, sfo_frame *f)
{
    const double *S = g->src + 3*view, *D = g->det_center + 3*view, *u = g->det_u + 3*view;
    double v[3] = {0.0, 0.0, 1.0};
    if (g->dim == 3) { v[0] = g->det_v[3*view]; v[1] = g->det_v[3*view+1]; v[2] = g->det_v[3*view+2]; }
    double n[3] = { u[1]*v[2] - u[2]*v[1], u[2]*v[0] - u[0]*v[2], u[0]*v[1] - u[1]*v[0] };
    double DS[3] = { D[0]-S[0], D[1]-S[1], D[2]-S[2] };
    if (dot3(DS, n) < 0.0) { n[0] = -n[0]; n[1] = -n[1]; n[2] = -n[2]; }   /* (D-S).n > 0 */
    for (int c = 0; c < 3; ++c) { f->S[c] = S[c]; f->u[c] = u[c]; f->v[c] = v[c]; f->n[c] = n[c]; }
    f->R  = dot3(DS, n);
    f->Du = dot3(DS, u);
    f->Dv = dot3(DS, v);
}

/* Detector coordinates (s, t) in mm of a world point P (SURVEY 8 "Notation").
 * Returns 0 if P is not in front of the source (a <= 0). */
static int det_coords(const sfo_geom *g, const sfo_frame *f, const double *P, double *s, double *t)
{
    double w[3] = { P[0]-f->S[0], P[1]-f->S[1], P[2]-f->S[2] };
    double a = dot3(w, f->n), b = dot3(w, f->u), c = dot3(w, f->v);
    if (!(a > 0.0)) return 0;
    if (g->det_type == 0) {            /* flat */
        *s = f->R * b / a - f->Du;
        *t = f->R * c / a - f->Dv;
    } else {                           /* arc: cylinder of radius R about the line through S along v */
        *s = f->R * atan2(b, a);
        *t = f->R * c / sqrt(a*a + b*b) - f->Dv;
    }
    return 1;
}

/* O4: CDF of the unit-height trapezoid with vertices tau[0] <= tau[1] <= tau[2] <= tau[3].
 * Half-open branches: a zero-width ramp is an empty branch, so no 0/0 is evaluated. */
double sfo_trap_cdf(const double *tau, double s)
{
    const double t0 = tau[0], t1 = tau[1], t2 = tau[2], t3 = tau[3];
    if (s <= t0) return 0.0;
    if (s <= t1) return (s - t0)*(s - t0) / (2.0*(t1 - t0));
    if (s <= t2) return (t1 - t0)/2.0 + (s - t1);
    if (s <= t3) return (t1 - t0)/2.0 + (t2 - t1) + (s - t2) - (s - t2)*(s - t2) / (2.0*(t3 - t2));
    return (t1 - t0)/2.0 + (t2 - t1) + (t3 - t2)/2.0;
}

static void sort4(double *a)
{
    for (int i = 1; i < 4; ++i) {
        double x = a[i]; int j = i - 1;
        while (j >= 0 && a[j] > x) { a[j+1] = a[j]; --j; }
        a[j+1] = x;
    }
}

/* O2-O6 for one (view, voxel).  Outputs the cell ranges [k_lo, k_hi], [l_lo, l_hi] (empty when
 * lo > hi), F1[k - k_lo], F2[l - l_lo] and the amplitude.  F1 must hold nu doubles, F2 nv doubles.
 * Returns 1 when the footprint touches the detector, 0 otherwise. */
static int footprint(const sfo_geom *g, const sfo_frame *f, int ix, int iy, int iz,
                     int *k_lo, int *k_hi, double *F1, int *l_lo, int *l_hi, double *F2,
                     double *amp, double *tau_out, double *sumF2_out)
{
    /* voxel centre (R9) */
    double Pc[3] = { g->ox + (ix - 0.5*(g->nx - 1))*g->dx,
                     g->oy + (iy - 0.5*(g->ny - 1))*g->dy,
                     g->dim == 3 ? g->oz + (iz - 0.5*(g->nz - 1))*g->dz : 0.0 };
    /* O3: transaxial corners at the voxel mid-plane (R4) */
    double tau[4]; int c = 0;
    for (int sx = -1; sx <= 1; sx += 2)
        for (int sy = -1; sy <= 1; sy += 2) {
            double P[3] = { Pc[0] + sx*0.5*g->dx, Pc[1] + sy*0.5*g->dy, Pc[2] };
            double t_unused;
            if (!det_coords(g, f, P, &tau[c], &t_unused)) return 0;       /* O2 */
            ++c;
        }
    if (g->model == 1) {
        /* R26, distance-driven (DD considers a "face-based voxel model"): the voxel is its
         * central face perpendicular to the axis the voxel-centre ray mostly runs along.  The face's two
         * in-plane edges -- (x_c +- dx/2, y_c) when the ray runs mostly along y, i.e. dy/|e_y| <= dx/|e_x|,
         * else (x_c, y_c +- dy/2) -- project to s_a <= s_b and the transaxial footprint is the RECTANGLE on
         * [s_a, s_b] (a trapezoid with zero-width ramps); the axial one stays the rectangle of O5 (the
         * face's two z edges); the amplitude O6 is the slab thickness along the ray, as for SF. */
        double ex = fabs(Pc[0] - f->S[0]), ey = fabs(Pc[1] - f->S[1]);
        int along_y = g->dy * ex <= g->dx * ey;                    /* dy/|e_y| <= dx/|e_x| */
        double Pa[3] = { Pc[0], Pc[1], Pc[2] }, Pb[3] = { Pc[0], Pc[1], Pc[2] };
        if (along_y) { Pa[0] -= 0.5*g->dx; Pb[0] += 0.5*g->dx; } else { Pa[1] -= 0.5*g->dy; Pb[1] += 0.5*g->dy; }
        double sa, sb, t_unused;
        if (!det_coords(g, f, Pa, &sa, &t_unused)) return 0;
        if (!det_coords(g, f, Pb, &sb, &t_unused)) return 0;
        tau[0] = tau[1] = sa < sb ? sa : sb;
        tau[2] = tau[3] = sa < sb ? sb : sa;
    }
    sort4(tau);
    if (tau_out) memcpy(tau_out, tau, sizeof tau);
    /* O4: transaxial cell range and cell-averaged weights (R3, R12, R15) */
    int klo = (int)floor(tau[0]/g->du + 0.5*g->nu), khi = (int)floor(tau[3]/g->du + 0.5*g->nu);
    if (klo < 0) klo = 0;
    if (khi > g->nu - 1) khi = g->nu - 1;
    *k_lo = klo; *k_hi = khi;
    if (klo > khi) return 0;
    for (int k = klo; k <= khi; ++k) {
        double uk = (k - 0.5*(g->nu - 1))*g->du;
        F1[k - klo] = (sfo_trap_cdf(tau, uk + 0.5*g->du) - sfo_trap_cdf(tau, uk - 0.5*g->du)) / g->du;
    }
    /* O5: axial footprint (R5) */
    if (g->dim == 3 && g->model >= 2) {
        /* R27 ("higher-cone-angle SF variants"): the axial footprint of a ray family at row
         * coordinate t is the fraction of the in-plane chord (length l_theta, from the voxel's near point to its far
         * point along the voxel-centre ray's in-plane direction) that lies between z_c - dz/2 and z_c + dz/2: a
         * TRAPEZOID whose vertices are the row coordinates of (near, far) x (z_c -+ dz/2).  model 3 additionally
         * evaluates the polar stretch |d| / |d_xy| of the amplitude per detector row instead of at the voxel centre. */
        double exy[2] = { Pc[0]-f->S[0], Pc[1]-f->S[1] };
        double nxy = sqrt(exy[0]*exy[0] + exy[1]*exy[1]);
        double ux = exy[0]/nxy, uy = exy[1]/nxy;
        double rx_ = g->dx / fabs(ux), ry_ = g->dy / fabs(uy);
        double lth = rx_ < ry_ ? rx_ : ry_;
        double xi[4]; int c4 = 0;
        for (int sn = -1; sn <= 1; sn += 2)
            for (int sz = -1; sz <= 1; sz += 2) {
                double P[3] = { Pc[0] + sn*0.5*lth*ux, Pc[1] + sn*0.5*lth*uy, Pc[2] + sz*0.5*g->dz };
                double s_unused;
                if (!det_coords(g, f, P, &s_unused, &xi[c4])) return 0;
                ++c4;
            }
        sort4(xi);
        if (sumF2_out) *sumF2_out = 0.5*(xi[3] + xi[2] - xi[1] - xi[0]) / g->dv;   /* area of the trapezoid */
        int llo = (int)floor(xi[0]/g->dv + 0.5*g->nv), lhi = (int)floor(xi[3]/g->dv + 0.5*g->nv);
        if (llo < 0) llo = 0;
        if (lhi > g->nv - 1) lhi = g->nv - 1;
        *l_lo = llo; *l_hi = lhi;
        if (llo > lhi) return 0;
        double e3[3] = { Pc[0]-f->S[0], Pc[1]-f->S[1], Pc[2]-f->S[2] };
        double polar_c = sqrt(e3[0]*e3[0] + e3[1]*e3[1] + e3[2]*e3[2]) / nxy;      /* |e| / |e_xy| at the voxel centre */
        double sc, tc_unused;
        det_coords(g, f, Pc, &sc, &tc_unused);
        for (int l = llo; l <= lhi; ++l) {
            double vl = (l - 0.5*(g->nv - 1))*g->dv;
            F2[l - llo] = (sfo_trap_cdf(xi, vl + 0.5*g->dv) - sfo_trap_cdf(xi, vl - 0.5*g->dv)) / g->dv;
            if (g->model == 3) {
                /* ray from the source to the detector point (s of the voxel centre, row centre v_l) */
                double d[3];
                if (g->det_type == 0) {
                    for (int q = 0; q < 3; ++q) d[q] = f->R*f->n[q] + (sc + f->Du)*f->u[q] + (vl + f->Dv)*f->v[q];
                } else {
                    double ga = sc / f->R;
                    for (int q = 0; q < 3; ++q) d[q] = f->R*(sin(ga)*f->u[q] + cos(ga)*f->n[q]) + (vl + f->Dv)*f->v[q];
                }
                double polar_l = sqrt(d[0]*d[0] + d[1]*d[1] + d[2]*d[2]) / sqrt(d[0]*d[0] + d[1]*d[1]);
                F2[l - llo] *= polar_l / polar_c;       /* the common amplitude below carries polar_c */
            }
        }
    } else if (g->dim == 3) {
        double Pm[3] = { Pc[0], Pc[1], Pc[2] - 0.5*g->dz }, Pp[3] = { Pc[0], Pc[1], Pc[2] + 0.5*g->dz };
        double s_unused, ta, tb;
        if (!det_coords(g, f, Pm, &s_unused, &ta)) return 0;
        if (!det_coords(g, f, Pp, &s_unused, &tb)) return 0;
        double tlo = ta < tb ? ta : tb, thi = ta < tb ? tb : ta;
        if (sumF2_out) *sumF2_out = (thi - tlo) / g->dv;
        int llo = (int)floor(tlo/g->dv + 0.5*g->nv), lhi = (int)floor(thi/g->dv + 0.5*g->nv);
        if (llo < 0) llo = 0;
        if (lhi > g->nv - 1) lhi = g->nv - 1;
        *l_lo = llo; *l_hi = lhi;
        if (llo > lhi) return 0;
        for (int l = llo; l <= lhi; ++l) {
            double vl = (l - 0.5*(g->nv - 1))*g->dv;
            double hi = vl + 0.5*g->dv < thi ? vl + 0.5*g->dv : thi;
            double lo = vl - 0.5*g->dv > tlo ? vl - 0.5*g->dv : tlo;
            F2[l - llo] = (hi - lo > 0.0 ? hi - lo : 0.0) / g->dv;
        }
    } else {
        *l_lo = 0; *l_hi = 0; F2[0] = 1.0;                                  /* R18 */
        if (sumF2_out) *sumF2_out = 1.0;
    }
    /* O6: amplitude along the voxel-centre ray (R2, R14) */
    double e[3] = { Pc[0]-f->S[0], Pc[1]-f->S[1], g->dim == 3 ? Pc[2]-f->S[2] : 0.0 };
    double norm = sqrt(e[0]*e[0] + e[1]*e[1] + e[2]*e[2]);
    double rx = g->dx / fabs(e[0]), ry = g->dy / fabs(e[1]);                /* x/0 = +inf */
    *amp = norm * (rx < ry ? rx : ry);
    return 1;
}

/* ---- public entry points (all arrays double, C-contiguous) ------------------------------- */

/* Footprint of one voxel in one view, for the pins.  F1 (nu doubles) and F2 (nv doubles) are
 * caller-allocated.  rng_out = {k_lo, k_hi, l_lo, l_hi}; tau_out = 4 sorted vertices. */
int sfo_footprint(const sfo_geom *g, int view, int ix, int iy, int iz,
                  int *rng_out, double *F1, double *F2, double *amp, double *tau_out)
{
    sfo_frame f; make_frame(g, view, &f);
    rng_out[0] = 0; rng_out[1] = -1; rng_out[2] = 0; rng_out[3] = -1;
    return footprint(g, &f, ix, iy, iz, &rng_out[0], &rng_out[1], F1, &rng_out[2], &rng_out[3], F2, amp, tau_out, NULL);
}

/* Detector coordinates of a world point in one view (for the brute-force pins). */
int sfo_det_coords(const sfo_geom *g, int view, const double *P, double *st)
{
    sfo_frame f; make_frame(g, view, &f);
    return det_coords(g, &f, P, &st[0], &st[1]);
}

/* O7, forward: one view of y += A x restricted to slices [z0, z1). y is [nv][nu]. */
static void fp_view_slab(const sfo_geom *g, const sfo_frame *f, const double *vol, double *y,
                         int z0, int z1, double *F1, double *F2)
{
    for (int iz = z0; iz < z1; ++iz)
        for (int iy = 0; iy < g->ny; ++iy)
            for (int ix = 0; ix < g->nx; ++ix) {
                double xv = vol[((size_t)iz*g->ny + iy)*g->nx + ix];
                int klo, khi, llo, lhi; double amp;
                if (!footprint(g, f, ix, iy, iz, &klo, &khi, F1, &llo, &lhi, F2, &amp, NULL, NULL)) continue;
                for (int l = llo; l <= lhi; ++l)
                    for (int k = klo; k <= khi; ++k)
                        y[(size_t)l*g->nu + k] += amp * F1[k - klo] * F2[l - llo] * xv;
            }
}

/* y[j] = (A x)[views[j]] for j < n_sel.  vol [nz][ny][nx]; proj [n_sel][nv][nu] (overwritten).
 * Deterministic for a fixed thread count.  Returns the number of threads used. */
int sfo_fp(const sfo_geom *g, const double *vol, const int *views, int n_sel, double *proj)
{
    const size_t ncell = (size_t)g->nu * g->nv;
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    memset(proj, 0, sizeof(double) * ncell * n_sel);
    if (g->nz < 2*nthreads || n_sel >= 4*nthreads) {
        /* parallel over views: every view's output is private */
        #pragma omp parallel
        {
            double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
            #pragma omp for schedule(dynamic, 1)
            for (int j = 0; j < n_sel; ++j) {
                sfo_frame f; make_frame(g, views[j], &f);
                fp_view_slab(g, &f, vol, proj + ncell*j, 0, g->nz, F1, F2);
            }
            free(F1); free(F2);
        }
    } else {
        /* few views, many slices: split slices statically, private partial images, ordered sum */
        double *part = malloc(sizeof(double) * ncell * nthreads);
        for (int j = 0; j < n_sel; ++j) {
            sfo_frame f; make_frame(g, views[j], &f);
            memset(part, 0, sizeof(double) * ncell * nthreads);
            #pragma omp parallel num_threads(nthreads)
            {
                int tid = 0, nt = 1;
#ifdef _OPENMP
                tid = omp_get_thread_num(); nt = omp_get_num_threads();
#endif
                double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
                int z0 = (int)((long)g->nz * tid / nt), z1 = (int)((long)g->nz * (tid+1) / nt);
                fp_view_slab(g, &f, vol, part + ncell*tid, z0, z1, F1, F2);
                free(F1); free(F2);
            }
            for (int t = 0; t < nthreads; ++t)
                for (size_t c = 0; c < ncell; ++c) proj[ncell*j + c] += part[ncell*t + c];
        }
        free(part);
    }
    return nthreads;
}

/* O7, adjoint, one voxel: sum over the selected views in order. proj is [n_sel][nv][nu]. */
static double bp_voxel(const sfo_geom *g, const sfo_frame *frames, const double *proj, int n_sel,
                       int ix, int iy, int iz, double *F1, double *F2)
{
    const size_t ncell = (size_t)g->nu * g->nv;
    double acc = 0.0;
    for (int j = 0; j < n_sel; ++j) {
        int klo, khi, llo, lhi; double amp;
        if (!footprint(g, &frames[j], ix, iy, iz, &klo, &khi, F1, &llo, &lhi, F2, &amp, NULL, NULL)) continue;
        const double *y = proj + ncell*j;
        for (int l = llo; l <= lhi; ++l)
            for (int k = klo; k <= khi; ++k)
                acc += amp * F1[k - klo] * F2[l - llo] * y[(size_t)l*g->nu + k];
    }
    return acc;
}

/* vol = A^T y over the selected views.  proj [n_sel][nv][nu]; vol [nz][ny][nx] (overwritten). */
int sfo_bp(const sfo_geom *g, const double *proj, const int *views, int n_sel, double *vol)
{
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    sfo_frame *frames = malloc(sizeof(sfo_frame) * (n_sel > 0 ? n_sel : 1));
    for (int j = 0; j < n_sel; ++j) make_frame(g, views[j], &frames[j]);
    #pragma omp parallel
    {
        double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
        #pragma omp for schedule(dynamic, 4) collapse(2)
        for (int iz = 0; iz < g->nz; ++iz)
            for (int iy = 0; iy < g->ny; ++iy)
                for (int ix = 0; ix < g->nx; ++ix)
                    vol[((size_t)iz*g->ny + iy)*g->nx + ix] = bp_voxel(g, frames, proj, n_sel, ix, iy, iz, F1, F2);
        free(F1); free(F2);
    }
    free(frames);
    return nthreads;
}

/* ---- "recon" mode ("depth-dependent weighting specifically for FBP
 * reconstruction", "discrete ramp filter").  The paper prints neither formula; DESIGN.md
 * readings R23 (backprojection) and R24 (filter) are followed step by step.  Pins: tests/test_oracle_recon.py
 * (filtered backprojection of analytic disk / sphere projections returns the attenuation value). ------- */

/* R24: q = du * sum_m p'[m] h[k-m] along every detector row of the selected views.
 * p' = p * R/sqrt(R^2 + s^2 + t^2) (flat; (s,t) measured from the foot of the source normal) or
 * p * cos(gamma) * R/sqrt(R^2 + t^2) (arc; gamma = u_k/R).  h[0] = 1/(4 du^2), h[even] = 0,
 * h[odd n] = -1/(pi n du)^2 (flat), -1/(pi R sin(n du/R))^2 (arc).  proj, out: [n_sel][nv][nu]. */
int sfo_fbp_filter(const sfo_geom *g, const double *proj, const int *views, int n_sel, double *out)
{
    const double PI = 3.14159265358979323846;
    for (int j = 0; j < n_sel; ++j) {
        sfo_frame f; make_frame(g, views[j], &f);
        double *pw = malloc(sizeof(double) * g->nu);
        for (int l = 0; l < g->nv; ++l) {
            const double *p = proj + ((size_t)j*g->nv + l)*g->nu;
            double *q = out + ((size_t)j*g->nv + l)*g->nu;
            double t = g->dim == 3 ? (l - 0.5*(g->nv - 1))*g->dv + f.Dv : 0.0;
            for (int k = 0; k < g->nu; ++k) {
                double uk = (k - 0.5*(g->nu - 1))*g->du;
                if (g->det_type == 0) { double s = uk + f.Du; pw[k] = p[k] * f.R / sqrt(f.R*f.R + s*s + t*t); }
                else                  { pw[k] = p[k] * cos(uk / f.R) * f.R / sqrt(f.R*f.R + t*t); }
            }
            for (int k = 0; k < g->nu; ++k) {
                double acc = 0.0;
                for (int m = 0; m < g->nu; ++m) {
                    int n = k - m; if (n < 0) n = -n;
                    double h;
                    if (n == 0) h = 1.0 / (4.0*g->du*g->du);
                    else if (n % 2 == 0) h = 0.0;
                    else if (g->det_type == 0) h = -1.0 / (PI*n*g->du * PI*n*g->du);
                    else { double sn = PI * f.R * sin(n*g->du / f.R); h = -1.0 / (sn*sn); }
                    acc += pw[m] * h;
                }
                q[k] = g->du * acc;
            }
        }
        free(pw);
    }
    return 0;
}

/* R23, one voxel: sum over views of W * sum_kl (F1/sumF1)(F2/sumF2) q, W = d R / a^2 (flat),
 * d R / (a^2 + b^2) (arc); d = in-plane distance of the rotation centre (world origin) from the
 * source: -S.n (flat), sqrt((S.n)^2 + (S.u)^2) (arc).  sumF1, sumF2: unclipped footprint sums. */
static double bp_voxel_recon(const sfo_geom *g, const sfo_frame *frames, const double *q, int n_sel,
                             int ix, int iy, int iz, double *F1, double *F2)
{
    const size_t ncell = (size_t)g->nu * g->nv;
    double Pc[3] = { g->ox + (ix - 0.5*(g->nx - 1))*g->dx, g->oy + (iy - 0.5*(g->ny - 1))*g->dy,
                     g->dim == 3 ? g->oz + (iz - 0.5*(g->nz - 1))*g->dz : 0.0 };
    double acc = 0.0;
    for (int j = 0; j < n_sel; ++j) {
        const sfo_frame *f = &frames[j];
        int klo, khi, llo, lhi; double amp, tau[4], sumF2 = 1.0;
        if (!footprint(g, f, ix, iy, iz, &klo, &khi, F1, &llo, &lhi, F2, &amp, tau, &sumF2)) continue;
        double sumF1 = 0.5*(tau[3] + tau[2] - tau[1] - tau[0]) / g->du;     /* sumF2: the axial factor's own unclipped sum */
        double w[3] = { Pc[0]-f->S[0], Pc[1]-f->S[1], Pc[2]-f->S[2] };
        double a = dot3(w, f->n), b = dot3(w, f->u);
        double Sn = dot3(f->S, f->n), Su = dot3(f->S, f->u);
        double W = g->det_type == 0 ? (-Sn) * f->R / (a*a) : sqrt(Sn*Sn + Su*Su) * f->R / (a*a + b*b);
        double sum = 0.0;
        const double *y = q + ncell*j;
        for (int l = llo; l <= lhi; ++l)
            for (int k = klo; k <= khi; ++k)
                sum += F1[k - klo] * F2[l - llo] * y[(size_t)l*g->nu + k];
        acc += W * sum / (sumF1 * sumF2);
    }
    return acc;
}

/* vol = B q over the selected views (recon-mode backprojection).  q [n_sel][nv][nu]; vol overwritten. */
int sfo_bp_recon(const sfo_geom *g, const double *q, const int *views, int n_sel, double *vol)
{
    sfo_frame *frames = malloc(sizeof(sfo_frame) * (n_sel > 0 ? n_sel : 1));
    for (int j = 0; j < n_sel; ++j) make_frame(g, views[j], &frames[j]);
    #pragma omp parallel
    {
        double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
        #pragma omp for schedule(dynamic, 4) collapse(2)
        for (int iz = 0; iz < g->nz; ++iz)
            for (int iy = 0; iy < g->ny; ++iy)
                for (int ix = 0; ix < g->nx; ++ix)
                    vol[((size_t)iz*g->ny + iy)*g->nx + ix] = bp_voxel_recon(g, frames, q, n_sel, ix, iy, iz, F1, F2);
        free(F1); free(F2);
    }
    free(frames);
    return 0;
}

/* (A^T y) at n listed voxels (ijk[3*i..] = ix, iy, iz), all views; y is the FULL [n_views][nv][nu]. */
int sfo_bp_voxels(const sfo_geom *g, const double *proj, const int *ijk, int n, double *out)
{
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    sfo_frame *frames = malloc(sizeof(sfo_frame) * g->n_views);
    for (int j = 0; j < g->n_views; ++j) make_frame(g, j, &frames[j]);
    #pragma omp parallel
    {
        double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
        #pragma omp for schedule(dynamic, 16)
        for (int i = 0; i < n; ++i)
            out[i] = bp_voxel(g, frames, proj, g->n_views, ijk[3*i], ijk[3*i+1], ijk[3*i+2], F1, F2);
        free(F1); free(F2);
    }
    free(frames);
    return nthreads;
}

/* Same as sfo_bp_voxels but the projections are given in float32 (the full-size config-4
 * projection set is 1.6 GB in fp32; widening all of it to float64 would need 3.4 GB more).
 * Each value is widened to double before use. */
int sfo_bp_voxels_f32(const sfo_geom *g, const float *proj, const int *ijk, int n, double *out)
{
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
#endif
    const size_t ncell = (size_t)g->nu * g->nv;
    sfo_frame *frames = malloc(sizeof(sfo_frame) * g->n_views);
    for (int j = 0; j < g->n_views; ++j) make_frame(g, j, &frames[j]);
    #pragma omp parallel
    {
        double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
        #pragma omp for schedule(dynamic, 16)
        for (int i = 0; i < n; ++i) {
            double acc = 0.0;
            for (int j = 0; j < g->n_views; ++j) {
                int klo, khi, llo, lhi; double amp;
                if (!footprint(g, &frames[j], ijk[3*i], ijk[3*i+1], ijk[3*i+2], &klo, &khi, F1, &llo, &lhi, F2, &amp, NULL, NULL)) continue;
                const float *y = proj + ncell*j;
                for (int l = llo; l <= lhi; ++l)
                    for (int k = klo; k <= khi; ++k)
                        acc += amp * F1[k - klo] * F2[l - llo] * (double)y[(size_t)l*g->nu + k];
            }
            out[i] = acc;
        }
        free(F1); free(F2);
    }
    free(frames);
    return nthreads;
}

/* Fraction of voxel x view pairs whose footprint touches the detector ("live"), on a strided
 * sample of voxels and views; reported by the bench next to GUPS. */
double sfo_live_fraction(const sfo_geom *g, int vox_stride, int view_stride)
{
    long live = 0, total = 0;
    double *F1 = malloc(sizeof(double)*g->nu), *F2 = malloc(sizeof(double)*g->nv);
    for (int j = 0; j < g->n_views; j += view_stride) {
        sfo_frame f; make_frame(g, j, &f);
        for (int iz = 0; iz < g->nz; iz += vox_stride)
            for (int iy = 0; iy < g->ny; iy += vox_stride)
                for (int ix = 0; ix < g->nx; ix += vox_stride) {
                    int klo, khi, llo, lhi; double amp;
                    live += footprint(g, &f, ix, iy, iz, &klo, &khi, F1, &llo, &lhi, F2, &amp, NULL, NULL);
                    ++total;
                }
    }
    free(F1); free(F2);
    return total ? (double)live / (double)total : 0.0;
}

int sfo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
