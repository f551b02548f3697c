// sf_params.h -- per-view kernel parameters of the SF-TR projector pair (internal to libctsf).
//
// Everything here is derived on the host in float64 by geom.cpp (step S0 of DESIGN.md) and rounded
// once to fp32.  Kernels work in INDEX space: a voxel is addressed by (p, q, z) where p is the
// index along the memory-fastest in-slab axis and q the slab index.  For the backprojector and for
// forward views whose rays run mostly along y, (p, q) = (ix, iy); for forward views whose rays run
// mostly along x the volume is read through its xy-transpose and (p, q) = (iy, ix).
#pragma once
#include <stdint.h>

struct SfView {
    // w = P - S expressed in the detector frame, affine in the voxel index:
    //   a = w.n = a0 + p*ap + q*aq + z*az   (depth, mm)      b = w.u,  c = w.v  likewise
    float a0, ap, aq, az;
    float b0, bp, bq, bz;
    float c0, cp, cq, cz;
    // detector coordinates in CELL units (cell k spans [k, k+1], row l spans [l, l+1]):
    //   flat: kf = Ru*b/a + ku0,            lf = Rv*c/a + lv0
    //   arc : kf = Ru*atan2(b,a) + ku0,     lf = Rv*c/sqrt(a^2+b^2) + lv0
    float Ru, ku0, Rv, lv0;
    // amplitude: l = sqrt(a^2+b^2+c^2) / max(|p + ep0| , |q + eq0|)   (e_x/dx = ix + (x0 - Sx)/dx)
    float ep0, eq0;
    // transaxial corner half-diagonals: corners (+,+)/(-,-) move (a,b) by +-(pa,pb), (+,-)/(-,+) by +-(qa,qb)
    float pa, pb, qa, qb;
    // half steps along z for the axial end points
    float haz, hbz, hcz;
    int32_t untilted;          // 1: az == bz == 0 and cp == cq == 0 (transaxial part independent of z)
    int32_t swap_xy;           // forward only: 1 when (p, q) = (iy, ix)
    // ---- forward projector only: tile -> voxel-region inverse map -------------------------------
    // ray through detector point (kf, lf), in index space: dir = Dm + (kf - ku0c)*U + (lf - lv0c)*V (flat)
    // arc: dir = sin(g)*U + cos(g)*Dm + (lf - lv0c)*V with g = (kf - ku0c)/Ru   (U, Dm scaled by R)
    float Sp, Sq, Sz;          // source in index space
    float Dp, Dq, Dz;
    float Up, Uq, Uz;
    float Vp, Vq, Vz;
    float ku0c, lv0c;          // detector coordinates (cells) of the point the Dm ray hits
    float ek, el;              // max footprint half extent (cells / rows) over the view, x1.1: host-side bound on K, L
    int32_t lane_stride;       // voxels p, p + lane_stride project >= 1 cell apart (conflict-free rounds)
    float recon_dR;            // recon mode (reading R23): d * R, d = distance source -> rotation centre (world origin)
    float lpad;                // SF-TT (MODEL 2): rows the axial trapezoid reaches beyond the rectangle (brick shadow margin)
    float zpad;                // ... the same in voxels along z (forward kernel's region halo)
};

struct SfProblem {
    int32_t dim, det_type;
    int32_t nx, ny, nz, nu, nv, n_views;
};
