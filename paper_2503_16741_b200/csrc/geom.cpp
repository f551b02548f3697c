// geom.cpp -- step S0: validate a scan description and pack per-view kernel parameters.
// Host only, float64 throughout; the single rounding to fp32 happens in pack_view().
// ("C++ projector function ... constructs C++ geometry objects"; Table 2.)
#include "ctsf_internal.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>

namespace {

struct V3 { double x, y, z; };
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline V3 ld3(const double *p, int i) { return {p[3 * i], p[3 * i + 1], p[3 * i + 2]}; }

// float64 model of one view in (p, q, z) index space, used for packing and for the bounds below
struct ViewD {
    double a0, ap, aq, az, b0, bp, bq, bz, c0, cp, cq, cz;
    double Ru, ku0, Rv, lv0;
    int arc, dim;
    void project(double p, double q, double z, double &kf, double &lf) const {
        double a = a0 + p * ap + q * aq + z * az;
        double b = b0 + p * bp + q * bq + z * bz;
        double c = c0 + p * cp + q * cq + z * cz;
        if (!arc) { kf = Ru * b / a + ku0; lf = Rv * c / a + lv0; }
        else      { kf = Ru * std::atan2(b, a) + ku0; lf = Rv * c / std::sqrt(a * a + b * b) + lv0; }
        if (dim == 2) lf = 0.5;
    }
};

}  // namespace

ct_status_t ctsf_build_views(const ct_geom_desc_t *d, ct_geom *g)
{
    const int nviews = d->n_views;
    const bool is3 = d->dim == 3;
    g->h_bp.resize(nviews);
    g->h_fp.resize(nviews);
    g->any_swap = 0;
    g->all_untilted = 1;
    int small_fp = 1;
    // world position of voxel (0,0,0)
    const V3 O = {d->ox - 0.5 * (d->nx - 1) * d->dx, d->oy - 0.5 * (d->ny - 1) * d->dy,
                  is3 ? d->oz - 0.5 * (d->nz - 1) * d->dz : 0.0};
    const V3 C = {d->ox, d->oy, is3 ? d->oz : 0.0};
    const V3 half = {0.5 * d->nx * d->dx, 0.5 * d->ny * d->dy, is3 ? 0.5 * d->nz * d->dz : 0.0};

    for (int i = 0; i < nviews; ++i) {
        V3 S = ld3(d->src, i), D = ld3(d->det_center, i), u = ld3(d->det_u, i);
        V3 v = (is3 || d->det_v) ? ld3(d->det_v ? d->det_v : d->det_u, i) : V3{0, 0, 1};
        if (!is3) {
            if (!d->det_v) v = V3{0, 0, 1};
            if (S.z != 0.0 || D.z != 0.0 || u.z != 0.0 || std::fabs(v.x) > 1e-9 || std::fabs(v.y) > 1e-9)
                return CT_ERR_GEOMETRY;
            v = V3{0, 0, 1};
        }
        if (std::fabs(dot(u, u) - 1.0) > 1e-9 || std::fabs(dot(v, v) - 1.0) > 1e-9 || std::fabs(dot(u, v)) > 1e-9)
            return CT_ERR_GEOMETRY;
        V3 n = cross(u, v);
        V3 DS = D - S;
        if (dot(DS, n) < 0.0) n = V3{-n.x, -n.y, -n.z};
        const double R = dot(DS, n), Du = dot(DS, u), Dv = dot(DS, v);
        if (!(R > 0.0) || !std::isfinite(R)) return CT_ERR_GEOMETRY;
        if (d->det_type == 1 && std::fabs(Du) > 1e-9 * R) return CT_ERR_GEOMETRY;
        // the whole voxel grid (outer faces) must lie strictly in front of the source plane
        double amin = std::numeric_limits<double>::infinity();
        for (int cx = -1; cx <= 1; cx += 2) for (int cy = -1; cy <= 1; cy += 2) for (int cz = -1; cz <= 1; cz += 2) {
            V3 P = {C.x + cx * half.x, C.y + cy * half.y, C.z + cz * half.z};
            amin = std::min(amin, dot(P - S, n));
        }
        if (!(amin > 0.0)) return CT_ERR_GEOMETRY;

        // affine coefficients in natural (ix, iy, iz) order
        V3 w0 = O - S;
        double A[4] = {dot(w0, n), d->dx * n.x, d->dy * n.y, is3 ? d->dz * n.z : 0.0};
        double B[4] = {dot(w0, u), d->dx * u.x, d->dy * u.y, is3 ? d->dz * u.z : 0.0};
        double Cc[4] = {dot(w0, v), d->dx * v.x, d->dy * v.y, is3 ? d->dz * v.z : 0.0};
        if (!is3) { Cc[0] = Cc[1] = Cc[2] = Cc[3] = 0.0; }
        const double Ru = R / d->du, Rv = R / d->dv;
        const double ku0 = (d->det_type == 0 ? -Du / d->du : 0.0) + 0.5 * d->nu;
        const double lv0 = -Dv / d->dv + 0.5 * d->nv;
        const double ex0 = (O.x - S.x) / d->dx, ey0 = (O.y - S.y) / d->dy;
        const bool untilted = std::fabs(A[3]) <= 1e-13 * d->dz && std::fabs(B[3]) <= 1e-13 * d->dz &&
                              std::fabs(Cc[1]) <= 1e-13 * d->dx && std::fabs(Cc[2]) <= 1e-13 * d->dy;
        if (!untilted) g->all_untilted = 0;
        // forward: rays mostly along x  <=>  |n.x| > |n.y|  -> read the volume through its transpose
        const bool swap = std::fabs(n.x) > std::fabs(n.y);
        if (swap) g->any_swap = 1;

        for (int pass = 0; pass < 2; ++pass) {
            if (pass == 1 && !swap) break;
            const bool sw = pass == 1 && swap;
            const int P = sw ? 2 : 1, Q = sw ? 1 : 2;       // which natural axis plays p / q
            SfView o;
            std::memset(&o, 0, sizeof o);
            ViewD m;
            m.a0 = A[0]; m.ap = A[P]; m.aq = A[Q]; m.az = A[3];
            m.b0 = B[0]; m.bp = B[P]; m.bq = B[Q]; m.bz = B[3];
            m.c0 = Cc[0]; m.cp = Cc[P]; m.cq = Cc[Q]; m.cz = Cc[3];
            m.Ru = Ru; m.ku0 = ku0; m.Rv = Rv; m.lv0 = lv0; m.arc = d->det_type; m.dim = d->dim;
            o.a0 = (float)m.a0; o.ap = (float)m.ap; o.aq = (float)m.aq; o.az = (float)m.az;
            o.b0 = (float)m.b0; o.bp = (float)m.bp; o.bq = (float)m.bq; o.bz = (float)m.bz;
            o.c0 = (float)m.c0; o.cp = (float)m.cp; o.cq = (float)m.cq; o.cz = (float)m.cz;
            o.Ru = (float)Ru; o.ku0 = (float)ku0; o.Rv = (float)Rv; o.lv0 = (float)lv0;
            o.ep0 = (float)(sw ? ey0 : ex0); o.eq0 = (float)(sw ? ex0 : ey0);
            o.pa = (float)(0.5 * (m.ap + m.aq)); o.pb = (float)(0.5 * (m.bp + m.bq));
            o.qa = (float)(0.5 * (m.ap - m.aq)); o.qb = (float)(0.5 * (m.bp - m.bq));
            o.haz = (float)(0.5 * m.az); o.hbz = (float)(0.5 * m.bz); o.hcz = (float)(0.5 * m.cz);
            o.untilted = untilted ? 1 : 0;
            {   // recon mode: depth weight numerator d * R (flat: d = -S.n; arc: in-plane distance of the origin)
                const V3 Sv = S;
                const double Sn = dot(Sv, n), Su = dot(Sv, u);
                o.recon_dR = (float)((d->det_type == 0 ? -Sn : std::sqrt(Sn * Sn + Su * Su)) * R);
            }
            o.swap_xy = sw ? 1 : 0;
            if (pass == 0) g->h_bp[i] = o;

            // ---- forward extras (computed for the fp ordering only) -------------------------------
            if (pass == 0 && swap) continue;     // fp copy of a swapped view is built in pass 1
            const double pitch[3] = {sw ? d->dy : d->dx, sw ? d->dx : d->dy, is3 ? d->dz : 1.0};
            const double Sn[3] = {S.x, S.y, S.z}, On[3] = {O.x, O.y, O.z};
            const double un[3] = {u.x, u.y, u.z}, vn[3] = {v.x, v.y, v.z}, nn[3] = {n.x, n.y, n.z};
            const int ax3[3] = {sw ? 1 : 0, sw ? 0 : 1, 2};
            double Sidx[3], Uidx[3], Vidx[3], Nidx[3];
            for (int c = 0; c < 3; ++c) {
                Sidx[c] = (Sn[ax3[c]] - On[ax3[c]]) / pitch[c];
                Uidx[c] = un[ax3[c]] / pitch[c];
                Vidx[c] = vn[ax3[c]] / pitch[c];
                Nidx[c] = nn[ax3[c]] / pitch[c];
            }
            if (!is3) { Sidx[2] = 0; Uidx[2] = 0; Nidx[2] = 0; Vidx[2] = 0; }
            o.Sp = (float)Sidx[0]; o.Sq = (float)Sidx[1]; o.Sz = (float)Sidx[2];
            if (d->det_type == 0) {
                // dir = (D - S) + s u + t v,  s = (kf - nu/2) du, t = (lf - nv/2) dv
                const double DSn[3] = {DS.x, DS.y, DS.z};
                o.Dp = (float)(DSn[ax3[0]] / pitch[0]); o.Dq = (float)(DSn[ax3[1]] / pitch[1]);
                o.Dz = (float)(is3 ? DSn[2] / pitch[2] : 0.0);
                o.Up = (float)(Uidx[0] * d->du); o.Uq = (float)(Uidx[1] * d->du); o.Uz = (float)(Uidx[2] * d->du);
                o.Vp = (float)(Vidx[0] * d->dv); o.Vq = (float)(Vidx[1] * d->dv); o.Vz = (float)(Vidx[2] * d->dv);
                o.ku0c = (float)(0.5 * d->nu); o.lv0c = (float)(0.5 * d->nv);
            } else {
                // dir = R sin(g) u + R cos(g) n + (t + Dv) v,  g = (kf - nu/2)/Ru, t + Dv = (lf - lv0) dv
                o.Up = (float)(Uidx[0] * R); o.Uq = (float)(Uidx[1] * R); o.Uz = (float)(Uidx[2] * R);
                o.Dp = (float)(Nidx[0] * R); o.Dq = (float)(Nidx[1] * R); o.Dz = (float)(Nidx[2] * R);
                o.Vp = (float)(Vidx[0] * d->dv); o.Vq = (float)(Vidx[1] * d->dv); o.Vz = (float)(Vidx[2] * d->dv);
                o.ku0c = (float)(0.5 * d->nu); o.lv0c = (float)lv0;
            }
            // bounds over the part of the volume that projects on or near the detector
            const int np = sw ? d->ny : d->nx, nq = sw ? d->nx : d->ny, nz = is3 ? d->nz : 1;
            const int NS = 9;
            double gp_min = 1e300, hk_max = 0, hl_max = 0, lpad_max = 0, zpad_max = 0;
            int used = 0;
            for (int sz = 0; sz < (is3 ? NS : 1); ++sz) for (int sq = 0; sq < NS; ++sq) for (int sp = 0; sp < NS; ++sp) {
                double p = (np - 1) * sp / double(NS - 1), q = (nq - 1) * sq / double(NS - 1);
                double z = is3 ? (nz - 1) * sz / double(NS - 1) : 0.0;
                double kc, lc;
                m.project(p, q, z, kc, lc);
                if (kc < -0.15 * d->nu - 4 || kc > 1.15 * d->nu + 4) continue;
                if (is3 && (lc < -0.15 * d->nv - 4 || lc > 1.15 * d->nv + 4)) continue;
                ++used;
                double k1, k2, l1, l2;
                m.project(p + 0.5, q, z, k1, l1); m.project(p - 0.5, q, z, k2, l2);
                gp_min = std::min(gp_min, std::fabs(k1 - k2));
                double klo = 1e300, khi = -1e300;
                for (int s1 = -1; s1 <= 1; s1 += 2) for (int s2 = -1; s2 <= 1; s2 += 2) {
                    m.project(p + 0.5 * s1, q + 0.5 * s2, z, k1, l1);
                    klo = std::min(klo, k1); khi = std::max(khi, k1);
                }
                hk_max = std::max(hk_max, std::max(khi - kc, kc - klo));
                if (is3) {
                    m.project(p, q, z + 0.5, k1, l1); m.project(p, q, z - 0.5, k2, l2);
                    const double hl_rect = std::max(std::fabs(l1 - lc), std::fabs(l2 - lc));
                    const double rows_per_z = std::fabs(l1 - l2);                 // rows one voxel spans along z
                    hl_max = std::max(hl_max, hl_rect);
                    if (d->algo == CT_ALGO_SFTT) {
                        // SF-TT (R27): the axial trapezoid's vertices are the rows of the in-plane chord's ends at z -+ 1/2
                        const double ep = p + (sw ? ey0 : ex0), eq = q + (sw ? ex0 : ey0);
                        const double hm = 0.5 / std::max(std::fabs(ep), std::fabs(eq));
                        double hl_trap = 0.0;
                        for (int sn = -1; sn <= 1; sn += 2) for (int sz = -1; sz <= 1; sz += 2) {
                            m.project(p + sn * ep * hm, q + sn * eq * hm, z + 0.5 * sz, k1, l1);
                            hl_trap = std::max(hl_trap, std::fabs(l1 - lc));
                        }
                        hl_max = std::max(hl_max, hl_trap);
                        const double extra = std::max(0.0, hl_trap - hl_rect);
                        lpad_max = std::max(lpad_max, extra);
                        zpad_max = std::max(zpad_max, extra / std::max(rows_per_z, 1e-6));
                    }
                }
            }
            // lane stride of the forward kernel: voxels p and p + stride must project >= 1 cell apart
            // (the kernel re-checks at run time and serialises if the bound is ever violated)
            int stride = 1;
            if (used > 0) {
                const double gp = gp_min / 1.10;           // margin for variation between samples
                stride = gp > 1e-6 ? (int)std::min<double>(np, std::ceil(1.02 / gp)) : np;
            } else {
                hk_max = 1.0; hl_max = 1.0;      // nothing of this view reaches the detector
            }
            o.lane_stride = std::max(stride, 1);
            o.ek = (float)(hk_max * 1.10 + 0.05);
            o.el = (float)(is3 ? hl_max * 1.10 + 0.05 : 0.0);
            // testing aid (CtsfDebug::tt_pad, read when the geometry is created): extra rows / voxels on top of the
            // sampled SF-TT margins -- a result that changes with it beyond summation order means they were too small
            const double tt_pad = g_ctsf_debug.tt_pad;
            o.lpad = (float)(d->algo == CT_ALGO_SFTT && is3 ? lpad_max * 1.25 + 0.1 + tt_pad : 0.0);
            o.zpad = (float)(d->algo == CT_ALGO_SFTT && is3 ? zpad_max * 1.25 + 0.1 + tt_pad : 0.0);
            g->h_bp[i].lpad = o.lpad;                  // the backprojector's brick shadow uses the same margin
            // columns / rows one footprint can span: floor(kc+t3) - floor(kc+t0) + 1 <= 2 ek + 2
            if (2.0 * o.ek + 2.0 > 6.0 || 2.0 * o.el + 2.0 > 8.0) small_fp = 0;
            g->h_fp[i] = o;
        }
    }
    g->fp_hoist_ok = (is3 && g->all_untilted && small_fp) ? 1 : 0;
    return CT_OK;
}
