"""Oracle pins, part 3: the places where one-line mutations of oracle/sf_oracle.c survived the earlier pins
(VERDICT round 1): the height at which the four transaxial corners are taken in a TILTED frame (reading R4; the
headline config 4 is the tilted case), the sign flip of make_frame when u x v points away from the detector,
and the arc detector in a tilted frame (reading R8; SURVEY 8(c) last pin row).  CPU only.

The detector model used here is an independent restatement: a world point is mapped to detector coordinates by
INTERSECTING the ray source -> point with the detector surface (plane / source-centred cylinder) and reading the
hit point's coordinates in the detector's own axes -- not the oracle's closed form R b / a - (D - S).u.
"""
import math

import numpy as np
import pytest

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import workloads as W

from test_oracle_pins import _brute_footprint, geom2d, geom3d


def _hit(g, view, P):
    """(s, t) [mm] of the point where the ray S -> P meets the detector of `view`."""
    S, D = g["src"][view], g["det_center"][view]
    u, v = g["det_u"][view], g["det_v"][view]
    n = np.cross(u, v)
    if np.dot(D - S, n) < 0:
        n = -n
    d = np.asarray(P, dtype=np.float64) - S
    if g["det_type"] == "flat":
        lam = np.dot(D - S, n) / np.dot(d, n)            # (S + lam d - D).n = 0
        H = S + lam * d
        return np.dot(H - D, u), np.dot(H - D, v)
    R = np.dot(D - S, n)
    dn, du_ = np.dot(d, n), np.dot(d, u)
    lam = R / math.hypot(dn, du_)                        # cylinder of radius R about the line S + R v
    H = S + lam * d
    ang = math.atan2(np.dot(H - S, u), np.dot(H - S, n))
    return R * ang, np.dot(H - D, v)


def _centre(g, ijk):
    return np.array([g["ox"] + (ijk[0] - 0.5 * (g["nx"] - 1)) * g["dx"],
                     g["oy"] + (ijk[1] - 0.5 * (g["ny"] - 1)) * g["dy"],
                     g["oz"] + (ijk[2] - 0.5 * (g["nz"] - 1)) * g["dz"] if g["dim"] == 3 else 0.0])


def _trap_integral(tau, a, b):
    """Integral over [a, b] of the unit-height trapezoid on tau, by exact piecewise-linear integration
    (Gauss-Legendre of order 2 on every piece between breakpoints)."""
    t0, t1, t2, t3 = tau

    def f(s):
        up = (s - t0) / (t1 - t0) if t1 > t0 else 1.0 * (s >= t0)
        dn = (t3 - s) / (t3 - t2) if t3 > t2 else 1.0 * (s <= t3)
        return max(0.0, min(1.0, up, dn)) if t0 <= s <= t3 else 0.0
    br = sorted(set([a, b] + [t for t in tau if a < t < b]))
    tot = 0.0
    for lo, hi in zip(br[:-1], br[1:]):
        m, h = 0.5 * (lo + hi), 0.5 * (hi - lo)
        tot += h * (f(m - h / math.sqrt(3.0)) + f(m + h / math.sqrt(3.0)))
    return tot


def _expected_footprint(g, view, ijk):
    """SF-TR weights of one voxel from the readings R1-R5 with the intersection model above: corners at the voxel
    MID-PLANE z = z_c, axial ends (x_c, y_c, z_c +- dz/2), amplitude along the centre ray."""
    Pc = _centre(g, ijk)
    hx, hy, hz = 0.5 * g["dx"], 0.5 * g["dy"], 0.5 * g["dz"]
    tau = sorted(_hit(g, view, Pc + np.array([sx * hx, sy * hy, 0.0]))[0] for sx in (-1, 1) for sy in (-1, 1))
    nu, nv, du, dv = g["nu"], g["nv"], g["du"], g["dv"]
    F1 = np.array([_trap_integral(tau, (k - 0.5 * nu) * du, (k + 1 - 0.5 * nu) * du) / du for k in range(nu)])
    if g["dim"] == 3:
        ta = _hit(g, view, Pc - np.array([0, 0, hz]))[1]
        tb = _hit(g, view, Pc + np.array([0, 0, hz]))[1]
        tlo, thi = min(ta, tb), max(ta, tb)
        F2 = np.array([max(0.0, min((l + 1 - 0.5 * nv) * dv, thi) - max((l - 0.5 * nv) * dv, tlo)) / dv
                       for l in range(nv)])
    else:
        F2 = np.ones(1)
    e = Pc - g["src"][view]
    amp = np.linalg.norm(e) * min(g["dx"] / abs(e[0]), g["dy"] / abs(e[1]))
    return np.array(tau), amp * np.outer(F2, F1)


def _expected_footprint_tt(g, view, ijk):
    """SF-TT weights of one voxel from reading R27 with the intersection model above: transaxial trapezoid and
    amplitude as SF-TR; the axial factor is the unit-height trapezoid whose four vertices are the row coordinates of
    the ends of the centre ray's in-plane chord, P_c -+ (l_theta / 2) e_xy / |e_xy|, taken at z_c - dz/2 and at
    z_c + dz/2.  Returns (xi, area of the trapezoid in rows, weights)."""
    Pc = _centre(g, ijk)
    hx, hy, hz = 0.5 * g["dx"], 0.5 * g["dy"], 0.5 * g["dz"]
    tau = sorted(_hit(g, view, Pc + np.array([sx * hx, sy * hy, 0.0]))[0] for sx in (-1, 1) for sy in (-1, 1))
    nu, nv, du, dv = g["nu"], g["nv"], g["du"], g["dv"]
    F1 = np.array([_trap_integral(tau, (k - 0.5 * nu) * du, (k + 1 - 0.5 * nu) * du) / du for k in range(nu)])
    e = Pc - g["src"][view]
    exy = e[:2] / np.hypot(e[0], e[1])
    l_theta = min(g["dx"] / abs(exy[0]), g["dy"] / abs(exy[1]))          # in-plane chord of the centre ray
    ends = [Pc + np.array([sn * 0.5 * l_theta * exy[0], sn * 0.5 * l_theta * exy[1], sz * hz])
            for sn in (-1, 1) for sz in (-1, 1)]
    xi = sorted(_hit(g, view, P)[1] for P in ends)
    F2 = np.array([_trap_integral(xi, (l - 0.5 * nv) * dv, (l + 1 - 0.5 * nv) * dv) / dv for l in range(nv)])
    amp = np.linalg.norm(e) * min(g["dx"] / abs(e[0]), g["dy"] / abs(e[1]))
    return np.array(xi), 0.5 * (xi[3] + xi[2] - xi[1] - xi[0]) / dv, amp * np.outer(F2, F1)


def _dense(f, nv, nu):
    w = np.zeros((nv, nu))
    w[f["l_lo"]:f["l_hi"] + 1, f["k_lo"]:f["k_hi"] + 1] = f["w"]
    return w


# ---- R4 / R6: corner height and the general frame, hand-worked through the intersection model -------------
@pytest.mark.parametrize("det", ["flat", "arc"])
def test_tilted_frame_footprint_from_ray_detector_intersection(det):
    """phi = 15 deg off-plane tilt, psi = 0.5 deg in-plane rotation, voxels far off the mid-plane: with a tilted
    frame the depth a depends on z, so corners taken at z_c -+ dz/2 instead of z_c move tau by ~1e-3 mm --
    1e9 times this test's tolerance."""
    g = geom3d([0.4, 2.5], det, n=(64, 64, 64), d=(2.0, 2.0, 2.0), nu=96, nv=96, du=3.2, dv=3.2,
               phi=np.radians([15.0, -15.0]), psi=np.radians([0.5, -0.5]))
    o = Oracle(g)
    for view, ijk in [(0, (40, 20, 50)), (1, (10, 50, 12)), (0, (30, 30, 5)), (1, (55, 9, 60))]:
        f = o.footprint(view, *ijk)
        tau, w = _expected_footprint(g, view, ijk)
        assert np.allclose(f["tau"], tau, atol=1e-11, rtol=0.0)
        assert np.abs(_dense(f, g["nv"], g["nu"]) - w).max() < 1e-12
    # and the corner height matters here: the same corners at z_c - dz/2 are measurably elsewhere
    Pc = _centre(g, (40, 20, 50))
    s_mid = _hit(g, 0, Pc + np.array([1.0, 1.0, 0.0]))[0]
    s_low = _hit(g, 0, Pc + np.array([1.0, 1.0, -1.0]))[0]
    assert abs(s_mid - s_low) > 1e-3


def test_tilted_frame_config4_shape():
    """The same at the headline config's own geometry (config 4 shrunk: sinusoidal tilt + seeded per-view jitter)."""
    c = W.make_config(4, nx=32, ny=32, nz=32, nu=48, nv=48, n_views=12)
    g = W.geom_keys(c)
    o = Oracle(g)
    rng = np.random.default_rng(3)
    checked = 0
    for view in (1, 4, 7, 10):
        for _ in range(3):
            ijk = tuple(int(v) for v in rng.integers(4, 28, 3))
            f = o.footprint(view, *ijk)
            if f is None:
                continue
            tau, w = _expected_footprint(g, view, ijk)
            assert np.allclose(f["tau"], tau, atol=1e-11, rtol=0.0)
            assert np.abs(_dense(f, g["nv"], g["nu"]) - w).max() < 1e-12
            checked += 1
    assert checked >= 8


# ---- R27: the trapezoid axial footprint (SF-TT), hand-worked through the intersection model ------------------
def _tt_geometry(det, algo="SF-TT"):
    """Short orbit (SAD 200, SDD 400), tall volume (z up to +-95 mm), tilted frames (phi = +-10 deg, psi = +-0.5 deg):
    the voxels used below see the source (itself 35 mm off the mid-plane) under polar angles of ~13 and ~25 degrees."""
    return dict(geom3d([0.4, 2.5], det, n=(40, 40, 96), d=(2.0, 2.0, 2.0), nu=128, nv=600, du=3.0, dv=1.0,
                       sad=200.0, sdd=400.0, phi=np.radians([10.0, -10.0]), psi=np.radians([0.5, -0.5])), algo=algo)


TT_VOXELS = [(0, (25, 14, 40)), (1, (12, 27, 7)), (0, (12, 27, 23)), (1, (25, 14, 76))]


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_sftt_footprint_from_ray_detector_intersection(det):
    """Reading R27 to 1e-12: chord ends at P_c -+ (l_theta/2) e_xy/|e_xy| (a half chord of 0.4 l_theta moves the weights
    by ~5 %), heights z_c -+ dz/2, vertices through the detector model of THIS file, trapezoid integrated piecewise.
    The first two voxels sit at ~13 degrees of polar angle, the last two at ~25."""
    g = _tt_geometry(det)
    o = Oracle(g)
    polar = []
    for view, ijk in TT_VOXELS:
        e = _centre(g, ijk) - g["src"][view]
        polar.append(math.degrees(math.atan2(abs(e[2]), math.hypot(e[0], e[1]))))
        f = o.footprint(view, *ijk)
        xi, _, w = _expected_footprint_tt(g, view, ijk)
        assert f is not None and 0 < f["l_lo"] and f["l_hi"] < g["nv"] - 1          # fully on the detector
        assert np.abs(_dense(f, g["nv"], g["nu"]) - w).max() < 1e-12
        # and it is not SF-TR's footprint: the rectangle between the rows of (x_c, y_c, z_c -+ dz/2) differs visibly
        w_tr = _expected_footprint(g, view, ijk)[1]
        assert np.abs(w - w_tr).max() > 0.02 * w.max(), np.abs(w - w_tr).max() / w.max()
        assert xi[1] - xi[0] > 0.05 * (xi[3] - xi[0])                              # real ramps at these angles
    assert 11.0 < polar[0] < 15.0 and 11.0 < polar[1] < 15.0 and 23.0 < polar[2] < 27.0 and 23.0 < polar[3] < 27.0


def test_sftt_axial_profile_is_the_chord_fraction_between_the_voxel_faces():
    """What R27's trapezoid stands for, by brute force, without its vertex formula: in the vertical plane through the
    source and the voxel centre, a ray of slope m = dz/drho crosses the voxel's in-plane chord rho_c -+ l_theta/2; the
    axial factor at that ray's detector row is the fraction of the chord on which the ray is between z_c - dz/2 and
    z_c + dz/2.  Untilted frame, flat detector (the row coordinate is then linear in m).  The trapezoid joins the
    exact values at its four vertices by straight lines where the truth is linear in 1/m: a per-cent-level difference
    at ~20 degrees; a wrong chord length or wrong face heights are tens of per cent."""
    g = dict(geom3d([0.4], "flat", n=(40, 40, 96), d=(2.0, 2.0, 2.0), nu=128, nv=1600, du=3.0, dv=0.25,
                    sad=200.0, sdd=400.0), algo="SF-TT")
    o = Oracle(g)
    view, ijk = 0, (24, 15, 82)
    f = o.footprint(view, *ijk)
    Pc, S = _centre(g, ijk), g["src"][view]
    e = Pc - S
    rho_c = math.hypot(e[0], e[1])
    exy = e[:2] / rho_c
    l_theta = min(g["dx"] / abs(exy[0]), g["dy"] / abs(exy[1]))
    t0 = _hit(g, view, S + np.array([exy[0], exy[1], 0.0]))[1]
    t1 = _hit(g, view, S + np.array([exy[0], exy[1], 1.0]))[1]            # row coordinate of slope 1

    def fraction(t):
        m = (t - t0) / (t1 - t0)
        lo, hi = sorted(((Pc[2] - 1.0 - S[2]) / m, (Pc[2] + 1.0 - S[2]) / m))          # dz/2 = 1 mm
        return max(0.0, min(hi, rho_c + 0.5 * l_theta) - max(lo, rho_c - 0.5 * l_theta)) / l_theta

    sub = (np.arange(8) + 0.5) / 8
    rows = np.arange(f["l_lo"], f["l_hi"] + 1)
    brute = np.array([np.mean([fraction((l - 0.5 * g["nv"] + u) * g["dv"]) for u in sub]) for l in rows])
    assert len(rows) > 20 and brute.max() > 0.99
    assert np.abs(f["F2"] - brute).max() < 0.02
    assert abs(f["F2"].sum() / brute.sum() - 1.0) < 5e-3


# ---- make_frame's sign flip: u x v pointing AWAY from the detector ------------------------------------------
@pytest.mark.parametrize("index,shrink", [(1, dict(nx=24, ny=24, nu=48, n_views=7)),
                                          (5, dict(nx=28, ny=28, nu=56, n_views=6, batch=1)),
                                          (2, dict(nx=14, ny=14, nz=10, nu=24, nv=20, n_views=5)),
                                          (3, dict(nx=16, ny=16, nz=6, nu=36, nv=8, n_views=5)),
                                          (4, dict(nx=12, ny=12, nz=12, nu=24, nv=24, n_views=6))])
def test_reversed_channel_axis_mirrors_the_projections(index, shrink):
    """det_u -> -det_u describes the same physical detector read out in the opposite channel order; u x v then
    points away from the detector and the frame normal must be flipped ((D - S).n > 0, SURVEY 8 Notation).
    y'[.., k] == y[.., nu-1-k] and A'^T y' == A^T y, to rounding."""
    c = W.make_config(index, **shrink)
    g = W.geom_keys(c)
    gm = dict(g, det_u=-g["det_u"])
    x = W.make_phantom(c)[0].astype(np.float64)
    o, om = Oracle(g), Oracle(gm)
    y, ym = o.fp(x), om.fp(x)
    assert np.abs(y).max() > 0
    assert np.abs(ym - y[..., ::-1]).max() < 1e-12 * np.abs(y).max()
    xb, xbm = o.bp(y), om.bp(np.ascontiguousarray(y[..., ::-1]))
    assert np.abs(xbm - xb).max() < 1e-12 * np.abs(xb).max()
    # one footprint, explicitly
    ijk = (c["nx"] // 3, c["ny"] // 2, c["nz"] // 2)
    f, fm = o.footprint(2, *ijk), om.footprint(2, *ijk)
    assert fm is not None and (fm["k_lo"], fm["k_hi"]) == (c["nu"] - 1 - f["k_hi"], c["nu"] - 1 - f["k_lo"])


def test_reversed_row_axis_mirrors_the_projections():
    """det_v -> -det_v: u x v flips as well; rows come out in the opposite order."""
    c = W.make_config(4, nx=12, ny=12, nz=12, nu=24, nv=24, n_views=6)
    g = W.geom_keys(c)
    gm = dict(g, det_v=-g["det_v"])
    x = W.make_phantom(c)[0].astype(np.float64)
    y, ym = Oracle(g).fp(x), Oracle(gm).fp(x)
    assert np.abs(ym - y[:, ::-1, :]).max() < 1e-12 * np.abs(y).max()


# ---- R8: arc detector in a tilted frame against exact ray / box chords (last pin row) ----------
def test_p6_brute_force_3d_tilted_arc():
    g = geom3d([0.4, 2.5], "arc", n=(64, 64, 64), d=(2.0, 2.0, 2.0), nu=96, nv=96, du=3.2, dv=3.2,
               phi=np.radians([15.0, -15.0]), psi=np.radians([0.5, -0.5]))
    o = Oracle(g)
    for view, ijk in [(0, (40, 20, 32)), (1, (10, 50, 40)), (0, (30, 30, 10))]:
        f = o.footprint(view, *ijk)
        ks = np.arange(f["k_lo"] - 1, f["k_hi"] + 2)
        ls = np.arange(f["l_lo"] - 1, f["l_hi"] + 2)
        bf = _brute_footprint(g, view, ijk, ks, ls, 120)
        w = np.zeros((len(ls), len(ks)))
        w[1:-1, 1:-1] = f["w"]
        assert np.abs(w - bf).max() < 1e-1 * bf.max()
        assert abs(w.sum() - bf.sum()) < 5e-3 * bf.sum()


def test_arc_equals_flat_to_second_order_near_the_detector_centre():
    """Near the piercing point of the central ray the arc (s = R atan(b/a), t = R c / rho) and the flat detector
    (s = R b/a, t = R c/a) agree to O(gamma^2): a voxel on the central ray gets the same footprint to 1e-5, in a
    tilted frame as well -- a transposed atan2 or a wrong radius in the arc branch breaks this."""
    kw = dict(n=(33, 33, 33), d=(1.0, 1.0, 1.0), nu=64, nv=64, du=1.5, dv=1.5,
              phi=np.radians([10.0]), psi=np.radians([0.3]))
    gf, ga = geom3d([0.9], "flat", **kw), geom3d([0.9], "arc", **kw)
    ff, fa = Oracle(gf).footprint(0, 16, 16, 16), Oracle(ga).footprint(0, 16, 16, 16)
    assert (ff["k_lo"], ff["k_hi"], ff["l_lo"], ff["l_hi"]) == (fa["k_lo"], fa["k_hi"], fa["l_lo"], fa["l_hi"])
    assert np.abs(ff["w"] - fa["w"]).max() < 1e-5 * ff["w"].max()
