"""Pins for the oracle's distance-driven model (reading R26).  PAPER.md:103 says
only that DD "consider[s] a ... face-based voxel model" and that its strict adjoint is implemented; the reading is
the textbook distance-driven construction written with the detector as the common axis: the voxel is its central
face perpendicular to the axis the ray mostly runs along, the face's edges project to a rectangle, a cell's
weight is its overlap with that rectangle divided by the cell size, times the slab thickness along the ray.
CPU only (-m "not gpu")."""
import math

import numpy as np
import pytest

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import workloads as W
from test_oracle_pins import geom2d, geom3d, _cell_points
from test_oracle_pins2 import _raster, _analytic_proj, _rel, _small


def dd(g):
    return dict(g, algo="DD")


def test_dd_hand_worked_2d():
    """Config-1 geometry, view theta = 0: S = (0, 500), detector at y = -500, u = (1, 0).  Pixel (64, 64) has
    centre (0.5, 0.5); the ray runs along y, so the face is the segment x in [0, 1] at y = 0.5, whose ends project
    to s = 1000 x / 499.5 = {0, 2.002002...}; amplitude = |e| dy/|e_y| = sqrt(0.25 + 499.5^2)/499.5."""
    o = Oracle(dd(geom2d([0.0])))
    f = o.footprint(0, 64, 64)
    s_b = 1000.0 / 499.5
    amp = math.hypot(0.5, 499.5) / 499.5
    assert np.allclose(f["tau"], [0.0, 0.0, s_b, s_b], atol=1e-12)
    assert abs(f["amp"] - amp) < 1e-12
    assert (f["k_lo"], f["k_hi"]) == (128, 130)
    assert np.allclose(f["w"][0], [amp, amp, amp * (s_b - 2.0)], rtol=1e-11)
    # a pixel whose ray runs mostly along x (view 90 degrees): the face is the y segment
    o = Oracle(dd(geom2d([math.pi / 2])))
    f = o.footprint(0, 64, 64)            # S = (-500, 0): e = (500.5, 0.5): along x
    assert abs(f["amp"] - math.hypot(500.5, 0.5) / 500.5) < 1e-12
    assert abs((f["tau"][2] - f["tau"][0]) - 1000.0 / 500.5) < 1e-9


def test_dd_exact_tie_takes_the_face_across_y():
    """R26's tie rule: when dx/|e_x| == dy/|e_y| exactly, the ray counts as running along y and the voxel is its face
    across y, the segment x_c -+ dx/2 at y_c.  Source at (400.5, 400.5), pixel (64, 64) centred at (0.5, 0.5): e =
    (-400, -400) in exact arithmetic.  n = -(1, 1)/sqrt(2), u = (1, -1)/sqrt(2), R = 1200: the segment's ends (0, 0.5)
    and (1, 0.5) project to s = R b / a = 1200 (-0.5)/800.5 and 1200 (0.5)/799.5; the OTHER face, (0.5, 0) - (0.5, 1),
    would give the mirror image, 1200 (0.5)/800.5 and 1200 (-0.5)/799.5 -- 1e-3 mm away."""
    r2 = math.sqrt(0.5)
    S = np.array([[400.5, 400.5, 0.0]])
    n = np.array([-r2, -r2, 0.0])
    g = dict(dim=2, nx=128, ny=128, nz=1, dx=1.0, dy=1.0, dz=1.0, ox=0.0, oy=0.0, oz=0.0, nu=64, nv=1, du=0.25, dv=1.0,
             det_type="flat", src=S, det_center=S + 1200.0 * n, det_u=np.array([[r2, -r2, 0.0]]),
             det_v=np.array([[0.0, 0.0, 1.0]]), algo="DD")
    f = Oracle(g).footprint(0, 64, 64)
    want = [1200.0 * -0.5 / 800.5, 1200.0 * 0.5 / 799.5]
    assert np.allclose(f["tau"], [want[0], want[0], want[1], want[1]], atol=1e-12, rtol=0.0)
    assert abs(want[1] + want[0]) > 9e-4                 # the two faces are distinguishable here
    assert abs(f["amp"] - math.sqrt(2.0)) < 1e-12        # |e| dy/|e_y| = 400 sqrt(2) / 400


def test_dd_parallel_limit_is_exact():
    """Parallel beam along y with nu = nx, du = dx: distance-driven projection is exactly dy x column sums;
    at 45 degrees with dx = dy the face model gives each pixel a rectangle of width dx/sqrt(2) and amplitude
    sqrt(2) dx (area dx^2)."""
    n = 16
    src, dc, u, v = W.trajectory(1, 1e9, 1e9 + 1.0, "flat", np.array([0.0]))
    g = dict(dim=2, nx=n, ny=n, nz=1, dx=1.5, dy=1.5, dz=1.0, ox=0.0, oy=0.0, oz=0.0, nu=n, nv=1,
             du=1.5, dv=1.0, det_type="flat", src=src, det_center=dc, det_u=u, det_v=v, algo="DD")
    x = np.random.default_rng(5).uniform(0, 1, (1, n, n))
    assert np.allclose(Oracle(g).fp(x)[0, 0], 1.5 * x[0].sum(axis=0), rtol=1e-6, atol=0)
    src, dc, u, v = W.trajectory(1, 1e9, 1e9 + 1.0, "flat", np.array([np.pi / 4 - 1e-3]))
    g = dict(g, src=src, det_center=dc, det_u=u, det_v=v, nu=64, du=0.4)
    f = Oracle(g).footprint(0, 5, 9)
    assert abs(f["w"].sum() * 0.4 - 1.5 ** 2) < 2e-3 * 2.25
    assert abs(f["amp"] - math.sqrt(2) * 1.5) < 3e-3 and abs(f["tau"][1] - f["tau"][0]) < 1e-12


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_dd_face_model_brute_force(det):
    """The model itself, by brute force: points spread uniformly over the voxel's central face are projected and
    binned into cells; distance-driven assumes the face's image is uniform on the detector, which holds up to the
    variation of the magnification across one voxel (O(voxel/SAD))."""
    g = dd(geom3d([0.4, 1.9, 3.0], det, n=(64, 64, 64), d=(2.0, 2.0, 2.0), nu=96, nv=96, du=3.2, dv=3.2))
    o = Oracle(g)
    rng = np.random.default_rng(0)
    for view, ijk in [(0, (40, 20, 32)), (1, (10, 50, 33)), (2, (50, 12, 60))]:
        f = o.footprint(view, *ijk)
        c = np.array([(ijk[0] - 31.5) * 2.0, (ijk[1] - 31.5) * 2.0, (ijk[2] - 31.5) * 2.0])
        e = c - g["src"][view]
        along_y = 2.0 * abs(e[0]) <= 2.0 * abs(e[1])
        n = 400000
        pts = np.tile(c, (n, 1))
        pts[:, 0 if along_y else 1] += rng.uniform(-1.0, 1.0, n)
        pts[:, 2] += rng.uniform(-1.0, 1.0, n)
        st = np.array([o.det_coords(view, p) for p in pts[:2000]])          # spot-check the helper on a subset
        S, D, u, v = g["src"][view], g["det_center"][view], g["det_u"][view], g["det_v"][view]
        nn = np.cross(u, v)
        nn = -nn if np.dot(D - S, nn) < 0 else nn
        R = np.dot(D - S, nn)
        w = pts - S
        a, b, cc = w @ nn, w @ u, w @ v
        s = R * b / a - np.dot(D - S, u) if det == "flat" else R * np.arctan2(b, a)
        t = R * cc / a - np.dot(D - S, v) if det == "flat" else R * cc / np.hypot(a, b) - np.dot(D - S, v)
        assert np.allclose(st[:, 0], s[:2000], atol=1e-9) and np.allclose(st[:, 1], t[:2000], atol=1e-9)
        k = np.floor(s / 3.2 + 48).astype(int)
        l = np.floor(t / 3.2 + 48).astype(int)
        H = np.zeros((96, 96))
        np.add.at(H, (l, k), 1.0 / n)
        # model: share of the face's image that falls into each cell
        got = f["w"] / f["w"].sum()
        ref = H[f["l_lo"]:f["l_hi"] + 1, f["k_lo"]:f["k_hi"] + 1]
        assert abs(ref.sum() - 1.0) < 1e-9                                    # the footprint covers the whole image
        assert np.abs(got - ref).max() < 6e-3, np.abs(got - ref).max()


def test_dd_mass_and_identities():
    g = dd(geom3d([0.9], "flat"))
    o = Oracle(g)
    f = o.footprint(0, 100, 140, 90)
    # sum_k F1 du = s_b - s_a exactly (rectangle); separable: w = amp F1 (x) F2
    assert abs(f["F1"].sum() * 0.8 - (f["tau"][3] - f["tau"][0])) < 1e-12
    assert np.allclose(f["w"], f["amp"] * np.outer(f["F2"], f["F1"]), rtol=1e-15)
    colsum = f["w"].sum(axis=0) / f["amp"]                      # F1[k] * sum_l F2
    rowsum = f["w"].sum(axis=1) / f["amp"]
    total = f["w"].sum() / f["amp"]
    assert abs(colsum.sum() - total) < 1e-12 and abs(rowsum.sum() - total) < 1e-12
    # 2-D: sum_k w du = amp (s_b - s_a)
    g2 = dd(geom2d([0.3, 2.0]))
    for view, (ix, iy) in [(0, (64, 64)), (1, (20, 100))]:
        f = Oracle(g2).footprint(view, ix, iy)
        assert abs(f["w"].sum() * 1.0 - f["amp"] * (f["tau"][3] - f["tau"][0])) < 1e-12


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_dd_adjoint(index):
    c = _small(index)
    o = Oracle(dd(W.geom_keys(c)))
    rng = np.random.default_rng(index)
    x = rng.uniform(0, 1, (c["nz"], c["ny"], c["nx"]))
    y = rng.uniform(0, 1, (c["n_views"], c["nv"], c["nu"]))
    lhs, rhs = np.vdot(o.fp(x), y), np.vdot(x, o.bp(y))
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs) and lhs > 0


def test_dd_dense_matrix():
    theta = 2 * np.pi * np.arange(5) / 5
    g = dd(geom2d(theta, "flat", nx=8, ny=8, dx=4.0, nu=16, du=5.0, sad=200.0, sdd=400.0))
    o = Oracle(g)
    A = np.zeros((5 * 16, 64))
    for j in range(64):
        e = np.zeros(64)
        e[j] = 1.0
        A[:, j] = o.fp(e.reshape(1, 8, 8)).ravel()
    assert A.min() >= -1e-14 and A.max() > 1.0
    y = np.random.default_rng(7).uniform(0, 1, (5, 1, 16))
    assert np.abs(o.bp(y).ravel() - A.T @ y.ravel()).max() < 1e-13
    # it is a different matrix from SF's, with the same column sums to first order
    Asf = np.zeros_like(A)
    osf = Oracle(geom2d(theta, "flat", nx=8, ny=8, dx=4.0, nu=16, du=5.0, sad=200.0, sdd=400.0))
    for j in range(64):
        e = np.zeros(64)
        e[j] = 1.0
        Asf[:, j] = osf.fp(e.reshape(1, 8, 8)).ravel()
    assert np.abs(A - Asf).max() > 1e-2
    assert np.abs(A.sum(axis=0) / Asf.sum(axis=0) - 1.0).max() < 2e-2


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_dd_analytic_chords_2d(det):
    """Against closed-form chords of an off-centre rotated ellipse: distance-driven is less accurate than the
    separable footprint (rectangle instead of trapezoid) but converges with the pixel size."""
    theta = [0.0, 0.5, 1.3, 2.9, 4.4]
    errs = []
    for n, d in ((128, 1.0), (256, 0.5)):
        g = dd(geom2d(theta, det, nx=n, ny=n, dx=d))
        args = ((12.0, -7.0, 0.0), np.array([37.0, 18.0, 1.0]), 0.6, 0.02)
        y = Oracle(g).fp(_raster(g, *args, 8))
        errs.append(_rel(y, _analytic_proj(g, np.array(args[0]), args[1], args[2], args[3], 32)))
    assert errs[0] < 3e-2 and errs[0] / errs[1] > 2.0, errs


def test_dd_2d_equals_one_slice_3d():
    theta = 2 * np.pi * np.arange(7) / 7
    g2 = dd(geom2d(theta, "flat", nx=24, ny=24, dx=2.0, nu=40, du=3.0))
    g3 = dict(g2, dim=3, nz=1, dz=10.0, nv=1, dv=1.0)
    x = np.random.default_rng(2).uniform(0, 1, (1, 24, 24))
    y2, y3 = Oracle(g2).fp(x), Oracle(g3).fp(x)
    assert np.abs(y2 - y3).max() <= 1e-13 * np.abs(y2).max()
