"""Oracle pins, part 2: analytic chords (P7), identities (P8), reductions (P9, P11), adjoint and
dense transpose (P12, P13), symmetries (P14).  See tests/test_oracle_pins.py for the preamble."""
import math

import numpy as np
import pytest

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import workloads as W
from test_oracle_pins import geom2d, geom3d, _cell_points


def _ellipsoid_chords(S, P, centre, semi, alpha=0.0):
    """Chord lengths of rays S->P through an ellipsoid rotated by alpha about z (textbook quadratic)."""
    ca, sa = math.cos(alpha), math.sin(alpha)
    Rm = np.array([[ca, sa, 0.0], [-sa, ca, 0.0], [0.0, 0.0, 1.0]])
    d = P - S[None, :]
    d = d / np.linalg.norm(d, axis=1)[:, None]
    dd = (Rm @ d.T).T / semi[None, :]
    oo = (Rm @ (S - centre)) / semi
    A = np.sum(dd * dd, axis=1)
    B = 2.0 * dd @ oo
    C = oo @ oo - 1.0
    disc = B * B - 4.0 * A * C
    return np.where(disc > 0, np.sqrt(np.maximum(disc, 0.0)) / A, 0.0)


def _raster(g, centre, semi, alpha, mu, ss):
    """Area/volume-fraction rasterisation with ss^dim sub-samples per voxel."""
    sub = (np.arange(ss) + 0.5) / ss - 0.5
    def axis(n, d):
        return ((np.arange(n) - 0.5 * (n - 1))[:, None] + sub[None, :]).ravel() * d
    x, y = axis(g["nx"], g["dx"]), axis(g["ny"], g["dy"])
    ca, sa = math.cos(alpha), math.sin(alpha)
    X, Y = x[None, :] - centre[0], y[:, None] - centre[1]
    q2 = ((ca * X + sa * Y) / semi[0]) ** 2 + ((-sa * X + ca * Y) / semi[1]) ** 2
    if g["dim"] == 2:
        ins = (q2 <= 1.0).astype(np.float64)
        return mu * ins.reshape(g["ny"], ss, g["nx"], ss).mean(axis=(1, 3))[None]
    z = axis(g["nz"], g["dz"])
    out = np.zeros((g["nz"], g["ny"], g["nx"]))
    for i, zz in enumerate(z):
        ins = (q2 + ((zz - centre[2]) / semi[2]) ** 2 <= 1.0).astype(np.float64)
        out[i // ss] += ins.reshape(g["ny"], ss, g["nx"], ss).mean(axis=(1, 3)) / ss
    return mu * out


def _analytic_proj(g, centre, semi, alpha, mu, ns):
    sub = (np.arange(ns) + 0.5) / ns - 0.5
    nv = g["nv"]
    out = np.zeros((g["src"].shape[0], nv, g["nu"]))
    s = ((np.arange(g["nu"]) - 0.5 * (g["nu"] - 1))[:, None] + sub[None, :]).ravel() * g["du"]
    for i in range(out.shape[0]):
        for l in range(nv):
            if g["dim"] == 3:
                t = ((l - 0.5 * (nv - 1)) + sub) * g["dv"]
                ss_, tt = [a.ravel() for a in np.meshgrid(s, t)]
            else:
                ss_, tt = s, np.zeros_like(s)
            ch = _ellipsoid_chords(g["src"][i], _cell_points(g, i, ss_, tt), centre, semi, alpha)
            if g["dim"] == 3:
                out[i, l] = ch.reshape(ns, g["nu"], ns).mean(axis=(0, 2))
            else:
                out[i, l] = ch.reshape(g["nu"], ns).mean(axis=1)
    return mu * out


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_p7_disk_and_ellipse_2d(det):
    theta = [0.0, 0.5, 1.3, 2.9, 4.4]
    # centred disk: y = 2 mu sqrt(r^2 - SOD^2 sin^2 gamma): every view identical, closed form
    g = geom2d(theta, det)
    disk = _raster(g, (0.0, 0.0), np.array([40.0, 40.0]), 0.0, 0.02, 8)
    y = Oracle(g).fp(disk)[:, 0, :]
    sub = (np.arange(64) + 0.5) / 64 - 0.5
    s = ((np.arange(256) - 127.5)[:, None] + sub[None, :]) * 1.0
    gam = np.arctan(s / 1000.0) if det == "flat" else s / 1000.0
    ref = (2 * 0.02 * np.sqrt(np.maximum(40.0 ** 2 - (500.0 * np.sin(gam)) ** 2, 0.0))).mean(axis=1)
    for i in range(len(theta)):
        assert _rel(y[i], ref) < 1e-2
    assert abs(y.sum(axis=1) / ref.sum() - 1.0).max() < 2e-4
    # off-centre rotated ellipse at two resolutions: error <= 2e-2 at config-1 sampling, drops >= 2.5x
    errs = []
    for n, d in ((128, 1.0), (256, 0.5)):
        g = geom2d(theta, det, nx=n, ny=n, dx=d)
        args = ((12.0, -7.0, 0.0), np.array([37.0, 18.0, 1.0]), 0.6, 0.02)
        y = Oracle(g).fp(_raster(g, *args, 8))
        errs.append(_rel(y, _analytic_proj(g, np.array(args[0]), args[1], args[2], args[3], 32)))
    assert errs[0] < 2e-2 and errs[0] / errs[1] > 2.5, errs


def test_p7_ellipsoid_3d():
    theta = [0.2, 1.7, 3.3]
    errs, mass = [], []
    args = (np.array([3.0, -2.0, 1.5]), np.array([14.0, 9.0, 11.0]), 0.5, 0.02)
    for n, d in ((48, 1.0), (96, 0.5)):
        g = geom3d(theta, "flat", n=(n, n, n), d=(d, d, d), nu=96, nv=96, du=0.8, dv=0.8)
        y = Oracle(g).fp(_raster(g, *args, 4))
        ref = _analytic_proj(g, *args, 6)
        errs.append(_rel(y, ref))
        mass.append(y.sum() / ref.sum())
    assert errs[1] < 2e-2 and errs[0] / errs[1] > 2.5, errs
    assert abs(mass[1] - 1.0) < 1e-4, mass


def test_p8_mass_identities():
    g = geom3d([0.9], "flat")
    o = Oracle(g)
    for ijk in [(128, 128, 128), (40, 200, 30), (250, 3, 250), (0, 0, 255)]:
        f = o.footprint(0, *ijk)
        if f is None or f["k_lo"] == 0 or f["k_hi"] == g["nu"] - 1 or f["l_lo"] == 0 or f["l_hi"] == g["nv"] - 1:
            continue
        tau = f["tau"]
        assert abs(f["F1"].sum() * g["du"] - 0.5 * (tau[3] + tau[2] - tau[1] - tau[0])) < 1e-12
        c = (np.array(ijk) - 127.5) * 0.5
        t0 = o.det_coords(0, c - [0, 0, 0.25])[1]
        t1 = o.det_coords(0, c + [0, 0, 0.25])[1]
        assert abs(f["F2"].sum() * g["dv"] - abs(t1 - t0)) < 1e-12
    # parallel limit: sum_kl w du dv = dx dy dz M^2 with M -> 1
    g = geom3d([0.7], "flat", sad=1e9, sdd=1e9 + 1.0)
    f = Oracle(g).footprint(0, 100, 140, 120)
    assert abs(f["w"].sum() * 0.64 / 0.125 - 1.0) < 1e-6      # float64 at 1e9 mm: ~1e-7


def test_p9_2d_equals_one_slice_3d():
    theta = 2 * np.pi * np.arange(7) / 7
    g2 = geom2d(theta, "flat", nx=24, ny=24, dx=2.0, nu=40, du=3.0)
    g3 = dict(g2, dim=3, nz=1, dz=10.0, nv=1, dv=1.0)
    rng = np.random.default_rng(3)
    x = rng.uniform(0, 1, (1, 24, 24))
    y2, y3 = Oracle(g2).fp(x), Oracle(g3).fp(x)
    assert np.abs(y2 - y3).max() <= 1e-13 * np.abs(y2).max()
    g2a, g3a = dict(g2, det_type="arc"), dict(g3, det_type="arc")
    assert np.abs(Oracle(g2a).fp(x) - Oracle(g3a).fp(x)).max() <= 1e-13 * np.abs(y2).max()
    assert np.abs(Oracle(g2a).fp(x) - y2).max() > 1e-4        # arc really differs from flat


def test_p11_parallel_limit_column_sums():
    n = 16
    src, dc, u, v = W.trajectory(1, 1e9, 1e9 + 1.0, "flat", np.array([0.0]))
    g = dict(dim=2, nx=n, ny=n, nz=1, dx=1.5, dy=1.5, dz=1.0, ox=0.0, oy=0.0, oz=0.0, nu=n, nv=1,
             du=1.5, dv=1.0, det_type="flat", src=src, det_center=dc, det_u=u, det_v=v)
    x = np.random.default_rng(5).uniform(0, 1, (1, n, n))
    y = Oracle(g).fp(x)[0, 0]
    assert np.allclose(y, 1.5 * x[0].sum(axis=0), rtol=1e-6, atol=0)
    # 45 degrees, dx = dy: each pixel's footprint is a triangle of area dx^2
    src, dc, u, v = W.trajectory(1, 1e9, 1e9 + 1.0, "flat", np.array([np.pi / 4]))
    g = dict(g, src=src, det_center=dc, det_u=u, det_v=v, nu=64, du=0.4)
    f = Oracle(g).footprint(0, 5, 9)
    assert abs(f["w"].sum() * 0.4 - 1.5 ** 2) < 1e-6 * 2.25
    assert abs(f["tau"][2] - f["tau"][1]) < 1e-6 and abs(f["amp"] - math.sqrt(2) * 1.5) < 1e-6


def _small(index):
    shr = {1: dict(nx=20, ny=18, nu=30, n_views=7),
           2: dict(nx=14, ny=12, nz=10, nu=22, nv=18, n_views=5),
           3: dict(nx=16, ny=16, nz=6, nu=40, nv=7, n_views=6),
           4: dict(nx=12, ny=12, nz=12, nu=14, nv=14, n_views=6),
           5: dict(nx=18, ny=18, nu=25, n_views=8, batch=2)}[index]
    return W.make_config(index, **shr)


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_p12_adjoint(index):
    c = _small(index)
    o = Oracle(W.geom_keys(c))
    rng = np.random.default_rng(index)
    x = rng.uniform(0, 1, (c["nz"], c["ny"], c["nx"]))
    y = rng.uniform(0, 1, (c["n_views"], c["nv"], c["nu"]))
    Ax, Aty = o.fp(x), o.bp(y)
    lhs, rhs = np.vdot(Ax, y), np.vdot(x, Aty)
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    assert lhs > 0
    if index in (3, 4):          # these shapes clip footprints at the detector edge (R12)
        live = o.live_fraction(1, 1)
        assert live < 0.999
    # view subsets and listed voxels agree with the full operators
    sel = np.array([c["n_views"] - 1, 0, 2])
    assert np.array_equal(o.fp(x, sel), Ax[sel])
    ijk = np.array([[1, 2, 0], [c["nx"] - 1, c["ny"] - 1, c["nz"] - 1], [3, 0, c["nz"] // 2]])
    got = o.bp_voxels(y, ijk)
    assert np.allclose(got, Aty[ijk[:, 2], ijk[:, 1], ijk[:, 0]], rtol=1e-14, atol=0)
    assert np.allclose(o.bp_voxels(y.astype(np.float32), ijk),
                       o.bp(y.astype(np.float32))[ijk[:, 2], ijk[:, 1], ijk[:, 0]], rtol=1e-14)


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_p13_dense_matrix(det):
    theta = 2 * np.pi * np.arange(5) / 5
    g = geom2d(theta, det, nx=8, ny=8, dx=4.0, nu=16, du=5.0, sad=200.0, sdd=400.0)
    o = Oracle(g)
    A = np.zeros((5 * 16, 64))
    for j in range(64):
        e = np.zeros(64)
        e[j] = 1.0
        A[:, j] = o.fp(e.reshape(1, 8, 8)).ravel()
    assert A.min() >= -1e-14 and A.max() > 1.0        # G differences round to ~-2e-15 at worst
    y = np.random.default_rng(7).uniform(0, 1, (5, 1, 16))
    assert np.abs(o.bp(y).ravel() - A.T @ y.ravel()).max() < 1e-13
    x = np.random.default_rng(8).uniform(0, 1, (1, 8, 8))
    assert np.abs(o.fp(x).ravel() - A @ x.ravel()).max() < 1e-13


def test_p14_symmetries():
    # 4-fold symmetric centred phantom: views at multiples of 90 degrees are identical
    theta = np.pi / 2 * np.arange(4)
    g = geom2d(theta, "flat", nx=32, ny=32, dx=2.0, nu=60, du=2.5)
    rng = np.random.default_rng(11)
    q = rng.uniform(0, 1, (16, 16))
    top = np.hstack([q, np.rot90(q, -1)])
    x = np.vstack([np.rot90(top, 2), top])[None]
    x = 0.25 * (x + np.rot90(x, 1, (1, 2)) + np.rot90(x, 2, (1, 2)) + np.rot90(x, 3, (1, 2)))
    y = Oracle(g).fp(x)
    for i in range(1, 4):
        assert np.abs(y[i] - y[0]).max() < 1e-12
    # linearity and length scaling
    x2 = rng.uniform(0, 1, (1, 32, 32))
    o = Oracle(g)
    assert np.abs(o.fp(2.0 * x + 3.0 * x2) - (2.0 * o.fp(x) + 3.0 * o.fp(x2))).max() < 1e-11
    gs = geom2d(theta, "flat", nx=32, ny=32, dx=6.0, nu=60, du=7.5, sad=1500.0, sdd=3000.0)
    assert np.abs(Oracle(gs).fp(x2) - 3.0 * o.fp(x2)).max() < 1e-11
    # z-mirror symmetry with the source in the mid-plane: y[i, l, k] = y[i, nv-1-l, k]
    g3 = geom3d([0.3, 2.0], "arc", n=(12, 12, 10), d=(4.0, 4.0, 3.0), nu=24, nv=16, du=5.0, dv=4.0)
    x3 = rng.uniform(0, 1, (10, 12, 12))
    x3 = 0.5 * (x3 + x3[::-1])
    y3 = Oracle(g3).fp(x3)
    assert np.abs(y3 - y3[:, ::-1, :]).max() < 1e-12
    # u-mirror: centred disk-like (x-symmetric) phantom at theta = 0 is symmetric in k
    xs = rng.uniform(0, 1, (1, 32, 32))
    xs = 0.5 * (xs + xs[:, :, ::-1])
    y0 = Oracle(geom2d([0.0], "flat", nx=32, ny=32, dx=2.0, nu=60, du=2.5)).fp(xs)[0, 0]
    assert np.abs(y0 - y0[::-1]).max() < 1e-12
