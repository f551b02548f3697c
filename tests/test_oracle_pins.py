"""Pins for the float64 CPU oracle (oracle/sf_oracle.c) against what the mathematics fixes.

Each test is chosen so that a plausible mistake in the oracle (dropped term, wrong sign or index,
transposed operand, wrong half-sample convention) fails at least one of them.  None of them calls
the CUDA path.  Pin numbers refer to SURVEY.md 8(c) / DESIGN.md "Oracle pins".
"""
import math
import os

import numpy as np
import pytest

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def geom2d(theta, det="flat", nx=128, ny=128, dx=1.0, nu=256, du=1.0, sad=500.0, sdd=1000.0):
    theta = np.atleast_1d(np.asarray(theta, dtype=np.float64))
    src, dc, u, v = W.trajectory(len(theta), sad, sdd, det, theta)
    return dict(dim=2, nx=nx, ny=ny, nz=1, dx=dx, dy=dx, dz=1.0, ox=0.0, oy=0.0, oz=0.0,
                nu=nu, nv=1, du=du, dv=1.0, det_type=det, src=src, det_center=dc, det_u=u, det_v=v)


def geom3d(theta, det="flat", n=(256, 256, 256), d=(0.5, 0.5, 0.5), nu=384, nv=384, du=0.8, dv=0.8,
           sad=600.0, sdd=1200.0, phi=None, psi=None):
    theta = np.atleast_1d(np.asarray(theta, dtype=np.float64))
    src, dc, u, v = W.trajectory(len(theta), sad, sdd, det, theta, phi, psi)
    return dict(dim=3, nx=n[0], ny=n[1], nz=n[2], dx=d[0], dy=d[1], dz=d[2], ox=0.0, oy=0.0, oz=0.0,
                nu=nu, nv=nv, du=du, dv=dv, det_type=det, src=src, det_center=dc, det_u=u, det_v=v)


# ---- P1: trapezoid CDF vs quadrature ---------------------------------------------------------
def _trap(tau, s):
    t0, t1, t2, t3 = tau
    up = np.where(t1 > t0, (s - t0) / np.where(t1 > t0, t1 - t0, 1.0), (s >= t0) * 1.0)
    dn = np.where(t3 > t2, (t3 - s) / np.where(t3 > t2, t3 - t2, 1.0), (s <= t3) * 1.0)
    return np.clip(np.minimum(up, dn), 0.0, 1.0) * (s >= t0) * (s <= t3)


def test_p1_trap_cdf_vs_quadrature():
    rng = np.random.default_rng(1)
    for case in range(40):
        tau = np.sort(rng.uniform(-3, 3, 4))
        if case % 4 == 1:
            tau[1] = tau[0]
        if case % 4 == 2:
            tau[3] = tau[2]
        if case % 4 == 3:
            tau[1] = tau[0]
            tau[3] = tau[2]
        for _ in range(5):
            a, b = np.sort(rng.uniform(-4, 4, 2))
            # integrate piecewise between the breakpoints with Gauss-Legendre (exact for degree 1)
            br = np.unique(np.clip(np.concatenate([[a, b], tau]), a, b))
            xg, wg = np.polynomial.legendre.leggauss(4)
            q = 0.0
            for lo, hi in zip(br[:-1], br[1:]):
                xm = 0.5 * (hi + lo) + 0.5 * (hi - lo) * xg
                q += 0.5 * (hi - lo) * np.sum(wg * _trap(tau, xm))
            got = Oracle.trap_cdf(tau, b) - Oracle.trap_cdf(tau, a)
            assert abs(got - q) < 1e-10
    # total area and monotonicity
    tau = np.array([-1.0, -0.25, 0.5, 2.0])
    assert abs(Oracle.trap_cdf(tau, 10.0) - 0.5 * (tau[3] + tau[2] - tau[1] - tau[0])) < 1e-15
    assert Oracle.trap_cdf(tau, -1.0) == 0.0


# ---- P2/P3: hand-worked and probe 2-D footprints -------------------------------------------
def test_p2_hand_worked_2d():
    # theta = 0: S = (0, 500), u = (1, 0), n = (0, -1).  Pixel (64, 64): centre (0.5, 0.5), corners
    # x in {0, 1}, y in {0, 1}; a = 500 - y, b = x, s = 1000 b / a -> {0, 0, 1000/500, 1000/499}.
    o = Oracle(geom2d(0.0))
    f = o.footprint(0, 64, 64)
    assert np.allclose(f["tau"], [0.0, 0.0, 2.0, 1000.0 / 499.0], atol=1e-12)
    amp = math.hypot(0.5, 499.5) * min(1.0 / 0.5, 1.0 / 499.5)
    assert abs(f["amp"] - amp) < 1e-12
    # cell k spans [k - 128, k - 127] mm: bins 128, 129 sit on the plateau, bin 130 holds the ramp
    assert (f["k_lo"], f["k_hi"]) == (128, 130)
    expect = amp * np.array([1.0, 1.0, 0.5 * (1000.0 / 499.0 - 2.0)])
    assert np.allclose(f["w"][0], expect, atol=1e-12)
    assert np.allclose(f["w"][0], [1.000000501, 1.000000501, 0.002004009], atol=1e-9)


def test_p3_golden_2d():
    for line in open(os.path.join(GOLD, "sf_footprints_2d.txt")):
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        det, theta, ix, iy, k0 = p[0], float(p[1]), int(p[2]), int(p[3]), int(p[4])
        vals = np.array([float(x) for x in p[5:]])
        f = Oracle(geom2d(theta, det)).footprint(0, ix, iy)
        w = np.zeros(256)
        w[f["k_lo"]:f["k_hi"] + 1] = f["w"][0]
        assert np.allclose(w[k0:k0 + len(vals)], vals, atol=1e-8), (line, w[k0 - 1:k0 + len(vals) + 1])
        rest = w.copy()
        rest[k0:k0 + len(vals)] = 0.0
        assert rest.max() < 1e-20          # e.g. bin 127 ~ 3e-28 at theta = 0.3


# ---- P4: hand-worked 3-D footprint ---------------------------------------------------------
def test_p4_golden_3d():
    for line in open(os.path.join(GOLD, "sf_footprints_3d.txt")):
        if line.startswith("#") or not line.strip():
            continue
        p = line.split()
        vals = np.array([float(x) for x in p[1:]]).reshape(2, 2)
        f = Oracle(geom3d(0.0, p[0])).footprint(0, 128, 128, 128)
        assert (f["k_lo"], f["l_lo"]) == (192, 192)
        assert np.allclose(f["w"][:2, :2], vals, atol=1e-8)
        assert f["w"].shape == (2, 2)
    # hand check (flat): voxel centre (.25,.25,.25); a in {600, 599.5}; s in {0, 0, 1.0, 1.000834};
    # cell 192 spans [0, 0.8] -> F1 = 1; cell 193 spans [0.8, 1.6] -> (0.2 + ~0.0004)/0.8 = 0.2505
    f = Oracle(geom3d(0.0)).footprint(0, 128, 128, 128)
    assert abs(f["F1"][0] - 1.0) < 1e-12 and abs(f["F1"][1] - 0.2505) < 3e-4
    assert abs(f["F2"][0] - 1.0) < 1e-12 and abs(f["F2"][1] - 0.2505) < 3e-4
    assert abs(f["amp"] - 0.5) < 1e-6


# ---- brute force: exact ray / box chords averaged over a detector cell -------------------
def _cell_points(g, view, s, t):
    """World points on the detector at detector coordinates (s, t) [mm]; independent restatement
    of the detector model (flat plane / source-centred cylinder)."""
    S = g["src"][view]
    D = g["det_center"][view]
    u = g["det_u"][view]
    v = g["det_v"][view]
    n = np.cross(u, v)
    if np.dot(D - S, n) < 0:
        n = -n
    if g["det_type"] == "flat":
        return D[None, :] + s[:, None] * u[None, :] + t[:, None] * v[None, :]
    R = np.dot(D - S, n)
    gam = s / R
    return (S[None, :] + R * (np.sin(gam)[:, None] * u[None, :] + np.cos(gam)[:, None] * n[None, :])
            + (t + np.dot(D - S, v))[:, None] * v[None, :])


def _chords(S, P, lo, hi):
    """Slab-method chord lengths of rays S->P through the box [lo, hi]."""
    d = P - S[None, :]
    L = np.linalg.norm(d, axis=1)
    d = d / L[:, None]
    with np.errstate(divide="ignore", invalid="ignore"):
        t1 = (lo[None, :] - S[None, :]) / d
        t2 = (hi[None, :] - S[None, :]) / d
    tmin = np.nanmax(np.minimum(t1, t2), axis=1)
    tmax = np.nanmin(np.maximum(t1, t2), axis=1)
    return np.maximum(tmax - tmin, 0.0)


def _brute_footprint(g, view, ijk, ks, ls, nsub):
    nx, ny, nz = g["nx"], g["ny"], g["nz"]
    c = np.array([(ijk[0] - 0.5 * (nx - 1)) * g["dx"], (ijk[1] - 0.5 * (ny - 1)) * g["dy"],
                  (ijk[2] - 0.5 * (nz - 1)) * g["dz"] if g["dim"] == 3 else 0.0])
    h = 0.5 * np.array([g["dx"], g["dy"], g["dz"] if g["dim"] == 3 else 1e9])
    sub = (np.arange(nsub) + 0.5) / nsub - 0.5
    out = np.zeros((len(ls), len(ks)))
    for a, l in enumerate(ls):
        for b, k in enumerate(ks):
            s = ((k - 0.5 * (g["nu"] - 1)) + sub) * g["du"]
            if g["dim"] == 3:
                t = ((l - 0.5 * (g["nv"] - 1)) + sub) * g["dv"]
                ss, tt = [x.ravel() for x in np.meshgrid(s, t)]
            else:
                ss, tt = s, np.zeros_like(s)
            P = _cell_points(g, view, ss, tt)
            out[a, b] = _chords(g["src"][view], P, c - h, c + h).mean()
    return out


def _analytic_mass(g, view, ijk):
    """Exact first-order total of a voxel's cell-averaged footprint, sum_kl w, from the change of
    variables (detector area <-> volume along rays); exact up to O((voxel size / distance)^2):
    flat: V R^2 |e| / a^3, arc: V R^2 |e| / rho^3 (rho^2 = a^2 + b^2); 2-D: A R |e| / a^2, A R / rho."""
    S, D, u, v = g["src"][view], g["det_center"][view], g["det_u"][view], g["det_v"][view]
    n = np.cross(u, v)
    if np.dot(D - S, n) < 0:
        n = -n
    R = np.dot(D - S, n)
    c = np.array([(ijk[0] - 0.5 * (g["nx"] - 1)) * g["dx"], (ijk[1] - 0.5 * (g["ny"] - 1)) * g["dy"],
                  (ijk[2] - 0.5 * (g["nz"] - 1)) * g["dz"] if g["dim"] == 3 else 0.0])
    e = c - S
    a, b = e @ n, e @ u
    rho = a if g["det_type"] == "flat" else math.hypot(a, b)
    if g["dim"] == 3:
        return g["dx"] * g["dy"] * g["dz"] * R * R * np.linalg.norm(e) / rho ** 3 / (g["du"] * g["dv"])
    return g["dx"] * g["dy"] * R * np.linalg.norm(e) / rho ** 2 / g["du"]


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_p6_brute_force_2d(det):
    g = geom2d([0.3, 0.7, 2.1, 4.0], det)
    o = Oracle(g)
    for view, (ix, iy) in [(0, (64, 64)), (1, (10, 120)), (2, (90, 40)), (3, (40, 45))]:
        f = o.footprint(view, ix, iy)
        ks = np.arange(f["k_lo"] - 1, f["k_hi"] + 2)
        bf = _brute_footprint(g, view, (ix, iy, 0), ks, [0], 4000)[0]
        w = np.zeros(len(ks))
        w[1:-1] = f["w"][0]
        assert np.abs(w - bf).max() < 5e-4 * bf.max()
        assert abs(w.sum() - bf.sum()) < 1e-5 * bf.sum()
        assert abs(w.sum() - _analytic_mass(g, view, (ix, iy, 0))) < 1e-5 * w.sum()


@pytest.mark.parametrize("det", ["flat", "arc"])
def test_p6_brute_force_3d_circular(det):
    g = geom3d([0.4, 1.9], det, n=(64, 64, 64), d=(2.0, 2.0, 2.0), nu=96, nv=96, du=3.2, dv=3.2)
    o = Oracle(g)
    # near the mid-plane (polar < 1 deg) and far off it (polar up to ~6 deg).  The brute-force
    # TOTAL converges only as O(1/nsub) near the mid-plane (a voxel face is almost parallel to the
    # rays), so the total is pinned to the closed form instead and the cells to brute force.
    for view, ijk, tol_cell in [(0, (40, 20, 32), 5e-3), (1, (10, 50, 33), 5e-3),
                                (0, (50, 12, 60), 5e-2), (1, (8, 8, 2), 5e-2)]:
        f = o.footprint(view, *ijk)
        ks = np.arange(f["k_lo"] - 1, f["k_hi"] + 2)
        ls = np.arange(f["l_lo"] - 1, f["l_hi"] + 2)
        bf = _brute_footprint(g, view, ijk, ks, ls, 120)
        w = np.zeros((len(ls), len(ks)))
        w[1:-1, 1:-1] = f["w"]
        assert np.abs(w - bf).max() < tol_cell * bf.max(), (ijk, np.abs(w - bf).max() / bf.max())
        assert abs(w.sum() - bf.sum()) < 5e-3 * bf.sum()
        assert abs(w.sum() - _analytic_mass(g, view, ijk)) < 2e-5 * w.sum()


def test_p6_brute_force_3d_tilted():
    # 15 deg off-plane tilt + 0.5 deg in-plane rotation (R6): SF-TR's known limit; gates 1e-1 / 5e-3
    g = geom3d([0.4, 2.5], "flat", n=(64, 64, 64), d=(2.0, 2.0, 2.0), nu=96, nv=96, du=3.2, dv=3.2,
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
