"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: no footprints, no weights, no projection -- only (a) scan trajectories written out as
per-view vectors (source, detector centre, detector axes) and (b) piecewise-constant ellipse /
ellipsoid phantoms.  It imports neither the product binding nor oracle/.

The paper's own data (bench CBCT scans, AAPM CT-MAR sinograms, XCAT head) are
not available; these phantoms take their shapes and sizes and stand in for them.  No item of any
public dataset is reproduced.  Recipe: DESIGN.md "Input recipe".
"""
import math

import numpy as np

SEED0 = 250316741


def _rot(axis, ang):
    c, s = math.cos(ang), math.sin(ang)
    if axis == "x":
        return np.array([[1, 0, 0], [0, c, -s], [0, s, c]], dtype=np.float64)
    if axis == "y":
        return np.array([[c, 0, s], [0, 1, 0], [-s, 0, c]], dtype=np.float64)
    return np.array([[c, -s, 0], [s, c, 0], [0, 0, 1]], dtype=np.float64)


def trajectory(n_views, sad, sdd, det_type, theta=None, phi=None, psi=None):
    """Per-view vectors of a scan with all offsets zero (Table 2; R11).

    Right-handed active rotations Q = Rz(theta) Rx(phi) Ry(psi); S = Q (0, SAD, 0);
    u = Q ex, v = Q ez; detector centre = Q (0, SAD - SDD, 0) (flat and arc alike when the
    lateral offset is zero).  Returns float64 arrays [n_views, 3]."""
    if theta is None:
        theta = 2.0 * math.pi * np.arange(n_views) / n_views
    phi = np.zeros(n_views) if phi is None else np.broadcast_to(phi, (n_views,))
    psi = np.zeros(n_views) if psi is None else np.broadcast_to(psi, (n_views,))
    src = np.zeros((n_views, 3))
    dc = np.zeros((n_views, 3))
    u = np.zeros((n_views, 3))
    v = np.zeros((n_views, 3))
    for i in range(n_views):
        Q = _rot("z", theta[i]) @ _rot("x", phi[i]) @ _rot("y", psi[i])
        src[i] = Q @ np.array([0.0, sad, 0.0])
        dc[i] = Q @ np.array([0.0, sad - sdd, 0.0])
        u[i] = Q @ np.array([1.0, 0.0, 0.0])
        v[i] = Q @ np.array([0.0, 0.0, 1.0])
    return src, dc, u, v


def _jitter(rng, src, dc, u, v):
    """Config 4: per view, in this draw order, dS ~ U(-1,1)^3 mm, dD ~ U(-1,1)^3 mm,
    dpsi ~ U(-0.5, 0.5) deg rotating (u, v) about n = u x v (in-plane)."""
    for i in range(src.shape[0]):
        src[i] += rng.uniform(-1.0, 1.0, 3)
        dc[i] += rng.uniform(-1.0, 1.0, 3)
        a = math.radians(rng.uniform(-0.5, 0.5))
        ui, vi = u[i].copy(), v[i].copy()
        u[i] = math.cos(a) * ui + math.sin(a) * vi
        v[i] = -math.sin(a) * ui + math.cos(a) * vi


_BASE = {
    1: dict(name="fan2d_flat_128", dim=2, nx=128, ny=128, nz=1, dx=1.0, dy=1.0, dz=1.0,
            nu=256, nv=1, du=1.0, dv=1.0, det_type="flat", n_views=180, sad=500.0, sdd=1000.0,
            batch=1, n_obj=10),
    2: dict(name="cone_circ_flat_256", dim=3, nx=256, ny=256, nz=256, dx=0.5, dy=0.5, dz=0.5,
            nu=384, nv=384, du=0.8, dv=0.8, det_type="flat", n_views=360, sad=600.0, sdd=1200.0,
            batch=1, n_obj=20),
    3: dict(name="cone_diag_arc_512x512x64", dim=3, nx=512, ny=512, nz=64, dx=0.7, dy=0.7, dz=1.0,
            nu=888, nv=64, du=1.0, dv=1.0, det_type="arc", n_views=984, sad=541.0, sdd=949.0,
            batch=1, n_obj=20),
    4: dict(name="cone_noncirc_flat_512", dim=3, nx=512, ny=512, nz=512, dx=0.5, dy=0.5, dz=0.5,
            nu=768, nv=768, du=0.388, dv=0.388, det_type="flat", n_views=720, sad=600.0, sdd=1200.0,
            batch=1, n_obj=20),
    5: dict(name="fan2d_arc_batch16_512", dim=2, nx=512, ny=512, nz=1, dx=0.5, dy=0.5, dz=1.0,
            nu=736, nv=1, du=1.0, dv=1.0, det_type="arc", n_views=720, sad=595.0, sdd=1085.6,
            batch=16, n_obj=10),
}


def make_config(index, **shrink):
    """Config `index` (1..5) of BASELINE.json as a flat dict: the problem-description keys
    (dim, nx.., dx.., ox.., nu, nv, du, dv, det_type, n_views, src, det_center, det_u, det_v)
    plus name, batch, index, seed.

    `shrink` may override the COUNTS nx, ny, nz, nu, nv, n_views, batch; pitches are rescaled so
    the physical extent of volume and detector (hence magnification, fan and cone angles and
    the footprint-to-cell ratios' order of magnitude) stays that of the full config."""
    c = dict(_BASE[index])
    c["index"] = index
    c["seed"] = SEED0 + index
    for key, pitch in (("nx", "dx"), ("ny", "dy"), ("nz", "dz"), ("nu", "du"), ("nv", "dv")):
        if key in shrink and c[key] > 1:
            c[pitch] = c[pitch] * c[key] / float(shrink[key])
            c[key] = int(shrink[key])
    for key in ("n_views", "batch"):
        if key in shrink:
            c[key] = int(shrink[key])
    c["ox"] = c["oy"] = c["oz"] = 0.0
    n = c["n_views"]
    theta = 2.0 * math.pi * np.arange(n) / n
    if index == 4:
        phi = np.radians(15.0) * np.sin(2.0 * theta)
        src, dc, u, v = trajectory(n, c["sad"], c["sdd"], c["det_type"], theta, phi)
        _jitter(np.random.default_rng(c["seed"] + 1000), src, dc, u, v)
    else:
        src, dc, u, v = trajectory(n, c["sad"], c["sdd"], c["det_type"], theta)
    c.update(src=src, det_center=dc, det_u=u, det_v=v)
    return c


def make_phantom(c, seed=None, batch=None):
    """Piecewise-constant phantom, float32 [batch, nz, ny, nx]; values computed in float64.

    2-D: per image n_obj ellipses, draw order per ellipse: cx, cy ~ U(-L/4, L/4); semi-axes a, b ~
    U(5, 50) mm scaled by L/128mm-equivalent of config 1 (i.e. U(0.04, 0.40) L); rotation ~ U(0, pi);
    mu ~ U(0.01, 0.03) /mm.  3-D: n_obj ellipsoids, centre per axis ~ U(-L_axis/4, L_axis/4),
    semi-axes per axis ~ U(0.04, 0.40) L_axis, rotation about z ~ U(0, pi), mu ~ U(0.01, 0.03).
    Pixel value = sum of mu over the objects containing the voxel CENTRE (overlaps add)."""
    rng = np.random.default_rng(c["seed"] if seed is None else seed)
    B = c["batch"] if batch is None else batch
    nx, ny, nz = c["nx"], c["ny"], c["nz"]
    xs = c["ox"] + (np.arange(nx) - 0.5 * (nx - 1)) * c["dx"]
    ys = c["oy"] + (np.arange(ny) - 0.5 * (ny - 1)) * c["dy"]
    zs = c["oz"] + (np.arange(nz) - 0.5 * (nz - 1)) * c["dz"]
    Lx, Ly, Lz = nx * c["dx"], ny * c["dy"], nz * c["dz"]
    out = np.zeros((B, nz, ny, nx), dtype=np.float64)
    for b in range(B):
        for _ in range(c["n_obj"]):
            cx = rng.uniform(-Lx / 4, Lx / 4)
            cy = rng.uniform(-Ly / 4, Ly / 4)
            cz = rng.uniform(-Lz / 4, Lz / 4) if c["dim"] == 3 else 0.0
            ax = rng.uniform(0.04, 0.40) * Lx
            ay = rng.uniform(0.04, 0.40) * Ly
            az = rng.uniform(0.04, 0.40) * Lz if c["dim"] == 3 else 1.0
            al = rng.uniform(0.0, math.pi)
            mu = rng.uniform(0.01, 0.03)
            ca, sa = math.cos(al), math.sin(al)
            # bounding box in index space (conservative), to keep 512^3 cheap
            rxy = max(ax, ay)
            ix0, ix1 = np.searchsorted(xs, cx - rxy), np.searchsorted(xs, cx + rxy, side="right")
            iy0, iy1 = np.searchsorted(ys, cy - rxy), np.searchsorted(ys, cy + rxy, side="right")
            X = xs[ix0:ix1][None, :] - cx
            Y = ys[iy0:iy1][:, None] - cy
            xr = (ca * X + sa * Y) / ax
            yr = (-sa * X + ca * Y) / ay
            q2 = xr * xr + yr * yr                           # [ny', nx']
            if c["dim"] == 3:
                iz0, iz1 = np.searchsorted(zs, cz - az), np.searchsorted(zs, cz + az, side="right")
                for iz in range(iz0, iz1):
                    zz = ((zs[iz] - cz) / az) ** 2
                    out[b, iz, iy0:iy1, ix0:ix1] += mu * (q2 + zz <= 1.0)
            else:
                out[b, 0, iy0:iy1, ix0:ix1] += mu * (q2 <= 1.0)
    return out.astype(np.float32)


def geom_keys(c):
    """The problem-description subset of a config dict (what oracle and binding both take)."""
    keys = ("dim", "nx", "ny", "nz", "dx", "dy", "dz", "ox", "oy", "oz", "nu", "nv", "du", "dv",
            "det_type", "src", "det_center", "det_u", "det_v")
    return {k: c[k] for k in keys}


def n_updates(c):
    """Voxel x view updates of one operator application (the GUPS numerator)."""
    return c["batch"] * c["nx"] * c["ny"] * c["nz"] * c["n_views"]


def make_projections(c, seed=None, batch=None):
    """Smooth, positive, seeded projection-domain input for A^T at sizes where the oracle cannot
    produce A x in reasonable time: float32 [batch, n_views, nv, nu].  A sum of three low-frequency
    separable cosine products over (view, row, channel) on a positive offset -- sinogram-like in range
    and smoothness, but not derived from any projector."""
    rng = np.random.default_rng((c["seed"] if seed is None else seed) + 5000)
    B = c["batch"] if batch is None else batch
    nvw, nv, nu = c["n_views"], c["nv"], c["nu"]
    out = np.empty((B, nvw, nv, nu), dtype=np.float32)
    i = np.arange(nvw, dtype=np.float64)[:, None, None] / nvw
    l = (np.arange(nv, dtype=np.float64)[None, :, None] + 0.5) / nv
    k = (np.arange(nu, dtype=np.float64)[None, None, :] + 0.5) / nu
    for b in range(B):
        acc = np.full((nvw, nv, nu), 2.0)
        for _ in range(3):
            fi, fl, fk = rng.integers(1, 4), rng.integers(1, 4), rng.integers(1, 6)
            pi_, pl, pk = rng.uniform(0, 2 * math.pi, 3)
            amp = rng.uniform(0.2, 0.6)
            acc = acc + amp * (np.cos(2 * math.pi * fi * i + pi_) * np.cos(math.pi * fl * l + pl)
                               * np.cos(math.pi * fk * k + pk))
        out[b] = acc.astype(np.float32)
    return out
