"""CTorch-style scan parameters -> the per-view vectors the C ABI takes (Table 2).

The kernels never see these parameters; this is host-side convenience mirroring the paper's
`Geom2D` / 3-D circular / 3-D non-circular classes.  Every parameter may be a
scalar (shared by all views) or a length-n_views vector (view-specific).

Reading R11: world origin at the rotation centre; at theta = 0 the y axis is
perpendicular to the detector; right-handed active rotations Q = Rz(theta) Rx(phi) Ry(psi) (order
y -> x -> z); source S = Q (x_src, SAD, z_src); u = Q ex, v = Q ez; flat detector centre
D = Q (u_ofst, SAD - SDD, v_ofst) (the detector is shifted by +u_ofst, so the central ray pierces it
at detector coordinate -u_ofst, Table 2's "u_d = -u_ofst"); arc detector: (u, n) are rotated about v
through S by u_ofst / SDD and D = S + SDD n + v_ofst v.  A per-view object offset is folded into S and
D; a constant one becomes the volume centre (ox, oy, oz).
"""
import math

import numpy as np


def _vec(x, n):
    a = np.asarray(x, dtype=np.float64).reshape(-1)
    if a.size == 1:
        return np.full(n, a[0])
    if a.size != n:
        raise ValueError("parameter must be a scalar or have one entry per view (%d), got %d" % (n, a.size))
    return a


def _rz(t):
    c, s = math.cos(t), math.sin(t)
    return np.array([[c, -s, 0.0], [s, c, 0.0], [0.0, 0.0, 1.0]])


def _rx(t):
    c, s = math.cos(t), math.sin(t)
    return np.array([[1.0, 0.0, 0.0], [0.0, c, -s], [0.0, s, c]])


def _ry(t):
    c, s = math.cos(t), math.sin(t)
    return np.array([[c, 0.0, s], [0.0, 1.0, 0.0], [-s, 0.0, c]])


def make_geometry(dim, nx, ny, dx, dy, nu, du, view_angles, SAD, SDD, det_type="flat",
                  nz=1, dz=1.0, nv=1, dv=1.0, x_src=0.0, z_src=0.0, x_ofst=0.0, y_ofst=0.0, z_ofst=0.0,
                  u_ofst=0.0, v_ofst=0.0, phi=0.0, psi=0.0):
    """Returns the problem-description dict for binding.ct_geom_create / projector.Geometry."""
    theta = np.asarray(view_angles, dtype=np.float64).reshape(-1)
    n = theta.size
    SAD, SDD = _vec(SAD, n), _vec(SDD, n)
    x_src, z_src = _vec(x_src, n), _vec(z_src, n)
    xo, yo, zo = _vec(x_ofst, n), _vec(y_ofst, n), _vec(z_ofst, n)
    uo, vo = _vec(u_ofst, n), _vec(v_ofst, n)
    phi, psi = _vec(phi, n), _vec(psi, n)
    if dim == 2 and (np.any(z_src != 0) or np.any(zo != 0) or np.any(vo != 0) or np.any(phi != 0) or np.any(psi != 0)):
        raise ValueError("a 2-D geometry has no z_src, z_ofst, v_ofst, phi or psi")
    # constant part of the object offset -> volume centre; view-specific remainder -> shift of S and D
    ox, oy, oz = float(xo[0]), float(yo[0]), float(zo[0])
    src = np.zeros((n, 3))
    dc = np.zeros((n, 3))
    u = np.zeros((n, 3))
    v = np.zeros((n, 3))
    for i in range(n):
        Q = _rz(theta[i]) @ _rx(phi[i]) @ _ry(psi[i])
        S = Q @ np.array([x_src[i], SAD[i], z_src[i]])
        ui, vi = Q @ np.array([1.0, 0.0, 0.0]), Q @ np.array([0.0, 0.0, 1.0])
        ni = Q @ np.array([0.0, -1.0, 0.0])
        if det_type == "flat":
            D = Q @ np.array([uo[i], SAD[i] - SDD[i], vo[i]])
        else:
            a = uo[i] / SDD[i]
            ui, ni = math.cos(a) * ui + math.sin(a) * ni, -math.sin(a) * ui + math.cos(a) * ni
            D = S + SDD[i] * ni + vo[i] * vi
        shift = np.array([xo[i] - ox, yo[i] - oy, zo[i] - oz])
        src[i], dc[i], u[i], v[i] = S - shift, D - shift, ui, vi
    return dict(dim=dim, nx=nx, ny=ny, nz=nz, dx=dx, dy=dy, dz=dz, ox=ox, oy=oy, oz=oz, nu=nu, nv=nv,
                du=du, dv=dv, det_type=det_type, src=src, det_center=dc, det_u=u, det_v=v)


def Geom2D(nx, ny, dx, dy, nu, du, nView, viewAngles, detType="flat", SAD=500.0, SDD=1000.0,
           xOfst=0.0, yOfst=0.0, uOfst=0.0, xSrc=0.0):
    """Mirror of the paper's example constructor."""
    ang = np.asarray(viewAngles, dtype=np.float64).reshape(-1)
    if ang.size != nView:
        raise ValueError("viewAngles must have nView entries")
    return make_geometry(2, nx, ny, dx, dy, nu, du, ang, SAD, SDD, "arc" if detType in ("arc", "curved", "curve") else "flat",
                         x_src=xSrc, x_ofst=xOfst, y_ofst=yOfst, u_ofst=uOfst)


def shard_views(n_views, world_size, rank):
    """Contiguous view shard (view_begin, view_stride, view_count) of `rank`:
    A: each rank projects its own views of a replicated volume, no collective.
    A^T: each rank backprojects its views; the partial volumes are summed by one all-reduce."""
    base, rem = divmod(n_views, world_size)
    count = base + (1 if rank < rem else 0)
    begin = rank * base + min(rank, rem)
    return begin, 1, count
