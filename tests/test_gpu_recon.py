"""GPU parity for "recon" mode (readings R23, R24): ct_fbp_filter and
ct_bp_sf_recon through the C ABI against the float64 oracle, element by element, on shrunken versions of the
five BASELINE.json configs; plus the end-to-end FBP of analytic ball/disk projections on the GPU.
Tolerances as for the projector pair: rel-L2 <= 1e-5, max-abs <= 1e-4 max|oracle|."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import workloads as W

pytestmark = pytest.mark.gpu

SHRINK = {
    1: dict(nx=77, ny=70, nu=300, n_views=19),
    2: dict(nx=70, ny=66, nz=37, nu=150, nv=101, n_views=11),
    3: dict(nx=90, ny=84, nz=19, nu=301, nv=40, n_views=13),
    4: dict(nx=61, ny=64, nz=58, nu=140, nv=135, n_views=12),
    5: dict(nx=96, ny=90, nu=290, n_views=17, batch=3),
}


def _check(gpu, ref, what):
    gpu = gpu.double().cpu().numpy()
    rel = np.linalg.norm(gpu - ref) / np.linalg.norm(ref)
    mx = np.abs(gpu - ref).max() / np.abs(ref).max()
    assert rel <= 1e-5 and mx <= 1e-4, "%s: rel-L2 %.3e max-abs/max %.3e" % (what, rel, mx)


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_recon_parity_small(index):
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(index, **SHRINK[index])
    g = W.geom_keys(c)
    o, geom = Oracle(g), Geometry(g)
    p = o.fp(W.make_phantom(c)).astype(np.float32)               # sinogram-like input from the oracle
    q_ref = o.fbp_filter(p)
    q = geom.fbp_filter(torch.from_numpy(p).cuda())
    _check(q, q_ref, "filter config %d" % index)
    q32 = q_ref.astype(np.float32)
    x_ref = o.bp_recon(q32)
    x = geom.bp_recon(torch.from_numpy(q32).cuda())
    _check(x, x_ref, "recon BP config %d" % index)
    # ordered subset of the recon backprojection
    sel = np.arange(1, c["n_views"], 3)
    xs = geom.bp_recon(torch.from_numpy(q32[..., sel, :, :].copy()).cuda(), views=(1, 3, len(sel)))
    _check(xs, o.bp_recon(q32[..., sel, :, :], sel), "recon BP subset config %d" % index)
    geom.close()


def test_fbp_of_an_analytic_ball_on_the_gpu():
    """Whole chain on the GPU (Projector-level API): FDK of closed-form ball projections gives mu in the mid-plane."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(2, nx=64, ny=64, nz=32, nu=128, nv=96, n_views=180)
    mu, radius = 0.02, 0.22 * c["nx"] * c["dx"]
    centre = np.array([0.06 * c["nx"] * c["dx"], -0.04 * c["nx"] * c["dx"], 0.0])
    u = (np.arange(c["nu"]) - 0.5 * (c["nu"] - 1)) * c["du"]
    v = (np.arange(c["nv"]) - 0.5 * (c["nv"] - 1)) * c["dv"]
    p = np.empty((c["n_views"], c["nv"], c["nu"]), np.float32)
    for i in range(c["n_views"]):
        P = c["det_center"][i] + u[None, :, None] * c["det_u"][i] + v[:, None, None] * c["det_v"][i]
        d = P - c["src"][i]
        d /= np.linalg.norm(d, axis=-1, keepdims=True)
        oc = c["src"][i] - centre
        b = d @ oc
        p[i] = mu * 2.0 * np.sqrt(np.maximum(b * b - (oc @ oc - radius ** 2), 0.0))
    geom = Geometry(W.geom_keys(c))
    x = geom.fbp(torch.from_numpy(p).cuda()).cpu().numpy()
    xs = (np.arange(c["nx"]) - 0.5 * (c["nx"] - 1)) * c["dx"]
    X, Y = np.meshgrid(xs, xs)
    inside = np.hypot(X - centre[0], Y - centre[1]) < 0.75 * radius
    mid = 0.5 * (x[c["nz"] // 2 - 1] + x[c["nz"] // 2])
    assert abs(mid[inside].mean() / mu - 1.0) < 1e-2, mid[inside].mean() / mu
    geom.close()


def test_curved_detector_with_lateral_offset_all_operators():
    """PAPER.md:151 scenario (curved detector, 1.25-channel lateral offset) through the CTorch-style converter
    with clockwise view angles: A, A^T, the ramp filter and the recon backprojection against the oracle."""
    from paper_2503_16741_b200 import geometry as G
    from paper_2503_16741_b200.projector import Geometry
    n_views, nu, du = 31, 230, 1.2
    g = G.Geom2D(nx=100, ny=94, dx=0.5, dy=0.5, nu=nu, du=du, nView=n_views,
                 viewAngles=-np.linspace(0.0, 2.0 * math.pi, n_views, endpoint=False), detType="curved",
                 SAD=595.0, SDD=1085.6, uOfst=1.25 * du)
    c = W.make_config(5, nx=100, ny=94, nu=nu, n_views=n_views, batch=2)     # phantom recipe only
    x = W.make_phantom(c)
    o, geom = Oracle(g), Geometry(g)
    y_ref = o.fp(x)
    _check(geom.fp(torch.from_numpy(x).cuda()), y_ref, "A offset arc")
    y32 = y_ref.astype(np.float32)
    _check(geom.bp(torch.from_numpy(y32).cuda()), o.bp(y32), "A^T offset arc")
    q_ref = o.fbp_filter(y32)
    _check(geom.fbp_filter(torch.from_numpy(y32).cuda()), q_ref, "filter offset arc")
    q32 = q_ref.astype(np.float32)
    _check(geom.bp_recon(torch.from_numpy(q32).cuda()), o.bp_recon(q32), "recon BP offset arc")
    geom.close()
