"""GPU parity: ct_fp_sf / ct_bp_sf (through the C ABI) vs the float64 CPU oracle, element by element,
on the same seeded inputs.  Sizes are shrunken versions of BASELINE.json's five configs (same physical
extents, odd counts so that several tiles and a ragged tail are covered).

Tolerances (BASELINE.json north_star): rel-L2 <= 1e-5 and max-abs <= 1e-4 * max|oracle| for A and
A^T; GPU adjoint test 1e-5 relative with the inner products accumulated in float64."""
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
    5: dict(nx=96, ny=90, nu=290, n_views=17, batch=5),
}


def check(gpu, ref, what):
    gpu = gpu.double().cpu().numpy()
    rel = np.linalg.norm(gpu - ref) / np.linalg.norm(ref)
    mx = np.abs(gpu - ref).max() / np.abs(ref).max()
    assert rel <= 1e-5 and mx <= 1e-4, "%s: rel-L2 %.3e max-abs/max %.3e" % (what, rel, mx)
    return rel, mx


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_parity_small(index):
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(index, **SHRINK[index])
    g = W.geom_keys(c)
    x = W.make_phantom(c)                                    # [B, nz, ny, nx] fp32
    o = Oracle(g)
    y_ref = o.fp(x)                                          # float64
    geom = Geometry(g)
    xd = torch.from_numpy(x).cuda()
    y = geom.fp(xd)
    check(y, y_ref, "A  config %d" % index)
    y32 = y_ref.astype(np.float32)                           # A^T input: fp32(oracle A x)
    xb_ref = o.bp(y32)
    xb = geom.bp(torch.from_numpy(y32).cuda())
    check(xb, xb_ref, "A^T config %d" % index)
    # adjoint test on the GPU pair with U(0,1) inputs
    rng = np.random.default_rng(100 + index)
    xr = torch.from_numpy(rng.uniform(0, 1, x.shape).astype(np.float32)).cuda()
    yr = torch.from_numpy(rng.uniform(0, 1, y_ref.shape).astype(np.float32)).cuda()
    lhs = torch.sum(geom.fp(xr).double() * yr.double()).item()
    rhs = torch.sum(xr.double() * geom.bp(yr).double()).item()
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs), (lhs, rhs)
    geom.close()


def test_view_subsets_and_batch_independence():
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(2, nx=40, ny=36, nz=20, nu=80, nv=60, n_views=12, batch=3)
    g = W.geom_keys(c)
    x = torch.from_numpy(W.make_phantom(c)).cuda()
    geom = Geometry(g)
    y = geom.fp(x)
    ys = geom.fp(x, views=(1, 3, 4))
    assert torch.equal(ys, y[:, 1::3][:, :4])
    for b in range(3):
        assert torch.equal(geom.fp(x[b]), y[b])
    o = Oracle(g)
    sel = np.array([1, 4, 7, 10])
    ref = o.bp(ys.double().cpu().numpy(), sel)
    check(geom.bp(ys, views=(1, 3, 4)), ref, "A^T subset")
    geom.close()


def test_edge_cases():
    from paper_2503_16741_b200 import binding as B
    from paper_2503_16741_b200.projector import Geometry
    # detector much smaller than the object's shadow (heavy clipping) and a 1x1x1 volume
    c = W.make_config(2, nx=33, ny=31, nz=29, nu=24, nv=9, n_views=7)
    c["du"] *= 0.3
    c["dv"] *= 0.2
    g = W.geom_keys(c)
    x = W.make_phantom(c)
    o, geom = Oracle(g), Geometry(g)
    y_ref = o.fp(x)
    check(geom.fp(torch.from_numpy(x).cuda()), y_ref, "A clipped")
    check(geom.bp(torch.from_numpy(y_ref.astype(np.float32)).cuda()), o.bp(y_ref.astype(np.float32)), "A^T clipped")
    geom.close()
    c1 = W.make_config(2, nx=1, ny=1, nz=1, nu=16, nv=16, n_views=3)
    g1 = W.geom_keys(c1)
    geom = Geometry(g1)
    x1 = np.ones((1, 1, 1, 1), np.float32)
    y1_ref = Oracle(g1).fp(x1)
    check(geom.fp(torch.from_numpy(x1).cuda()), y1_ref, "A single voxel")
    y1 = y1_ref.astype(np.float32)
    check(geom.bp(torch.from_numpy(y1).cuda()), Oracle(g1).bp(y1), "A^T single voxel")
    geom.close()
    # error behaviour: bad descriptors are refused, nothing throws across the ABI
    bad = dict(g, det_u=np.array(g["det_u"]) * 1.1)
    with pytest.raises(B.CtError) as e:
        B.ct_geom_create(bad)
    assert e.value.status == 2
    with pytest.raises(B.CtError) as e:
        B.ct_geom_create(dict(g, nx=0))
    assert e.value.status == 1


def test_autograd_and_mbir_loop():
    """gradient descent on ||A x - y||^2 through autograd; the loss must fall."""
    from paper_2503_16741_b200.projector import Projector
    c = W.make_config(5, nx=64, ny=64, nu=120, n_views=24, batch=2)
    g = W.geom_keys(c)
    A = Projector(g, "proj", "SF", "forward")
    x_true = torch.from_numpy(W.make_phantom(c, seed=c["seed"] + 100)).cuda()[:, 0]     # [B, ny, nx]
    x_true = x_true[:, None]                                                             # [B, 1(nz), ny, nx]
    y = A(x_true)
    x = torch.zeros_like(x_true, requires_grad=True)
    ones = torch.ones_like(x_true)
    lr = 1.0 / (2.0 * A.geom.bp(A.geom.fp(ones)).max().item())
    losses = []
    for _ in range(10):
        loss = torch.sum((A(x) - y) ** 2)
        (grad,) = torch.autograd.grad(loss, [x])
        # autograd's gradient is 2 A^T (A x - y)
        manual = 2.0 * A.geom.bp(A.geom.fp(x.detach()) - y)
        assert torch.allclose(grad, manual, rtol=1e-5, atol=1e-6 * manual.abs().max().item())
        x.data -= lr * grad
        losses.append(loss.item())
    assert all(b < a for a, b in zip(losses, losses[1:])), losses
