"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot produce whole outputs at these sizes in reasonable time, so it computes sampled
outputs one by one: A on a few whole views (every cell of those views is compared), A^T on randomly
sampled voxels over all views.  Inputs: the seeded phantom (A) and a seeded smooth positive
projection field (A^T) from the workloads module -- never anything computed by the CUDA path."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import binding as B
from paper_2503_16741_b200 import workloads as W

pytestmark = pytest.mark.gpu

N_VIEWS = {1: 6, 2: 5, 3: 5, 4: 6, 5: 4}
N_VOX = {1: 4000, 2: 3000, 3: 3000, 4: 3000, 5: 3000}


@pytest.mark.parametrize("index", [1, 5, 2, 3, 4])
def test_parity_full_size_sampled(index):
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(index)
    g = W.geom_keys(c)
    o = Oracle(g)
    rng = np.random.default_rng(9000 + index)
    x = W.make_phantom(c)
    geom = Geometry(g)
    # ---- A: whole sampled views -------------------------------------------------------------
    xd = torch.from_numpy(x).cuda()
    y = geom.fp(xd)                                              # full operator, as bench.py runs it
    views = np.sort(rng.choice(c["n_views"], N_VIEWS[index], replace=False))
    views[0] = 0 if index != 4 else views[0]
    y_ref = o.fp(x, views)                                       # [B, n_sel, nv, nu] float64
    y_gpu = y[:, torch.from_numpy(views).cuda()].double().cpu().numpy()
    rel = np.linalg.norm(y_gpu - y_ref) / np.linalg.norm(y_ref)
    mx = np.abs(y_gpu - y_ref).max() / np.abs(y_ref).max()
    assert rel <= 1e-5 and mx <= 1e-4, "A config %d: rel-L2 %.3e max %.3e" % (index, rel, mx)
    # every output element is written (overwrite semantics): poison the buffer first
    y.fill_(float("nan"))
    geom.fp(xd, out=y)
    assert not torch.isnan(y).any()
    del y, xd
    # ---- A^T: sampled voxels over all views -----------------------------------------------
    p = W.make_projections(c)
    pd = torch.from_numpy(p).cuda()
    xb = geom.bp(pd)
    ijk = np.stack([rng.integers(0, c["nx"], N_VOX[index]), rng.integers(0, c["ny"], N_VOX[index]),
                    rng.integers(0, c["nz"], N_VOX[index])], axis=1)
    ijk[0] = (0, 0, 0)
    ijk[1] = (c["nx"] - 1, c["ny"] - 1, c["nz"] - 1)
    for b in range(c["batch"]):                     # all 16 images of config 5
        ref = o.bp_voxels(p[b], ijk)
        got = xb[b, ijk[:, 2], ijk[:, 1], ijk[:, 0]].double().cpu().numpy()
        rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
        mx = np.abs(got - ref).max() / np.abs(ref).max()
        assert rel <= 1e-5 and mx <= 1e-4, "A^T config %d: rel-L2 %.3e max %.3e" % (index, rel, mx)
    geom.close()


def test_sftt_full_size_sampled():
    """SF-TT (row f3) at config 4's full size: A on whole sampled views, A^T on sampled voxels over all 720 views,
    against the oracle's algo='SF-TT' -- the sizes at which its sampled margins (lpad, zpad) have to hold."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4)
    g = dict(W.geom_keys(c), algo="SF-TT")
    o = Oracle(g)
    rng = np.random.default_rng(9400)
    x = W.make_phantom(c)
    geom = Geometry(g)
    xd = torch.from_numpy(x).cuda()
    y = geom.fp(xd)
    views = np.sort(rng.choice(c["n_views"], 4, replace=False))
    y_ref = o.fp(x, views)
    y_gpu = y[:, torch.from_numpy(views).cuda()].double().cpu().numpy()
    rel = np.linalg.norm(y_gpu - y_ref) / np.linalg.norm(y_ref)
    mx = np.abs(y_gpu - y_ref).max() / np.abs(y_ref).max()
    assert rel <= 1e-5 and mx <= 1e-4, "SF-TT A config 4: rel-L2 %.3e max %.3e" % (rel, mx)
    del y, xd
    p = W.make_projections(c)
    xb = geom.bp(torch.from_numpy(p).cuda())
    n = 2000
    ijk = np.stack([rng.integers(0, c["nx"], n), rng.integers(0, c["ny"], n), rng.integers(0, c["nz"], n)], axis=1)
    ijk[0] = (0, 0, 0)
    ijk[1] = (c["nx"] - 1, c["ny"] - 1, c["nz"] - 1)
    ref = o.bp_voxels(p[0], ijk)
    got = xb[0, ijk[:, 2], ijk[:, 1], ijk[:, 0]].double().cpu().numpy()
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / np.abs(ref).max()
    assert rel <= 1e-5 and mx <= 1e-4, "SF-TT A^T config 4: rel-L2 %.3e max %.3e" % (rel, mx)
    geom.close()


def test_sftt_margins_are_conservative_full_size():
    """SF-TT's trapezoid reaches beyond the rectangle's rows; how far is SAMPLED when the geometry is created (a 9x9x9
    probe x 1.25: lpad for the backprojector's brick shadow, zpad for the forward kernel's region).  Nothing re-checks
    it at run time, so it is checked here where it matters: at config 4's full volume and detector (96 of its views),
    two more rows / voxels of margin (testing switch tt_pad) may change A and A^T by summation order only."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4, n_views=96)
    g = dict(W.geom_keys(c), algo="SF-TT")
    rng = np.random.default_rng(81)
    x = torch.from_numpy(rng.uniform(0.5, 1.5, (1, c["nz"], c["ny"], c["nx"])).astype(np.float32)).cuda()
    y = torch.from_numpy(rng.uniform(0.5, 1.5, (1, c["n_views"], c["nv"], c["nu"])).astype(np.float32)).cuda()
    geom = Geometry(g)
    B.debug_set("tt_pad", 2.0)
    wide = Geometry(g)                                  # the switch is read when the geometry is created
    B.debug_set("tt_pad", 0.0)
    y_t, y_w = geom.fp(x), wide.fp(x)
    assert (y_t - y_w).abs().max().item() <= 3e-6 * y_w.abs().max().item()
    del y_t, y_w
    x_t, x_w = geom.bp(y), wide.bp(y)
    assert (x_t - x_w).abs().max().item() <= 3e-6 * x_w.abs().max().item()
    geom.close()
    wide.close()


def test_recon_mode_full_size_few_views():
    """Recon mode (row f2) on config 4's full volume and detector: the RECON instantiation of the packed backprojector
    has its own register allocation, and the shrunken configs of test_gpu_recon.py never fill a brick grid of 32^3.
    Six of the trajectory's views, so that the oracle can backproject the WHOLE volume: every voxel is compared."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4, n_views=6)
    g = W.geom_keys(c)
    o, geom = Oracle(g), Geometry(g)
    q = W.make_projections(c)
    got = geom.bp_recon(torch.from_numpy(q).cuda()).double().cpu().numpy()
    ref = o.bp_recon(q)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.abs(got - ref).max() / np.abs(ref).max()
    assert rel <= 1e-5 and mx <= 1e-4, "recon A^T config 4, 6 views: rel-L2 %.3e max %.3e" % (rel, mx)
    geom.close()


@pytest.mark.parametrize("algo", ["SF", "DD", "SF-TT"])
@pytest.mark.parametrize("index", [4, 3, 2])
def test_forward_region_is_conservative(index, algo, monkeypatch):
    """The forward kernel sweeps, per slab, only the voxels its tile's frustum can touch (exact half-voxel halo).
    Property that holds at any size: widening that region by a whole voxel (debug switch fp_pad) may only change the
    summation order.  Checked on EVERY cell of every view of the full-size operator (a missed voxel would
    shift a cell by ~1e-3 of its value)."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(index)
    if index == 4:
        c = W.make_config(index, n_views=96)          # every 7.5th view of the trajectory, full volume/detector
    g = dict(W.geom_keys(c), algo=algo)
    rng = np.random.default_rng(77 + index)
    x = torch.from_numpy(rng.uniform(0.5, 1.5, (1, c["nz"], c["ny"], c["nx"])).astype(np.float32)).cuda()
    geom = Geometry(g)
    B.debug_set("fp_pad", 0)
    y_tight = geom.fp(x)
    torch.cuda.synchronize()
    B.debug_set("fp_pad", 1.0)
    y_wide = geom.fp(x)
    torch.cuda.synchronize()
    B.debug_set("fp_pad", 0)
    diff = (y_tight - y_wide).abs().max().item()
    assert diff <= 3e-6 * y_wide.abs().max().item(), diff
    geom.close()


@pytest.mark.parametrize("algo", ["SF", "DD"])
@pytest.mark.parametrize("index", [2, 5])
def test_run_to_run_determinism(index, algo):
    """Both operators fix their summation order (no atomics; the forward kernel's conflict-free rounds), so
    repeated calls are bit-identical.  A shared-memory race in the forward tile would show up here."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(index)
    g = dict(W.geom_keys(c), algo=algo)
    rng = np.random.default_rng(5 + index)
    x = torch.from_numpy(rng.uniform(0, 1, (c["batch"], c["nz"], c["ny"], c["nx"])).astype(np.float32)).cuda()
    geom = Geometry(g)
    y0 = geom.fp(x)
    xb0 = geom.bp(y0)
    for _ in range(2):
        assert torch.equal(geom.fp(x), y0)
        assert torch.equal(geom.bp(y0), xb0)
    geom.close()
