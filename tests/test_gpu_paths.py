"""GPU parity on the kernels' special code paths (each case names the path it forces):
footprints much larger / much smaller than a detector cell, arc detector in a tilted frame (reading R8),
off-centre anisotropic volumes, regions too small for multi-row passes, view-specific magnification.
Same tolerances as test_gpu_parity.py (BASELINE.json north_star)."""
import math

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle.sf_oracle import Oracle
from paper_2503_16741_b200 import binding as B
from paper_2503_16741_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _check(gpu, ref, what, rel_tol=1e-5, max_tol=1e-4):
    gpu = gpu.double().cpu().numpy()
    rel = np.linalg.norm(gpu - ref) / np.linalg.norm(ref)
    mx = np.abs(gpu - ref).max() / np.abs(ref).max()
    assert rel <= rel_tol and mx <= max_tol, "%s: rel-L2 %.3e max-abs/max %.3e" % (what, rel, mx)


def _pair(c, what, seed=0):
    """A and A^T against the oracle plus the GPU adjoint identity, for config dict c."""
    from paper_2503_16741_b200.projector import Geometry
    g = W.geom_keys(c)
    x = W.make_phantom(c)
    o, geom = Oracle(g), Geometry(g)
    y_ref = o.fp(x)
    y = geom.fp(torch.from_numpy(x).cuda())
    _check(y, y_ref, "A " + what)
    y32 = y_ref.astype(np.float32)
    _check(geom.bp(torch.from_numpy(y32).cuda()), o.bp(y32), "A^T " + what)
    rng = np.random.default_rng(seed)
    xr = torch.from_numpy(rng.uniform(0, 1, x.shape).astype(np.float32)).cuda()
    yr = torch.from_numpy(rng.uniform(0, 1, y_ref.shape).astype(np.float32)).cuda()
    lhs = torch.sum(geom.fp(xr).double() * yr.double()).item()
    rhs = torch.sum(xr.double() * geom.bp(yr).double()).item()
    assert abs(lhs - rhs) <= 1e-5 * abs(lhs), (what, lhs, rhs)
    geom.close()


def test_large_footprints():
    """Cells 8x smaller than a voxel's shadow: K, L ~ 20 (FP: more than 8 footprint rows -> row-chunk loop;
    BP: several row chunks per voxel, shadows larger than one TMA box)."""
    c = W.make_config(2, nx=24, ny=22, nz=20, nu=320, nv=300, n_views=7)
    _pair(c, "large footprints (3-D flat)")
    c = W.make_config(1, nx=30, ny=28, nu=500, n_views=9)
    _pair(c, "large footprints (2-D flat)")


def test_small_footprints_lane_stride():
    """Cells 4x larger than a voxel's shadow: neighbouring voxels fall into the same cell, so the forward
    kernel must use a lane stride > 1 (and its run-time conflict check must hold)."""
    c = W.make_config(2, nx=96, ny=90, nz=40, nu=40, nv=36, n_views=9)
    _pair(c, "small footprints (3-D flat)")
    c = W.make_config(5, nx=200, ny=190, nu=60, n_views=11, batch=3)
    _pair(c, "small footprints (2-D arc, batch 3)")
    c = W.make_config(3, nx=120, ny=110, nz=24, nu=90, nv=16, n_views=9)
    _pair(c, "small footprints (3-D arc)")


def test_arc_detector_in_tilted_frame():
    """Reading R8: arc detector with view-specific tilt and in-plane rotation (no BASELINE config has it)."""
    c = W.make_config(3, nx=48, ny=44, nz=30, nu=150, nv=40, n_views=8)
    n = c["n_views"]
    theta = 2.0 * math.pi * np.arange(n) / n
    phi = np.radians(12.0) * np.sin(2.0 * theta + 0.3)
    psi = np.radians(0.4) * np.cos(theta)
    src, dc, u, v = W.trajectory(n, c["sad"], c["sdd"], c["det_type"], theta, phi, psi)
    c.update(src=src, det_center=dc, det_u=u, det_v=v)
    _pair(c, "arc, tilted")


def test_offcentre_anisotropic_volume():
    c = W.make_config(4, nx=40, ny=52, nz=28, nu=120, nv=96, n_views=9)
    c["dx"] *= 1.3
    c["dz"] *= 0.6
    c["ox"], c["oy"], c["oz"] = 7.5, -11.0, 4.0
    _pair(c, "off-centre anisotropic (3-D flat, jittered)")
    c = W.make_config(1, nx=50, ny=36, nu=200, n_views=10)
    c["dy"] *= 1.7
    c["ox"], c["oy"] = -9.0, 6.0
    _pair(c, "off-centre anisotropic (2-D flat)")


def test_thin_volumes_and_detectors():
    """Few slices / few rows: the forward sweep has too few region rows for multi-row passes; the
    backprojector's brick is mostly empty in z."""
    c = W.make_config(2, nx=64, ny=60, nz=3, nu=150, nv=5, n_views=7)
    _pair(c, "3 slices, 5 rows")
    c = W.make_config(3, nx=70, ny=66, nz=2, nu=160, nv=3, n_views=6)
    _pair(c, "2 slices, 3 rows (arc)")


def test_host_buffer_entry_points():
    """ct_fp_sf_host / ct_bp_sf_host (the e2e path of bench.py): view-chunked copy/compute pipeline for
    3-D batch 1 (A^T: 6 chunks at >= 64 views, accumulating chunk by chunk; A: chunks of >= 18 waves of CTAs, i.e.
    one chunk at test sizes -- 5 chunks are forced here to exercise the pipeline), plain path otherwise; results
    must equal the device-pointer operators bit for bit (A) / to rounding of the chunked sum (A^T) and
    match the oracle within the usual tolerances."""
    from paper_2503_16741_b200 import binding as B
    from paper_2503_16741_b200.projector import Geometry
    for index, shrink, fp_chunks in ((4, dict(nx=36, ny=40, nz=30, nu=100, nv=90, n_views=67), 5),
                                     (4, dict(nx=36, ny=40, nz=30, nu=100, nv=90, n_views=67), 0),
                                     (2, dict(nx=30, ny=30, nz=20, nu=64, nv=60, n_views=9), 0),
                                     (5, dict(nx=64, ny=60, nu=150, n_views=20, batch=3), 0)):
        B.debug_set("host_fp_chunks", fp_chunks)
        c = W.make_config(index, **shrink)
        g = W.geom_keys(c)
        x = W.make_phantom(c)
        o, geom = Oracle(g), Geometry(g)
        y_ref = o.fp(x)
        hx = torch.from_numpy(x).pin_memory()
        hy = torch.empty(y_ref.shape, dtype=torch.float32).pin_memory()
        B.ct_fp_sf_host(geom.handle, hx.data_ptr(), hy.data_ptr(), c["batch"], 0)
        assert geom.last_launch_count() > 0
        y_dev = geom.fp(torch.from_numpy(x).cuda())
        torch.cuda.synchronize()
        assert torch.equal(hy, y_dev.cpu()), "A host != device, config %d" % index
        _check(hy, y_ref, "A host config %d" % index)
        y32 = y_ref.astype(np.float32)
        hp = torch.from_numpy(y32).pin_memory()
        hxb = torch.empty(x.shape, dtype=torch.float32).pin_memory()
        B.ct_bp_sf_host(geom.handle, hp.data_ptr(), hxb.data_ptr(), c["batch"], 0)
        _check(hxb, o.bp(y32), "A^T host config %d" % index)
        # pageable host memory is accepted too
        out = np.empty(y_ref.shape, np.float32)
        B.ct_fp_sf_host(geom.handle, x.ctypes.data, out.ctypes.data, c["batch"], 0)
        assert np.array_equal(out, hy.numpy())
        geom.close()


def test_config5_gradient_descent_against_oracle():
    """BASELINE.json config 5 (shrunken): 10 steps of x <- x - lr * 2 A^T (A x - y), y = fp32(oracle A x_true),
    lr = 1 / (2 max_j [A^T A 1]_j) from the oracle; the GPU loop (fp32, through the C ABI) must track the
    float64 oracle loop: every loss within 1e-4 relative, x_10 within rel-L2 1e-4 (ten operator pairs deep,
    so ten times the single-operator budget)."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(5, nx=72, ny=70, nu=150, n_views=30, batch=3)
    g = W.geom_keys(c)
    o, geom = Oracle(g), Geometry(g)
    x_true = W.make_phantom(c, seed=c["seed"] + 100)
    y = o.fp(x_true).astype(np.float32)
    ones = np.ones_like(x_true)
    lr = 1.0 / (2.0 * o.bp(o.fp(ones)).max())
    # oracle loop, float64
    xo = np.zeros(x_true.shape, np.float64)
    losses_o = []
    for _ in range(10):
        r = o.fp(xo) - y
        losses_o.append(float((r ** 2).sum()))
        xo = xo - lr * 2.0 * o.bp(r)
    # GPU loop, fp32
    yd = torch.from_numpy(y).cuda()
    xg = torch.zeros(x_true.shape, device="cuda")
    losses_g = []
    for _ in range(10):
        r = geom.fp(xg) - yd
        losses_g.append(float((r.double() ** 2).sum().item()))
        xg = xg - float(lr) * 2.0 * geom.bp(r)
    assert all(b < a for a, b in zip(losses_g, losses_g[1:])), losses_g
    for a, b in zip(losses_g, losses_o):
        assert abs(a - b) <= 1e-4 * abs(b), (losses_g, losses_o)
    _check(xg, xo, "x_10 of the config-5 loop", rel_tol=1e-4, max_tol=1e-3)
    geom.close()


def test_untilted_fast_path_overflow_and_equivalence(monkeypatch):
    """The forward kernel's untilted fast path keeps <= 6 footprint columns / <= 8 rows in registers and is only
    chosen when the host's bound says that is enough.  Forced on geometries with larger footprints
    (debug switch fp_forcehoist) its overflow branch must still give the oracle's answer; and on a geometry where both
    paths apply, fast path and general path must agree to summation order."""
    from paper_2503_16741_b200.projector import Geometry
    for index, shrink in ((2, dict(nx=24, ny=22, nz=20, nu=320, nv=300, n_views=7)),     # K, L ~ 20
                          (3, dict(nx=40, ny=36, nz=10, nu=400, nv=60, n_views=6))):     # arc, K ~ 10
        c = W.make_config(index, **shrink)
        g = W.geom_keys(c)
        x = W.make_phantom(c)
        o, geom = Oracle(g), Geometry(g)
        B.debug_set("fp_forcehoist", 1)
        B.debug_set("bp_forcehoist", 1)
        y = geom.fp(torch.from_numpy(x).cuda())
        y_ref = o.fp(x)
        y32 = y_ref.astype(np.float32)
        xb = geom.bp(torch.from_numpy(y32).cuda())
        torch.cuda.synchronize()
        B.debug_set("fp_forcehoist", 0)
        B.debug_set("bp_forcehoist", 0)
        _check(y, y_ref, "A forced fast path, config %d" % index)
        _check(xb, o.bp(y32), "A^T forced fast path, config %d" % index)
        geom.close()
    c = W.make_config(2, nx=70, ny=66, nz=37, nu=150, nv=101, n_views=11)
    geom = Geometry(W.geom_keys(c))
    x = torch.from_numpy(W.make_phantom(c)).cuda()
    y_fast = geom.fp(x)
    torch.cuda.synchronize()
    B.debug_set("fp_nohoist", 1)
    y_gen = geom.fp(x)
    torch.cuda.synchronize()
    B.debug_set("fp_nohoist", 0)
    assert (y_fast - y_gen).abs().max().item() <= 3e-6 * y_gen.abs().max().item()
    xb_gen = geom.bp(y_gen)
    torch.cuda.synchronize()
    B.debug_set("bp_nohoist", 1)
    xb_gen2 = geom.bp(y_gen)
    torch.cuda.synchronize()
    B.debug_set("bp_nohoist", 0)
    assert (xb_gen - xb_gen2).abs().max().item() <= 3e-6 * xb_gen2.abs().max().item()
    geom.close()


def test_forward_lane_serial_branch(monkeypatch):
    """If a pass ever fails its conflict check the forward kernel adds the lanes' footprints one lane at a time.
    The branch is never expected to run; forced (debug switch fp_serial) it must give the same answer."""
    from paper_2503_16741_b200.projector import Geometry
    for index, shrink in ((4, dict(nx=30, ny=28, nz=26, nu=70, nv=66, n_views=5)),
                          (2, dict(nx=30, ny=28, nz=20, nu=64, nv=60, n_views=4)),
                          (5, dict(nx=40, ny=36, nu=90, n_views=6, batch=2))):
        c = W.make_config(index, **shrink)
        g = W.geom_keys(c)
        x = W.make_phantom(c)
        o, geom = Oracle(g), Geometry(g)
        B.debug_set("fp_serial", 1)
        y = geom.fp(torch.from_numpy(x).cuda())
        torch.cuda.synchronize()
        B.debug_set("fp_serial", 0)
        _check(y, o.fp(x), "A lane-serial, config %d" % index)
        geom.close()


def test_empty_view_subset():
    """view_count == 0: A writes nothing (empty projection tensor), A^T is the empty sum (zeros)."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(2, nx=20, ny=18, nz=12, nu=40, nv=30, n_views=6)
    geom = Geometry(W.geom_keys(c))
    x = torch.from_numpy(W.make_phantom(c)).cuda()
    y = geom.fp(x, views=(2, 1, 0))
    assert tuple(y.shape) == (1, 0, 30, 40)
    xb = torch.full_like(x, float("nan"))
    geom.bp(y, views=(2, 1, 0), out=xb)
    assert torch.count_nonzero(xb).item() == 0
    geom.bp_recon(y, views=(0, 1, 0), out=xb.fill_(float("nan")))
    assert torch.count_nonzero(xb).item() == 0
    assert tuple(geom.fbp_filter(y, views=(0, 1, 0)).shape) == (1, 0, 30, 40)
    geom.close()


@pytest.mark.parametrize("env", [{"bp_tma": 0}, {"bp_chunk": 3}, {"bp_tma": 0, "bp_chunk": 5}, {"bp_scalar": 1},
                                 {"bp_scalar": 1, "bp_chunk": 4}])
def test_backprojector_alternate_staging_and_chunking(env, monkeypatch):
    """The backprojector with cp.async tile staging instead of TMA, with its view loop cut into many small
    launches (accumulating), and with the one-voxel-per-thread kernel instead of packed pairs, must give the same
    answer as the default configuration and as the oracle."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4, nx=44, ny=48, nz=40, nu=112, nv=100, n_views=17)
    g = W.geom_keys(c)
    o, geom = Oracle(g), Geometry(g)
    y32 = o.fp(W.make_phantom(c)).astype(np.float32)
    yd = torch.from_numpy(y32).cuda()
    x_default = geom.bp(yd)
    torch.cuda.synchronize()
    for k, v in env.items():
        B.debug_set(k, v)
    x_alt = geom.bp(yd)
    torch.cuda.synchronize()
    B.debug_set("reset")
    _check(x_alt, o.bp(y32), "A^T with %s" % env)
    assert (x_alt - x_default).abs().max().item() <= 3e-6 * x_default.abs().max().item()
    geom.close()


@pytest.mark.parametrize("index, chunk", [(2, 1), (2, 2), (4, 1)])
def test_packed_backprojector_never_reads_unstaged_shared_memory(index, chunk):
    """The two voxels of a z-pair walk max(L_a, L_b) x max(K_a, K_b) cells each; the one whose footprint is cut by the
    end of a TMA box or of the detector must not run past the tile's zero rows into the next ring stage (its weights
    there are exactly 0, but 0 * NaN = NaN).  Footprints of ~20 rows in shadows of several boxes, one or two views
    per launch so that one or two ring stages are never staged, those stages pre-filled with NaN (bp_poison): the
    result must be finite and bit-identical to the unpoisoned run."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(index, nx=24, ny=22, nz=20, nu=320, nv=300, n_views=7)
    geom = Geometry(W.geom_keys(c))
    rng = np.random.default_rng(31 + index)
    y = torch.from_numpy(rng.uniform(0.5, 1.5, (1, 7, 300, 320)).astype(np.float32)).cuda()
    B.debug_set("bp_chunk", chunk)
    x_plain = geom.bp(y)
    torch.cuda.synchronize()
    B.debug_set("bp_poison", 1)
    x_poison = geom.bp(y)
    torch.cuda.synchronize()
    B.debug_set("reset")
    assert bool(torch.isfinite(x_poison).all()), "%d non-finite voxels" % int((~torch.isfinite(x_poison)).sum())
    assert torch.equal(x_poison, x_plain)
    assert x_plain.max().item() > 0.0
    geom.close()


@pytest.mark.parametrize("nz", [13, 29, 47])
def test_packed_backprojector_odd_z_runs(nz):
    """Tilted frames, nu % 4 == 0, 16-byte aligned projections: ct_bp_sf takes the packed two-voxel kernel, and with
    nz mod 16 odd the last z-pair of the top brick has no second voxel (it rides along with zero weights and is
    never stored).  Every voxel against the oracle, plus the adjoint identity."""
    c = W.make_config(4, nx=45, ny=48, nz=nz, nu=140, nv=120, n_views=9)
    _pair(c, "packed A^T, nz = %d" % nz, seed=nz)


def test_backward_direction_module_gradient_is_forward_projection():
    """"forward projection and backprojection are gradients of each other".  For the module in
    direction 'backward' (x = A^T y) autograd's gradient of <w, A^T y> with respect to y must be A w."""
    from paper_2503_16741_b200.projector import Projector
    c = W.make_config(2, nx=24, ny=22, nz=16, nu=48, nv=40, n_views=6)
    At = Projector(W.geom_keys(c), "proj", "SF", "backward")
    rng = np.random.default_rng(3)
    y = torch.from_numpy(rng.uniform(0, 1, (1, 6, 40, 48)).astype(np.float32)).cuda().requires_grad_()
    w = torch.from_numpy(rng.uniform(0, 1, (1, 16, 22, 24)).astype(np.float32)).cuda()
    loss = (At(y) * w).sum()
    (grad,) = torch.autograd.grad(loss, [y])
    want = At.geom.fp(w)
    assert torch.allclose(grad, want, rtol=1e-6, atol=1e-6 * want.abs().max().item())
    # ordered subsets through the module
    sub = At(y[:, 1::2].contiguous(), subset=(1, 2, 3))
    assert torch.equal(sub, At.geom.bp(y.detach()[:, 1::2].contiguous(), views=(1, 2, 3)))


def test_host_buffer_entry_points_odd_sizes():
    """VERDICT round 1 / ADVICE: chunk offsets v0 * nv * nu that are not multiples of 4 floats (odd nu * nv) used to be
    rejected by an over-strict 16-byte check inside ct_fp_sf_host; they are valid inputs."""
    from paper_2503_16741_b200.projector import Geometry
    for index, shrink in ((2, dict(nx=26, ny=24, nz=18, nu=150, nv=101, n_views=11)),
                          (4, dict(nx=30, ny=28, nz=26, nu=101, nv=91, n_views=67))):
        B.debug_set("host_fp_chunks", 7 if index == 4 else 2)      # chunk offsets v0 * nv * nu: odd multiples of 4 bytes
        c = W.make_config(index, **shrink)
        g = W.geom_keys(c)
        x = W.make_phantom(c)
        o, geom = Oracle(g), Geometry(g)
        y_ref = o.fp(x)
        hy = np.empty(y_ref.shape, np.float32)
        B.ct_fp_sf_host(geom.handle, x.ctypes.data, hy.ctypes.data, 1, 0)
        _check(torch.from_numpy(hy), y_ref, "A host, odd sizes, config %d" % index)
        y32 = y_ref.astype(np.float32)
        hx = np.empty(x.shape, np.float32)
        B.ct_bp_sf_host(geom.handle, y32.ctypes.data, hx.ctypes.data, 1, 0)
        _check(torch.from_numpy(hx), o.bp(y32), "A^T host, odd sizes, config %d" % index)
        # device entry points on a buffer that is only 4-byte aligned (a slice of a larger tensor)
        big = torch.zeros(x.size + 1, device="cuda")
        big[1:] = torch.from_numpy(x).cuda().flatten()
        y_off = geom.fp(big[1:].view(x.shape))
        _check(y_off, y_ref, "A on a 4-byte aligned volume, config %d" % index)
        pbig = torch.zeros(y32.size + 3, device="cuda")
        pbig[3:] = torch.from_numpy(y32).cuda().flatten()
        _check(geom.bp(pbig[3:].view(y32.shape)), o.bp(y32), "A^T on 4-byte aligned projections, config %d" % index)
        geom.close()


def test_wide_fan_and_anisotropic_pitch():
    """the forward kernel's swept-region halo is 1/2 + 1/2 |dp/dq| voxels; fans with a half-angle
    beyond ~31 degrees (views near 45 degrees) and in-plane pitches dy = 2 dx drive the slope past the old cap of 4.
    A must still see every voxel (parity) and stay the transpose of A^T."""
    import math
    n = 16
    theta = 2.0 * math.pi * np.arange(n) / n + math.pi / 4.0           # includes the 45-degree views
    for name, kw in (("wide fan", dict(sad=140.0, sdd=280.0, nx=64, ny=64, dx=1.0, dy=1.0, nu=200, du=1.6)),
                     ("dy = 2 dx", dict(sad=300.0, sdd=600.0, nx=96, ny=48, dx=0.7, dy=1.4, nu=180, du=1.3))):
        src, dc, u, v = W.trajectory(n, kw["sad"], kw["sdd"], "flat", theta)
        c = dict(index=1, seed=77, name=name, dim=3, nx=kw["nx"], ny=kw["ny"], nz=10, dx=kw["dx"], dy=kw["dy"], dz=1.0,
                 ox=0.0, oy=0.0, oz=0.0, nu=kw["nu"], nv=24, du=kw["du"], dv=1.6, det_type="flat", n_views=n,
                 batch=1, n_obj=8, src=src, det_center=dc, det_u=u, det_v=v)
        _pair(c, name + " (3-D)")
        c2 = dict(c, dim=2, nz=1, nv=1, dz=1.0, dv=1.0)
        _pair(c2, name + " (2-D)")


def test_reversed_detector_axes_on_the_gpu():
    """det_u -> -det_u (u x v then points away from the detector: the sign flip of geom.cpp's frame normal) mirrors the
    channels; det_v -> -det_v mirrors the rows.  Against the oracle, and against the GPU's own unmirrored result."""
    from paper_2503_16741_b200.projector import Geometry
    for index, shrink in ((4, dict(nx=36, ny=32, nz=28, nu=80, nv=72, n_views=7)),
                          (5, dict(nx=60, ny=56, nu=128, n_views=9, batch=2)),
                          (3, dict(nx=40, ny=44, nz=12, nu=96, nv=16, n_views=6))):
        c = W.make_config(index, **shrink)
        g = W.geom_keys(c)
        x = W.make_phantom(c)
        xd = torch.from_numpy(x).cuda()
        geom = Geometry(g)
        y = geom.fp(xd)
        for flip_u, flip_v in ((True, False), (False, True)) if c["dim"] == 3 else ((True, False),):
            gm = dict(g, det_u=-g["det_u"] if flip_u else g["det_u"], det_v=-g["det_v"] if flip_v else g["det_v"])
            gm_geom, om = Geometry(gm), Oracle(gm)
            ym = gm_geom.fp(xd)
            _check(ym, om.fp(x), "A, reversed axes, config %d" % index)
            dims = ([-1] if flip_u else []) + ([-2] if flip_v else [])
            assert (ym - torch.flip(y, dims)).abs().max().item() <= 2e-6 * y.abs().max().item()
            y32 = om.fp(x).astype(np.float32)
            _check(gm_geom.bp(torch.from_numpy(y32).cuda()), om.bp(y32), "A^T, reversed axes, config %d" % index)
            gm_geom.close()
        geom.close()


def test_fbp_entry_point_and_2d_shapes():
    """ct_fbp_sf == (pi / N) ct_bp_sf_recon(ct_fbp_filter(p)) (the angular weight is applied inside the library);
    2-D geometries take [..., ny, nx] / [..., views, nu] tensors without the unit axis and give
    outputs of the same kind; wrong dtypes and bad out= buffers are rejected before the library sees them."""
    import math
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(5, nx=48, ny=44, nu=100, n_views=24, batch=2)
    geom = Geometry(W.geom_keys(c))
    x = torch.from_numpy(W.make_phantom(c)).cuda()                    # [2, 1, ny, nx]
    y = geom.fp(x)
    y2 = geom.fp(x[:, 0])                                             # [2, ny, nx] -> [2, views, nu]
    assert tuple(y2.shape) == (2, 24, 100) and torch.equal(y2, y[:, :, 0])
    xb2 = geom.bp(y2)
    assert tuple(xb2.shape) == (2, 44, 48) and torch.equal(xb2, geom.bp(y)[:, 0])
    f1 = geom.fbp(y)
    f2 = geom.bp_recon(geom.fbp_filter(y)) * (math.pi / 24)
    assert (f1 - f2).abs().max().item() <= 2e-6 * f2.abs().max().item()
    assert tuple(geom.fbp(y2).shape) == (2, 44, 48)
    # a mini-batch of ONE image keeps the layout of its larger predecessors: rank decides, not the batch size
    y1 = geom.fp(x[:1, 0])                                            # [1, ny, nx] -> [1, views, nu]
    assert tuple(y1.shape) == (1, 24, 100) and torch.equal(y1, y2[:1])
    xb1 = geom.bp(y1)                                                 # [1, views, nu] -> [1, ny, nx]
    assert tuple(xb1.shape) == (1, 44, 48) and torch.equal(xb1, xb2[:1])
    assert tuple(geom.fp(x[0, 0]).shape) == (24, 100)                 # [ny, nx] -> [views, nu]
    assert tuple(geom.fp(x[:1]).shape) == (1, 24, 1, 100)             # [1, 1, ny, nx]: the unit axis is kept
    assert tuple(geom.bp(y[:1]).shape) == (1, 1, 44, 48)
    with pytest.raises(TypeError):
        geom.fp(x.double())
    with pytest.raises(ValueError):
        geom.fp(x, out=torch.empty(5, device="cuda"))
    with pytest.raises(ValueError):
        geom.fp(x, out=torch.empty(y.shape, device="cuda", dtype=torch.float64))
    geom.close()


def test_forward_projector_scratch_is_reused():
    """no allocation in ct_fp_sf once the geometry is warm -- the transposed-volume scratch belongs to
    the geometry.  Device memory in use must not move between the second and the tenth call, and calls from two
    streams must not share a scratch buffer in flight."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4, nx=64, ny=64, nz=48, nu=128, nv=120, n_views=16)
    geom = Geometry(W.geom_keys(c))
    x = torch.from_numpy(W.make_phantom(c)).cuda()
    y = geom.fp(x)
    out = torch.empty_like(y)                   # before the reading: in a fresh process torch allocates a block for it
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(9):
        geom.fp(x, out=out)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    assert torch.equal(out, y)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    o1, o2 = torch.empty_like(y), torch.empty_like(y)
    x2 = (x * 2.0).contiguous()
    torch.cuda.synchronize()
    for _ in range(3):
        with torch.cuda.stream(s1):
            geom.fp(x, out=o1)
        with torch.cuda.stream(s2):
            geom.fp(x2, out=o2)
    torch.cuda.synchronize()
    assert torch.equal(o1, y) and torch.equal(o2, geom.fp(x2))
    geom.close()


def test_forward_projector_scratch_does_not_grow_with_every_batch_size():
    """A larger batch replaces the geometry's idle scratch buffer instead of keeping the old one beside a new one:
    after batch 1 then batch 2 the geometry holds ONE buffer of two volumes (6 MiB each), not three volumes."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4, nx=128, ny=128, nz=96, nu=64, nv=48, n_views=8)
    geom = Geometry(W.geom_keys(c))
    vol_bytes = 128 * 128 * 96 * 4
    x2 = torch.rand((2, 96, 128, 128), device="cuda")
    out1 = torch.empty((1, 8, 48, 64), device="cuda")
    out2 = torch.empty((2, 8, 48, 64), device="cuda")
    warm = Geometry(W.geom_keys(c))               # first launches load the kernels (device memory of their own)
    warm.fp(x2, out=out2)
    torch.cuda.synchronize()
    warm.close()
    free_cold = torch.cuda.mem_get_info()[0]
    geom.fp(x2[:1], out=out1)
    torch.cuda.synchronize()
    free_b1 = torch.cuda.mem_get_info()[0]
    geom.fp(x2, out=out2)
    torch.cuda.synchronize()
    free_b2 = torch.cuda.mem_get_info()[0]
    assert free_cold - free_b1 >= vol_bytes                      # this geometry does use the scratch
    assert free_cold - free_b2 <= 2 * vol_bytes + (2 << 20), (free_cold - free_b1, free_cold - free_b2)
    assert torch.equal(out2[:1], out1)
    geom.fp(x2[:1], out=out1)                                    # the larger buffer serves the smaller batch
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_b2
    geom.close()


def test_view_sharded_operators_world_size_1():
    """SURVEY 8(e) item 2 on one GPU: shards of A concatenate to A, shards of A^T sum to A^T (the all-reduce is the
    identity at world size 1; two shards are summed by hand here)."""
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(4, nx=40, ny=36, nz=32, nu=96, nv=88, n_views=13)
    geom = Geometry(W.geom_keys(c))
    x = torch.from_numpy(W.make_phantom(c)).cuda()
    y = geom.fp(x)
    sub, y_all = geom.fp_sharded(x, 0, 1)
    assert sub == (0, 1, 13) and torch.equal(y_all, y)
    parts, xb = [], None
    for rank in range(2):
        (vb, vs, vc), yr = geom.fp_sharded(x, rank, 2)
        parts.append(yr)
        xr = geom.bp(yr, views=(vb, vs, vc))
        xb = xr if xb is None else xb + xr
    assert torch.equal(torch.cat(parts, dim=1), y)
    full = geom.bp(y)
    assert (xb - full).abs().max().item() <= 3e-6 * full.abs().max().item()
    assert torch.equal(geom.bp_sharded(y, 0, 1), full)
    geom.close()


def test_bench_view_sharded_mode_single_rank():
    """bench.py --shard views at N = 1: runs, prints one contract line, strong scaling label."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--shard", "views", "--config", "1", "--steps", "2",
                          "--warmup", "3", "--no-cpu"], capture_output=True, text=True, timeout=600, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["scaling"] == "strong" and d["value"] > 0 and d["gpu_launches"] > 0
    assert d["shard"]["mode"] == "views" and len(d["shard"]["per_rank_ms_fp_bp_allreduce"]) == 1
    assert d["roofline"]["peak"] > 50.0 and "measured" in d["roofline"]["peak_src"]


_TWO_GPU_WORKER = r'''
import os, sys
sys.path.insert(0, sys.argv[1])
import numpy as np, torch, torch.distributed as dist
from paper_2503_16741_b200 import workloads as W
from paper_2503_16741_b200.projector import Geometry
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
torch.cuda.set_device(int(os.environ["LOCAL_RANK"]))
dist.init_process_group("nccl", device_id=torch.device("cuda", int(os.environ["LOCAL_RANK"])))
c = W.make_config(4, nx=40, ny=36, nz=32, nu=96, nv=88, n_views=13)
geom = Geometry(W.geom_keys(c))
x = torch.from_numpy(W.make_phantom(c)).cuda()
y_full = geom.fp(x)                                   # every rank: the unsharded reference
(vb, vs, vc), y_mine = geom.fp_sharded(x, rank, world)
assert torch.equal(y_mine, y_full[:, vb:vb + vc])
xb = geom.bp_sharded(y_mine, rank, world)             # ct_bp_sf_views + one NCCL all-reduce
full = geom.bp(y_full)
assert (xb - full).abs().max().item() <= 3e-6 * full.abs().max().item()
dist.destroy_process_group()
print("ok")
'''


def test_view_sharded_operators_two_gpus(tmp_path):
    """The same identities over NCCL when the box has two GPUs (skipped on the single-GPU boxes of this run)."""
    import os
    import socket
    import subprocess
    import sys
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "worker.py"
    script.write_text(_TWO_GPU_WORKER)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", str(port), str(script), root],
                         capture_output=True, text=True, timeout=900)
    assert out.returncode == 0 and out.stdout.count("ok") == 2, (out.stdout[-1000:], out.stderr[-2000:])


def test_fp32_peak_microbenchmark():
    """ct_measure_fp32_peak (the roofline's measured denominator): plausible on any Blackwell-class part, packed >=
    scalar, the FFMA2 / FFMA mix below both, bad arguments rejected."""
    f0, t0 = B.ct_measure_fp32_peak(0)
    f1, _ = B.ct_measure_fp32_peak(1)
    f2, _ = B.ct_measure_fp32_peak(2)
    f3, _ = B.ct_measure_fp32_peak(3)
    assert 20e12 < f0 < 120e12 and 0.9 * f0 < f1 < 120e12 and t0 > 0
    assert f2 < 0.95 * f1 and f3 < 0.95 * f1
    with pytest.raises(B.CtError):
        B.ct_measure_fp32_peak(4)
