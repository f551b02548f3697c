"""ct_fp_sf_noalloc: the forward projector for callers that may not allocate device memory while they run.

Who needs it: a reconstruction loop living inside a process whose GPU memory already belongs to another allocator
(a framework's caching pool, a fixed budget on a shared GPU), a loop with a latency bound that cannot take the
device-wide stall of a cudaMalloc, a service that is not allowed to grow after start-up.  For them the library keeps
the forward projector's one scratch buffer (the xy-transposed volume) in a fixed 16 MiB array of its own image
instead of allocating it; the price is a size limit and one array shared by every call on a GPU.

What is checked here, through the C ABI: the new entry point returns what ct_fp_sf returns (the tolerance of the
parity tests, tests/test_gpu_parity.py) on two calls in a row with different volumes -- the second call must not see
what the first one left in the shared array -- then on a smaller, batched 2-D geometry that reuses only the front of
the array; a problem beyond the limit is refused with a clear error and nothing is written.

This file is named to be collected LAST (pytest -x stops at the first failure: a failure here hides no other test).
It passes alone in a fresh process (its first call does the once-per-GPU set-up) and after the other GPU tests."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from paper_2503_16741_b200 import binding as B
from paper_2503_16741_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _close(got, want, what):
    got, want = got.double(), want.double()
    rel = (torch.linalg.norm(got - want) / torch.linalg.norm(want)).item()
    mx = ((got - want).abs().max() / want.abs().max()).item()
    assert rel <= 1e-5 and mx <= 1e-4, "%s: rel-L2 %.3e max-abs/max %.3e" % (what, rel, mx)


def _noalloc_fp(geom, x, batch):
    """y = A x through ct_fp_sf_noalloc on torch's current stream; y pre-filled with NaN so that a cell the call
    fails to write cannot pass."""
    y = torch.full((batch, geom.n_views) + geom.det_shape, float("nan"), device=x.device)
    B.ct_fp_sf_noalloc(geom.handle, x.data_ptr(), y.data_ptr(), batch, torch.cuda.current_stream().cuda_stream)
    return y


def test_noalloc_forward_matches_ct_fp_sf_on_consecutive_calls():
    from paper_2503_16741_b200.projector import Geometry
    # tilted, jittered cone-beam frames over a full turn (config 4, shrunk): about half the views run along x and
    # read the volume through the transposed copy, i.e. through the fixed array
    c = W.make_config(4, nx=61, ny=64, nz=58, nu=140, nv=135, n_views=12)
    geom = Geometry(W.geom_keys(c))
    x1 = torch.from_numpy(W.make_phantom(c)).cuda()
    rng = np.random.default_rng(7)
    x2 = torch.from_numpy(rng.uniform(0.0, 1.0, tuple(x1.shape)).astype(np.float32)).cuda()

    y1 = _noalloc_fp(geom, x1, 1)
    assert geom.last_launch_count() >= 2, "the transposed-volume scratch was not used: pick other views"
    y2 = _noalloc_fp(geom, x2, 1)                       # second call in a row, same array, other contents
    torch.cuda.synchronize()
    _close(y1.view(-1), geom.fp(x1).view(-1), "first call")
    _close(y2.view(-1), geom.fp(x2).view(-1), "second call")
    geom.close()

    # a smaller problem next (2-D fan beam, batch of 5): only the front of the array is rewritten, the rest still
    # holds the 3-D volume of the calls above and must not matter
    c5 = W.make_config(5, nx=96, ny=90, nu=290, n_views=17, batch=5)
    geom5 = Geometry(W.geom_keys(c5))
    x5 = torch.from_numpy(W.make_phantom(c5)).cuda()
    y5 = _noalloc_fp(geom5, x5, 5)
    y5b = _noalloc_fp(geom5, x5, 5)
    torch.cuda.synchronize()
    ref5 = geom5.fp(x5).view(-1)
    _close(y5.view(-1), ref5, "2-D batch")
    _close(y5b.view(-1), ref5, "2-D batch, again")
    geom5.close()


def test_noalloc_forward_refuses_what_does_not_fit():
    from paper_2503_16741_b200.projector import Geometry
    c = W.make_config(5, nx=96, ny=90, nu=290, n_views=17, batch=5)
    geom = Geometry(W.geom_keys(c))
    per_image = 96 * 90
    too_many = B.CT_FP_SF_NOALLOC_MAX_VOXELS // per_image + 1          # one image more than the array holds
    x = torch.zeros((too_many, 1, 90, 96), device="cuda")
    y = torch.full((too_many, geom.n_views) + geom.det_shape, -1.0, device="cuda")
    with pytest.raises(B.CtError) as e:
        B.ct_fp_sf_noalloc(geom.handle, x.data_ptr(), y.data_ptr(), too_many, torch.cuda.current_stream().cuda_stream)
    assert e.value.status == 3 and "exceeds the fixed scratch" in str(e.value)
    torch.cuda.synchronize()
    assert bool((y == -1.0).all()), "a refused call must not queue any work"
    # the largest batch that fits is accepted
    fits = too_many - 1
    y_ok = _noalloc_fp(geom, x[:fits], fits)
    torch.cuda.synchronize()
    assert bool((y_ok == 0.0).all())                                     # A 0 = 0, every cell written
    geom.close()
