"""torch-facing layer: geometry handle, autograd Functions, and an nn.Module.

PyTorch supplies device memory, streams and the autograd tape only; the arithmetic is in libctsf.
`FP.backward` is ct_bp_sf and `BP.backward` is ct_fp_sf because the pair is matched
("forward projection and backprojection are gradients of each other").
"""
import torch

from . import binding as B


class Geometry:
    """Owns a ct_geom_t.  `g` is a problem-description dict (see binding.ct_geom_create)."""

    def __init__(self, g):
        if not torch.cuda.is_available():
            raise RuntimeError("ctsf needs a CUDA device (no CPU fallback)")
        torch.cuda.current_device()          # make sure a context exists before libctsf allocates
        torch.zeros(1, device="cuda")
        self.handle = B.ct_geom_create(g)
        self.algo = {0: "SF", 1: "DD"}.get(g.get("algo", "SF"), g.get("algo", "SF"))
        self.dim = int(g["dim"])
        self.vol_shape = (int(g.get("nz", 1)), int(g["ny"]), int(g["nx"]))
        self.n_views = len(g["src"])
        self.det_shape = (int(g.get("nv", 1)), int(g["nu"]))

    def close(self):
        if getattr(self, "handle", None):
            B.ct_geom_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- raw operators on contiguous fp32 CUDA tensors -------------------------------------------
    def _views(self, views):
        if views is None:
            return 0, 1, self.n_views
        vb, vs, vc = views
        return int(vb), int(vs), int(vc)

    def fp(self, vol, views=None, out=None):
        """vol [..., nz, ny, nx] -> proj [..., n_sel, nv, nu]."""
        vb, vs, vc = self._views(views)
        lead, batch, vol = _prep(vol, self.vol_shape)
        if out is None:
            out = torch.empty((batch, vc) + self.det_shape, device=vol.device, dtype=torch.float32)
        B.ct_fp_sf_views(self.handle, vol.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                         torch.cuda.current_stream(vol.device).cuda_stream)
        return out.view(lead + (vc,) + self.det_shape)

    def bp(self, proj, views=None, out=None):
        """proj [..., n_sel, nv, nu] -> vol [..., nz, ny, nx]."""
        vb, vs, vc = self._views(views)
        lead, batch, proj = _prep(proj, (vc,) + self.det_shape)
        if out is None:
            out = torch.empty((batch,) + self.vol_shape, device=proj.device, dtype=torch.float32)
        B.ct_bp_sf_views(self.handle, proj.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                         torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + self.vol_shape)

    # ---- recon mode (readings R23, R24) --------------------------------
    def fbp_filter(self, proj, views=None, out=None):
        """Cosine pre-weight + discrete ramp filter along the channels; proj [..., n_sel, nv, nu] -> same shape."""
        vb, vs, vc = self._views(views)
        lead, batch, proj = _prep(proj, (vc,) + self.det_shape)
        if out is None:
            out = torch.empty_like(proj)
        B.ct_fbp_filter_views(self.handle, proj.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                              torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + (vc,) + self.det_shape)

    def bp_recon(self, proj, views=None, out=None):
        """Recon-mode backprojection (normalised footprints x depth weight); proj [..., n_sel, nv, nu] -> volume."""
        vb, vs, vc = self._views(views)
        lead, batch, proj = _prep(proj, (vc,) + self.det_shape)
        if out is None:
            out = torch.empty((batch,) + self.vol_shape, device=proj.device, dtype=torch.float32)
        B.ct_bp_sf_recon_views(self.handle, proj.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                               torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + self.vol_shape)

    def fbp(self, proj):
        """Filtered backprojection of N equi-angular views over 360 degrees: (pi / N) B(filter(p))."""
        import math
        return self.bp_recon(self.fbp_filter(proj)).mul_(math.pi / self.n_views)

    def last_launch_count(self):
        return B.ct_last_launch_count(self.handle)


def _prep(t, tail):
    if not t.is_cuda:
        raise RuntimeError("ctsf operators take CUDA tensors (no CPU fallback)")
    nd = len(tail)
    if tuple(t.shape[-nd:]) != tuple(tail):
        raise ValueError("expected trailing shape %s, got %s" % (tail, tuple(t.shape)))
    lead = tuple(t.shape[:-nd])
    t = t.detach().to(torch.float32).contiguous()
    batch = 1
    for s in lead:
        batch *= s
    if batch < 1:
        raise ValueError("empty batch")
    return lead, batch, t.view((batch,) + tuple(tail))


class FP(torch.autograd.Function):
    """y = A x; backward: grad_x = A^T grad_y."""

    @staticmethod
    def forward(ctx, vol, geom, views=None):
        ctx.geom, ctx.views = geom, views
        return geom.fp(vol, views)

    @staticmethod
    def backward(ctx, grad):
        return ctx.geom.bp(grad, ctx.views), None, None


class BP(torch.autograd.Function):
    """x = A^T y; backward: grad_y = A grad_x."""

    @staticmethod
    def forward(ctx, proj, geom, views=None):
        ctx.geom, ctx.views = geom, views
        return geom.bp(proj, views)

    @staticmethod
    def backward(ctx, grad):
        return ctx.geom.fp(grad, ctx.views), None, None


class Projector(torch.nn.Module):
    """`A = Projector(geom, 'proj', 'SF', 'forward'); sino = A(img)`.
    Algorithm 'SF' (separable footprint) or 'DD' (distance-driven); mode 'proj' (matched pair, differentiable) or 'recon' (FBP backprojection of
    PAPER.md:103, direction 'backward' only); direction is 'forward' or 'backward'.
    `subset=(view_begin, view_stride, view_count)` restricts to an ordered subset."""

    def __init__(self, geom, mode="proj", algo="SF", direction="forward"):
        super().__init__()
        if mode not in ("proj", "recon") or algo not in ("SF", "DD"):
            raise NotImplementedError("algo 'SF' or 'DD' with mode 'proj' or 'recon' is built (see DESIGN.md)")
        if direction not in ("forward", "backward"):
            raise ValueError(direction)
        if mode == "recon" and direction != "backward":
            raise NotImplementedError("'recon' mode is the FBP backprojection: direction must be 'backward'")
        self.mode = mode
        if isinstance(geom, Geometry):
            if geom.algo != algo:
                raise ValueError("the Geometry was created for algo=%r, not %r" % (geom.algo, algo))
            self.geom = geom
        else:
            self.geom = Geometry(dict(geom, algo=algo))
        self.direction = direction

    def forward(self, x, subset=None):
        if self.mode == "recon":            # not differentiable: FBP is used for reconstruction only
            return self.geom.bp_recon(x, subset)
        return (FP if self.direction == "forward" else BP).apply(x, self.geom, subset)
