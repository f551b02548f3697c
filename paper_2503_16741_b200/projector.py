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
        self.algo = {0: "SF", 1: "DD", 2: "SF-TT"}.get(g.get("algo", "SF"), g.get("algo", "SF"))
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
        lead, batch, vol, sq = _prep(vol, self.vol_shape, -3 if self.dim == 2 else None)
        out = _out(out, (batch, vc) + self.det_shape, vol.device)
        B.ct_fp_sf_views(self.handle, vol.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                         torch.cuda.current_stream(vol.device).cuda_stream)
        return out.view(lead + self._tail((vc,) + self.det_shape, -2, sq))

    def bp(self, proj, views=None, out=None):
        """proj [..., n_sel, nv, nu] -> vol [..., nz, ny, nx]."""
        vb, vs, vc = self._views(views)
        lead, batch, proj, sq = _prep(proj, (vc,) + self.det_shape, -2 if self.dim == 2 else None)
        out = _out(out, (batch,) + self.vol_shape, proj.device)
        B.ct_bp_sf_views(self.handle, proj.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                         torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + self._tail(self.vol_shape, -3, sq))

    # ---- recon mode (readings R23, R24) --------------------------------
    def fbp_filter(self, proj, views=None, out=None):
        """Cosine pre-weight + discrete ramp filter along the channels; proj [..., n_sel, nv, nu] -> same shape."""
        vb, vs, vc = self._views(views)
        lead, batch, proj, sq = _prep(proj, (vc,) + self.det_shape, -2 if self.dim == 2 else None)
        out = _out(out, tuple(proj.shape), proj.device)
        B.ct_fbp_filter_views(self.handle, proj.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                              torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + self._tail((vc,) + self.det_shape, -2, sq))

    def bp_recon(self, proj, views=None, out=None):
        """Recon-mode backprojection (normalised footprints x depth weight); proj [..., n_sel, nv, nu] -> volume."""
        vb, vs, vc = self._views(views)
        lead, batch, proj, sq = _prep(proj, (vc,) + self.det_shape, -2 if self.dim == 2 else None)
        out = _out(out, (batch,) + self.vol_shape, proj.device)
        B.ct_bp_sf_recon_views(self.handle, proj.data_ptr(), out.data_ptr(), batch, vb, vs, vc,
                               torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + self._tail(self.vol_shape, -3, sq))

    def fbp(self, proj, out=None):
        """Filtered backprojection of N equi-angular views over 360 degrees: (pi / N) B(filter(p)) (ct_fbp_sf)."""
        lead, batch, proj, sq = _prep(proj, (self.n_views,) + self.det_shape, -2 if self.dim == 2 else None)
        out = _out(out, (batch,) + self.vol_shape, proj.device)
        work = torch.empty_like(proj)
        B.ct_fbp_sf(self.handle, proj.data_ptr(), work.data_ptr(), out.data_ptr(), batch,
                    torch.cuda.current_stream(proj.device).cuda_stream)
        return out.view(lead + self._tail(self.vol_shape, -3, sq))

    def _tail(self, tail, unit_axis, squeezed):
        """Output tail shape: 2-D inputs given without their unit axis ([..., ny, nx] / [..., views, nu], the paper's
        own usage; `squeezed` as reported by _prep) get outputs without theirs too."""
        tail = tuple(tail)
        if self.dim == 2 and squeezed:
            i = len(tail) + unit_axis
            return tail[:i] + tail[i + 1:]
        return tail

    def last_launch_count(self):
        return B.ct_last_launch_count(self.handle)

    # ---- view-sharded operators -------------------------------
    def fp_sharded(self, vol, rank, world_size, out=None):
        """This rank's views of A x (volume replicated): returns ((view_begin, view_stride, view_count), projections)."""
        from .geometry import shard_views
        sub = shard_views(self.n_views, world_size, rank)
        return sub, self.fp(vol, views=sub, out=out)

    def bp_sharded(self, proj_shard, rank, world_size, group=None, out=None):
        """A^T y with the views sharded over the ranks of `group`: every rank backprojects its own shard
        (ct_bp_sf_views) into a full-size partial volume; ONE sum all-reduce (NCCL) makes them the result."""
        import torch.distributed as dist
        from .geometry import shard_views
        sub = shard_views(self.n_views, world_size, rank)
        x = self.bp(proj_shard, views=sub, out=out)
        if world_size > 1:
            dist.all_reduce(x, op=dist.ReduceOp.SUM, group=group)
        return x


def _prep(t, tail, unit_axis=None):
    """(lead, batch, view, squeezed): the contiguous fp32 view [batch, *tail] of a CUDA tensor whose trailing dims are
    `tail`, the leading dims it had, and whether the unit axis was missing.  unit_axis (2-D geometries): index in `tail`
    of the unit z / row axis, which may be left out: [..., ny, nx] and [..., views, nu] are accepted.
    One shape reads both ways -- a rank-3 [1, ny, nx] is "one image with its unit z axis" and "a batch of one image
    without it".  Rank decides, never the batch size: a tensor of exactly len(tail) dims given to a 2-D geometry is
    [batch, ny, nx] (so the last mini-batch of a loop, of size 1, comes back as [1, views, nu] like its predecessors
    came back as [B, views, nu]); the unit axis counts from rank len(tail) + 1 on ([B, 1, ny, nx])."""
    if not t.is_cuda:
        raise RuntimeError("ctsf operators take CUDA tensors (no CPU fallback)")
    if t.dtype != torch.float32:
        raise TypeError("ctsf operators compute in float32; got %s (cast explicitly)" % t.dtype)
    tail = tuple(tail)
    nd = len(tail)
    full = t.dim() >= nd and tuple(t.shape[-nd:]) == tail
    i = nd + unit_axis if unit_axis is not None else None
    short = tail[:i] + tail[i + 1:] if i is not None and tail[i] == 1 else None
    squeezed = short is not None and t.dim() >= nd - 1 and tuple(t.shape[-(nd - 1):]) == short and \
        (not full or t.dim() == nd)
    if squeezed:
        t = t.unsqueeze(t.dim() - (nd - 1) + i)
    elif not full:
        raise ValueError("expected trailing shape %s, got %s" % (tail, tuple(t.shape)))
    lead = tuple(t.shape[:-nd])
    t = t.detach().contiguous()
    batch = 1
    for s in lead:
        batch *= s
    if batch < 1:
        raise ValueError("empty batch")
    return lead, batch, t.view((batch,) + tail), squeezed


def _out(out, shape, device):
    """A fresh output, or the caller's after checking what the library cannot: dtype, device, size, contiguity."""
    if out is None:
        return torch.empty(shape, device=device, dtype=torch.float32)
    n = 1
    for s in shape:
        n *= s
    if out.dtype != torch.float32 or out.device != device or out.numel() != n or not out.is_contiguous():
        raise ValueError("out= must be a contiguous float32 tensor of %d elements on %s" % (n, device))
    return out


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
    Algorithm 'SF' (separable footprint, SF-TR), 'SF-TT' (trapezoid axial factor) or 'DD' (distance-driven); mode 'proj' (matched pair, differentiable) or 'recon' (FBP backprojection of
    PAPER.md:103, direction 'backward' only); direction is 'forward' or 'backward'.
    `subset=(view_begin, view_stride, view_count)` restricts to an ordered subset."""

    def __init__(self, geom, mode="proj", algo="SF", direction="forward"):
        super().__init__()
        if mode not in ("proj", "recon") or algo not in ("SF", "DD", "SF-TT"):
            raise NotImplementedError("algo 'SF', 'SF-TT' or 'DD' with mode 'proj' or 'recon' is built (see DESIGN.md)")
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
