"""ctypes wrapper around oracle/sf_oracle.c -- the float64 CPU oracle.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module.  It imports nothing from the product package and the product imports nothing from here.
All arithmetic lives in sf_oracle.c (readings in DESIGN.md); this file only
marshals numpy arrays.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sf_oracle.c")
_LIB = os.path.join(_HERE, "libsf_oracle.so")


def build(force=False):
    """Compile sf_oracle.c with gcc (-O2, OpenMP).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Geom(ctypes.Structure):
    _fields_ = [("dim", ctypes.c_int), ("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int),
                ("dx", ctypes.c_double), ("dy", ctypes.c_double), ("dz", ctypes.c_double),
                ("ox", ctypes.c_double), ("oy", ctypes.c_double), ("oz", ctypes.c_double),
                ("nu", ctypes.c_int), ("nv", ctypes.c_int),
                ("du", ctypes.c_double), ("dv", ctypes.c_double),
                ("det_type", ctypes.c_int), ("n_views", ctypes.c_int),
                ("src", ctypes.c_void_p), ("det_center", ctypes.c_void_p),
                ("det_u", ctypes.c_void_p), ("det_v", ctypes.c_void_p), ("model", ctypes.c_int)]


_lib = None


def _declare(lib):
    lib.sfo_trap_cdf.restype = ctypes.c_double
    lib.sfo_trap_cdf.argtypes = [ctypes.c_void_p, ctypes.c_double]
    lib.sfo_live_fraction.restype = ctypes.c_double
    P, I = ctypes.c_void_p, ctypes.c_int
    lib.sfo_live_fraction.argtypes = [P, I, I]
    lib.sfo_footprint.argtypes = [P, I, I, I, I, P, P, P, P, P]
    lib.sfo_det_coords.argtypes = [P, I, P, P]
    lib.sfo_fp.argtypes = [P, P, P, I, P]
    lib.sfo_bp.argtypes = [P, P, P, I, P]
    lib.sfo_fbp_filter.argtypes = [P, P, P, I, P]
    lib.sfo_bp_recon.argtypes = [P, P, P, I, P]
    lib.sfo_bp_voxels.argtypes = [P, P, P, I, P]
    lib.sfo_bp_voxels_f32.argtypes = [P, P, P, I, P]
    return lib


def load_library(path):
    """A build of sf_oracle.c other than the in-tree one (tests/test_oracle_mutations.py loads deliberately
    broken copies through this to prove that the pins notice)."""
    return _declare(ctypes.CDLL(path))


def _load():
    global _lib
    if _lib is None:
        _lib = _declare(ctypes.CDLL(build()))
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    """One scan geometry.  `g` is a plain dict with the keys of the problem description:
    dim, nx, ny, nz, dx, dy, dz, ox, oy, oz, nu, nv, du, dv, det_type ('flat'|'arc' or 0|1),
    src, det_center, det_u, det_v (each [n_views, 3], float64); optional algo 'SF' (default) | 'DD' | 'SF-TT' | 'SF-TT-A2'
    (the last two: row f3 variants, oracle only)."""

    def __init__(self, g):
        self.lib = _load()
        self.src = _f64(g["src"]).reshape(-1, 3)
        self.n_views = self.src.shape[0]
        self.dc = _f64(g["det_center"]).reshape(-1, 3)
        self.du_vec = _f64(g["det_u"]).reshape(-1, 3)
        dv = g.get("det_v")
        if dv is None:
            dv = np.tile(np.array([0.0, 0.0, 1.0]), (self.n_views, 1))
        self.dv_vec = _f64(dv).reshape(-1, 3)
        det = g["det_type"]
        det = {"flat": 0, "arc": 1}.get(det, det)
        self.dim = int(g["dim"])
        self.nx, self.ny, self.nz = int(g["nx"]), int(g["ny"]), int(g.get("nz", 1))
        self.nu, self.nv = int(g["nu"]), int(g.get("nv", 1))
        self.g = _Geom(self.dim, self.nx, self.ny, self.nz,
                       float(g["dx"]), float(g["dy"]), float(g.get("dz", 1.0)),
                       float(g.get("ox", 0.0)), float(g.get("oy", 0.0)), float(g.get("oz", 0.0)),
                       self.nu, self.nv, float(g["du"]), float(g.get("dv", 1.0)),
                       int(det), self.n_views,
                       self.src.ctypes.data, self.dc.ctypes.data,
                       self.du_vec.ctypes.data, self.dv_vec.ctypes.data,
                       {"SF": 0, "DD": 1, "SF-TT": 2, "SF-TT-A2": 3}.get(g.get("algo", "SF"), g.get("algo", 0)))
        self.threads = 0

    # -- pins ------------------------------------------------------------------------------
    @staticmethod
    def trap_cdf(tau, s):
        tau = _f64(tau)
        return _load().sfo_trap_cdf(tau.ctypes.data, float(s))

    def footprint(self, view, ix, iy, iz=0):
        """-> dict(k_lo, k_hi, l_lo, l_hi, F1, F2, amp, tau, w[l, k]) or None if off-detector."""
        rng = np.zeros(4, dtype=np.int32)
        F1 = np.zeros(self.nu)
        F2 = np.zeros(self.nv)
        amp = ctypes.c_double(0.0)
        tau = np.zeros(4)
        ok = self.lib.sfo_footprint(ctypes.byref(self.g), int(view), int(ix), int(iy), int(iz),
                                    rng.ctypes.data, F1.ctypes.data, F2.ctypes.data,
                                    ctypes.byref(amp), tau.ctypes.data)
        if not ok:
            return None
        k_lo, k_hi, l_lo, l_hi = [int(v) for v in rng]
        f1 = F1[:k_hi - k_lo + 1].copy()
        f2 = F2[:l_hi - l_lo + 1].copy()
        return dict(k_lo=k_lo, k_hi=k_hi, l_lo=l_lo, l_hi=l_hi, F1=f1, F2=f2, amp=amp.value, tau=tau,
                    w=amp.value * np.outer(f2, f1))

    def det_coords(self, view, P):
        P = _f64(P)
        st = np.zeros(2)
        ok = self.lib.sfo_det_coords(ctypes.byref(self.g), int(view), P.ctypes.data, st.ctypes.data)
        return (st[0], st[1]) if ok else None

    # -- operators ---------------------------------------------------------------------------
    def _views(self, views):
        if views is None:
            views = np.arange(self.n_views)
        return np.ascontiguousarray(views, dtype=np.int32)

    def fp(self, vol, views=None):
        """y = A x.  vol [..., nz, ny, nx] (leading dims = batch); returns [..., n_sel, nv, nu] float64."""
        views = self._views(views)
        vol = _f64(vol)
        lead = vol.shape[:-3] if vol.ndim > 3 else ()
        v = vol.reshape((-1, self.nz, self.ny, self.nx))
        out = np.empty((v.shape[0], len(views), self.nv, self.nu))
        for b in range(v.shape[0]):
            self.threads = self.lib.sfo_fp(ctypes.byref(self.g), v[b].ctypes.data, views.ctypes.data,
                                           len(views), out[b].ctypes.data)
        return out.reshape(lead + (len(views), self.nv, self.nu))

    def bp(self, proj, views=None):
        """x = A^T y.  proj [..., n_sel, nv, nu]; returns [..., nz, ny, nx] float64."""
        views = self._views(views)
        proj = _f64(proj)
        lead = proj.shape[:-3] if proj.ndim > 3 else ()
        p = proj.reshape((-1, len(views), self.nv, self.nu))
        out = np.empty((p.shape[0], self.nz, self.ny, self.nx))
        for b in range(p.shape[0]):
            self.threads = self.lib.sfo_bp(ctypes.byref(self.g), p[b].ctypes.data, views.ctypes.data,
                                           len(views), out[b].ctypes.data)
        return out.reshape(lead + (self.nz, self.ny, self.nx))

    def fbp_filter(self, proj, views=None):
        """Recon mode, reading R24: cosine pre-weight + discrete ramp filter along u.
        proj [..., n_sel, nv, nu] -> same shape, float64."""
        views = self._views(views)
        proj = _f64(proj)
        p = proj.reshape((-1, len(views), self.nv, self.nu))
        out = np.empty_like(p)
        for b in range(p.shape[0]):
            self.lib.sfo_fbp_filter(ctypes.byref(self.g), p[b].ctypes.data, views.ctypes.data, len(views),
                                    out[b].ctypes.data)
        return out.reshape(proj.shape)

    def bp_recon(self, q, views=None):
        """Recon mode, reading R23: x = B q (normalised footprints x depth weight d R / a^2).
        q [..., n_sel, nv, nu]; returns [..., nz, ny, nx] float64."""
        views = self._views(views)
        q = _f64(q)
        lead = q.shape[:-3] if q.ndim > 3 else ()
        p = q.reshape((-1, len(views), self.nv, self.nu))
        out = np.empty((p.shape[0], self.nz, self.ny, self.nx))
        for b in range(p.shape[0]):
            self.lib.sfo_bp_recon(ctypes.byref(self.g), p[b].ctypes.data, views.ctypes.data, len(views),
                                  out[b].ctypes.data)
        return out.reshape(lead + (self.nz, self.ny, self.nx))

    def bp_voxels(self, proj, ijk):
        """(A^T y) at listed voxels; proj is the full [n_views, nv, nu] (float64, or float32 which is
        widened value by value inside the C loop); ijk [n, 3] = (ix, iy, iz)."""
        ijk = np.ascontiguousarray(ijk, dtype=np.int32).reshape(-1, 3)
        out = np.empty(len(ijk))
        assert proj.shape[-3:] == (self.n_views, self.nv, self.nu)
        if proj.dtype == np.float32:
            p = np.ascontiguousarray(proj)
            self.threads = self.lib.sfo_bp_voxels_f32(ctypes.byref(self.g), p.ctypes.data, ijk.ctypes.data,
                                                      len(ijk), out.ctypes.data)
        else:
            p = _f64(proj)
            self.threads = self.lib.sfo_bp_voxels(ctypes.byref(self.g), p.ctypes.data, ijk.ctypes.data,
                                                  len(ijk), out.ctypes.data)
        return out

    def live_fraction(self, vox_stride=8, view_stride=8):
        return self.lib.sfo_live_fraction(ctypes.byref(self.g), int(vox_stride), int(view_stride))

    def num_threads(self):
        return int(self.lib.sfo_num_threads())
