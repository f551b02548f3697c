"""Thin ctypes binding of libctsf.so (include/ctsf.h): argument marshalling only.

Every step of the hot path runs inside the library's CUDA kernels.  There is no CPU fallback: if the
shared library is missing or fails to load, importing a function from here raises.
PyTorch is used by callers for device memory and streams only; this module does not need it.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libctsf.so")

CT_OK = 0
STATUS_NAMES = {0: "CT_OK", 1: "CT_ERR_INVALID_ARG", 2: "CT_ERR_GEOMETRY", 3: "CT_ERR_UNSUPPORTED",
                4: "CT_ERR_ALLOC", 5: "CT_ERR_CUDA"}
EXPORTS = ("ct_geom_create", "ct_geom_destroy", "ct_fp_sf", "ct_bp_sf", "ct_fp_sf_views", "ct_bp_sf_views",
           "ct_fp_sf_host", "ct_bp_sf_host", "ct_fbp_filter", "ct_fbp_filter_views", "ct_bp_sf_recon",
           "ct_bp_sf_recon_views", "ct_fbp_sf", "ct_measure_fp32_peak", "ct_last_launch_count", "ct_status_string",
           "ct_fp_sf_noalloc")
CT_FP_SF_NOALLOC_MAX_VOXELS = 4194304          # include/ctsf.h


class CtError(RuntimeError):
    def __init__(self, status, what):
        self.status = status
        super().__init__("%s failed: %s" % (what, ct_status_string(status)))


class ct_geom_desc_t(ctypes.Structure):
    _fields_ = [("dim", ctypes.c_int32), ("nx", ctypes.c_int32), ("ny", ctypes.c_int32), ("nz", ctypes.c_int32),
                ("dx", ctypes.c_double), ("dy", ctypes.c_double), ("dz", ctypes.c_double),
                ("ox", ctypes.c_double), ("oy", ctypes.c_double), ("oz", ctypes.c_double),
                ("nu", ctypes.c_int32), ("nv", ctypes.c_int32),
                ("du", ctypes.c_double), ("dv", ctypes.c_double),
                ("det_type", ctypes.c_int32), ("n_views", ctypes.c_int32),
                ("src", ctypes.c_void_p), ("det_center", ctypes.c_void_p),
                ("det_u", ctypes.c_void_p), ("det_v", ctypes.c_void_p), ("algo", ctypes.c_int32)]


_lib = None


def lib():
    """The loaded libctsf.so; raises (loudly) when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libctsf.so is not built: run `python -m paper_2503_16741_b200.build` "
                              "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        P, I = ctypes.c_void_p, ctypes.c_int32
        L.ct_geom_create.argtypes = [ctypes.POINTER(ct_geom_desc_t), ctypes.POINTER(P)]
        L.ct_geom_destroy.argtypes = [P]
        L.ct_fp_sf.argtypes = [P, P, P, I, P]
        L.ct_bp_sf.argtypes = [P, P, P, I, P]
        L.ct_fp_sf_views.argtypes = [P, P, P, I, I, I, I, P]
        L.ct_bp_sf_views.argtypes = [P, P, P, I, I, I, I, P]
        L.ct_fp_sf_host.argtypes = [P, P, P, I, P]
        L.ct_bp_sf_host.argtypes = [P, P, P, I, P]
        L.ct_fbp_filter.argtypes = [P, P, P, I, P]
        L.ct_bp_sf_recon.argtypes = [P, P, P, I, P]
        L.ct_fbp_filter_views.argtypes = [P, P, P, I, I, I, I, P]
        L.ct_bp_sf_recon_views.argtypes = [P, P, P, I, I, I, I, P]
        L.ct_fbp_sf.argtypes = [P, P, P, P, I, P]
        L.ctsf_debug_set.argtypes = [ctypes.c_char_p, ctypes.c_double]
        L.ctsf_debug_set.restype = ctypes.c_int
        L.ctsf_debug_get.argtypes = [ctypes.c_char_p]
        L.ctsf_debug_get.restype = ctypes.c_double
        L.ct_measure_fp32_peak.argtypes = [I, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), P]
        L.ct_last_launch_count.argtypes = [P]
        L.ct_last_launch_count.restype = I
        L.ct_status_string.argtypes = [ctypes.c_int]
        L.ct_status_string.restype = ctypes.c_char_p
        for name in EXPORTS[:14]:
            getattr(L, name).restype = ctypes.c_int
        L.ct_fp_sf_noalloc.argtypes = [P, P, P, I, P]
        L.ct_fp_sf_noalloc.restype = ctypes.c_int
        _lib = L
    return _lib


def ct_status_string(status):
    return lib().ct_status_string(int(status)).decode()


def _check(status, what):
    if status != CT_OK:
        raise CtError(status, what)


def ct_geom_create(g):
    """g: dict with the ct_geom_desc_t keys (det_type 'flat'|'arc' or 0|1; vectors as [n_views,3]
    float64 arrays; optional algo 'SF' (default) | 'DD' | 'SF-TT').  Returns an opaque handle (int) for the calls below."""
    src = np.ascontiguousarray(g["src"], dtype=np.float64).reshape(-1, 3)
    dc = np.ascontiguousarray(g["det_center"], dtype=np.float64).reshape(-1, 3)
    du = np.ascontiguousarray(g["det_u"], dtype=np.float64).reshape(-1, 3)
    dv = g.get("det_v")
    dv = None if dv is None else np.ascontiguousarray(dv, dtype=np.float64).reshape(-1, 3)
    det = {"flat": 0, "arc": 1}.get(g["det_type"], g["det_type"])
    n_views = src.shape[0]
    if dc.shape[0] != n_views or du.shape[0] != n_views or (dv is not None and dv.shape[0] != n_views):
        raise CtError(1, "ct_geom_create (per-view arrays of different lengths)")
    d = ct_geom_desc_t(int(g["dim"]), int(g["nx"]), int(g["ny"]), int(g.get("nz", 1)),
                       float(g["dx"]), float(g["dy"]), float(g.get("dz", 1.0)),
                       float(g.get("ox", 0.0)), float(g.get("oy", 0.0)), float(g.get("oz", 0.0)),
                       int(g["nu"]), int(g.get("nv", 1)), float(g["du"]), float(g.get("dv", 1.0)),
                       int(det), int(n_views), src.ctypes.data, dc.ctypes.data, du.ctypes.data,
                       None if dv is None else dv.ctypes.data,
                       int({"SF": 0, "DD": 1, "SF-TT": 2}.get(g.get("algo", "SF"), g.get("algo", 0))))
    out = ctypes.c_void_p()
    _check(lib().ct_geom_create(ctypes.byref(d), ctypes.byref(out)), "ct_geom_create")
    return out.value


def ct_geom_destroy(handle):
    _check(lib().ct_geom_destroy(handle), "ct_geom_destroy")


def ct_fp_sf(handle, d_vol, d_proj, batch, stream=0):
    """Device pointers as ints (tensor.data_ptr()); stream as int (torch stream .cuda_stream)."""
    _check(lib().ct_fp_sf(handle, d_vol, d_proj, int(batch), stream), "ct_fp_sf")


def ct_bp_sf(handle, d_proj, d_vol, batch, stream=0):
    _check(lib().ct_bp_sf(handle, d_proj, d_vol, int(batch), stream), "ct_bp_sf")


def ct_fp_sf_noalloc(handle, d_vol, d_proj, batch, stream=0):
    """ct_fp_sf for callers that may not allocate device memory while running (GPU memory owned by another pool, a
    latency-bound loop, a no-growth policy): same arguments and results, scratch in a fixed 16 MiB array of the library
    instead of a cudaMalloc.  Refuses batch * nz * ny * nx > CT_FP_SF_NOALLOC_MAX_VOXELS; all calls on a GPU share the
    array, so keep them on one stream (overlapping calls race).  Make the first call on a GPU outside stream capture."""
    status = lib().ct_fp_sf_noalloc(handle, d_vol, d_proj, int(batch), stream)
    if status == 3:
        raise CtError(status, "ct_fp_sf_noalloc (batch * nz * ny * nx exceeds the fixed scratch of %d voxels; "
                              "use ct_fp_sf)" % CT_FP_SF_NOALLOC_MAX_VOXELS)
    _check(status, "ct_fp_sf_noalloc")


def ct_fp_sf_views(handle, d_vol, d_proj, batch, view_begin, view_stride, view_count, stream=0):
    _check(lib().ct_fp_sf_views(handle, d_vol, d_proj, int(batch), int(view_begin), int(view_stride),
                                int(view_count), stream), "ct_fp_sf_views")


def ct_bp_sf_views(handle, d_proj, d_vol, batch, view_begin, view_stride, view_count, stream=0):
    _check(lib().ct_bp_sf_views(handle, d_proj, d_vol, int(batch), int(view_begin), int(view_stride),
                                int(view_count), stream), "ct_bp_sf_views")


def ct_fp_sf_host(handle, h_vol, h_proj, batch, stream=0):
    """Host pointers as ints (ndarray.ctypes.data or a pinned tensor's data_ptr())."""
    _check(lib().ct_fp_sf_host(handle, h_vol, h_proj, int(batch), stream), "ct_fp_sf_host")


def ct_bp_sf_host(handle, h_proj, h_vol, batch, stream=0):
    _check(lib().ct_bp_sf_host(handle, h_proj, h_vol, int(batch), stream), "ct_bp_sf_host")


def ct_fbp_filter_views(handle, d_proj, d_out, batch, view_begin, view_stride, view_count, stream=0):
    _check(lib().ct_fbp_filter_views(handle, d_proj, d_out, batch, view_begin, view_stride, view_count, stream),
           "ct_fbp_filter_views")


def ct_bp_sf_recon_views(handle, d_proj, d_vol, batch, view_begin, view_stride, view_count, stream=0):
    _check(lib().ct_bp_sf_recon_views(handle, d_proj, d_vol, batch, view_begin, view_stride, view_count, stream),
           "ct_bp_sf_recon_views")


def ct_fbp_filter(handle, d_proj, d_out, batch, stream=0):
    _check(lib().ct_fbp_filter(handle, d_proj, d_out, batch, stream), "ct_fbp_filter")


def ct_bp_sf_recon(handle, d_proj, d_vol, batch, stream=0):
    _check(lib().ct_bp_sf_recon(handle, d_proj, d_vol, batch, stream), "ct_bp_sf_recon")


def ct_fbp_sf(handle, d_proj, d_work, d_vol, batch, stream=0):
    _check(lib().ct_fbp_sf(handle, d_proj, d_work, d_vol, int(batch), stream), "ct_fbp_sf")


def debug_set(name, value=1):
    """Testing aid (ctsf_debug_set, not part of include/ctsf.h): force a rarely taken code path of the launchers;
    debug_set('reset') restores the defaults.  Used by tests only."""
    if lib().ctsf_debug_set(name.encode(), float(value)) != 0:
        raise KeyError(name)


DEBUG_DEFAULTS = {"fp_pad": 0.0, "tt_pad": 0.0, "fp_nohoist": 0, "fp_forcehoist": 0, "fp_serial": 0, "bp_nohoist": 0,
                  "bp_forcehoist": 0, "bp_tma": -1, "bp_chunk": 0, "bp_scalar": 0, "bp_poison": 0,
                  "host_fp_chunks": 0, "host_bp_chunks": 0}


def debug_state():
    """The testing switches that are NOT at their defaults, as {name: value} (ctsf_debug_get); {} = product paths."""
    out = {}
    for name, default in DEBUG_DEFAULTS.items():
        v = lib().ctsf_debug_get(name.encode())
        if v != v:
            raise KeyError(name)
        if v != default:
            out[name] = v
    return out


def ct_measure_fp32_peak(kind=0, stream=0):
    """Measured fp32 FMA throughput of the current device: (flop/s, seconds of the timed launch).
    kind 0: scalar FFMA, 1: packed FFMA2; 2, 3 (design record): FFMA2 interleaved with scalar FFMA / with FMNMX."""
    f, t = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(lib().ct_measure_fp32_peak(int(kind), ctypes.byref(f), ctypes.byref(t), stream), "ct_measure_fp32_peak")
    return f.value, t.value


def ct_last_launch_count(handle):
    return int(lib().ct_last_launch_count(handle))
