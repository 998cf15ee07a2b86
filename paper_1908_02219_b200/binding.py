"""Thin ctypes binding of liborb_b200.so (include/orb.h): same names, argument
marshalling only.  Every step of the deposition runs in the library's CUDA
kernels; there is no CPU fallback, and loading fails loudly if the library has
not been built (``python -m paper_1908_02219_b200.build``).
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liborb_b200.so")

ORB_OK, ORB_E_INVAL, ORB_E_STATE, ORB_E_NOMEM, ORB_E_CUDA = 0, -1, -2, -3, -4
ORB_NL_FIXED, ORB_NL_ADAPTIVE = 0, 1
ORB_DEPOSIT_ZERO_FIRST = 0x1
ORB_DEPOSIT_NO_BIN = 0x2
ORB_DEPOSIT_ALGO_ATOMIC = 0x4
ORB_DEPOSIT_ALGO_TILE_V4 = 0x8
ORB_DEPOSIT_ALGO_TILE_WS = 0x10
ORB_DEPOSIT_ALGO_RING_DATA = 0x20
ORB_DEPOSIT_ALGO_TILE_WS2 = 0x40
ORB_MARKERS_SORTED = 0x1
ORB_MARKERS_TILE_BINS = 0x2
ORB_MAX_NL = 32
ORB_MAX_FIELDS = 8
ORB_NOALLOC_MAX_NS = 1024

# every symbol include/orb.h declares
SYMBOLS = ("orb_grid_create", "orb_grid_destroy", "orb_grid_shape", "orb_markers_bind",
           "orb_reserve", "orb_ring_reserve", "orb_markers_bin", "orb_markers_refresh", "orb_markers_rebin", "orb_last_moved",
           "orb_markers_layout", "orb_debug_tilebins", "orb_deposit", "orb_gather", "orb_grid_zero", "orb_last_points", "orb_last_fallback_points", "orb_deposit_host",
           "orb_launch_count", "orb_debug_counters", "orb_debug_binned", "orb_probe_dfma", "orb_deposit_noalloc", "orb_spline_table_radial", "orb_strerror", "orb_last_error", "orb_version")


class OrbError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("liborb_b200: %s (code %d)" % (msg, code))
        self.code = code


class GridDesc(C.Structure):
    _fields_ = [("ns", C.c_int32), ("ntheta", C.c_int32), ("nphi", C.c_int32),
                ("r0", C.c_double), ("a", C.c_double), ("b0", C.c_double),
                ("rho_star", C.c_double), ("q", C.c_double),
                ("theta_map", C.c_int32), ("device", C.c_int32)]


class NlPolicy(C.Structure):
    _fields_ = [("mode", C.c_int32), ("n_fixed", C.c_int32), ("n_max", C.c_int32),
                ("flags", C.c_uint32), ("rho_ref", C.c_double), ("alpha0", C.c_double)]


class MarkerLayout(C.Structure):
    _fields_ = [("records", C.c_void_p), ("count", C.c_void_p), ("record_doubles", C.c_int32),
                ("capacity", C.c_uint32), ("n_bins", C.c_uint32), ("tiles_s", C.c_int32),
                ("tiles_theta", C.c_int32)]


_lib = None


def lib():
    """Loads the C-ABI library.  Raises if it is missing: the CUDA path is the only path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise OrbError(ORB_E_STATE, "liborb_b200.so is not built at %s; run "
                       "`python -m paper_1908_02219_b200.build` (nvcc, sm_100a)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, dp, i64p = C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)
    L.orb_grid_create.argtypes = [C.POINTER(GridDesc), C.POINTER(vp)]
    L.orb_grid_destroy.argtypes = [vp]
    L.orb_grid_shape.argtypes = [vp, C.POINTER(C.c_int64 * 3)]
    L.orb_markers_bind.argtypes = [vp, C.c_int64, dp, dp, dp, dp, dp, dp, C.c_uint32]
    L.orb_reserve.argtypes = [vp, C.c_int64]
    L.orb_ring_reserve.argtypes = [vp, C.c_int64, C.c_int64]
    L.orb_markers_bin.argtypes = [vp, vp]
    L.orb_markers_refresh.argtypes = [vp, vp]
    L.orb_markers_rebin.argtypes = [vp, vp]
    L.orb_last_moved.argtypes = [vp, i64p, i64p]
    L.orb_markers_layout.argtypes = [vp, C.POINTER(MarkerLayout)]
    L.orb_debug_tilebins.argtypes = [vp, dp, dp]
    L.orb_deposit.argtypes = [vp, dp, dp, C.POINTER(NlPolicy), vp]
    L.orb_gather.argtypes = [vp, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_void_p),
                             C.POINTER(NlPolicy), vp]
    L.orb_grid_zero.argtypes = [vp, dp, dp, vp]
    L.orb_last_points.argtypes = [vp, i64p]
    L.orb_last_fallback_points.argtypes = [vp, i64p]
    L.orb_deposit_host.argtypes = [vp, C.c_int64, dp, dp, dp, dp, dp, dp, dp, dp,
                                   C.POINTER(NlPolicy), i64p, i64p, i64p]
    L.orb_launch_count.argtypes = [vp, i64p]
    L.orb_deposit_noalloc.argtypes = [C.POINTER(GridDesc), C.c_int64, dp, dp, dp, dp, dp, dp, dp, dp,
                                      C.POINTER(NlPolicy), vp, i64p, C.c_char_p, C.c_int32]
    L.orb_debug_binned.argtypes = [vp, dp, dp, C.POINTER(C.c_int32)]
    L.orb_spline_table_radial.argtypes = [C.c_int32, dp]
    L.orb_strerror.argtypes = [C.c_int]
    L.orb_strerror.restype = C.c_char_p
    L.orb_last_error.argtypes = [vp]
    L.orb_last_error.restype = C.c_char_p
    L.orb_version.argtypes = []
    for name in SYMBOLS:
        if name not in ("orb_strerror", "orb_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L


def _check(code, handle=None):
    if code != ORB_OK:
        L = lib()
        msg = L.orb_last_error(handle).decode() if handle else ""
        raise OrbError(code, msg or L.orb_strerror(code).decode())


def _ptr(t):
    """Address of a torch tensor / numpy array / raw int / None."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def policy(n_fixed=4, *, adaptive=False, n_max=None, rho_ref=1.0, alpha0=0.0, flags=0) -> NlPolicy:
    return NlPolicy(ORB_NL_ADAPTIVE if adaptive else ORB_NL_FIXED, n_fixed,
                    n_max if n_max is not None else n_fixed, flags, rho_ref, alpha0)


def probe_dfma(device: int = 0) -> float:
    """Measured fp64 FMA rate of the device, TFLOP/s (harness aid)."""
    v = C.c_double()
    _check(lib().orb_probe_dfma(device, C.byref(v)))
    return v.value


def spline_table_radial(ns: int):
    """(ns, 4, 4) numpy array: [cell, basis offset a, power of t] (host-only diagnostic)."""
    import numpy as np
    out = np.empty((ns, 4, 4), dtype=np.float64)
    _check(lib().orb_spline_table_radial(ns, out.ctypes.data))
    return out


def deposit_noalloc(desc: GridDesc, s, theta, phi, vpar, mu, w, rho, jpar, pol: NlPolicy,
                    stream=None, n=None, want_points=False):
    """orb_deposit_noalloc: handle-free deposit that allocates nothing (static device scratch,
    ns <= ORB_NOALLOC_MAX_NS).  Device arrays in, device grids added to.  Returns the sum of N_L
    if want_points (the call then waits for the stream), else None (asynchronous)."""
    if n is None:
        n = s.numel() if hasattr(s, "numel") else len(s)
    err = C.create_string_buffer(512)
    pts = C.c_int64(0)
    code = lib().orb_deposit_noalloc(C.byref(desc), n, _ptr(s), _ptr(theta), _ptr(phi), _ptr(vpar),
                                     _ptr(mu), _ptr(w), _ptr(rho), _ptr(jpar), C.byref(pol), stream,
                                     C.byref(pts) if want_points else None, err, len(err))
    if code != ORB_OK:
        raise OrbError(code, err.value.decode() or lib().orb_strerror(code).decode())
    return pts.value if want_points else None


class Grid:
    """RAII wrapper of an orb_grid_t handle; method names follow the C calls."""

    def __init__(self, ns, ntheta, nphi, *, r0=1.0, a=0.3, b0=1.0, rho_star=1.0 / 180.0, q=1.0,
                 theta_map=1, device=0):
        self._h = C.c_void_p()
        self.desc = GridDesc(ns, ntheta, nphi, r0, a, b0, rho_star, q, theta_map, device)
        _check(lib().orb_grid_create(C.byref(self.desc), C.byref(self._h)))
        self._keep = None

    def shape(self):
        dims = (C.c_int64 * 3)()
        _check(lib().orb_grid_shape(self._h, C.byref(dims)), self._h)
        return tuple(dims)

    def markers_bind(self, s, theta, phi, vpar, mu, w, flags=0, n=None):
        if n is None:
            n = s.numel() if hasattr(s, "numel") else len(s)
        self._keep = (s, theta, phi, vpar, mu, w)   # the library borrows the pointers
        _check(lib().orb_markers_bind(self._h, n, _ptr(s), _ptr(theta), _ptr(phi), _ptr(vpar),
                                      _ptr(mu), _ptr(w), flags), self._h)

    def reserve(self, n):
        _check(lib().orb_reserve(self._h, n), self._h)

    def ring_reserve(self, n_markers, n_points):
        _check(lib().orb_ring_reserve(self._h, n_markers, n_points), self._h)

    def markers_bin(self, stream=None):
        _check(lib().orb_markers_bin(self._h, stream), self._h)

    def markers_refresh(self, stream=None):
        _check(lib().orb_markers_refresh(self._h, stream), self._h)

    def markers_rebin(self, stream=None):
        _check(lib().orb_markers_rebin(self._h, stream), self._h)

    def last_moved(self):
        """-> (markers moved by the last rebin, movers left in place)."""
        a, b = C.c_int64(), C.c_int64()
        _check(lib().orb_last_moved(self._h, C.byref(a), C.byref(b)), self._h)
        return a.value, b.value

    def markers_layout(self) -> MarkerLayout:
        out = MarkerLayout()
        _check(lib().orb_markers_layout(self._h, C.byref(out)), self._h)
        return out

    def debug_tilebins(self, n):
        """-> (records (n, 8) packed tile by tile, count per tile)."""
        import numpy as np
        lay = self.markers_layout()
        cnt = np.empty(lay.n_bins, dtype=np.uint32)
        rec = np.zeros((n, 8), dtype=np.float64)
        _check(lib().orb_debug_tilebins(self._h, rec.ctypes.data, cnt.ctypes.data), self._h)
        return rec, cnt

    def deposit(self, rho, jpar, pol: NlPolicy, stream=None):
        _check(lib().orb_deposit(self._h, _ptr(rho), _ptr(jpar), C.byref(pol), stream), self._h)

    def gather(self, fields, out, pol: NlPolicy, stream=None):
        """fields: sequence of device grids; out: sequence of device arrays of n doubles."""
        nf = len(fields)
        fa = (C.c_void_p * nf)(*[_ptr(f) for f in fields])
        oa = (C.c_void_p * nf)(*[_ptr(o) for o in out])
        _check(lib().orb_gather(self._h, nf, fa, oa, C.byref(pol), stream), self._h)

    def grid_zero(self, rho, jpar, stream=None):
        _check(lib().orb_grid_zero(self._h, _ptr(rho), _ptr(jpar), stream), self._h)

    def last_points(self) -> int:
        v = C.c_int64()
        _check(lib().orb_last_points(self._h, C.byref(v)), self._h)
        return v.value

    def last_fallback_points(self) -> int:
        v = C.c_int64()
        _check(lib().orb_last_fallback_points(self._h, C.byref(v)), self._h)
        return v.value

    def debug_counters(self):
        out = (C.c_uint64 * 16)()
        _check(lib().orb_debug_counters(self._h, out), self._h)
        return list(out)

    def debug_binned(self, n):
        """-> (records (n, 8) float64 or None for ORB_MARKERS_SORTED bindings, cell_start uint32)."""
        import numpy as np
        ncells = self.desc.ns * self.desc.ntheta * self.desc.nphi
        cs = np.empty(ncells + 1, dtype=np.uint32)
        rec = np.empty((n, 8), dtype=np.float64)
        stride = C.c_int32()
        _check(lib().orb_debug_binned(self._h, rec.ctypes.data, cs.ctypes.data, C.byref(stride)),
               self._h)
        return (rec if stride.value else None), cs

    def launch_count(self) -> int:
        v = C.c_int64()
        _check(lib().orb_launch_count(self._h, C.byref(v)), self._h)
        return v.value

    def deposit_host(self, s, theta, phi, vpar, mu, w, rho_host, jpar_host, pol: NlPolicy, n=None):
        """Host arrays in, host grids out (overwritten). -> (n_points, h2d_bytes, d2h_bytes)."""
        if n is None:
            n = s.numel() if hasattr(s, "numel") else len(s)
        npts, up, down = C.c_int64(), C.c_int64(), C.c_int64()
        _check(lib().orb_deposit_host(self._h, n, _ptr(s), _ptr(theta), _ptr(phi), _ptr(vpar),
                                      _ptr(mu), _ptr(w), _ptr(rho_host), _ptr(jpar_host),
                                      C.byref(pol), C.byref(npts), C.byref(up), C.byref(down)),
               self._h)
        return npts.value, up.value, down.value

    def destroy(self):
        if self._h:
            lib().orb_grid_destroy(self._h)
            self._h = C.c_void_p()
            self._keep = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def grid_for(cfg, device=0) -> Grid:
    """Grid handle for a workloads.Config."""
    return Grid(cfg.ns, cfg.ntheta, cfg.nphi, r0=cfg.r0, a=cfg.a, b0=cfg.b0, rho_star=cfg.rho_star,
                q=cfg.q, device=device)


def policy_for(cfg, flags=0) -> NlPolicy:
    return policy(cfg.n_fixed, adaptive=cfg.adaptive, n_max=cfg.n_max if cfg.adaptive else None,
                  rho_ref=cfg.rho_ref, flags=flags)
