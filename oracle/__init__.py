"""ORACLE — TEST INFRASTRUCTURE ONLY.

ctypes driver for ``orb_oracle.c``: the plain single-threaded CPU statement of
the gyro-averaged deposition (see that file's header for the passages of
/root/reference/PAPER.md it follows and for its pins).  Nothing under
``paper_1908_02219_b200/`` imports this package; only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "orb_oracle.c")
_SO = os.path.join(_HERE, "liborb_oracle.so")
MAX_NL = 64

CFLAGS = ["-O2", "-ffp-contract=off", "-fPIC", "-shared", "-std=c99"]


class Geom(C.Structure):
    _fields_ = [("ns", C.c_int32), ("ntheta", C.c_int32), ("nphi", C.c_int32),
                ("theta_map", C.c_int32), ("r0", C.c_double), ("a", C.c_double),
                ("b0", C.c_double), ("rho_star", C.c_double), ("q", C.c_double)]


class Policy(C.Structure):
    _fields_ = [("mode", C.c_int32), ("n_fixed", C.c_int32), ("n_max", C.c_int32),
                ("pad_", C.c_int32), ("rho_ref", C.c_double), ("alpha0", C.c_double)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        L.oracle_wrap_2pi.restype = C.c_double
        L.oracle_wrap_2pi.argtypes = [C.c_double]
        for f in (L.oracle_thetastar_from_theta, L.oracle_theta_from_thetastar):
            f.restype = C.c_double
            f.argtypes = [C.c_double, C.c_double]
        for f in (L.oracle_periodic_cubic, L.oracle_clamped_cubic):
            f.restype = None
            f.argtypes = [C.c_double, C.c_int32, C.POINTER(C.c_int32), dp]
        L.oracle_larmor_radius.restype = C.c_double
        L.oracle_larmor_radius.argtypes = [C.POINTER(Geom), C.c_double, C.c_double, C.c_double]
        L.oracle_nl.restype = C.c_int32
        L.oracle_nl.argtypes = [C.POINTER(Policy), C.c_double]
        L.oracle_ring_points.restype = C.c_int32
        L.oracle_ring_points.argtypes = [C.POINTER(Geom), C.POINTER(Policy), C.c_double,
                                         C.c_double, C.c_double, dp, dp, dp, dp]
        L.oracle_deposit.restype = C.c_int64
        L.oracle_deposit.argtypes = [C.POINTER(Geom), C.POINTER(Policy), C.c_int64,
                                     dp, dp, dp, dp, dp, dp, dp, dp]
        L.oracle_gather.restype = C.c_int64
        L.oracle_gather.argtypes = [C.POINTER(Geom), C.POINTER(Policy), C.c_int64,
                                    dp, dp, dp, dp, dp, dp]
        L.oracle_nl_histogram.restype = C.c_int64
        L.oracle_nl_histogram.argtypes = [C.POINTER(Geom), C.POINTER(Policy), C.c_int64,
                                          dp, dp, dp, C.POINTER(C.c_int64)]
        _lib = L
    return _lib


def geom(ns, ntheta, nphi, *, r0=1.0, a=0.3, b0=1.0, rho_star=1.0 / 180.0, q=1.0,
         theta_map=1) -> Geom:
    return Geom(ns, ntheta, nphi, theta_map, r0, a, b0, rho_star, q)


def policy_fixed(n, alpha0=0.0) -> Policy:
    return Policy(0, n, n, 0, 1.0, alpha0)


def policy_adaptive(n_min, n_max, rho_ref, alpha0=0.0) -> Policy:
    return Policy(1, n_min, n_max, 0, rho_ref, alpha0)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def wrap_2pi(u):
    return lib().oracle_wrap_2pi(float(u))


def thetastar_from_theta(th, e):
    return lib().oracle_thetastar_from_theta(float(th), float(e))


def theta_from_thetastar(ts, e):
    return lib().oracle_theta_from_thetastar(float(ts), float(e))


def periodic_cubic(u, n):
    j0 = C.c_int32()
    w = np.zeros(4)
    lib().oracle_periodic_cubic(float(u), int(n), C.byref(j0), _dp(w))
    return j0.value, w


def clamped_cubic(s, n):
    i0 = C.c_int32()
    w = np.zeros(4)
    lib().oracle_clamped_cubic(float(s), int(n), C.byref(i0), _dp(w))
    return i0.value, w


def larmor_radius(g: Geom, s, thetastar, mu):
    return lib().oracle_larmor_radius(C.byref(g), float(s), float(thetastar), float(mu))


def nl(pol: Policy, rho_l):
    return lib().oracle_nl(C.byref(pol), float(rho_l))


def ring_points(g: Geom, pol: Policy, s, thetastar, mu):
    """-> dict(n, s, thetastar, x, z) for one marker."""
    sl, tsl, x, z = (np.zeros(MAX_NL) for _ in range(4))
    n = lib().oracle_ring_points(C.byref(g), C.byref(pol), float(s), float(thetastar), float(mu),
                                 _dp(sl), _dp(tsl), _dp(x), _dp(z))
    return dict(n=n, s=sl[:n].copy(), thetastar=tsl[:n].copy(), x=x[:n].copy(), z=z[:n].copy())


def grid_shape(g: Geom):
    return (g.ns + 3, g.ntheta, g.nphi)


def deposit(g: Geom, pol: Policy, s, thetastar, phi, vpar, mu, w, *, current=True,
            rho=None, jpar=None):
    """Single-threaded oracle deposition.  Returns (rho, jpar or None, n_points)."""
    s, thetastar, phi, mu, w = map(_f64, (s, thetastar, phi, mu, w))
    n = s.shape[0]
    shape = grid_shape(g)
    if rho is None:
        rho = np.zeros(shape)
    if current:
        vpar = _f64(vpar)
        if jpar is None:
            jpar = np.zeros(shape)
        jp, vp = _dp(jpar), _dp(vpar)
    else:
        jpar = None
        jp = C.POINTER(C.c_double)()
        vp = C.POINTER(C.c_double)()
    npts = lib().oracle_deposit(C.byref(g), C.byref(pol), n, _dp(s), _dp(thetastar), _dp(phi),
                                vp, _dp(mu), _dp(w), _dp(rho), jp)
    if npts < 0:
        raise ValueError("oracle_deposit: N_L > %d" % MAX_NL)
    return rho, jpar, int(npts)


def deposit_ranges(g: Geom, pol: Policy, s, thetastar, phi, vpar, mu, w, *, current=True,
                   workers=None):
    """The same oracle_deposit run on contiguous marker ranges, one private grid
    per range, the grids summed in range order afterwards (the replica scheme of
    PAPER.md:81).  Only the summation order differs from ``deposit``; used by the
    full-size parity tests so they finish in minutes.  Returns (rho, jpar, n_points, workers).
    """
    s, thetastar, phi, mu, w = map(_f64, (s, thetastar, phi, mu, w))
    if current:
        vpar = _f64(vpar)
    n = s.shape[0]
    workers = workers or min(os.cpu_count() or 1, 64)
    workers = max(1, min(workers, (n + 4095) // 4096 or 1))
    if workers == 1:
        r, j, npts = deposit(g, pol, s, thetastar, phi, vpar, mu, w, current=current)
        return r, j, npts, 1
    bounds = np.linspace(0, n, workers + 1).astype(np.int64)

    def run(i):
        a, b = int(bounds[i]), int(bounds[i + 1])
        return deposit(g, pol, s[a:b], thetastar[a:b], phi[a:b],
                       vpar[a:b] if current else None, mu[a:b], w[a:b], current=current)

    lib()
    with ThreadPoolExecutor(workers) as ex:
        parts = list(ex.map(run, range(workers)))
    rho = parts[0][0]
    jpar = parts[0][1]
    npts = parts[0][2]
    for r, j, k in parts[1:]:
        rho += r
        if current:
            jpar += j
        npts += k
    return rho, jpar, npts, workers


def gather(g: Geom, pol: Policy, s, thetastar, phi, mu, field, *, workers=1):
    """Get fields + gyroaverage (oracle_gather): field (ns+3, ntheta, nphi) -> out[n].
    Markers are independent, so ``workers`` > 1 only splits the marker range over threads and
    gives bit-identical results.  Returns (out, n_points)."""
    s, thetastar, phi, mu = map(_f64, (s, thetastar, phi, mu))
    field = _f64(field)
    assert field.shape == grid_shape(g), (field.shape, grid_shape(g))
    n = s.shape[0]
    out = np.empty(n)
    L = lib()

    def run(a, b):
        r = L.oracle_gather(C.byref(g), C.byref(pol), b - a, _dp(s[a:b]), _dp(thetastar[a:b]),
                            _dp(phi[a:b]), _dp(mu[a:b]), _dp(field), _dp(out[a:b]))
        if r < 0:
            raise ValueError("oracle_gather: N_L > %d" % MAX_NL)
        return int(r)

    workers = max(1, min(workers or (os.cpu_count() or 1), (n + 4095) // 4096 or 1))
    if workers == 1:
        return out, run(0, n)
    bounds = np.linspace(0, n, workers + 1).astype(np.int64)
    with ThreadPoolExecutor(workers) as ex:
        npts = sum(ex.map(lambda i: run(int(bounds[i]), int(bounds[i + 1])), range(workers)))
    return out, npts


def nl_histogram(g: Geom, pol: Policy, s, thetastar, mu):
    s, thetastar, mu = map(_f64, (s, thetastar, mu))
    hist = np.zeros(MAX_NL + 1, dtype=np.int64)
    npts = lib().oracle_nl_histogram(C.byref(g), C.byref(pol), s.shape[0], _dp(s), _dp(thetastar),
                                     _dp(mu), hist.ctypes.data_as(C.POINTER(C.c_int64)))
    if npts < 0:
        raise ValueError("oracle_nl_histogram: N_L > %d" % MAX_NL)
    return hist, int(npts)
