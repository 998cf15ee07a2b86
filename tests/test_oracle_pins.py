"""Pins for the CPU oracle (oracle/orb_oracle.c) against what the paper's
definition and the mathematics fix -- never against the oracle itself and never
against the CUDA path.  P-numbers refer to DESIGN.md "Pins".
"""
import math
import os

import numpy as np
import pytest
from scipy import integrate, interpolate, optimize, special

import oracle as O
from paper_1908_02219_b200 import workloads as W

TWO_PI = 2 * math.pi
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def small_markers(n, seed=1, s_lo=0.1, s_hi=0.9):
    cfg = W.scaled(W.CONFIGS["cfg0"], n)
    cfg = W.dataclasses.replace(cfg, seed=seed, s_lo=s_lo, s_hi=s_hi)
    return W.generate(cfg, workers=1)


def dep(g, pol, m, current=True, **kw):
    return O.deposit(g, pol, m["s"], m["theta"], m["phi"], m["vpar"], m["mu"], m["w"],
                     current=current, **kw)


# ---------------------------------------------------------------- splines ---

def beta3(v):
    """Cardinal centred cubic B-spline (textbook definition)."""
    v = np.abs(v)
    return np.where(v < 1, 2 / 3 - v * v + v ** 3 / 2, np.where(v < 2, (2 - v) ** 3 / 6, 0.0))


def periodic_basis(j, u, n):
    """Lambda_j(u) = sum_m beta3(u n/2pi - j - m n): function definition, no index logic."""
    x = (u % TWO_PI) * n / TWO_PI
    return sum(beta3(x - j - m * n) for m in (-2, -1, 0, 1, 2))


def cox_de_boor(i, p, T, x):
    """Recursive definition of B-spline i of degree p on knot vector T (right-closed at the end)."""
    if p == 0:
        if T[i] <= x < T[i + 1]:
            return 1.0
        if x == T[-1] and T[i] < T[i + 1] == T[-1]:
            return 1.0
        return 0.0
    a = 0.0
    if T[i + p] > T[i]:
        a = (x - T[i]) / (T[i + p] - T[i]) * cox_de_boor(i, p - 1, T, x)
    b = 0.0
    if T[i + p + 1] > T[i + 1]:
        b = (T[i + p + 1] - x) / (T[i + p + 1] - T[i + 1]) * cox_de_boor(i + 1, p - 1, T, x)
    return a + b


def open_knots(n):
    return np.array([0.0] * 3 + list(range(n + 1)) + [float(n)] * 3)


def test_clamped_golden_values():
    """Closed-form rationals of the open-knot cubic basis (tests/golden/clamped_cubic_n8.txt)."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "clamped_cubic_n8.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) >= 6
    for r in rows:
        x, cell = float(r[0]), int(r[1])
        want = [float(eval(v, {"__builtins__": {}})) for v in r[2:6]]
        i0, w = O.clamped_cubic(x / 8.0, 8)
        assert i0 == cell
        np.testing.assert_allclose(w, want, rtol=0, atol=2e-16)


@pytest.mark.parametrize("n", [4, 5, 8, 16])
def test_clamped_matches_scipy_and_cox_de_boor(n):
    """Library pin: scipy's BSpline on the same open knot vector; and the recursive definition."""
    T = open_knots(n)
    rng = np.random.default_rng(3)
    xs = np.concatenate([rng.uniform(0, n, 200), np.arange(n + 1.0), [0.5, n - 0.5, 1e-9, n - 1e-9]])
    dm = interpolate.BSpline.design_matrix(np.clip(xs, 0, n), T, 3).toarray()
    for x, row in zip(xs, dm):
        i0, w = O.clamped_cubic(x / n, n)
        full = np.zeros(n + 3)
        full[i0:i0 + 4] = w
        np.testing.assert_allclose(full, row, rtol=0, atol=1e-14)
    for x in xs[:40]:
        i0, w = O.clamped_cubic(x / n, n)
        for i in range(n + 3):
            want = cox_de_boor(i, 3, T, x * (1 - 1e-16) if False else x)
            got = w[i - i0] if i0 <= i < i0 + 4 else 0.0
            assert abs(got - want) < 1e-13


def test_clamped_ends():
    """P2: s = 0 -> basis 0 carries everything; s = 1 -> basis N+2."""
    for n in (4, 16, 128):
        i0, w = O.clamped_cubic(0.0, n)
        assert i0 == 0 and w[0] == 1.0 and np.all(w[1:] == 0)
        i0, w = O.clamped_cubic(1.0, n)
        assert i0 == n - 1 and w[3] == 1.0 and np.all(w[:3] == 0)


@pytest.mark.parametrize("n", [4, 5, 32])
def test_periodic_matches_definition(n):
    rng = np.random.default_rng(5)
    us = np.concatenate([rng.uniform(-10, 10, 200), TWO_PI * np.arange(n) / n, [0.0, TWO_PI, -1e-17]])
    for u in us:
        j0, w = O.periodic_cubic(u, n)
        full = np.zeros(n)
        for b in range(4):
            full[(j0 + b) % n] += w[b]
        want = np.array([periodic_basis(j, u, n) for j in range(n)])
        np.testing.assert_allclose(full, want, rtol=0, atol=1e-14)
        assert abs(w.sum() - 1) < 1e-15


# -------------------------------------------------------------- geometry ---

def test_thetastar_map_quadrature_and_roundtrip():
    """P5: closed form of R3 == integral of sqrt(1-e^2)/(1+e cos t); fixed points; round trip."""
    for e in (0.0, 0.03, 0.15, 0.3):
        for th in np.linspace(0.05, TWO_PI - 0.05, 23):
            want, _ = integrate.quad(lambda t: math.sqrt(1 - e * e) / (1 + e * math.cos(t)), 0, th,
                                     epsabs=1e-14, epsrel=1e-14)
            got = O.thetastar_from_theta(th, e)
            assert abs(got - want) < 1e-12
            back = O.theta_from_thetastar(got, e)
            assert abs(back - th) < 5e-15
        assert O.thetastar_from_theta(0.0, e) == 0.0
        assert abs(O.thetastar_from_theta(math.pi, e) - math.pi) < 1e-15
    for th in np.linspace(0, 6, 13):
        assert abs(O.thetastar_from_theta(th, 0.0) - th) < 1e-15   # e -> 0: identity
    # straight field lines make theta* lag behind theta on the outboard side (e > 0)
    assert O.thetastar_from_theta(1.0, 0.3) < 1.0


def theta_by_root_finding(ts, e):
    """Independent route to theta(theta*): invert the quadrature numerically."""
    f = lambda th: integrate.quad(lambda t: math.sqrt(1 - e * e) / (1 + e * math.cos(t)), 0, th,
                                  epsabs=1e-14, epsrel=1e-14)[0] - ts
    return optimize.brentq(f, 0.0, TWO_PI, xtol=1e-15, rtol=1e-15)


def test_ring_geometry():
    """P6 (+R1,R2,R6): every point at distance rho_L from the guiding centre, centroid at the
    guiding centre, N_L=4 points at (+-rho, 0), (0, +-rho); rho_L = rho* sqrt(2 mu/B) with
    B = 1/(1 + eps s cos theta) computed by an independent route."""
    g = O.geom(16, 32, 16, rho_star=1 / 20.0)
    rng = np.random.default_rng(11)
    for n in (2, 3, 4, 8, 32):
        pol = O.policy_fixed(n)
        for _ in range(10):
            s, ts, mu = rng.uniform(0.2, 0.7), rng.uniform(0.1, 6.1), rng.uniform(0.1, 2.0)
            e = 0.3 * s
            th = theta_by_root_finding(ts, e)
            B = 1.0 / (1.0 + e * math.cos(th))
            rho = (1 / 20.0) * math.sqrt(2 * mu / B)
            assert abs(O.larmor_radius(g, s, ts, mu) - rho) < 1e-13
            r = O.ring_points(g, pol, s, ts, mu)
            assert r["n"] == n
            x0, z0 = s * math.cos(th), s * math.sin(th)
            d = np.hypot(r["x"] - x0, r["z"] - z0)
            np.testing.assert_allclose(d, rho, rtol=0, atol=1e-12)
            assert abs(r["x"].mean() - x0) < 1e-12 and abs(r["z"].mean() - z0) < 1e-12
            if n == 4:
                np.testing.assert_allclose(r["x"], [x0 + rho, x0, x0 - rho, x0], atol=1e-12)
                np.testing.assert_allclose(r["z"], [z0, z0 + rho, z0, z0 - rho], atol=1e-12)
            # magnetic coordinates of the points: s_l = |(x,z)|, theta*_l from theta_l by quadrature
            np.testing.assert_allclose(r["s"], np.hypot(r["x"], r["z"]), atol=1e-15)
            for xl, zl, sl, tsl in zip(r["x"], r["z"], r["s"], r["thetastar"]):
                thl = math.atan2(zl, xl) % TWO_PI
                el = 0.3 * sl
                want, _ = integrate.quad(lambda t: math.sqrt(1 - el * el) / (1 + el * math.cos(t)),
                                         0, thl, epsabs=1e-14, epsrel=1e-14)
                assert abs(tsl - want) < 1e-11
    # gyro-phase offset alpha0 rotates the ring
    pol = O.policy_fixed(4, alpha0=math.pi / 2)
    r = O.ring_points(g, pol, 0.5, 1.0, 1.0)
    r0 = O.ring_points(g, O.policy_fixed(4), 0.5, 1.0, 1.0)
    np.testing.assert_allclose(r["x"], np.roll(r0["x"], -1), atol=1e-15)


def independent_ring(s, ts, mu, n, *, r0, a, b0, rho_star, alpha0=0.0):
    """Larmor points by a route that shares nothing with the oracle: theta by root-finding on the
    quadrature of the straight-field-line relation, B = B0 R0 / R with R = R0 + a s cos(theta) (R1,
    R2), rho_L = rho* sqrt(2 mu / B) in units of a (R6), ring in the (x, z) plane (R5, R7), theta*
    of every point by quadrature again (R3) with e_l = (a / R0) s_l.  -> (rho_L, x, z, s_l, ts_l)"""
    eps = a / r0
    th = theta_by_root_finding(ts, eps * s)
    R = r0 + a * s * math.cos(th)
    B = b0 * r0 / R
    rho = rho_star * math.sqrt(2 * mu / B)
    x0, z0 = s * math.cos(th), s * math.sin(th)
    al = alpha0 + TWO_PI * np.arange(n) / n
    x, z = x0 + rho * np.cos(al), z0 + rho * np.sin(al)
    sl = np.minimum(np.hypot(x, z), 1.0)
    tsl = []
    for xl, zl, s_l in zip(x, z, sl):
        thl = math.atan2(zl, xl) % TWO_PI
        el = eps * s_l
        v, _ = integrate.quad(lambda t: math.sqrt(1 - el * el) / (1 + el * math.cos(t)), 0, thl,
                              epsabs=1e-14, epsrel=1e-14)
        tsl.append(v)
    return rho, x, z, sl, np.array(tsl)


@pytest.mark.parametrize("r0,a,b0", [(1.7, 0.5, 2.5), (3.0, 0.9, 0.4), (1.0, 0.3, 1.0)])
def test_ring_geometry_nondefault_r0_a_b0(r0, a, b0):
    """R1, R2, R6 away from the defaults: oracle_larmor_radius and oracle_ring_points against the
    independent route (a mistake such as eps = a * r0, or a dropped B0, fails here)."""
    rs = 1 / 15.0
    g = O.geom(16, 32, 16, r0=r0, a=a, b0=b0, rho_star=rs)
    rng = np.random.default_rng(5)
    for n in (4, 7):
        pol = O.policy_fixed(n, alpha0=0.3)
        for _ in range(6):
            s, ts, mu = rng.uniform(0.25, 0.7), rng.uniform(0.1, 6.1), rng.uniform(0.1, 1.5)
            rho, x, z, sl, tsl = independent_ring(s, ts, mu, n, r0=r0, a=a, b0=b0, rho_star=rs,
                                                  alpha0=0.3)
            assert abs(O.larmor_radius(g, s, ts, mu) - rho) < 1e-13
            r = O.ring_points(g, pol, s, ts, mu)
            np.testing.assert_allclose(r["x"], x, rtol=0, atol=1e-12)
            np.testing.assert_allclose(r["z"], z, rtol=0, atol=1e-12)
            np.testing.assert_allclose(r["s"], sl, rtol=0, atol=1e-12)
            d = np.abs(r["thetastar"] - tsl)
            assert np.minimum(d, TWO_PI - d).max() < 1e-11


def test_brute_force_nondefault_geometry():
    """P4 with r0, a, b0, q, rho*, alpha0 all away from their defaults and the Larmor points taken
    from the independent route, not from the oracle: a node-centric gather with the function
    definitions of the splines."""
    ns, nt, nph = 6, 7, 5
    r0, a, b0, q, rs, alpha0, nl = 1.7, 0.5, 2.5, -1.3, 0.06, 0.37, 4
    m = small_markers(60, seed=9, s_lo=0.1, s_hi=0.9)
    g = O.geom(ns, nt, nph, r0=r0, a=a, b0=b0, rho_star=rs, q=q)
    rho, jp, npts = dep(g, O.policy_fixed(nl, alpha0=alpha0), m)
    assert npts == 60 * nl
    T = open_knots(ns)
    want = np.zeros((ns + 3, nt, nph))
    wantj = np.zeros_like(want)
    for p in range(60):
        _, _, _, sl_, tsl_ = independent_ring(m["s"][p], m["theta"][p], m["mu"][p], nl, r0=r0, a=a,
                                              b0=b0, rho_star=rs, alpha0=alpha0)
        lp = np.array([periodic_basis(k, m["phi"][p], nph) for k in range(nph)])
        for sl, tsl in zip(sl_, tsl_):
            ls = np.array([cox_de_boor(i, 3, T, sl * ns) for i in range(ns + 3)])
            lt = np.array([periodic_basis(j, tsl, nt) for j in range(nt)])
            t3 = ls[:, None, None] * lt[None, :, None] * lp[None, None, :]
            want += q * m["w"][p] / nl * t3
            wantj += q * m["w"][p] / nl * m["vpar"][p] * t3
    scale = np.abs(want).max()
    assert np.abs(rho - want).max() < 1e-10 * scale
    assert np.abs(jp - wantj).max() < 1e-10 * np.abs(wantj).max()


def test_ring_clamp_and_axis():
    """R11 (ii): points beyond the edge are moved to s = 1; a ring enclosing the axis is legal."""
    g = O.geom(16, 32, 16, rho_star=0.2)
    r = O.ring_points(g, O.policy_fixed(8), 0.95, 0.3, 1.0)
    assert r["s"].max() == 1.0 and (np.hypot(r["x"], r["z"]) > 1).any()
    r = O.ring_points(g, O.policy_fixed(8), 0.05, 2.0, 1.0)
    assert (r["s"] >= 0).all()
    assert np.ptp(np.sort(r["thetastar"])) > math.pi           # wraps around the axis


def test_discrete_gyroaverage_closed_forms():
    """P7: ring average of cos(kappa x): 4 points -> cos(k x0)(1+cos(k rho))/2; many -> J0."""
    g = O.geom(16, 32, 16, rho_star=1 / 10.0, theta_map=1)
    s, ts, mu = 0.45, 2.2, 0.8
    rho = O.larmor_radius(g, s, ts, mu)
    x0 = O.ring_points(g, O.policy_fixed(1), s, ts, mu)["x"][0]
    for kappa in (1.0, 5.0, 12.0):
        r = O.ring_points(g, O.policy_fixed(4), s, ts, mu)
        got = np.cos(kappa * r["x"]).mean()
        assert abs(got - math.cos(kappa * x0) * (1 + math.cos(kappa * rho)) / 2) < 1e-14
        r = O.ring_points(g, O.policy_fixed(32), s, ts, mu)
        got = np.cos(kappa * r["x"]).mean()
        assert kappa * rho <= 2
        assert abs(got - special.j0(kappa * rho) * math.cos(kappa * x0)) < 1e-10


def test_adaptive_rule():
    """R9: N = min(n_max, n_min * max(1, ceil(rho/rho_ref)))."""
    pol = O.policy_adaptive(4, 32, 0.01)
    assert O.nl(pol, 0.0) == 4
    assert O.nl(pol, 0.0099) == 4
    assert O.nl(pol, 0.0101) == 8
    assert O.nl(pol, 0.035) == 16
    assert O.nl(pol, 1.0) == 32
    assert O.nl(O.policy_adaptive(4, 16, 0.01), 0.079) == 16
    assert O.nl(O.policy_fixed(7), 123.0) == 7


def test_adaptive_histogram_rayleigh():
    """P12: with rho_ref = rho*, N_L = 4 ceil(v_perp/B); for B == 1 and Rayleigh v_perp,
    P(N = 4m) = exp(-(m-1)^2/2) - exp(-m^2/2).  B varies by +-30 %, so compare loosely and
    check the survey's Monte-Carlo mix to 1 %."""
    cfg = W.scaled(W.CONFIGS["cfg2"], 200_000)
    m = W.generate(cfg, workers=1)
    g = O.geom(cfg.ns, cfg.ntheta, cfg.nphi, rho_star=cfg.rho_star)
    pol = O.policy_adaptive(4, 32, cfg.rho_ref)
    hist, npts = O.nl_histogram(g, pol, m["s"], m["theta"], m["mu"])
    frac = hist / hist.sum()
    assert hist.sum() == cfg.n_markers and npts == (hist * np.arange(len(hist))).sum()
    assert set(np.nonzero(hist)[0]) <= {4, 8, 12, 16, 20, 24, 28, 32}
    for mm in (1, 2, 3):
        closed = math.exp(-(mm - 1) ** 2 / 2) - math.exp(-mm ** 2 / 2)
        assert abs(frac[4 * mm] - closed) < 0.04
    np.testing.assert_allclose(frac[[4, 8, 12, 16]], [0.410, 0.458, 0.118, 0.0129], atol=0.01)
    assert abs(npts / cfg.n_markers - 6.94) < 0.1


# ------------------------------------------------------------ deposition ---

def test_conservation_all_policies():
    """P1: sum rho = q sum w, sum jpar = q sum w vpar -- fixed, adaptive, clamped rings, both maps."""
    m = small_markers(3000, s_lo=0.02, s_hi=0.99)
    for tm in (1, 0):
        for rs in (1 / 180.0, 1 / 20.0, 0.3):
            g = O.geom(16, 32, 16, rho_star=rs, q=1.7, theta_map=tm)
            for pol in (O.policy_fixed(1), O.policy_fixed(4), O.policy_fixed(7),
                        O.policy_adaptive(4, 32, rs)):
                rho, jp, npts = dep(g, pol, m)
                scale = np.abs(m["w"]).sum() * 1.7
                assert abs(rho.sum() - 1.7 * m["w"].sum()) < 1e-13 * scale
                assert abs(jp.sum() - 1.7 * (m["w"] * m["vpar"]).sum()) < 3e-13 * scale


def test_point_on_node():
    """P2: one marker on a node, N_L = 1 -> 27 nodes = q w {1/6,4/6,1/6}^3, 4th weight 0."""
    ns, nt, nph = 16, 32, 16
    g = O.geom(ns, nt, nph, q=2.0)
    for (i, j, k) in [(5, 7, 3), (2, 0, 0), (14, 31, 15), (8, 1, 15)]:
        one = lambda v: np.array([v])
        rho, _, npts = O.deposit(g, O.policy_fixed(1), one(i / ns), one(TWO_PI * j / nt),
                                 one(TWO_PI * k / nph), one(0.5), one(1.0), one(0.25), current=False)
        assert npts == 1
        want = np.zeros_like(rho)
        c = [1 / 6, 4 / 6, 1 / 6]
        # cardinal basis i+1 peaks at knot i: bases i, i+1, i+2 carry 1/6, 4/6, 1/6
        for a in range(3):
            for b in range(3):
                for d in range(3):
                    want[i + a, (j - 1 + b) % nt, (k - 1 + d) % nph] += 2.0 * 0.25 * c[a] * c[b] * c[d]
        np.testing.assert_allclose(rho, want, rtol=0, atol=1e-15)
        assert np.count_nonzero(np.abs(rho) > 1e-18) == 27
    for sval, basis in ((0.0, 0), (1.0, ns + 2)):
        rho, _, _ = O.deposit(g, O.policy_fixed(1), np.array([sval]), np.array([0.0]),
                              np.array([0.0]), None, np.array([1.0]), np.array([1.0]), current=False)
        assert abs(rho[basis].sum() - 2.0) < 1e-15 and abs(rho.sum() - 2.0) < 1e-15


def test_nl1_is_guiding_centre_and_zero_radius_limit():
    """P3: N_L = 1 deposits the guiding centre; rho* = 0 gives the same grid for any N_L."""
    m = small_markers(500)
    g = O.geom(16, 32, 16)
    g0 = O.geom(16, 32, 16, rho_star=0.0)
    ref, jref, _ = dep(g, O.policy_fixed(1), m)
    # guiding-centre deposition written from the spline definitions (no ring code involved)
    want = np.zeros_like(ref)
    for p in range(200):
        i0, ws = O.clamped_cubic(m["s"][p], 16)
        for i in range(19):
            li = ws[i - i0] if i0 <= i < i0 + 4 else 0.0
            if li == 0:
                continue
            lt = np.array([periodic_basis(j, m["theta"][p], 32) for j in range(32)])
            lp = np.array([periodic_basis(k, m["phi"][p], 16) for k in range(16)])
            want[i] += m["w"][p] * li * np.outer(lt, lp)
    got, _, _ = O.deposit(g, O.policy_fixed(1), *(m[f][:200] for f in W.FIELDS), current=False)
    np.testing.assert_allclose(got, want, rtol=0, atol=1e-16)
    for n in (4, 8):
        r, j, _ = dep(g0, O.policy_fixed(n), m)
        assert np.abs(r - ref).max() < 2e-15 * np.abs(ref).max() * 10
        assert np.abs(j - jref).max() < 2e-15 * np.abs(jref).max() * 10


@pytest.mark.parametrize("nl", [1, 4, 8])
def test_brute_force_node_centric(nl):
    """P4: every node as a gather over all Larmor points using the FUNCTION definitions
    (Cox-de Boor on the open knot vector; periodised beta3), tiny grid with N_theta, N_phi
    barely above 4 and markers in the end cells."""
    ns, nt, nph = 6, 5, 5
    m = small_markers(200, seed=7, s_lo=0.0, s_hi=1.0)
    g = O.geom(ns, nt, nph, rho_star=0.08, q=1.3)
    pol = O.policy_fixed(nl)
    rho, jp, npts = dep(g, pol, m)
    assert npts == 200 * nl
    T = open_knots(ns)
    want = np.zeros((ns + 3, nt, nph))
    wantj = np.zeros_like(want)
    for p in range(200):
        r = O.ring_points(g, pol, m["s"][p], m["theta"][p], m["mu"][p])
        lp = np.array([periodic_basis(k, m["phi"][p], nph) for k in range(nph)])
        for sl, tsl in zip(r["s"], r["thetastar"]):
            ls = np.array([cox_de_boor(i, 3, T, sl * ns) for i in range(ns + 3)])
            lt = np.array([periodic_basis(j, tsl, nt) for j in range(nt)])
            c = 1.3 * m["w"][p] / nl
            t3 = ls[:, None, None] * lt[None, :, None] * lp[None, None, :]
            want += c * t3
            wantj += c * m["vpar"][p] * t3
    np.testing.assert_allclose(rho, want, rtol=0, atol=1e-15)
    np.testing.assert_allclose(jp, wantj, rtol=0, atol=1e-15)


def test_first_moment_greville():
    """P8: cubic splines reproduce linear functions: sum_n xi_i rho[n] = sum_p (q w/N) sum_l s_pl."""
    ns = 16
    m = small_markers(2000, s_lo=0.0, s_hi=1.0)
    g = O.geom(ns, 32, 16, rho_star=0.05)
    pol = O.policy_fixed(4)
    rho, _, _ = dep(g, pol, m, current=False)
    T = open_knots(ns)
    xi = np.array([(T[i + 1] + T[i + 2] + T[i + 3]) / (3 * ns) for i in range(ns + 3)])
    lhs = (xi[:, None, None] * rho).sum()
    rhs = 0.0
    for p in range(2000):
        r = O.ring_points(g, pol, m["s"][p], m["theta"][p], m["mu"][p])
        rhs += m["w"][p] / 4 * r["s"].sum()
    assert abs(lhs - rhs) < 1e-13 * np.abs(m["w"]).sum()


def test_discrete_rotation():
    """P9: shifting phi by one cell rotates rho by one k index; same for theta* at N_L = 1."""
    m = small_markers(800)
    g = O.geom(16, 32, 16)
    rho, _, _ = dep(g, O.policy_fixed(4), m, current=False)
    m2 = dict(m, phi=m["phi"] + TWO_PI / 16)
    rho2, _, _ = dep(g, O.policy_fixed(4), m2, current=False)
    assert np.abs(np.roll(rho, 1, axis=2) - rho2).max() < 1e-12 * np.abs(rho).max()
    r1, _, _ = dep(g, O.policy_fixed(1), m, current=False)
    m3 = dict(m, theta=m["theta"] + TWO_PI / 32)
    r3, _, _ = dep(g, O.policy_fixed(1), m3, current=False)
    assert np.abs(np.roll(r1, 1, axis=1) - r3).max() < 1e-12 * np.abs(r1).max()


def test_linearity_and_current():
    """P10: additive in w; jpar with vpar == 1 equals rho; q scales both."""
    m = small_markers(800)
    g = O.geom(16, 32, 16)
    pol = O.policy_fixed(4)
    rho, jp, _ = dep(g, pol, m)
    w2 = np.roll(m["w"], 17)
    ra, _, _ = dep(g, pol, dict(m, w=w2), current=False)
    rs, _, _ = dep(g, pol, dict(m, w=m["w"] + w2), current=False)
    assert np.abs(rs - (rho + ra)).max() < 1e-15
    r1, j1, _ = dep(g, pol, dict(m, vpar=np.ones_like(m["w"])))
    assert np.array_equal(r1, j1)
    g2 = O.geom(16, 32, 16, q=2.0)
    r2, j2, _ = dep(g2, pol, m)
    np.testing.assert_allclose(r2, 2 * rho, rtol=0, atol=1e-16)
    np.testing.assert_allclose(j2, 2 * jp, rtol=0, atol=1e-16)
    # deposit ADDS into the arrays it is given
    r3, _, _ = dep(g, pol, m, current=False, rho=rho.copy())
    np.testing.assert_allclose(r3, 2 * rho, rtol=0, atol=1e-16)


def test_permutation_invariance_and_ranges():
    """P11: marker order changes rho by rounding only; the range-split driver agrees."""
    cfg = W.scaled(W.CONFIGS["cfg0"], 20_000)
    m = W.generate(cfg, workers=1)
    g = O.geom(16, 32, 16)
    pol = O.policy_fixed(4)
    rho, jp, n0 = dep(g, pol, m)
    perm = np.argsort(W.cell_key(cfg, m["s"], m["theta"], m["phi"]), kind="stable")
    ms = {f: m[f][perm] for f in W.FIELDS}
    rs, js, n1 = dep(g, pol, ms)
    assert n0 == n1 == 80_000
    assert np.abs(rs - rho).max() < 1e-13 * np.abs(rho).max()
    assert np.abs(js - jp).max() < 1e-13 * np.abs(jp).max()
    rr, jr, n2, workers = O.deposit_ranges(g, pol, *(m[f] for f in W.FIELDS), workers=3)
    assert n2 == n0 and workers == 3
    assert np.abs(rr - rho).max() < 1e-13 * np.abs(rho).max()
    assert np.abs(jr - jp).max() < 1e-13 * np.abs(jp).max()


def test_cfg0_regression_golden():
    """Stored summary of the oracle on the first 4096 markers of cfg 0, written by
    tests/golden/make_cfg0_golden.py (which calls only oracle/): guards against silent edits."""
    import json
    want = json.load(open(os.path.join(GOLDEN, "cfg0_first4096.json")))
    cfg = W.scaled(W.CONFIGS["cfg0"], 4096)
    m = W.generate(cfg, workers=1)
    g = O.geom(cfg.ns, cfg.ntheta, cfg.nphi, rho_star=cfg.rho_star)
    rho, _, npts = dep(g, O.policy_fixed(4), m, current=False)
    assert npts == want["n_points"]
    assert abs(rho.sum() - want["sum"]) < 1e-15
    assert abs(np.abs(rho).max() - want["max_abs"]) < 1e-16
    for (i, j, k), v in zip(want["nodes"], want["values"]):
        assert abs(rho[i, j, k] - v) < 1e-16


# ------------------------------------------- NEXT-1: get fields + gyroaverage (oracle_gather) ---

def gat(g, pol, m, field, n=None):
    n = n or len(m["s"])
    return O.gather(g, pol, m["s"][:n], m["theta"][:n], m["phi"][:n], m["mu"][:n], field)


@pytest.mark.parametrize("policy", ["fixed1", "fixed4", "fixed7", "adaptive"])
def test_gather_is_the_adjoint_of_deposit(policy):
    """G1: <deposit(w), F> = q sum_p w_p gather(F)_p for any field F --
    ties every index, weight and 1/N_L of oracle_gather to the (pinned) oracle_deposit, markers in
    the radial end cells and rings clamped at s = 1 included."""
    m = small_markers(3000, seed=11, s_lo=0.0, s_hi=1.0)
    g = O.geom(12, 9, 7, r0=1.4, a=0.45, b0=1.8, rho_star=0.06, q=-1.7)
    pol = {"fixed1": O.policy_fixed(1), "fixed4": O.policy_fixed(4), "fixed7": O.policy_fixed(7, 0.3),
           "adaptive": O.policy_adaptive(4, 16, 0.06)}[policy]
    rng = np.random.default_rng(5)
    F = rng.standard_normal(O.grid_shape(g))
    rho, _, npts = dep(g, pol, m, current=False)
    out, npts_g = gat(g, pol, m, F)
    assert npts_g == npts
    lhs = float((rho * F).sum())
    rhs = float(g.q * (m["w"] * out).sum())
    scale = abs(g.q) * np.abs(m["w"]).sum() * np.abs(F).max()
    assert abs(lhs - rhs) < 1e-13 * scale


def test_gather_constant_and_greville_fields():
    """G2: partition of unity -- a constant field is returned exactly for every marker (also
    those whose ring is clamped at s = 1 or encloses the axis).  G3: cubic splines reproduce
    linear functions: with F[i,j,k] = Greville abscissa xi_i the gather returns the mean of
    s_pl over the ring (ring_points is pinned by P6)."""
    ns = 10
    m = small_markers(1500, seed=3, s_lo=0.0, s_hi=1.0)
    g = O.geom(ns, 12, 6, rho_star=0.09)
    for pol in (O.policy_fixed(1), O.policy_fixed(4), O.policy_adaptive(4, 32, 0.09)):
        out, _ = gat(g, pol, m, np.full(O.grid_shape(g), 2.5))
        np.testing.assert_allclose(out, 2.5, rtol=0, atol=1e-14)
        T = open_knots(ns)
        xi = np.array([(T[i + 1] + T[i + 2] + T[i + 3]) / (3 * ns) for i in range(ns + 3)])
        F = np.broadcast_to(xi[:, None, None], O.grid_shape(g)).copy()
        out, _ = gat(g, pol, m, F)
        want = np.array([O.ring_points(g, pol, m["s"][p], m["theta"][p], m["mu"][p])["s"].mean()
                         for p in range(1500)])
        np.testing.assert_allclose(out, want, rtol=0, atol=2e-15)


@pytest.mark.parametrize("nl", [1, 4, 8])
def test_gather_dense_tensor_product_evaluation(nl):
    """G4: out[p] = mean_l sum_ijk F[ijk] Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p) with the basis
    FUNCTIONS evaluated densely -- scipy BSpline on the open knot vector in s, the periodised
    beta^3 definition in theta*, phi -- no index logic shared with the oracle.  For N_L = 1 this
    is plain tensor-product spline interpolation at (s, theta*, phi)."""
    ns, nt, nph = 6, 5, 7
    m = small_markers(150, seed=9, s_lo=0.0, s_hi=1.0)
    g = O.geom(ns, nt, nph, rho_star=0.08)
    pol = O.policy_fixed(nl)
    rng = np.random.default_rng(1)
    F = rng.standard_normal((ns + 3, nt, nph))
    T = open_knots(ns)
    basis = [interpolate.BSpline(T, np.eye(ns + 3)[i], 3, extrapolate=False) for i in range(ns + 3)]
    out, npts = gat(g, pol, m, F)
    assert npts == 150 * nl
    want = np.zeros(150)
    for p in range(150):
        r = O.ring_points(g, pol, m["s"][p], m["theta"][p], m["mu"][p])
        lp = np.array([periodic_basis(k, m["phi"][p], nph) for k in range(nph)])
        for sl, tsl in zip(r["s"], r["thetastar"]):
            x = min(sl * ns, ns * (1 - 1e-16))
            ls = np.nan_to_num(np.array([float(b(x)) for b in basis]))
            lt = np.array([periodic_basis(j, tsl, nt) for j in range(nt)])
            want[p] += np.einsum("i,j,k,ijk->", ls, lt, lp, F) / nl
    np.testing.assert_allclose(out, want, rtol=0, atol=2e-14)


def test_gather_linearity_rotation_and_threads():
    """Linear in the field; rotating field and markers by one phi cell leaves the result
    unchanged (wrap direction, cf. P9); marker ranges on threads are bit-identical."""
    m = small_markers(5000, seed=2)
    g = O.geom(16, 32, 16, rho_star=0.03)
    pol = O.policy_fixed(4)
    rng = np.random.default_rng(0)
    F1, F2 = rng.standard_normal((2,) + O.grid_shape(g))
    o1, _ = gat(g, pol, m, F1)
    o2, _ = gat(g, pol, m, F2)
    o12, _ = gat(g, pol, m, 2.0 * F1 - 3.0 * F2)
    np.testing.assert_allclose(o12, 2.0 * o1 - 3.0 * o2, rtol=0, atol=1e-14)
    m2 = dict(m)
    m2["phi"] = m["phi"] + TWO_PI / 16
    o1r, _ = gat(g, pol, m2, np.roll(F1, 1, axis=2))
    np.testing.assert_allclose(o1r, o1, rtol=0, atol=1e-13)
    ot, npts = O.gather(g, pol, m["s"], m["theta"], m["phi"], m["mu"], F1, workers=3)
    assert npts == 20000 and (ot == o1).all()
