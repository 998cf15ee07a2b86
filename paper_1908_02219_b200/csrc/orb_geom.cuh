// Device-side geometry and spline weights of the deposition (hot-path steps a2-a6
// of DESIGN.md): guiding-centre geometry, N_L policy, Larmor-ring generator,
// map back to (s, theta*), cubic B-spline weights.  fp64 throughout.
//
// Written for the GPU, not a transcription of the CPU oracle: the theta* <-> theta
// map (R3) is used in its algebraic ("eccentric anomaly") form
//   cos(theta)  = (cos(theta*) - e) / (1 - e cos(theta*)),
//   sin(theta)  = sqrt(1-e^2) sin(theta*) / (1 - e cos(theta*)),
//   theta*_l    = atan2( sqrt(1-e_l^2) z_l , x_l + e_l r_l ),
// which needs one sincos per marker and one atan2 per Larmor point instead of
// the four trigonometric calls per point of the textbook form.
#pragma once
#include "orb_internal.h"

namespace orb {

struct GuidingCentre {
  double s, ts;    // s, wrapped theta* in [0, 2pi]
  double x0, z0;   // position in the poloidal plane relative to the axis, units of a
  double rho;      // Larmor radius, units of a
  double cg, sg;   // cos, sin of the wrapped theta*
  int n;           // N_L
};

__device__ __forceinline__ double wrap_2pi(double u) {
  return u - kTwoPi * floor(u * (1.0 / kTwoPi));
}

// a2 + a3: geometry at the guiding centre and number of Larmor points.
__device__ __forceinline__ GuidingCentre guiding_centre(const Params& P, double s, double th,
                                                        double mu) {
  GuidingCentre g;
  s = fmin(fmax(s, 0.0), 1.0);          // precondition 0 <= s <= 1; outside values deposit at the bound
  g.s = s;
  double ts = wrap_2pi(th);
  if (ts < 0.0) ts += kTwoPi;           // rounding of the reciprocal multiply
  if (ts > kTwoPi) ts -= kTwoPi;
  g.ts = ts;
  const double e = P.eps * s;
  double sn, cs;
  sincos(ts, &sn, &cs);
  g.cg = cs;
  g.sg = sn;
  double two_mu_over_b;
  if (P.theta_map) {
    const double d = fma(-e, cs, 1.0);          // 1 - e cos(theta*)
    const double om = fma(-e, e, 1.0);          // 1 - e^2
    const double inv_d = 1.0 / d;
    const double cth = (cs - e) * inv_d;
    const double sth = sqrt(om) * sn * inv_d;
    g.x0 = s * cth;
    g.z0 = s * sth;
    two_mu_over_b = 2.0 * mu * om * inv_d * P.inv_b0;   // 1/B = (1-e^2) / (B0 (1 - e cos theta*))
  } else {
    g.x0 = s * cs;
    g.z0 = s * sn;
    two_mu_over_b = 2.0 * mu * fma(e, cs, 1.0) * P.inv_b0;
  }
  g.rho = P.rho_star * sqrt(two_mu_over_b);
  int n = P.n_fixed;
  if (P.adaptive) {
    double m = ceil(g.rho * P.inv_rho_ref);
    m = fmax(m, 1.0);
    double nn = fmin((double)P.n_fixed * m, (double)P.n_max);
    n = (int)nn;
  }
  g.n = n;
  return g;
}

// a4 + a5: Larmor point l of the ring -> magnetic coordinates (s_l, theta*_l in (-pi, pi]).
__device__ __forceinline__ void larmor_point(const Params& P, const GuidingCentre& g, double2 cs_l,
                                             double& s_l, double& ts_l) {
  const double x = fma(g.rho, cs_l.x, g.x0);
  const double z = fma(g.rho, cs_l.y, g.z0);
  const double r = sqrt(fma(x, x, z * z));
  s_l = fmin(r, 1.0);                                   // R11: clamp to the edge
  if (P.theta_map) {
    const double e = P.eps * s_l;
    const double q = sqrt(fma(-e, e, 1.0));
    ts_l = atan2(q * z, fma(e, r, x));
  } else {
    ts_l = atan2(z, x);
  }
}

// ---- branch-free fp64 building blocks of the per-point geometry.  The library sqrt / division /
// atan2 carry special-case branches; straight-line code lets the compiler interleave the four
// Larmor points a producer lane works on (the path is bound by fp64 latency, not by operation count).

// sqrt(x) for normal positive x (<= 1 ulp): MUFU seed (about 20 bits) + two coupled Newton steps
// + one residual correction.  *half_inv receives 0.5 / sqrt(x).
__device__ __forceinline__ double sqrt_pos(double x, double* half_inv) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  double g = x * y, h = 0.5 * y;
  double r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  r = fma(-g, h, 0.5);
  g = fma(g, r, g);
  h = fma(h, r, h);
  const double d = fma(-g, g, x);
  *half_inv = h;
  return fma(d, h, g);
}

// a / b for normal b (<= 1 ulp): MUFU seed + two Newton steps + one residual correction
__device__ __forceinline__ double div_fast(double a, double b) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(b));
  double e = fma(-b, y, 1.0);
  y = fma(y, e, y);
  e = fma(-b, y, 1.0);
  y = fma(y, e, y);
  const double t = a * y;
  return fma(fma(-b, t, a), y, t);
}

// atan(t) for |t| <= 1/4: t * P(t^2), Taylor coefficients (-1)^k / (2k+1) up to k = 12
// (truncation error <= (1/16)^13 / 27 < 1e-17 relative)
constexpr double kAtanSmallMax = 0.25;
__device__ __forceinline__ double atan_small(double t) {
  const double u = t * t;
  double p = 1.0 / 25.0;
  p = fma(p, u, -1.0 / 23.0);
  p = fma(p, u, 1.0 / 21.0);
  p = fma(p, u, -1.0 / 19.0);
  p = fma(p, u, 1.0 / 17.0);
  p = fma(p, u, -1.0 / 15.0);
  p = fma(p, u, 1.0 / 13.0);
  p = fma(p, u, -1.0 / 11.0);
  p = fma(p, u, 1.0 / 9.0);
  p = fma(p, u, -1.0 / 7.0);
  p = fma(p, u, 1.0 / 5.0);
  p = fma(p, u, -1.0 / 3.0);
  return fma(t * u, p, t);
}

// a4 + a5, fast form: Larmor point -> (s_l, theta*_l) with theta*_l = theta*_gc + atan(cross / dot),
// where (X, Y) = (x + e r, sqrt(1-e^2) z) points along theta*_l (see the header of this file) and
// (cg, sg) = (cos, sin)(theta*_gc): the ring is small against the minor radius, so the angle between
// the two is small and a short odd polynomial replaces atan2.  *ok is false when it is not (rings
// that come near the axis); the caller then takes atan2(Y, X) from (*X, *Y).
__device__ __forceinline__ void larmor_point_fast(const Params& P, double x0, double z0, double rho,
                                                  double ts_gc, double cg, double sg, double2 cs_l,
                                                  double& s_l, double& ts_l, double& X, double& Y,
                                                  bool& ok) {
  const double x = fma(rho, cs_l.x, x0);
  const double z = fma(rho, cs_l.y, z0);
  const double r2 = fmax(fma(x, x, z * z), 1e-280);
  double hinv;
  const double r = sqrt_pos(r2, &hinv);
  s_l = fmin(r, 1.0);                                   // R11: clamp to the edge
  const double e = (P.theta_map ? P.eps : 0.0) * s_l;
  const double q = sqrt_pos(fma(-e, e, 1.0), &hinv);
  X = fma(e, r, x);
  Y = q * z;
  const double dot = fma(X, cg, Y * sg);
  const double cross = fma(Y, cg, -(X * sg));
  ok = fabs(cross) <= kAtanSmallMax * dot && dot > 0.0;   // false for NaN
  const double t = div_fast(cross, fmax(dot, 1e-280));
  ts_l = ts_gc + atan_small(ok ? t : 0.0);
}

// Periodic cardinal cubic B-spline weights at cell-unit coordinate x in [0, n]:
// cell c = floor(x) (may equal n by rounding: wraps), first node c-1.
__device__ __forceinline__ void cardinal_weights(double t, double w[4]) {
  const double omt = 1.0 - t;
  const double t2 = t * t;
  w[0] = omt * omt * omt * (1.0 / 6.0);
  w[1] = fma(t2, fma(0.5, t, -1.0), 2.0 / 3.0);
  w[2] = fma(t, fma(t, fma(-0.5, t, 0.5), 0.5), 1.0 / 6.0);
  w[3] = t2 * t * (1.0 / 6.0);
}

// a6, radial: the 4 weights of bases c..c+3 on radial cell c at in-cell coordinate t.  Cells
// 2..ns-3 carry the cardinal pieces; the two cells at each end of the clamped (open knot vector)
// basis differ and come from the host-built table of polynomial pieces (orb_spline_table.cu).
__device__ __forceinline__ void radial_cell_weights(const Params& P, int c, double t, double w[4]) {
  if (c >= 2 && c <= P.ns - 3) {
    cardinal_weights(t, w);
  } else {
    const double* tb = P.scoef + (size_t)c * 16;
#pragma unroll
    for (int a = 0; a < 4; ++a)
      w[a] = fma(fma(fma(__ldg(tb + a * 4 + 3), t, __ldg(tb + a * 4 + 2)), t, __ldg(tb + a * 4 + 1)),
                 t, __ldg(tb + a * 4));
  }
}

// a6, radial: cell i0 (= first basis index) and the 4 weights of bases i0..i0+3.
__device__ __forceinline__ int radial_weights(const Params& P, double s_l, double w[4]) {
  const double x = s_l * (double)P.ns;
  const int c = min(max((int)x, 0), P.ns - 1);
  radial_cell_weights(P, c, x - (double)c, w);
  return c;
}

// a6, periodic: angle u (any value in [-2pi, 4pi]) -> first node index j0 = cell-1 in
// [-1, n-1] (caller wraps j0+b into [0,n)) and weights.
__device__ __forceinline__ int periodic_weights(double u, double scale, int n, double w[4]) {
  double x = u * scale;
  if (x < 0.0) x += (double)n;
  double c = floor(x);
  const double t = x - c;
  int ci = (int)c;
  if (ci >= n) ci -= n;
  cardinal_weights(t, w);
  return ci - 1;
}

__device__ __forceinline__ int wrap_index(int j, int n) {
  j = (j < 0) ? j + n : j;
  return (j >= n) ? j - n : j;
}

// Marker load: SoA in bound order, or the library's binned 6-double records.
struct MarkerData {
  double s, th, ph, vpar, mu, w;
};
__device__ __forceinline__ MarkerData load_marker(const Markers& M, int64_t p) {
  MarkerData m;
  if (M.rec) {
    const double2* r = reinterpret_cast<const double2*>(M.rec + p * kRecDoubles);
    const double2 a = __ldg(r), b = __ldg(r + 1), c = __ldg(r + 2);
    m.s = a.x; m.th = a.y; m.ph = b.x; m.vpar = b.y; m.mu = c.x; m.w = c.y;
  } else {
    m.s = __ldg(M.s + p);
    m.th = __ldg(M.th + p);
    m.ph = __ldg(M.ph + p);
    m.vpar = M.vpar ? __ldg(M.vpar + p) : 0.0;
    m.mu = __ldg(M.mu + p);
    m.w = __ldg(M.w + p);
  }
  return m;
}

// The markers of grid tile (tj, ti, k) (8 radial x 16 poloidal cells of toroidal slab k), as up to
// 8 runs of binned records: run r = radial row r of the tile in the dense cell-sorted layout
// (orb_bin.cu: one contiguous run per row), or the tile's kTileBinSubs bins as runs 0.. in the
// slack-tile layout (orb_tilebin.cu).  -> first record and number of records of run r.
__device__ __forceinline__ void tile_run(const Params& P, const uint32_t* __restrict__ cell_start,
                                         const TileBins& TB, int tj, int ti, int k, int r, uint32_t& b,
                                         uint32_t& n) {
  b = 0;
  n = 0;
  if (TB.count) {
    if (r < kTileBinSubs) {
      const uint32_t t = ((uint32_t)k * (uint32_t)TB.tiles_i + (uint32_t)ti) * (uint32_t)TB.tiles_j + (uint32_t)tj;
      const uint32_t bin = t * (uint32_t)kTileBinSubs + (uint32_t)r;
      b = bin * TB.cap;
      n = min(__ldg(TB.count + bin), TB.cap);
    }
    return;
  }
  const int i = ti * 8 + r;
  if (i < P.ns) {
    const int j_lo = tj * 16, j_hi = min(j_lo + 16, P.nth);
    const int64_t c0 = ((int64_t)k * P.ns + i) * P.nth;
    b = __ldg(cell_start + c0 + j_lo);
    n = __ldg(cell_start + c0 + j_hi) - b;
  }
}

__device__ __forceinline__ double2 ring_entry(const Params& P, int n, int l) {
  return __ldg(P.ring + (n * (n - 1) / 2 + l));
}

}  // namespace orb
