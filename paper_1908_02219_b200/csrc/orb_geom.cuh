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
  int n;           // N_L
};

__device__ __forceinline__ double wrap_2pi(double u) {
  return u - kTwoPi * floor(u * (1.0 / kTwoPi));
}

// a2 + a3: geometry at the guiding centre and number of Larmor points.
__device__ __forceinline__ GuidingCentre guiding_centre(const Params& P, double s, double th,
                                                        double mu) {
  GuidingCentre g;
  g.s = s;
  double ts = wrap_2pi(th);
  if (ts < 0.0) ts += kTwoPi;           // rounding of the reciprocal multiply
  if (ts > kTwoPi) ts -= kTwoPi;
  g.ts = ts;
  const double e = P.eps * s;
  double sn, cs;
  sincos(ts, &sn, &cs);
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

__device__ __forceinline__ double open_knot(int i, int n) { return (double)min(max(i - 3, 0), n); }

// Clamped (open knot vector) cubic B-splines, general cell: triangular Cox-de Boor
// scheme.  Only the two cells at each end differ from the cardinal polynomials.
static __device__ __noinline__ void clamped_end_weights(double x, int c, int n, double w[4]) {
  const int span = c + 3;
  double left[4], right[4];
  w[0] = 1.0;
#pragma unroll
  for (int j = 1; j <= 3; ++j) {
    left[j] = x - open_knot(span + 1 - j, n);
    right[j] = open_knot(span + j, n) - x;
    double saved = 0.0;
#pragma unroll
    for (int r = 0; r < j; ++r) {
      const double tmp = w[r] / (right[r + 1] + left[j - r]);
      w[r] = fma(right[r + 1], tmp, saved);
      saved = left[j - r] * tmp;
    }
    w[j] = saved;
  }
}

// a6, radial: cell i0 (= first basis index) and the 4 weights of bases i0..i0+3.
__device__ __forceinline__ int radial_weights(const Params& P, double s_l, double w[4]) {
  const double x = s_l * (double)P.ns;
  int c = min((int)x, P.ns - 1);       // s_l >= 0
  if (c >= 2 && c <= P.ns - 3) {
    cardinal_weights(x - (double)c, w);
  } else {
    clamped_end_weights(x, c, P.ns, w);
  }
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

__device__ __forceinline__ double2 ring_entry(const Params& P, int n, int l) {
  return __ldg(P.ring + (n * (n - 1) / 2 + l));
}

}  // namespace orb
