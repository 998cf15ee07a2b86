/*
 * orb_oracle.c -- ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded CPU statement of what the hot path computes:
 * gyro-averaged charge and parallel-current deposition of delta-f markers onto
 * a 3-D cubic B-spline finite-element grid in magnetic coordinates
 * (s, theta*, phi).  It shares no code, header, table or helper with the CUDA
 * path under paper_1908_02219_b200/csrc and is never called by it.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this file.
 *
 * The paper (arxiv 1908.02219, /root/reference/PAPER.md) gives the operation
 * in prose only; there is no equation or worked example.  Each function below
 * cites the passage it follows and, where the paper is silent, the reading
 * (R-number) of DESIGN.md "Readings of the paper" that it takes.
 *
 *   rho [i,j,k] = sum_p (q w_p        / N_L(p)) sum_l  Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p)
 *   jpar[i,j,k] = sum_p (q w_p vpar_p / N_L(p)) sum_l  Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p)
 *
 *   - markers in (s, theta*, phi), fields on 3-D finite-element B-splines up to
 *     third order
 *   - theta* = straight-field-line poloidal angle
 *   - Larmor points on a ring in the poloidal plane, number fixed or
 *     proportional to the ring size
 *   - Larmor ring data = real-space positions + guiding-centre weights
 *                                                              PAPER.md:73
 *   - "loops over the markers and then over the finite elements they
 *     contribute to" (unsorted deposition)
 *   - charge and current deposited together
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): partition of unity /
 * conservation, on-node 1/6-4/6-1/6 weights, clamped ends vs scipy BSpline,
 * N_L = 1 and rho* = 0 limits, node-centric brute force with Cox-de Boor and
 * periodised beta^3, theta* map vs quadrature, ring geometry, discrete
 * gyro-average vs closed form and Bessel J0, Greville first moment, discrete
 * rotation, linearity, permutation invariance, adaptive-N_L histogram vs the
 * Rayleigh closed form.
 * Choices the paper neither confirms nor contradicts (alpha0 = 0, clamped vs
 * ghost-node end treatment, rho_L in units of a) are "unpinned by the paper":
 * self-consistent and tested, listed in DESIGN.md.
 *
 * Arithmetic: IEEE double, textbook order; build with
 *   gcc -O2 -ffp-contract=off -fPIC -shared   (no FMA contraction).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define ORACLE_TWO_PI 6.283185307179586476925286766559
#define ORACLE_MAX_NL 64

typedef struct {
  int32_t ns, ntheta, nphi; /* CELLS; basis functions = (ns+3, ntheta, nphi)   */
  int32_t theta_map;        /* 1: theta* straight-field-line (R3); 0: theta*==theta */
  double r0, a, b0;         /* circular geometry (R1, R2)                       */
  double rho_star;          /* thermal Larmor radius / a (R6)                   */
  double q;                 /* species charge                                   */
} oracle_geom_t;

typedef struct {
  int32_t mode;    /* 0 fixed, 1 adaptive (R9)                                  */
  int32_t n_fixed; /* fixed: N_L ; adaptive: n_min                              */
  int32_t n_max;   /* adaptive cap                                              */
  int32_t pad_;
  double rho_ref;  /* adaptive reference radius, units of a                     */
  double alpha0;   /* gyro-phase of point 0 (R7)                                */
} oracle_policy_t;

/* R13: x - 2*pi*floor(x / 2*pi), result in [0, 2*pi] (2*pi only by rounding). */
double oracle_wrap_2pi(double u) { return u - ORACLE_TWO_PI * floor(u / ORACLE_TWO_PI); }

/* R3 ("modified from the geometric poloidal angle so that field
 * lines are straight"): for B ~ e_phi/R + (r/(qbar R0)) e_theta / R on
 * concentric circles, d(theta*)/d(theta) = sqrt(1-e^2)/(1+e cos theta), e = eps*s,
 * whose integral is theta* = 2 atan( sqrt((1-e)/(1+e)) tan(theta/2) ).
 * Written with atan2 so there is no pole at theta = pi. */
double oracle_thetastar_from_theta(double th, double e) {
  return oracle_wrap_2pi(2.0 * atan2(sqrt(1.0 - e) * sin(0.5 * th), sqrt(1.0 + e) * cos(0.5 * th)));
}
double oracle_theta_from_thetastar(double ts, double e) {
  return oracle_wrap_2pi(2.0 * atan2(sqrt(1.0 + e) * sin(0.5 * ts), sqrt(1.0 - e) * cos(0.5 * ts)));
}

/* Periodic cardinal cubic B-spline on [0, 2*pi) with n cells, node j at angle
 * 2*pi*j/n ("B-splines up to third order"; R13).  Returns the first
 * node index j0 = cell-1 (NOT wrapped; caller takes mod n) and the 4 weights of
 * nodes j0..j0+3. */
void oracle_periodic_cubic(double u, int32_t n, int32_t *j0, double w[4]) {
  double x = oracle_wrap_2pi(u) * (double)n / ORACLE_TWO_PI;
  double c = floor(x);
  double t = x - c;
  double omt = 1.0 - t;
  w[0] = omt * omt * omt / 6.0;
  w[1] = (3.0 * t * t * t - 6.0 * t * t + 4.0) / 6.0;
  w[2] = (-3.0 * t * t * t + 3.0 * t * t + 3.0 * t + 1.0) / 6.0;
  w[3] = t * t * t / 6.0;
  *j0 = (int32_t)c - 1;
}

/* Knot i of the open (clamped) knot vector T = {0,0,0,0, 1,2,...,n-1, n,n,n,n}. */
static double oracle_knot(int32_t i, int32_t n) {
  int32_t v = i - 3;
  if (v < 0) v = 0;
  if (v > n) v = n;
  return (double)v;
}

/* Clamped cubic B-splines on [0,1] with n cells, n+3 basis functions (R11 (i)).
 * Piegl & Tiller, The NURBS Book, algorithm A2.2 "BasisFuns" on T.
 * Returns cell c = min(floor(s*n), n-1) in *i0; the four non-zero functions are
 * the basis indices c..c+3. */
void oracle_clamped_cubic(double s, int32_t n, int32_t *i0, double w[4]) {
  double x = s * (double)n;
  int32_t c = (int32_t)floor(x);
  if (c > n - 1) c = n - 1;
  if (c < 0) c = 0;
  int32_t span = c + 3;
  double left[4], right[4];
  w[0] = 1.0;
  for (int j = 1; j <= 3; ++j) {
    left[j] = x - oracle_knot(span + 1 - j, n);
    right[j] = oracle_knot(span + j, n) - x;
    double saved = 0.0;
    for (int r = 0; r < j; ++r) {
      double temp = w[r] / (right[r + 1] + left[j - r]);
      w[r] = saved + right[r + 1] * temp;
      saved = left[j - r] * temp;
    }
    w[j] = saved;
  }
  *i0 = c;
}

/* O1-O2: Larmor radius in units of a at the guiding centre.
 * R2: B = B0 / (1 + eps s cos theta), theta the geometric angle;
 * R6: rho_L = rho* sqrt(2 mu / B). */
double oracle_larmor_radius(const oracle_geom_t *g, double s, double thetastar, double mu) {
  double e = (g->a / g->r0) * s;
  double th = g->theta_map ? oracle_theta_from_thetastar(thetastar, e) : thetastar;
  double B = g->b0 / (1.0 + e * cos(th));
  return g->rho_star * sqrt(2.0 * mu / B);
}

/* O3 / R9: number of Larmor points ("fixed or proportional to the
 * ring size", "fixed or adaptive (scaling with the ring size)"). */
int32_t oracle_nl(const oracle_policy_t *pol, double rho_l) {
  if (pol->mode == 0) return pol->n_fixed;
  double m = ceil(rho_l / pol->rho_ref);
  if (m < 1.0) m = 1.0;
  double n = (double)pol->n_fixed * m;
  if (n > (double)pol->n_max) n = (double)pol->n_max;
  return (int32_t)n;
}

/* O4-O5: the Larmor points of one marker.  Ring of radius rho_L in the poloidal
 * plane at the marker's phi (R5), equally spaced gyro-phases
 * (R7), mapped back to (s, theta*) (R1, R3), s clamped to <= 1 (R11 (ii)).
 * N_L = 1 is the guiding centre itself (R8).
 * Outputs (each may be NULL): magnetic coordinates sl, tsl and poloidal-plane
 * positions x, z relative to the magnetic axis in units of a.  Returns N_L. */
int32_t oracle_ring_points(const oracle_geom_t *g, const oracle_policy_t *pol, double s,
                           double thetastar, double mu, double *sl, double *tsl, double *x,
                           double *z) {
  double eps0 = g->a / g->r0;
  double e = eps0 * s;
  double th = g->theta_map ? oracle_theta_from_thetastar(thetastar, e) : thetastar;
  double B = g->b0 / (1.0 + e * cos(th));
  double rho = g->rho_star * sqrt(2.0 * mu / B);
  int32_t N = oracle_nl(pol, rho);
  double x0 = s * cos(th), z0 = s * sin(th);
  if (N == 1) {
    if (sl) sl[0] = s;
    if (tsl) tsl[0] = oracle_wrap_2pi(thetastar);
    if (x) x[0] = x0;
    if (z) z[0] = z0;
    return 1;
  }
  for (int32_t l = 0; l < N; ++l) {
    double al = pol->alpha0 + ORACLE_TWO_PI * (double)l / (double)N;
    double xl = x0 + rho * cos(al);
    double zl = z0 + rho * sin(al);
    double s_l = sqrt(xl * xl + zl * zl);
    if (s_l > 1.0) s_l = 1.0;
    double thl = atan2(zl, xl);
    double ts_l = g->theta_map ? oracle_thetastar_from_theta(thl, eps0 * s_l) : oracle_wrap_2pi(thl);
    if (sl) sl[l] = s_l;
    if (tsl) tsl[l] = ts_l;
    if (x) x[l] = xl;
    if (z) z[l] = zl;
  }
  return N;
}

static int32_t oracle_mod(int32_t a, int32_t n) { return ((a % n) + n) % n; }

/* O1-O7: the deposition.  Adds into rho (and jpar unless NULL), both dense
 * double arrays in C order over (i_s, j_theta, k_phi), k fastest (R14), i_s in
 * [0, ns+3).  The value carried by each Larmor point is q w / N_L (times vpar
 * for the current): no cell volume, no Jacobian (R10).  Marker order p = 0..n-1,
 * then l, then the 4x4x4 nodes.  Returns sum_p N_L(p), or -1 if a marker asks
 * for more than ORACLE_MAX_NL points. */
int64_t oracle_deposit(const oracle_geom_t *g, const oracle_policy_t *pol, int64_t n,
                       const double *s, const double *thetastar, const double *phi,
                       const double *vpar, const double *mu, const double *w, double *rho,
                       double *jpar) {
  int64_t npts = 0;
  double sl[ORACLE_MAX_NL], tsl[ORACLE_MAX_NL];
  for (int64_t p = 0; p < n; ++p) {
    {
      double rl = oracle_larmor_radius(g, s[p], thetastar[p], mu[p]);
      if (oracle_nl(pol, rl) > ORACLE_MAX_NL) return -1;
    }
    int32_t N = oracle_ring_points(g, pol, s[p], thetastar[p], mu[p], sl, tsl, NULL, NULL);
    double c = g->q * w[p] / (double)N;
    double cj = jpar ? c * vpar[p] : 0.0;
    int32_t k0;
    double wphi[4];
    oracle_periodic_cubic(phi[p], g->nphi, &k0, wphi);
    for (int32_t l = 0; l < N; ++l) {
      int32_t i0, j0;
      double ws[4], wt[4];
      oracle_clamped_cubic(sl[l], g->ns, &i0, ws);
      oracle_periodic_cubic(tsl[l], g->ntheta, &j0, wt);
      for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b)
          for (int d = 0; d < 4; ++d) {
            int64_t node = ((int64_t)(i0 + a) * g->ntheta + oracle_mod(j0 + b, g->ntheta)) *
                               (int64_t)g->nphi +
                           oracle_mod(k0 + d, g->nphi);
            double v = ws[a] * wt[b] * wphi[d];
            rho[node] += c * v;
            if (jpar) jpar[node] += cj * v;
          }
    }
    npts += N;
  }
  return npts;
}

/* Histogram of N_L over a marker set (pin P12, bench bookkeeping).
 * hist has ORACLE_MAX_NL+1 entries. */
int64_t oracle_nl_histogram(const oracle_geom_t *g, const oracle_policy_t *pol, int64_t n,
                            const double *s, const double *thetastar, const double *mu,
                            int64_t *hist) {
  int64_t npts = 0;
  for (int i = 0; i <= ORACLE_MAX_NL; ++i) hist[i] = 0;
  for (int64_t p = 0; p < n; ++p) {
    int32_t N = oracle_nl(pol, oracle_larmor_radius(g, s[p], thetastar[p], mu[p]));
    if (N > ORACLE_MAX_NL) return -1;
    hist[N] += 1;
    npts += N;
  }
  return npts;
}

/* ------------------------------------------------------------------------------------------
 * NEXT-1: 'get fields' + 'gyroaverage' -- the transpose of the deposition.
 *
 *   out[p] = (1 / N_L(p)) sum_l  sum_{i,j,k} field[i,j,k] Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p)
 *
 *   - stage (3) of the PIC step: "the interpolation of the field at particle positions"
 *     (PAPER.md:71); with the Larmor ring data it splits into 'get fields' at the Larmor
 *     points and 'gyroaveraging' back to the guiding centre;
 *   - the field is the finite-element cubic B-spline expansion on the same grid as the
 *     deposited arrays, same layout (R14);
 *   - same ring, same points, same splines as oracle_deposit (O1-O6).
 * Reading R20 (the paper prints no formula): the value at a Larmor point is the spline
 * expansion evaluated there; the gyro-average is the arithmetic mean over the marker's N_L
 * points -- the discrete gyro-average whose weights 1/N_L the deposition uses, so that
 *   sum_n rho[n] field[n] = q sum_p w_p out[p]          (adjointness; pinned)
 * One field per call (several fields = several calls).  Field gradients are not formed here.
 * Marker order p = 0..n-1, then l, then the 4x4x4 nodes.  Returns sum_p N_L(p) or -1.
 * Pins (tests/test_oracle_pins.py): adjointness with oracle_deposit, constant field -> 1,
 * Greville (linear-in-s) field -> mean of s_pl, dense tensor-product evaluation with scipy
 * BSpline / periodised beta^3 at the ring points for N_L = 1, 4, 8, linearity in the field.
 */
int64_t oracle_gather(const oracle_geom_t *g, const oracle_policy_t *pol, int64_t n,
                      const double *s, const double *thetastar, const double *phi,
                      const double *mu, const double *field, double *out) {
  int64_t npts = 0;
  double sl[ORACLE_MAX_NL], tsl[ORACLE_MAX_NL];
  for (int64_t p = 0; p < n; ++p) {
    {
      double rl = oracle_larmor_radius(g, s[p], thetastar[p], mu[p]);
      if (oracle_nl(pol, rl) > ORACLE_MAX_NL) return -1;
    }
    int32_t N = oracle_ring_points(g, pol, s[p], thetastar[p], mu[p], sl, tsl, NULL, NULL);
    int32_t k0;
    double wphi[4];
    oracle_periodic_cubic(phi[p], g->nphi, &k0, wphi);
    double acc = 0.0;
    for (int32_t l = 0; l < N; ++l) {
      int32_t i0, j0;
      double ws[4], wt[4];
      oracle_clamped_cubic(sl[l], g->ns, &i0, ws);
      oracle_periodic_cubic(tsl[l], g->ntheta, &j0, wt);
      for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b)
          for (int d = 0; d < 4; ++d) {
            int64_t node = ((int64_t)(i0 + a) * g->ntheta + oracle_mod(j0 + b, g->ntheta)) *
                               (int64_t)g->nphi +
                           oracle_mod(k0 + d, g->nphi);
            acc += ws[a] * wt[b] * wphi[d] * field[node];
          }
    }
    out[p] = acc / (double)N;
    npts += N;
  }
  return npts;
}
