// Host-side table of the radial (clamped, open-knot-vector) cubic B-spline pieces as
// polynomials in the in-cell coordinate t = s*ns - cell (hot-path step a6, PAPER.md:19, 39;
// DESIGN.md R11).  For every radial cell c the four basis functions c..c+3 that are non-zero on
// it are cubics  p_a(t) = k0 + k1 t + k2 t^2 + k3 t^3 ; the tile kernel evaluates ONE of them per
// lane with lane-constant coefficients (3 FMA, Horner) instead of running the Cox-de Boor
// recursion per Larmor point.  Only the two cells at each end differ from the cardinal pieces.
//
// The pieces are obtained by running the Cox-de Boor recursion on polynomial coefficients:
//   N_{i,0} = 1 on the cell,   N_{i,p} = (x - T_i)/(T_{i+p} - T_i) N_{i,p-1}
//                                       + (T_{i+p+1} - x)/(T_{i+p+1} - T_{i+1}) N_{i+1,p-1},
// T = {0,0,0,0, 1, ..., ns-1, ns,ns,ns,ns}, 0/0 := 0, with x = c + t.
#include <vector>

#include "orb_internal.h"

namespace orb {

namespace {

struct Poly {
  double k[4];
};

double knot(int m, int ns) {
  int v = m - 3;
  if (v < 0) v = 0;
  if (v > ns) v = ns;
  return (double)v;
}

// (alpha + beta t) * p, truncated at degree 3 (never exceeded: p has degree <= 2 when called)
Poly mul_linear(const Poly& p, double alpha, double beta) {
  Poly r;
  r.k[0] = alpha * p.k[0];
  for (int d = 1; d < 4; ++d) r.k[d] = alpha * p.k[d] + beta * p.k[d - 1];
  return r;
}

}  // namespace

// out[(c*4 + a)*4 + d] = coefficient of t^d of basis c+a on cell c;  c = 0..ns-1
void build_radial_table(int ns, std::vector<double>& out) {
  out.assign((size_t)ns * 16, 0.0);
  for (int c = 0; c < ns; ++c) {
    const int span = c + 3;
    // N[j] = N_{span-p+j, p} for j = 0..p
    Poly N[4] = {};
    N[0].k[0] = 1.0;
    for (int p = 1; p <= 3; ++p) {
      Poly next[4] = {};
      for (int j = 0; j <= p; ++j) {
        const int i = span - p + j;
        Poly acc = {};
        // left term: uses N_{i,p-1} = previous index j-1
        if (j >= 1) {
          const double den = knot(i + p, ns) - knot(i, ns);
          if (den > 0.0) {
            const Poly t = mul_linear(N[j - 1], ((double)c - knot(i, ns)) / den, 1.0 / den);
            for (int d = 0; d < 4; ++d) acc.k[d] += t.k[d];
          }
        }
        // right term: uses N_{i+1,p-1} = previous index j
        if (j <= p - 1) {
          const double den = knot(i + p + 1, ns) - knot(i + 1, ns);
          if (den > 0.0) {
            const Poly t = mul_linear(N[j], (knot(i + p + 1, ns) - (double)c) / den, -1.0 / den);
            for (int d = 0; d < 4; ++d) acc.k[d] += t.k[d];
          }
        }
        next[j] = acc;
      }
      for (int j = 0; j <= p; ++j) N[j] = next[j];
    }
    for (int a = 0; a < 4; ++a)
      for (int d = 0; d < 4; ++d) out[((size_t)c * 4 + a) * 4 + d] = N[a].k[d];
  }
}

}  // namespace orb
