// Ring table of the Larmor-ring generator (hot-path step a4; R7: equally spaced gyro-phases
// alpha_l = alpha0 + 2 pi l / N measured from +R towards +Z): entry N(N-1)/2 + l holds
// (cos, sin)(alpha_l) for N = 1..ORB_MAX_NL, l < N.  Built by one small block on the caller's
// stream whenever alpha0 changes, so that orb_deposit never synchronises the host.
#include "orb_internal.h"

namespace orb {

__global__ void k_ring_table(double2* __restrict__ ring, double alpha0) {
  constexpr int total = ORB_MAX_NL * (ORB_MAX_NL + 1) / 2;
  for (int e = threadIdx.x; e < total; e += blockDim.x) {
    // N with N(N-1)/2 <= e < N(N+1)/2
    int n = (int)((1.0 + sqrt(1.0 + 8.0 * (double)e)) * 0.5);
    while (n * (n - 1) / 2 > e) --n;
    while (n * (n + 1) / 2 <= e) ++n;
    const int l = e - n * (n - 1) / 2;
    const double al = alpha0 + kTwoPi * (double)l / (double)n;
    double sn, cs;
    sincos(al, &sn, &cs);
    ring[e] = make_double2(cs, sn);
  }
}

int launch_ring_table(double2* ring, double alpha0, cudaStream_t st) {
  k_ring_table<<<1, 256, 0, st>>>(ring, alpha0);
  return 1;
}

}  // namespace orb
