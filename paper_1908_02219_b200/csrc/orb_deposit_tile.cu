// placeholder until the tile kernel lands: binned markers through the atomics kernel
#include "orb_internal.h"
namespace orb {
int launch_deposit_tile(const Params& P, const Markers& M, const uint32_t* cell_start, double* rho,
                        double* jpar, unsigned long long* d_points, cudaStream_t st) {
  (void)cell_start;
  return launch_deposit_atomic(P, M, rho, jpar, d_points, st);
}
}  // namespace orb
