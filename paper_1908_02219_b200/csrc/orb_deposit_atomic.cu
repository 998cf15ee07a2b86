// Global-atomics deposition: one thread per marker, every one of the 64 nodes of
// every Larmor point goes to the grid with a hardware fp64 reduction (RED.ADD.F64
// in L2).  This is the GPU algorithm the paper describes for P100/V100
// ("OpenACC atomic directives around accumulation instructions") and
// the correctness anchor / performance baseline of this library; the tile kernel
// (orb_deposit_tile.cu) replaces it on the fast path.
#include "orb_geom.cuh"

namespace orb {

__global__ void __launch_bounds__(256)
k_deposit_atomic(const Params P, const Markers M, double* __restrict__ rho,
                 double* __restrict__ jpar, unsigned long long* __restrict__ d_points) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int my_points = 0;
  if (p < M.n) {
    const MarkerData m = load_marker(M, p);
    const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
    const int n = g.n;
    my_points = (unsigned int)n;
    const double c = P.q * m.w / (double)n;
    const double cj = c * m.vpar;

    double wp[4];
    const int k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
    int kk[4];
    double cw[4], cjw[4];
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      kk[d] = wrap_index(k0 + d, P.nph);
      cw[d] = c * wp[d];
      cjw[d] = cj * wp[d];
    }

    for (int l = 0; l < n; ++l) {
      double s_l, ts_l;
      if (n == 1) {            // R8: the guiding centre itself
        s_l = g.s;
        ts_l = g.ts;
      } else {
        larmor_point(P, g, ring_entry(P, n, l), s_l, ts_l);
      }
      double ws[4], wt[4];
      const int i0 = radial_weights(P, s_l, ws);
      const int j0 = periodic_weights(ts_l, P.nth_scale, P.nth, wt);
#pragma unroll
      for (int a = 0; a < 4; ++a) {
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          const double v = ws[a] * wt[b];
          const int64_t row =
              ((int64_t)(i0 + a) * P.nth + wrap_index(j0 + b, P.nth)) * (int64_t)P.nph;
#pragma unroll
          for (int d = 0; d < 4; ++d) {
            atomicAdd(rho + row + kk[d], v * cw[d]);
            if (jpar) atomicAdd(jpar + row + kk[d], v * cjw[d]);
          }
        }
      }
    }
  }
  // sum of N_L over the launch: warp shuffle, then one atomic per warp
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) my_points += __shfl_down_sync(0xffffffffu, my_points, o);
  if ((threadIdx.x & 31) == 0 && my_points) atomicAdd(d_points, (unsigned long long)my_points);
}

int launch_deposit_atomic(const Params& P, const Markers& M, double* rho, double* jpar,
                          unsigned long long* d_points, cudaStream_t st) {
  if (M.n == 0) return 0;
  const int threads = 256;
  const int64_t blocks = (M.n + threads - 1) / threads;
  k_deposit_atomic<<<(unsigned int)blocks, threads, 0, st>>>(P, M, rho, jpar, d_points);
  return 1;
}

}  // namespace orb
