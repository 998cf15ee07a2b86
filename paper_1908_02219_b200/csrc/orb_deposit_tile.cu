// Tile deposition (hot-path steps a1-a6, a8, a9): one thread block per grid tile
//   (1 toroidal cell slab k) x (TILE_I radial cells) x (TILE_J poloidal cells),
// the markers of the tile found through the binning pass's per-cell offsets
// (orb_bin.cu; key phi-major, so every radial row of the tile is one contiguous
// run of markers).  The block accumulates into a shared-memory copy of the tile's
// nodes -- 4 phi planes x (rho, jpar) per (s, theta*) node, with a halo for the
// spline support and the Larmor ring -- and flushes it ONCE with fp64 RED.ADD to
// global memory.  Points whose 4x4 (s, theta*) footprint leaves the halo go
// straight to global atomics (rare: ring radius ~0.7 cells in s).
//
// Shared-memory accumulation uses atomicAdd(double) on shared memory, which on
// sm_100a is a CAS loop (ATOMS.CAST.SPIN.64): measured 5.2 conflict-free
// updates/clk/SM against 0.78 lane-RED/clk/SM for global fp64 atomics
// (profiles/r01_microbench.md).  Threads take contiguous chunks of the tile's
// marker list so that the lanes of a warp work in different cells and rarely
// meet at the same node in the same instruction.
#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr int kTileThreads = 256;
constexpr int kTileI = 8;    // radial cells per tile
constexpr int kTileJ = 32;   // poloidal cells per tile
constexpr int kHaloS = 2;    // ring reach in s covered by the tile, cells
constexpr int kHaloT = 4;    // ring reach in theta* covered by the tile, cells
constexpr int kTileH = kTileI + 3 + 2 * kHaloS;   // node rows held in shared memory
constexpr int kTileW = kTileJ + 3 + 2 * kHaloT;   // node columns held in shared memory

template <int G>   // G = 1: rho only; G = 2: rho and jpar
__global__ void __launch_bounds__(kTileThreads)
k_deposit_tile(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
               double* __restrict__ rho, double* __restrict__ jpar,
               unsigned long long* __restrict__ d_points, int tiles_i, int tiles_j) {
  constexpr int NC = 4 * G;                       // values per (s, theta*) node: 4 phi planes x G
  extern __shared__ double tile[];                // [4][G][kTileH][kTileW]: plane-major, so that the
                                                  // lanes of one atomic (same plane, different nodes) spread over the banks
  __shared__ uint32_t row_begin[kTileI], row_off[kTileI + 1];

  const int tj = blockIdx.x % tiles_j;
  const int ti = (blockIdx.x / tiles_j) % tiles_i;
  const int k = blockIdx.x / (tiles_j * tiles_i);
  const int i_lo = ti * kTileI, j_lo = tj * kTileJ;
  const int i_hi = min(i_lo + kTileI, P.ns), j_hi = min(j_lo + kTileJ, P.nth);
  const int row_base = i_lo - kHaloS;             // node row of tile row 0 (may be < 0)
  const int col_base = j_lo - 1 - kHaloT;         // node column of tile column 0 (may be < 0)

  for (int x = threadIdx.x; x < kTileH * kTileW * NC; x += kTileThreads) tile[x] = 0.0;
  if (threadIdx.x == 0) {
    uint32_t off = 0;
    for (int r = 0; r < kTileI; ++r) {
      uint32_t b = 0, e = 0;
      if (i_lo + r < i_hi) {
        const int64_t c0 = ((int64_t)k * P.ns + (i_lo + r)) * P.nth;
        b = cell_start[c0 + j_lo];
        e = cell_start[c0 + j_hi];
      }
      row_begin[r] = b;
      row_off[r] = off;
      off += e - b;
    }
    row_off[kTileI] = off;
  }
  __syncthreads();

  const uint32_t n_tile = row_off[kTileI];
  // contiguous chunk per thread
  const uint32_t per = (n_tile + kTileThreads - 1) / kTileThreads;
  const uint32_t q_begin = min(threadIdx.x * per, n_tile);
  const uint32_t q_end = min(q_begin + per, n_tile);
  unsigned int my_points = 0, my_fallback = 0;

  int r_cur = 0;
  for (uint32_t qi = q_begin; qi < q_end; ++qi) {
    while (qi >= row_off[r_cur + 1]) ++r_cur;
    const int64_t p = (int64_t)row_begin[r_cur] + (qi - row_off[r_cur]);
    const MarkerData m = load_marker(M, p);
    const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
    const int n = g.n;
    my_points += (unsigned int)n;
    const double c = P.q * m.w / (double)n;

    double wp[4];
    const int k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
    double cw[NC];
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      cw[d * G] = c * wp[d];
      if (G == 2) cw[d * G + 1] = c * m.vpar * wp[d];
    }
    // the marker was binned into slab k, so k0 == k - 1 up to rounding at a cell boundary
    const bool k_ok = (k0 == k - 1);

    for (int l = 0; l < n; ++l) {
      double s_l, ts_l;
      if (n == 1) {
        s_l = g.s;
        ts_l = g.ts;
      } else {
        larmor_point(P, g, ring_entry(P, n, l), s_l, ts_l);
      }
      double ws[4], wt[4];
      const int i0 = radial_weights(P, s_l, ws);
      const int j0 = periodic_weights(ts_l, P.nth_scale, P.nth, wt);
      const int lr = i0 - row_base;
      int lc = j0 - col_base;
      if (lc >= P.nth) lc -= P.nth;
      if (lc < 0) lc += P.nth;
      if (k_ok && lr >= 0 && lr <= kTileH - 4 && lc >= 0 && lc <= kTileW - 4) {
#pragma unroll
        for (int a = 0; a < 4; ++a) {
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const double v = ws[a] * wt[b];
            double* t = tile + (lr + a) * kTileW + (lc + b);
#pragma unroll
            for (int x = 0; x < NC; ++x) atomicAdd(t + x * (kTileH * kTileW), v * cw[x]);
          }
        }
      } else {
        // footprint leaves the tile (long ring, or phi rounding): global atomics
        ++my_fallback;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const double v = ws[a] * wt[b];
            const int64_t row =
                ((int64_t)(i0 + a) * P.nth + wrap_index(j0 + b, P.nth)) * (int64_t)P.nph;
#pragma unroll
            for (int d = 0; d < 4; ++d) {
              const int kk = wrap_index(k0 + d, P.nph);
              atomicAdd(rho + row + kk, v * cw[d * G]);
              if (G == 2) atomicAdd(jpar + row + kk, v * cw[d * G + 1]);
            }
          }
        }
      }
    }
  }
  __syncthreads();

  // a9: one flush of the tile; lanes run along (column, phi plane) so that a warp
  // touches runs of 4 consecutive doubles (one 32-byte sector) per node
  int kk[4];
#pragma unroll
  for (int d = 0; d < 4; ++d) kk[d] = wrap_index(k - 1 + d, P.nph);
  for (int x = threadIdx.x; x < kTileH * kTileW * 4; x += kTileThreads) {
    const int d = x & 3;
    const int node = x >> 2;
    const int lr = node / kTileW, lc = node - lr * kTileW;
    const int gi = row_base + lr;
    if (gi < 0 || gi > P.ns + 2) continue;
    int gj = col_base + lc;
    gj %= P.nth;
    if (gj < 0) gj += P.nth;
    const int64_t idx = ((int64_t)gi * P.nth + gj) * (int64_t)P.nph + kk[d];
    const double vr = tile[(d * G) * (kTileH * kTileW) + node];
    if (vr != 0.0) atomicAdd(rho + idx, vr);
    if (G == 2) {
      const double vj = tile[(d * G + 1) * (kTileH * kTileW) + node];
      if (vj != 0.0) atomicAdd(jpar + idx, vj);
    }
  }

#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    my_points += __shfl_down_sync(0xffffffffu, my_points, o);
    my_fallback += __shfl_down_sync(0xffffffffu, my_fallback, o);
  }
  if ((threadIdx.x & 31) == 0) {
    if (my_points) atomicAdd(d_points, (unsigned long long)my_points);
    if (my_fallback) atomicAdd(d_points + 1, (unsigned long long)my_fallback);
  }
}

}  // namespace

int launch_deposit_tile(const Params& P, const Markers& M, const uint32_t* cell_start, double* rho,
                        double* jpar, unsigned long long* d_points, cudaStream_t st) {
  if (M.n == 0) return 0;
  const int tiles_i = (P.ns + kTileI - 1) / kTileI;
  const int tiles_j = (P.nth + kTileJ - 1) / kTileJ;
  const int64_t blocks = (int64_t)tiles_i * tiles_j * P.nph;
  if (jpar) {
    const size_t smem = (size_t)kTileH * kTileW * 8 * sizeof(double);
    if (cudaFuncSetAttribute(k_deposit_tile<2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)smem) != cudaSuccess)
      return -1;
    k_deposit_tile<2><<<(unsigned int)blocks, kTileThreads, smem, st>>>(
        P, M, cell_start, rho, jpar, d_points, tiles_i, tiles_j);
  } else {
    const size_t smem = (size_t)kTileH * kTileW * 4 * sizeof(double);
    k_deposit_tile<1><<<(unsigned int)blocks, kTileThreads, smem, st>>>(
        P, M, cell_start, rho, jpar, d_points, tiles_i, tiles_j);
  }
  return 1;
}

}  // namespace orb
