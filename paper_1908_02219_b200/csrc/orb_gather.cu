// Get fields + gyroaverage ("the interpolation of the field
// at particle positions", PAPER.md:73, 89 'get fields' and 'gyroaverage'): the transpose of the
// deposition,
//
//   out_f[p] = (1 / N_L(p)) sum_l sum_{a,b,d} field_f[i0+a, j0+b, k0+d] ws_a(s_pl) wt_b(ts_pl) wphi_d(phi_p)
//
// with the same ring, map and cubic B-spline weights as the deposit (orb_geom.cuh), for up to
// kMaxFields fields per launch.  The grid is only read, so there is no accumulation race, no retire
// and no flush; the cost is the geometry (fp64 pipe) and the 64 node values per Larmor point and
// field (load path).
//
//   k_gather_tile<F>   one block per grid tile (1 toroidal slab x 8 radial x 16 poloidal cells +
//                      halo, the deposit's tile): the tile's 15 x 27 nodes x 4 phi planes x F
//                      fields are staged in shared memory ONCE (periodic wrap resolved there), the
//                      tile's markers are found through the binning pass's per-cell offsets, one
//                      lane per marker walks its ring.  The phi contraction is hoisted out of the
//                      ring: the lane accumulates acc[f][d] += ws_a wt_b * node[f][d] and applies
//                      the marker's 4 phi weights once at the end (all Larmor points of a marker
//                      share phi, R5).  Points whose footprint leaves the tile read the grid
//                      directly (rare; counted).
//   k_gather_direct<F> one thread per marker in bound order, node values through the read-only
//                      global path: used for unbinned markers (ORB_DEPOSIT_NO_BIN /
//                      ORB_DEPOSIT_ALGO_ATOMIC) and as the comparison kernel.
//
// Results are written in BOUND marker order: the binned record carries the marker's original
// index (orb_bin.cu).
#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr int kThreads = 256;
constexpr int kTileI = 8;
constexpr int kTileJ = 16;
constexpr int kHaloS = 2;
constexpr int kHaloT = 4;
constexpr int kCH = kTileI + 2 * kHaloS;   // cell rows held (12)
constexpr int kCW = kTileJ + 2 * kHaloT;   // cell columns held (24)
constexpr int kNH = kCH + 3;               // node rows (15)
constexpr int kNW = kCW + 3;               // node columns (27)
constexpr unsigned kFull = 0xffffffffu;
constexpr int kSortCap = 2048;             // markers of a tile that the on-chip sort handles
constexpr int kSortClasses = 8;            // N_L classes of the sort key: N_L <= 4, <= 8, ..., > 28
constexpr int kSortBins = kSortClasses * kTileI * kTileJ;   // (N_L class, cell) bins: 1024

template <int F>
struct Fields {
  const double* f[F];
  double* out[F];
};

// One Larmor point read straight from the grid: acc[f][d] += ws_a wt_b field_f[.., k0+d]
template <int F>
__device__ __forceinline__ void gather_point_global(const Params& P, const Fields<F>& fl, double s_l,
                                                    double ts_l, int k0, double (&acc)[F][4]) {
  double ws[4], wt[4];
  const int i0 = radial_weights(P, s_l, ws);
  const int j0 = periodic_weights(ts_l, P.nth_scale, P.nth, wt);
  int kk[4];
#pragma unroll
  for (int d = 0; d < 4; ++d) kk[d] = wrap_index(k0 + d, P.nph);
#pragma unroll
  for (int a = 0; a < 4; ++a) {
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const double v = ws[a] * wt[b];
      const int64_t row = ((int64_t)(i0 + a) * P.nth + wrap_index(j0 + b, P.nth)) * (int64_t)P.nph;
#pragma unroll
      for (int f = 0; f < F; ++f)
#pragma unroll
        for (int d = 0; d < 4; ++d) acc[f][d] = fma(v, __ldg(fl.f[f] + row + kk[d]), acc[f][d]);
    }
  }
}

// the same out of line, for the tile kernel's rare out-of-tile points (its accumulators live in
// local memory, apart from the lane's register accumulators)
template <int F>
__device__ __noinline__ void gather_point_global_rare(const Params& P, const Fields<F>& fl, double s_l,
                                                      double ts_l, int k0, double (&acc)[F][4]) {
  gather_point_global<F>(P, fl, s_l, ts_l, k0, acc);
}

// Larmor point l of the ring of g (fast small-angle form, full-range atan2 when the ring comes
// near the axis); N_L = 1 is the guiding centre itself (R8)
__device__ __forceinline__ void ring_point(const Params& P, const GuidingCentre& g, int l,
                                           double& s_l, double& ts_l) {
  if (g.n == 1) {
    s_l = g.s;
    ts_l = g.ts;
    return;
  }
  double X, Y;
  bool ok;
  larmor_point_fast(P, g.x0, g.z0, g.rho, g.ts, g.cg, g.sg, ring_entry(P, g.n, l), s_l, ts_l, X, Y,
                    ok);
  if (!ok) ts_l = atan2(Y, X);
}

__device__ __forceinline__ int64_t original_index(const Markers& M, int64_t p) {
  return M.rec ? (int64_t)__double_as_longlong(__ldg(M.rec + p * kRecDoubles + 6)) : p;
}

template <int F>
__device__ __forceinline__ void store_result(const Fields<F>& fl, int64_t idx, const double (&acc)[F][4],
                                             const double (&wp)[4], int n) {
  const double inv_n = 1.0 / (double)n;
#pragma unroll
  for (int f = 0; f < F; ++f) {
    const double v = fma(wp[0], acc[f][0], fma(wp[1], acc[f][1], fma(wp[2], acc[f][2], wp[3] * acc[f][3])));
    fl.out[f][idx] = v * inv_n;
  }
}

template <int F>
__global__ void __launch_bounds__(kThreads)
k_gather_direct(const Params P, const Markers M, const Fields<F> fl,
                unsigned long long* __restrict__ d_points) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int my_points = 0;
  if (p < M.n) {
    const MarkerData m = load_marker(M, p);
    const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
    my_points = (unsigned)g.n;
    double wp[4];
    const int k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
    double acc[F][4];
#pragma unroll
    for (int f = 0; f < F; ++f)
#pragma unroll
      for (int d = 0; d < 4; ++d) acc[f][d] = 0.0;
    for (int l = 0; l < g.n; ++l) {
      double s_l, ts_l;
      ring_point(P, g, l, s_l, ts_l);
      gather_point_global<F>(P, fl, s_l, ts_l, k0, acc);
    }
    store_result<F>(fl, original_index(M, p), acc, wp, g.n);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) my_points += __shfl_down_sync(kFull, my_points, o);
  if ((threadIdx.x & 31) == 0 && my_points) atomicAdd(d_points, (unsigned long long)my_points);
}

template <int F>
__global__ void __launch_bounds__(kThreads, 3)
k_gather_tile(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
              const TileBins TB, const Fields<F> fl, unsigned long long* __restrict__ d_points) {
    // [field][node row][node col][plane], the two 16-byte halves of a node swapped on every other
  // group of 4 nodes: lanes of a quarter-warp read the same half of (mostly) different nodes, and
  // the swap spreads them over all eight 16-byte bank groups instead of four
  __shared__ __align__(16) double tile[F * kNH * kNW * 4];
  __shared__ uint32_t row_begin[kTileI], row_off[kTileI + 1];
  __shared__ unsigned int hist[kSortBins];
  __shared__ unsigned int warp_tot[kThreads / 32];
  __shared__ unsigned int key_rank[kSortCap];
  __shared__ unsigned short order[kSortCap];
  const int tid = threadIdx.x;
  const int tj = blockIdx.x, ti = blockIdx.y, k = blockIdx.z;
  const int row_base = ti * kTileI - kHaloS;        // radial cell (= first basis index) of cell row 0
  const int cellcol_base = tj * kTileJ - kHaloT;    // theta* cell of cell column 0 (may be < 0)

  // the tile's markers: one contiguous run per radial row (key phi-major, orb_bin.cu)
  if (tid < kTileI) {
    uint32_t b, n;
    tile_run(P, cell_start, TB, tj, ti, k, tid, b, n);
    row_begin[tid] = b;
    row_off[tid + 1] = n;
  }
  __syncthreads();
  if (tid == 0) {
    uint32_t acc = 0;
    row_off[0] = 0;
    for (int r = 0; r < kTileI; ++r) {
      acc += row_off[r + 1];
      row_off[r + 1] = acc;
    }
  }
  __syncthreads();
  const uint32_t n_tile = row_off[kTileI];
  if (n_tile == 0) return;

  // stage the tile's nodes: 4 phi planes (k-1 .. k+2, wrapped) of every field
  for (int x = tid; x < kNH * kNW * F; x += kThreads) {
    const int f = x % F, node = x / F;
    const int nr = node / kNW, nc = node - nr * kNW;
    const int gi = row_base + nr;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    if (gi >= 0 && gi < P.ns + 3) {
      int gj = cellcol_base - 1 + nc;
      while (gj < 0) gj += P.nth;
      while (gj >= P.nth) gj -= P.nth;
      const double* src = fl.f[f] + ((int64_t)gi * P.nth + gj) * (int64_t)P.nph;
#pragma unroll
      for (int d = 0; d < 4; ++d) v[d] = __ldg(src + wrap_index(k - 1 + d, P.nph));
    }
    double2* dst = reinterpret_cast<double2*>(tile + (f * kNH * kNW + node) * 4);
    const int sw = (node >> 2) & 1;
    dst[sw] = make_double2(v[0], v[1]);
    dst[sw ^ 1] = make_double2(v[2], v[3]);
  }
  __syncthreads();

  unsigned int my_points = 0, my_fallback = 0;
  // (uniform over the tile) only tiles that reach the two end cells of the clamped radial basis
  // need the tabulated pieces
  const bool edge = row_base < 2 || row_base + kCH - 1 > P.ns - 3;
  // Order of work inside the tile.  Lanes of a warp that work on markers of the same cell read the
  // same nodes (shared-memory broadcast), and lanes whose markers have the same N_L leave the ring
  // loop together.  The dense cell-sorted layout gives the first for free; for slack bins (markers
  // of a tile row in any order) and for adaptive N_L the tile's markers are first put in
  // (N_L class, cell) order with a small counting sort on chip.  Measured: cfg3 from slack bins
  // 20.2 -> 14.5 ms (13.4 ms from the dense layout); cfg4 (N_L = 4..16) 112 -> see DESIGN.md 6.4.
  const bool resort = (TB.count != nullptr || P.adaptive) && n_tile <= (uint32_t)kSortCap;
  if (resort) {
    for (int x = tid; x < kSortBins; x += kThreads) hist[x] = 0;
    __syncthreads();
    for (uint32_t v = tid; v < n_tile; v += kThreads) {
      int r = 0;
#pragma unroll
      for (int x = 1; x < kTileI; ++x) r += (v >= row_off[x]) ? 1 : 0;
      const int64_t p = (int64_t)row_begin[r] + (v - row_off[r]);
      const MarkerData m = load_marker(M, p);
      int ci = (int)(fmin(fmax(m.s, 0.0), 1.0) * (double)P.ns) - ti * kTileI;
      int cj = (int)(wrap_2pi(m.th) * P.nth_scale) - tj * kTileJ;
      ci = min(max(ci, 0), kTileI - 1);      // (a mis-binned marker just lands in an edge cell)
      cj = min(max(cj, 0), kTileJ - 1);
      int cls = 0;
      if (P.adaptive) cls = min((guiding_centre(P, m.s, m.th, m.mu).n - 1) >> 2, kSortClasses - 1);
      const int c = (cls * kTileI + ci) * kTileJ + cj;
      const unsigned int rank = atomicAdd(&hist[c], 1u);
      key_rank[v] = (unsigned int)c | (rank << 16);
    }
    __syncthreads();
    {   // exclusive scan of the kSortBins counts: 4 per thread, warp scan, warp totals
      static_assert(kSortBins == 4 * kThreads, "one thread scans 4 bins");
      unsigned int c4[4], sum = 0;
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        c4[x] = hist[tid * 4 + x];
        sum += c4[x];
      }
      unsigned int inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(kFull, inc, o);
        if ((tid & 31) >= o) inc += t;
      }
      if ((tid & 31) == 31) warp_tot[tid >> 5] = inc;
      __syncthreads();
      unsigned int base = 0;
      for (int w = 0; w < (tid >> 5); ++w) base += warp_tot[w];
      unsigned int ex = base + inc - sum;
#pragma unroll
      for (int x = 0; x < 4; ++x) {
        hist[tid * 4 + x] = ex;
        ex += c4[x];
      }
    }
    __syncthreads();
    for (uint32_t v = tid; v < n_tile; v += kThreads) {
      const unsigned int kr = key_rank[v];
      order[hist[kr & 0xffffu] + (kr >> 16)] = (unsigned short)v;
    }
    __syncthreads();
  }
  for (uint32_t x = tid; x < n_tile; x += kThreads) {
    const uint32_t v = resort ? (uint32_t)order[x] : x;
    int r = 0;
#pragma unroll
    for (int y = 1; y < kTileI; ++y) r += (v >= row_off[y]) ? 1 : 0;
    const int64_t p = (int64_t)row_begin[r] + (v - row_off[r]);
    const MarkerData m = load_marker(M, p);
    const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
    my_points += (unsigned)g.n;
    double wp[4];
    const int k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
    const bool k_ok = (k0 == k - 1);
    double acc[F][4], facc[F][4];
    bool any_fallback = false;
#pragma unroll
    for (int f = 0; f < F; ++f)
#pragma unroll
      for (int d = 0; d < 4; ++d) acc[f][d] = 0.0;
    for (int l = 0; l < g.n; ++l) {
      double s_l, ts_l;
      ring_point(P, g, l, s_l, ts_l);
      const double xs = s_l * (double)P.ns;
      const int ci = min((int)xs, P.ns - 1);
      const double t_s = xs - (double)ci;
      double x = ts_l * P.nth_scale;
      if (x < 0.0) x += (double)P.nth;
      const double c = floor(x);
      const double t_t = x - c;
      int cj = (int)c;
      if (cj >= P.nth) cj -= P.nth;
      const int lr = ci - row_base;
      int lc = cj - cellcol_base;
      if (lc >= P.nth) lc -= P.nth;
      if (lc < 0) lc += P.nth;
      if (k_ok && lr >= 0 && lr < kCH && lc >= 0 && lc < kCW) {
        double ws[4], wt[4];
        if (edge) {
          radial_cell_weights(P, ci, t_s, ws);
        } else {
          cardinal_weights(t_s, ws);
        }
        cardinal_weights(t_t, wt);
        const int node0 = lr * kNW + lc;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
#pragma unroll
          for (int b = 0; b < 4; ++b) {
            const double w = ws[a] * wt[b];
            const int node = node0 + a * kNW + b;
            const int sw = (node >> 2) & 1;
            const double2* nd = reinterpret_cast<const double2*>(tile) + node * 2;
#pragma unroll
            for (int f = 0; f < F; ++f) {
              const double2 lo = nd[f * kNH * kNW * 2 + sw], hi = nd[f * kNH * kNW * 2 + (sw ^ 1)];
              acc[f][0] = fma(w, lo.x, acc[f][0]);
              acc[f][1] = fma(w, lo.y, acc[f][1]);
              acc[f][2] = fma(w, hi.x, acc[f][2]);
              acc[f][3] = fma(w, hi.y, acc[f][3]);
            }
          }
        }
      } else {
        if (!any_fallback) {
          any_fallback = true;
#pragma unroll
          for (int f = 0; f < F; ++f)
#pragma unroll
            for (int d = 0; d < 4; ++d) facc[f][d] = 0.0;
        }
        ++my_fallback;
        gather_point_global_rare<F>(P, fl, s_l, ts_l, k0, facc);
      }
    }
    if (any_fallback) {
#pragma unroll
      for (int f = 0; f < F; ++f)
#pragma unroll
        for (int d = 0; d < 4; ++d) acc[f][d] += facc[f][d];
    }
    store_result<F>(fl, original_index(M, p), acc, wp, g.n);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    my_points += __shfl_down_sync(kFull, my_points, o);
    my_fallback += __shfl_down_sync(kFull, my_fallback, o);
  }
  if ((tid & 31) == 0) {
    if (my_points) atomicAdd(d_points, (unsigned long long)my_points);
    if (my_fallback) atomicAdd(d_points + 1, (unsigned long long)my_fallback);
  }
}

template <int F>
int launch(const Params& P, const Markers& M, const uint32_t* cell_start, const TileBins& TB,
           const double* const* fields,
           double* const* out, unsigned long long* d_points, bool tiled, cudaStream_t st) {
  Fields<F> fl;
  for (int f = 0; f < F; ++f) {
    fl.f[f] = fields[f];
    fl.out[f] = out[f];
  }
  if (tiled) {
    const dim3 grid((P.nth + kTileJ - 1) / kTileJ, (P.ns + kTileI - 1) / kTileI, P.nph);
    k_gather_tile<F><<<grid, kThreads, 0, st>>>(P, M, cell_start, TB, fl, d_points);
  } else {
    const int64_t blocks = (M.n + kThreads - 1) / kThreads;
    k_gather_direct<F><<<(unsigned int)blocks, kThreads, 0, st>>>(P, M, fl, d_points);
  }
  return 1;
}

}  // namespace

int launch_gather(const Params& P, const Markers& M, const uint32_t* cell_start, const TileBins& TB,
                  int n_fields,
                  const double* const* fields, double* const* out, unsigned long long* d_points,
                  bool tiled, cudaStream_t st) {
  if (M.n == 0) return 0;
  int launches = 0;
  for (int f0 = 0; f0 < n_fields; f0 += 2) {   // two fields per launch (16 accumulators per lane)
    const int nf = n_fields - f0 >= 2 ? 2 : 1;
    launches += nf == 2 ? launch<2>(P, M, cell_start, TB, fields + f0, out + f0, d_points, tiled, st)
                        : launch<1>(P, M, cell_start, TB, fields + f0, out + f0, d_points, tiled, st);
    d_points = d_points + 2;   // only the first launch counts the points ([2], [3]: scratch)
  }
  return launches;
}

}  // namespace orb
