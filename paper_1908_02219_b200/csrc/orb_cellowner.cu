// Materialised Larmor ring data + cell-owner deposition: the organisation
// the paper itself describes, built to be measured against the fused tile kernels.
//
//   PAPER.md:73  "a new data structure ..., named 'Larmor ring data', containing the positions in
//                real space of the Larmor markers and guiding center weights"
//   PAPER.md:75  "It also allows for the sorting of the Larmor markers by cells before depositing
//                them ... with sorting the outermost loop can be on the grid cells and the
//                innermost one on the particles in that cell."
//   PAPER.md:97  sorting "avoid[s] race conditions"
//
// Four steps, all on the caller's stream, Larmor ring data in HBM (library scratch reserved with
// orb_ring_reserve; 48 bytes per Larmor point, twice: unsorted and sorted):
//   1. k_ring_count   'build Larmor', pass 1: N_L per marker (bound order, no marker binning at
//                     all), then an exclusive scan -> first point slot of every marker.
//   2. k_ring_build   'build Larmor', pass 2: every Larmor point -> its field cell and in-cell
//                     coordinates; record {t_s, t_theta, t_phi, c = q w / N_L, c v_par, key|rank}
//                     at the marker's slots; the rank inside its cell comes from an integer atomic
//                     on the per-cell counter (the counting sort's histogram pass, fused in).
//   3. scan + k_ring_sort   exclusive scan of the per-cell counts; records to their sorted slots:
//                     the bucket sort of Larmor points by cell.
//   4. k_deposit_cellowner  outer loop over grid cells, inner loop over the points of the cell:
//                     one warp owns a run of cells of one radial row and toroidal slab and walks
//                     it along theta*.  All points of a cell hit the same 4 x 4 x 4 nodes (x 2
//                     grids): their sum is the contraction C[16 nodes][8 channels] = A . B issued
//                     as two fp64 MMAs (m8n8k4) per 4 points with register accumulators; each lane
//                     evaluates its own operands from (t_s, t_theta, t_phi).  Stepping to the next
//                     cell finishes one node column, which goes to the grid with fp64 RED.ADD: 32
//                     per cell instead of 128 per POINT.  No shared memory, no tile, no flush.
//                     The paper's cell loop is race-free on its CPUs because one thread owns a
//                     cell's elements; with cubic splines neighbouring cells (and the four radial
//                     rows that meet in a node) share nodes, so the column sums of different warps
//                     still meet in the grid through atomics.
#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr unsigned kFull = 0xffffffffu;
constexpr int kRingDoubles = 6;   // t_s, t_theta, t_phi, c, c*vpar, key|rank (sorted: 0)
constexpr int kWalk = 32;         // cells per warp walk

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(256)
k_ring_count(const Params P, const Markers M, uint32_t* __restrict__ off) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= M.n) return;
  const GuidingCentre g = guiding_centre(P, __ldg(M.s + p), __ldg(M.th + p), __ldg(M.mu + p));
  off[p] = (uint32_t)g.n;
}

// angle u (any value in [-2pi, 4pi]) -> cell in [0, n) and in-cell coordinate
__device__ __forceinline__ int angle_cell(double u, double scale, int n, double& t) {
  double x = u * scale;
  if (x < 0.0) x += (double)n;
  const double c = floor(x);
  t = x - c;
  int ci = (int)c;
  if (ci >= n) ci -= n;
  return ci;
}

__global__ void __launch_bounds__(256)
k_ring_build(const Params P, const Markers M, const uint32_t* __restrict__ off, int64_t capacity,
             uint32_t* __restrict__ cell_count, double* __restrict__ ring, double* __restrict__ rho,
             double* __restrict__ jpar, unsigned long long* __restrict__ d_points) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int my_points = 0, my_fallback = 0;
  if (p < M.n) {
    const MarkerData m = load_marker(M, p);
    const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
    my_points = (unsigned)g.n;
    const double c = P.q * m.w / (double)g.n;
    const double cj = c * m.vpar;
    double t_p;
    const int k = angle_cell(wrap_2pi(m.ph), P.nph_scale, P.nph, t_p);
    const int64_t first = off[p];
    for (int l = 0; l < g.n; ++l) {
      double s_l, ts_l;
      if (g.n == 1) {   // R8: the guiding centre itself
        s_l = g.s;
        ts_l = g.ts;
      } else {
        larmor_point(P, g, ring_entry(P, g.n, l), s_l, ts_l);
      }
      const double xs = s_l * (double)P.ns;
      const int i = min((int)xs, P.ns - 1);
      const double t_s = xs - (double)i;
      double t_t;
      const int j = angle_cell(ts_l, P.nth_scale, P.nth, t_t);
      if (first + l < capacity) {
        const uint32_t key = ((uint32_t)k * (uint32_t)P.ns + (uint32_t)i) * (uint32_t)P.nth + (uint32_t)j;
        const uint32_t rank = atomicAdd(cell_count + key, 1u);
        double* r = ring + (first + l) * kRingDoubles;
        const double2 a = make_double2(t_s, t_t), b = make_double2(t_p, c);
        const double2 d = make_double2(cj, __longlong_as_double((long long)(((uint64_t)key << 32) | rank)));
        reinterpret_cast<double2*>(r)[0] = a;
        reinterpret_cast<double2*>(r)[1] = b;
        reinterpret_cast<double2*>(r)[2] = d;
      } else {
        // beyond the reserved ring-data capacity: this point goes to the grid directly
        ++my_fallback;
        double ws[4], wt[4], wp[4];
        radial_cell_weights(P, i, t_s, ws);
        cardinal_weights(t_t, wt);
        cardinal_weights(t_p, wp);
        for (int a = 0; a < 4; ++a)
          for (int b = 0; b < 4; ++b) {
            const double v = ws[a] * wt[b];
            const int64_t row = ((int64_t)(i + a) * P.nth + wrap_index(j - 1 + b, P.nth)) * (int64_t)P.nph;
            for (int d = 0; d < 4; ++d) {
              const int kk = wrap_index(k - 1 + d, P.nph);
              atomicAdd(rho + row + kk, v * c * wp[d]);
              if (jpar) atomicAdd(jpar + row + kk, v * cj * wp[d]);
            }
          }
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    my_points += __shfl_down_sync(kFull, my_points, o);
    my_fallback += __shfl_down_sync(kFull, my_fallback, o);
  }
  if ((threadIdx.x & 31) == 0) {
    if (my_points) atomicAdd(d_points, (unsigned long long)my_points);
    if (my_fallback) atomicAdd(d_points + 1, (unsigned long long)my_fallback);
  }
}

__global__ void __launch_bounds__(256)
k_ring_sort(const uint32_t* __restrict__ off, int64_t n_markers, int64_t capacity,
            const uint32_t* __restrict__ cell_start, const double* __restrict__ ring,
            double* __restrict__ sorted) {
  const int64_t n_points = min((int64_t)off[n_markers], capacity);
  for (int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; x < n_points;
       x += (int64_t)gridDim.x * blockDim.x) {
    const double2* r = reinterpret_cast<const double2*>(ring + x * kRingDoubles);
    const double2 a = r[0], b = r[1];
    double2 d = r[2];
    const uint64_t kr = (uint64_t)__double_as_longlong(d.y);
    const int64_t dst = (int64_t)__ldg(cell_start + (uint32_t)(kr >> 32)) + (uint32_t)kr;
    d.y = 0.0;
    double2* o = reinterpret_cast<double2*>(sorted + dst * kRingDoubles);
    o[0] = a;
    o[1] = b;
    o[2] = d;
  }
}

// cardinal cubic B-spline piece b (weight of node cell-1+b) at in-cell coordinate t: pieces 0 / 3
// are y^3/6 and pieces 2 / 1 are 2/3 - y^2 + y^3/2, at y = 1 - t / t
__device__ __forceinline__ double cardinal_piece(int b, double t) {
  const double y = (b == 0 || b == 2) ? 1.0 - t : t;
  const double y2 = y * y;
  const double outer = y2 * y * (1.0 / 6.0);
  const double mid = fma(y2, fma(0.5, y, -1.0), 2.0 / 3.0);
  return (b == 0 || b == 3) ? outer : mid;
}

template <int G>
__global__ void __launch_bounds__(256)
k_deposit_cellowner(const Params P, const uint32_t* __restrict__ cell_start,
                    const double* __restrict__ pts, double* __restrict__ rho,
                    double* __restrict__ jpar, int walks_per_row) {
  const int lane = threadIdx.x & 31;
  const int64_t w = (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int64_t n_rows = (int64_t)P.nph * P.ns;
  if (w >= n_rows * walks_per_row) return;
  const int seg = (int)(w % walks_per_row);
  const int64_t row = w / walks_per_row;
  const int i = (int)(row % P.ns), k = (int)(row / P.ns);
  const int j_lo = seg * kWalk, j_hi = min(j_lo + kWalk, P.nth);
  const uint32_t* cs = cell_start + row * P.nth;
  if (__ldg(cs + j_lo) == __ldg(cs + j_hi)) return;   // no point in this run of cells

  const int g = lane >> 2, kk = lane & 3, hi = lane >> 4, a = g & 3;
  // radial piece a on cell row i: lane-constant cubic (tabulated pieces of the clamped basis)
  const double* tb = P.scoef + ((size_t)i * 4 + a) * 4;
  const double r0 = __ldg(tb), r1 = __ldg(tb + 1), r2 = __ldg(tb + 2), r3 = __ldg(tb + 3);
  const int dphi = g & 3;                     // phi plane of this lane's B element
  const bool use_cj = g >= 4;                 // channels 4..7 carry the current
  // this lane's retire targets: node row i + a, channels 2kk and 2kk + 1
  double* out0 = ((G == 2 && kk >= 2) ? jpar : rho) + wrap_index(k - 1 + ((2 * kk) & 3), P.nph);
  double* out1 = ((G == 2 && kk >= 2) ? jpar : rho) + wrap_index(k - 1 + ((2 * kk + 1) & 3), P.nph);
  const int64_t node_row = (int64_t)(i + a) * P.nth;
  const bool writes = (G == 2) || kk < 2;

  double c0a = 0.0, c0b = 0.0, c1a = 0.0, c1b = 0.0;   // slots hi and hi + 2
  auto retire = [&](int slot, int node_col) {   // slot's column is finished: add it to the grid
    const bool mine = (slot & 1) == hi;
    double va, vb;
    if (slot < 2) {
      va = c0a; vb = c0b;
      if (mine) { c0a = 0.0; c0b = 0.0; }
    } else {
      va = c1a; vb = c1b;
      if (mine) { c1a = 0.0; c1b = 0.0; }
    }
    if (mine && writes) {
      const int64_t o = (node_row + wrap_index(node_col, P.nth)) * (int64_t)P.nph;
      if (va != 0.0) atomicAdd(out0 + o, va);
      if (vb != 0.0) atomicAdd(out1 + o, vb);
    }
  };

  uint32_t begin = __ldg(cs + j_lo);
  for (int j = j_lo; j < j_hi; ++j) {
    const uint32_t end = __ldg(cs + j + 1);
    const int U = j & 3;
    // node column j - 1 + b lives in slot (U + b) & 3: this lane's slots hi, hi + 2 carry pieces
    const int b0 = (hi - U) & 3, b1 = (hi + 2 - U) & 3;
    for (uint32_t q = begin; q < end; q += 4) {
      double t_s = 0.0, t_t = 0.0, bval = 0.0;
      if (q + kk < end) {
        const double* r = pts + (size_t)(q + kk) * kRingDoubles;
        const double2 st = __ldg(reinterpret_cast<const double2*>(r));
        t_s = st.x;
        t_t = st.y;
        if (G == 2 || g < 4) {
          const double t_p = __ldg(r + 2);
          const double cw = __ldg(r + (use_cj ? 4 : 3));
          bval = cw * cardinal_piece(dphi, t_p);
        }
      }
      const bool live = q + kk < end;
      const double ws = live ? fma(fma(fma(r3, t_s, r2), t_s, r1), t_s, r0) : 0.0;
      const double a0 = ws * cardinal_piece(b0, t_t), a1 = ws * cardinal_piece(b1, t_t);
      __syncwarp();
      dmma884(c0a, c0b, a0, bval);
      dmma884(c1a, c1b, a1, bval);
    }
    begin = end;
    retire(U, j - 1);
  }
  // the three node columns beyond the last cell
  const int jl = j_hi - 1;
  retire((jl + 1) & 3, jl);
  retire((jl + 2) & 3, jl + 1);
  retire((jl + 3) & 3, jl + 2);
}

}  // namespace

// exclusive scan in place (orb_bin.cu): count[0..n) -> offsets, count[n] = total
int launch_scan(uint32_t* count, int64_t n, uint32_t* block_sums, cudaStream_t st);

int launch_deposit_ringdata(const Params& P, const Markers& M, const RingScratch& R, double* rho,
                            double* jpar, unsigned long long* d_points, cudaStream_t st) {
  if (M.n == 0) return 0;
  int launches = 0;
  const int64_t ncells = (int64_t)P.ns * P.nth * P.nph;
  if (cudaMemsetAsync(R.cell_start, 0, (size_t)(ncells + 1) * sizeof(uint32_t), st) != cudaSuccess)
    return -1;
  const int64_t mblocks = (M.n + 255) / 256;
  k_ring_count<<<(unsigned int)mblocks, 256, 0, st>>>(P, M, R.off);
  launches += 1 + launch_scan(R.off, M.n, R.block_sums, st);
  k_ring_build<<<(unsigned int)mblocks, 256, 0, st>>>(P, M, R.off, R.capacity, R.cell_start, R.ring, rho,
                                                       jpar, d_points);
  launches += 1 + launch_scan(R.cell_start, ncells, R.block_sums, st);
  k_ring_sort<<<148 * 16, 256, 0, st>>>(R.off, M.n, R.capacity, R.cell_start, R.ring, R.sorted);
  const int walks = (P.nth + kWalk - 1) / kWalk;
  const int64_t warps = (int64_t)P.nph * P.ns * walks;
  const unsigned int blocks = (unsigned int)((warps + 7) / 8);
  if (jpar)
    k_deposit_cellowner<2><<<blocks, 256, 0, st>>>(P, R.cell_start, R.sorted, rho, jpar, walks);
  else
    k_deposit_cellowner<1><<<blocks, 256, 0, st>>>(P, R.cell_start, R.sorted, rho, jpar, walks);
  return launches + 2;
}

}  // namespace orb
