// Tile deposition, v2 (hot-path steps a1-a6, a8, a9): register accumulation through the fp64
// MMA unit, no shared-memory atomics on the per-point path.
//
// One thread block per grid tile = (1 toroidal cell slab k) x (kTileI radial cells) x (kTileJ
// poloidal cells); its markers are found through the binning pass's per-cell offsets
// (orb_bin.cu; key phi-major, so every radial row of the tile is one contiguous run).  The tile's
// markers are processed in chunks of <= kPCap Larmor points; per chunk
//
//   phase 1  (one lane per marker, then one lane per Larmor point -- the ring expansion is
//            warp-cooperative so that adaptive N_L = 4..32 keeps every lane busy):
//            marker -> guiding-centre geometry, N_L, c = q w / N_L, c * phi-weights, v_par
//            (a 40-byte entry of a shared-memory marker table);  Larmor point -> (s_l, theta*_l)
//            -> (s, theta*) cell + in-cell coordinates (t_s, t_theta), appended as a 16-byte
//            record; a per-cell counter is bumped (native 32-bit shared atomics).
//   phase 1c exclusive scan of the per-cell counts and an index permutation: the chunk's points
//            are now grouped by (s, theta*) cell.  (This is the paper's "sorting Larmor points by
//            cell", done per tile in shared memory instead of in HBM.)
//   phase 2  warps walk rows of cells along theta*.  All points of one cell hit the same 4 x 4
//            (s, theta*) nodes x 4 phi planes x {rho, jpar}; their sum is the dense contraction
//                 C[node(a,b)][channel(d,grid)] = sum_pts  ws_a(pt) wt_b(pt) * cw_d(pt) {1, vpar(pt)}
//            = A (16 x npts) . B (npts x 8), issued as two DMMA m8n8k4 per 4 points with the
//            accumulators in registers.  Each lane prepares ONE spline value per step (a cubic in
//            t with lane-constant coefficients, 3 FMA), the operands are exchanged by shuffles.
//            Stepping to the next cell shifts the accumulators by one node column (shuffle) and
//            retires the column that can receive nothing more into the shared-memory tile.
//
// and at the end the tile (nodes incl. halo x 4 planes x {rho, jpar}) is flushed ONCE with fp64
// RED.ADD to global memory.  Points whose cell leaves the tile's halo (long rings, rounding at a
// slab boundary) are deposited directly with global atomics (rare; counted).
//
// Why this shape: profiles/r01_microbench.md -- shared-memory fp64 atomics are CAS loops
// (1.5 updates/clk/SM at this access pattern) and global fp64 REDs issue at 0.78 lanes/clk/SM,
// while the path needs 128 node updates per Larmor point; only register accumulators keep up with
// the fp64 pipe (64 FMA/clk/SM).  DMMA runs on that same pipe at the same FMA rate (measured
// 18.5 TFMA/s either way) but needs one operand pair per 8 FMAs, which is what makes the operand
// traffic fit.
#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr int kThreads = 512;
constexpr int kWarps = kThreads / 32;
constexpr int kTileI = 8;     // radial cells per tile
constexpr int kTileJ = 32;    // poloidal cells per tile
constexpr int kHaloS = 2;     // ring reach in s covered by the tile, cells
constexpr int kHaloT = 4;     // ring reach in theta* covered by the tile, cells
constexpr int kCH = kTileI + 2 * kHaloS;   // cell rows held (12)
constexpr int kCW = kTileJ + 2 * kHaloT;   // cell columns held (40)
constexpr int kNH = kCH + 3;               // node rows (15)
constexpr int kNW = kCW + 3;               // node columns (43)
constexpr int kCells = kCH * kCW;
constexpr int kPCap = 4096;   // Larmor points per chunk
constexpr int kMCap = 1024;   // markers per chunk
constexpr int kSegW = 10;     // cells per walk segment
constexpr int kSegs = kCW / kSegW;
constexpr int kItems = kCH * kSegs;
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned short kNoCell = 0xffffu;
static_assert(kCW % kSegW == 0, "segments must tile the row");
static_assert(kPCap >= 32 * ORB_MAX_NL && kPCap <= 65535 && kMCap <= 65535 && kMCap % 32 == 0, "caps");
static_assert(kCells < kNoCell, "cell id must fit 16 bits");

template <int G>
struct Smem {
  double tile[kNH * kNW * 4 * G];     // [node row][node col][grid][phi plane]
  double2 rec[kPCap];                 // (t_s, t_theta) of a Larmor point
  double mtab[kMCap * 5];             // per marker: c*wphi[0..3], vpar
  unsigned short pmark[kPCap];        // marker-table slot of a point
  unsigned short pcell[kPCap];        // tile-local cell of a point, kNoCell if deposited directly
  unsigned short perm[kPCap];         // points grouped by cell
  unsigned int count[kCells + 1];     // per-cell counts, then running cursors
  unsigned int cstart[kCells + 1];    // exclusive scan of count
  unsigned int row_begin[kTileI], row_off[kTileI + 1];
  int deferred[2][kWarps];
  int n_deferred[2];
  int take_deferred;
  int next_group;
  unsigned int npts, nmark, pts_end;
  int full;
  int next_item;
};

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// angle u in [-2pi, 4pi] -> cell in [0, n) and in-cell coordinate
__device__ __forceinline__ int periodic_cell(double u, double scale, int n, double& t) {
  double x = u * scale;
  if (x < 0.0) x += (double)n;
  const double c = floor(x);
  t = x - c;
  int ci = (int)c;
  if (ci >= n) ci -= n;
  return ci;
}

// Direct deposition of one Larmor point with global atomics (points outside the tile's halo).
template <int G>
__device__ __noinline__ void deposit_point_global(const Params& P, double s_l, double ts_l, int k0,
                                                  const double* cw, double vpar,
                                                  double* __restrict__ rho,
                                                  double* __restrict__ jpar) {
  double ws[4], wt[4];
  const int i0 = radial_weights(P, s_l, ws);
  const int j0 = periodic_weights(ts_l, P.nth_scale, P.nth, wt);
#pragma unroll
  for (int a = 0; a < 4; ++a) {
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const double v = ws[a] * wt[b];
      const int64_t row = ((int64_t)(i0 + a) * P.nth + wrap_index(j0 + b, P.nth)) * (int64_t)P.nph;
#pragma unroll
      for (int d = 0; d < 4; ++d) {
        const int kk = wrap_index(k0 + d, P.nph);
        atomicAdd(rho + row + kk, v * cw[d]);
        if (G == 2) atomicAdd(jpar + row + kk, v * cw[d] * vpar);
      }
    }
  }
}

template <int G>   // G = 1: rho only; G = 2: rho and jpar
__global__ void __launch_bounds__(kThreads, 1)
k_deposit_tile(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
               double* __restrict__ rho, double* __restrict__ jpar,
               unsigned long long* __restrict__ d_points, int tiles_i, int tiles_j) {
  constexpr int NC = 4 * G;   // channels per (s, theta*) node: channel = grid*4 + phi plane
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<G>& S = *reinterpret_cast<Smem<G>*>(smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int tj = blockIdx.x % tiles_j;
  const int ti = (blockIdx.x / tiles_j) % tiles_i;
  const int k = blockIdx.x / (tiles_j * tiles_i);
  const int i_lo = ti * kTileI, j_lo = tj * kTileJ;
  const int i_hi = min(i_lo + kTileI, P.ns), j_hi = min(j_lo + kTileJ, P.nth);
  const int row_base = i_lo - kHaloS;        // radial cell (= first basis index) of cell row 0
  const int cellcol_base = j_lo - kHaloT;    // theta* cell of cell column 0 (may be < 0)

  if (tid == 0) {
    uint32_t off = 0;
    for (int r = 0; r < kTileI; ++r) {
      uint32_t b = 0, e = 0;
      if (i_lo + r < i_hi) {
        const int64_t c0 = ((int64_t)k * P.ns + (i_lo + r)) * P.nth;
        b = cell_start[c0 + j_lo];
        e = cell_start[c0 + j_hi];
      }
      S.row_begin[r] = b;
      S.row_off[r] = off;
      off += e - b;
    }
    S.row_off[kTileI] = off;
    S.n_deferred[0] = S.n_deferred[1] = 0;
    S.take_deferred = 0;
    S.next_group = 0;
    S.npts = 0;
    S.nmark = 0;
    S.pts_end = 0xffffffffu;
    S.full = 0;
    S.next_item = 0;
  }
  __syncthreads();
  const uint32_t n_tile = S.row_off[kTileI];
  if (n_tile == 0) return;
  const int n_groups = (int)((n_tile + 31) / 32);

  for (int x = tid; x < kNH * kNW * NC; x += kThreads) S.tile[x] = 0.0;
  for (int x = tid; x <= kCells; x += kThreads) S.count[x] = 0;
  __syncthreads();

  unsigned int my_points = 0, my_fallback = 0;
  int cur = 0;   // which deferred list is being consumed this chunk

  for (;;) {
    // ------------------------------------------------------------------ phase 1
    for (;;) {
      int grp = -1;
      if (lane == 0) {
        const int di = atomicAdd(&S.take_deferred, 1);
        if (di < S.n_deferred[cur]) {
          grp = S.deferred[cur][di];
        } else if (!*(volatile int*)&S.full) {
          const int gi = atomicAdd(&S.next_group, 1);
          if (gi < n_groups) grp = gi;
        }
      }
      grp = __shfl_sync(kFull, grp, 0);
      if (grp < 0) break;

      // a1-a3: one lane per marker
      const uint32_t v = (uint32_t)grp * 32u + (uint32_t)lane;
      const bool have = v < n_tile;
      int n = 0, k0 = 0;
      double ga = 0.0, gb = 0.0, grho = 0.0;   // (x0, z0, rho_L), or (s, theta*, -) when N_L = 1
      double cw[4] = {0.0, 0.0, 0.0, 0.0}, vpar = 0.0;
      if (have) {
        int r = 0;
        while (v >= S.row_off[r + 1]) ++r;
        const int64_t p = (int64_t)S.row_begin[r] + (v - S.row_off[r]);
        const MarkerData m = load_marker(M, p);
        const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
        n = g.n;
        const double c = P.q * m.w / (double)n;
        double wp[4];
        k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
#pragma unroll
        for (int d = 0; d < 4; ++d) cw[d] = c * wp[d];
        vpar = (G == 2) ? m.vpar : 0.0;
        if (n == 1) {   // R8: the guiding centre itself
          ga = g.s;
          gb = g.ts;
        } else {
          ga = g.x0;
          gb = g.z0;
        }
        grho = g.rho;
      }
      // the marker was binned into slab k, so k0 == k - 1 up to rounding at a cell boundary
      const int k_ok = have && (k0 == k - 1);

      int incl = n;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(kFull, incl, o);
        if (lane >= o) incl += t;
      }
      const int total = __shfl_sync(kFull, incl, 31);

      // capacity: marker slots first, then points (so that failed point allocations are a tail)
      unsigned int mb = 0, pb = 0;
      int ok = 1;
      if (lane == 0) {
        mb = atomicAdd(&S.nmark, 32u);
        if (mb + 32u > (unsigned)kMCap) {
          ok = 0;
        } else {
          pb = atomicAdd(&S.npts, (unsigned)total);
          if (pb + (unsigned)total > (unsigned)kPCap) {
            ok = 0;
            atomicMin(&S.pts_end, pb);
          }
        }
        if (!ok) {
          S.full = 1;
          const int slot = atomicAdd(&S.n_deferred[cur ^ 1], 1);
          S.deferred[cur ^ 1][slot] = grp;
        }
      }
      ok = __shfl_sync(kFull, ok, 0);
      if (!ok) break;
      mb = __shfl_sync(kFull, mb, 0);
      pb = __shfl_sync(kFull, pb, 0);
      my_points += (unsigned)n;

      {
        double* e = S.mtab + (size_t)(mb + lane) * 5;
        e[0] = cw[0]; e[1] = cw[1]; e[2] = cw[2]; e[3] = cw[3]; e[4] = vpar;
      }
      __syncwarp();

      // a4-a6: one lane per Larmor point of the group's 32 markers
      const int uniform_n = P.adaptive ? 0 : P.n_fixed;
      for (int q0 = 0; q0 < total; q0 += 32) {
        const int q = q0 + lane;
        const bool pvalid = q < total;
        const int qq = pvalid ? q : total - 1;
        int owner;
        if (uniform_n) {
          owner = qq / uniform_n;
        } else {
          owner = 0;
#pragma unroll
          for (int step = 16; step >= 1; step >>= 1) {
            const int t = __shfl_sync(kFull, incl, owner + step - 1);
            if (t <= qq) owner += step;
          }
        }
        const int o_incl = __shfl_sync(kFull, incl, owner);
        const int o_n = __shfl_sync(kFull, n, owner);
        const double o_a = __shfl_sync(kFull, ga, owner);
        const double o_b = __shfl_sync(kFull, gb, owner);
        const double o_rho = __shfl_sync(kFull, grho, owner);
        const int o_kok = __shfl_sync(kFull, k_ok, owner);
        const int o_k0 = __shfl_sync(kFull, k0, owner);
        if (!pvalid) continue;
        const int l = qq - (o_incl - o_n);
        double s_l, ts_l;
        if (o_n == 1) {
          s_l = o_a;
          ts_l = o_b;
        } else {
          GuidingCentre g;
          g.x0 = o_a;
          g.z0 = o_b;
          g.rho = o_rho;
          larmor_point(P, g, ring_entry(P, o_n, l), s_l, ts_l);
        }
        const double xs = s_l * (double)P.ns;
        const int ci = min((int)xs, P.ns - 1);
        const double t_s = xs - (double)ci;
        double t_t;
        const int cj = periodic_cell(ts_l, P.nth_scale, P.nth, t_t);
        const int lr = ci - row_base;
        int lc = cj - cellcol_base;
        if (lc >= P.nth) lc -= P.nth;
        if (lc < 0) lc += P.nth;
        const unsigned int slot = pb + (unsigned)q;
        if (o_kok && lr >= 0 && lr < kCH && lc >= 0 && lc < kCW) {
          const int cell = lr * kCW + lc;
          S.rec[slot] = make_double2(t_s, t_t);
          S.pmark[slot] = (unsigned short)(mb + owner);
          S.pcell[slot] = (unsigned short)cell;
          atomicAdd(&S.count[cell], 1u);
        } else {
          // footprint leaves the tile (long ring, or phi rounding): global atomics
          S.pcell[slot] = kNoCell;
          ++my_fallback;
          const double* e = S.mtab + (size_t)(mb + owner) * 5;
          deposit_point_global<G>(P, s_l, ts_l, o_k0, e, e[4], rho, jpar);
        }
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ phase 1c
    const unsigned int n_rec = min(S.npts, S.pts_end);
    if (wid == 0) {
      // exclusive scan of the kCells counts: 15 consecutive cells per lane
      constexpr int per = (kCells + 31) / 32;
      unsigned int loc[per];
      unsigned int sum = 0;
#pragma unroll
      for (int x = 0; x < per; ++x) {
        const int c = lane * per + x;
        loc[x] = c < kCells ? S.count[c] : 0;
        sum += loc[x];
      }
      unsigned int inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(kFull, inc, o);
        if (lane >= o) inc += t;
      }
      unsigned int ex = inc - sum;
#pragma unroll
      for (int x = 0; x < per; ++x) {
        const int c = lane * per + x;
        if (c < kCells) {
          S.cstart[c] = ex;
          S.count[c] = ex;   // running cursor for the permutation
        }
        ex += loc[x];
      }
      if (lane == 31) S.cstart[kCells] = inc;
    }
    __syncthreads();
    for (unsigned int q = tid; q < n_rec; q += kThreads) {
      const unsigned short c = S.pcell[q];
      if (c != kNoCell) {
        const unsigned int pos = atomicAdd(&S.count[c], 1u);
        S.perm[pos] = (unsigned short)q;
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ phase 2
    {
      const int g = lane >> 2, kk = lane & 3;
      // lane's spline piece: g < 4 -> radial basis g of the current row's cell (coefficients
      // loaded per row); g >= 4 -> cardinal theta* piece g - 4
      double k0c, k1c, k2c, k3c;
      {
        const int b = g & 3;
        k0c = (b == 0 || b == 2) ? (1.0 / 6.0) : (b == 1 ? (2.0 / 3.0) : 0.0);
        k1c = (b == 0) ? -0.5 : (b == 2 ? 0.5 : 0.0);
        k2c = (b == 0 || b == 2) ? 0.5 : (b == 1 ? -1.0 : 0.0);
        k3c = (b == 0) ? (-1.0 / 6.0) : (b == 1 ? 0.5 : (b == 2 ? -0.5 : (1.0 / 6.0)));
      }
      const int src_ws0 = 4 * (g >> 2) + kk;         // lane holding ws[a = g>>2] of point kk
      const int src_ws1 = 4 * (2 + (g >> 2)) + kk;   // ws[a = 2 + (g>>2)]
      const int src_wt = 4 * (4 + (g & 3)) + kk;     // wt[b = g&3]
      for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(&S.next_item, 1);
        item = __shfl_sync(kFull, item, 0);
        if (item >= kItems) break;
        const int lr = item / kSegs, sg = item - lr * kSegs;
        const int c_first = lr * kCW + sg * kSegW;
        if (S.cstart[c_first + kSegW] == S.cstart[c_first]) continue;   // no point in the segment
        const int irow = row_base + lr;   // radial cell; points exist only where 0 <= irow < ns
        double q0 = k0c, q1 = k1c, q2 = k2c, q3 = k3c;
        if (g < 4) {
          const double* tb = P.scoef + ((size_t)irow * 4 + g) * 4;
          q0 = __ldg(tb); q1 = __ldg(tb + 1); q2 = __ldg(tb + 2); q3 = __ldg(tb + 3);
        }
        double c00 = 0.0, c01 = 0.0, c10 = 0.0, c11 = 0.0;
        int live = 0;   // node columns of the accumulators that may be non-zero
        for (int step = 0; step < kSegW + 3; ++step) {
          const int lc = sg * kSegW + step;
          if (step < kSegW) {
            const int cell = c_first + step;
            const unsigned int start = S.cstart[cell];
            const int cnt = (int)(S.cstart[cell + 1] - start);
            if (cnt > 0) live = 4;
            for (int p0 = 0; p0 < cnt; p0 += 4) {
              const bool valid = p0 + kk < cnt;
              const unsigned int qi = valid ? S.perm[start + p0 + kk] : S.perm[start];
              const double2 t = S.rec[qi];
              const unsigned int mk = S.pmark[qi];
              const double tt = (g < 4) ? t.x : t.y;
              const double val = fma(fma(fma(q3, tt, q2), tt, q1), tt, q0);
              const double ws0 = __shfl_sync(kFull, val, src_ws0);
              const double ws1 = __shfl_sync(kFull, val, src_ws1);
              const double wt = __shfl_sync(kFull, val, src_wt);
              double b = S.mtab[mk * 5 + (g & 3)];
              if (G == 2 && g >= 4) b *= S.mtab[mk * 5 + 4];
              if (!valid || (G == 1 && g >= 4)) b = 0.0;
              dmma884(c00, c01, ws0 * wt, b);
              dmma884(c10, c11, ws1 * wt, b);
            }
          }
          if (live > 0) {
            // retire node column lc (b = 0): nodes (lr + a, lc), a = 2m + (g>>2), channels 2kk, 2kk+1
            if ((g & 3) == 0 && kk < 2 * G) {
              double* t0 = S.tile + ((size_t)(lr + (g >> 2)) * kNW + lc) * NC + 2 * kk;
              atomicAdd(t0, c00);
              atomicAdd(t0 + 1, c01);
              double* t1 = t0 + (size_t)2 * kNW * NC;
              atomicAdd(t1, c10);
              atomicAdd(t1 + 1, c11);
            }
            c00 = __shfl_down_sync(kFull, c00, 4);
            c01 = __shfl_down_sync(kFull, c01, 4);
            c10 = __shfl_down_sync(kFull, c10, 4);
            c11 = __shfl_down_sync(kFull, c11, 4);
            if ((g & 3) == 3) c00 = c01 = c10 = c11 = 0.0;
            --live;
          }
        }
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ next chunk?
    const bool more = S.n_deferred[cur ^ 1] > 0 || S.next_group < n_groups;
    __syncthreads();
    if (!more) break;
    cur ^= 1;
    if (tid == 0) {
      S.n_deferred[cur ^ 1] = 0;
      S.take_deferred = 0;
      S.npts = 0;
      S.nmark = 0;
      S.pts_end = 0xffffffffu;
      S.full = 0;
      S.next_item = 0;
    }
    for (int x = tid; x <= kCells; x += kThreads) S.count[x] = 0;
    __syncthreads();
  }

  // a9: one flush of the tile; consecutive lanes run along the 4 phi planes of a node (one
  // 32-byte sector of the k-fastest grid)
  int kpl[4];
#pragma unroll
  for (int d = 0; d < 4; ++d) kpl[d] = wrap_index(k - 1 + d, P.nph);
  for (int x = tid; x < kNH * kNW * 4; x += kThreads) {
    const int d = x & 3;
    const int node = x >> 2;
    const int nr = node / kNW, ncol = node - nr * kNW;
    const int gi = row_base + nr;
    if (gi < 0 || gi > P.ns + 2) continue;
    int gj = (cellcol_base - 1 + ncol) % P.nth;
    if (gj < 0) gj += P.nth;
    const int64_t idx = ((int64_t)gi * P.nth + gj) * (int64_t)P.nph + kpl[d];
    const double vr = S.tile[(size_t)node * NC + d];
    if (vr != 0.0) atomicAdd(rho + idx, vr);
    if (G == 2) {
      const double vj = S.tile[(size_t)node * NC + 4 + d];
      if (vj != 0.0) atomicAdd(jpar + idx, vj);
    }
  }

#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    my_points += __shfl_down_sync(kFull, my_points, o);
    my_fallback += __shfl_down_sync(kFull, my_fallback, o);
  }
  if (lane == 0) {
    if (my_points) atomicAdd(d_points, (unsigned long long)my_points);
    if (my_fallback) atomicAdd(d_points + 1, (unsigned long long)my_fallback);
  }
}

template <int G>
int launch(const Params& P, const Markers& M, const uint32_t* cell_start, double* rho, double* jpar,
           unsigned long long* d_points, cudaStream_t st) {
  const int tiles_i = (P.ns + kTileI - 1) / kTileI;
  const int tiles_j = (P.nth + kTileJ - 1) / kTileJ;
  const int64_t blocks = (int64_t)tiles_i * tiles_j * P.nph;
  const size_t smem = sizeof(Smem<G>);
  if (cudaFuncSetAttribute(k_deposit_tile<G>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)smem) != cudaSuccess)
    return -1;
  k_deposit_tile<G><<<(unsigned int)blocks, kThreads, smem, st>>>(P, M, cell_start, rho, jpar,
                                                                   d_points, tiles_i, tiles_j);
  return 1;
}

}  // namespace

int launch_deposit_tile(const Params& P, const Markers& M, const uint32_t* cell_start, double* rho,
                        double* jpar, unsigned long long* d_points, cudaStream_t st) {
  if (M.n == 0) return 0;
  return jpar ? launch<2>(P, M, cell_start, rho, jpar, d_points, st)
              : launch<1>(P, M, cell_start, rho, jpar, d_points, st);
}

}  // namespace orb
