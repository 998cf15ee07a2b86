// Tile deposition, v4 (hot-path steps a1-a6, a8, a9): register accumulation through the fp64
// MMA unit, several small thread blocks per SM so that the phases of different tiles overlap.
//
// One thread block per grid tile = (1 toroidal cell slab k) x (kTileI radial cells) x (kTileJ
// poloidal cells); its markers are found through the binning pass's per-cell offsets
// (orb_bin.cu; key phi-major, so every radial row of the tile is one contiguous run).  The tile's
// markers are processed in chunks of <= kPCap Larmor points, in bin order (a chunk is a few cell
// rows of markers, so its points fall on a compact window of cells); per chunk
//
//   phase 1a (one lane per marker): marker -> guiding-centre geometry, N_L, c = q w / N_L, then
//            c * phi-weights and c * v_par * phi-weights (the 8 channel values of the marker)
//            into a shared-memory marker table; a prefix sum of N_L over the warp's 32 markers
//            allocates the slots of their Larmor points.
//   phase 1b (one lane per Larmor point, all threads, evenly -- adaptive N_L = 4..32 keeps every
//            lane busy): point -> (s_l, theta*_l) -> (s, theta*) cell + in-cell coordinates
//            (t_s, t_theta), a 16-byte record; a per-cell counter is bumped (native 32-bit shared
//            atomic) and its return value is the point's rank inside its cell.
//   phase 1c exclusive scan of the per-cell counts, each rounded up to a multiple of 4, and an
//            index permutation: the chunk's points are now grouped by (s, theta*) cell, padded
//            with a zero-weight dummy point.  (This is the paper's "sorting Larmor points by
//            cell", done per tile in shared memory instead of in HBM.)
//   phase 2  each warp owns a row segment of kSegW cells and walks it along theta*.  All points of
//            one cell hit the same 4 x 4 (s, theta*) nodes x 4 phi planes x {rho, jpar}; their sum
//            is the dense contraction
//                 C[node(a,b)][channel(d,grid)] = sum_pts  ws_a(pt) wt_b(pt) * cw_d(pt) {1, vpar(pt)}
//            = A (16 x npts) . B (npts x 8), issued as two DMMA m8n8k4 per 4 points with the
//            accumulators in registers.  Every lane evaluates its own A operands from (t_s,
//            t_theta) -- one radial cubic and the two cardinal theta* pieces of its slots, which
//            are y^3/6 and 2/3 - y^2 + y^3/2 at y = t or 1 - t -- so no operand crosses lanes (the
//            shuffle unit shares the 128 B/clk/SM load-store path, which is as scarce here as the
//            fp64 pipe).  The four node columns of the accumulator window live in four fixed
//            "slots" (half-warp x DMMA); stepping to the next cell retires the slot of the
//            finished column into the shared tile (fp64 CAS add, 2 per lane of a half-warp) and
//            re-uses it for the new column -- no data moves, only the piece a lane evaluates
//            rotates (the walk is unrolled by 4).
//
// and at the end the tile is flushed ONCE with fp64 RED.ADD to global memory.  Points whose cell
// leaves the tile's halo (long rings, rounding at a slab boundary) are deposited directly with
// global atomics (rare; counted).
//
// Why this shape (profiles/r01_microbench.md, profiles/r01_final_deposit_ncu.md):
// shared-memory fp64 atomics are CAS loops (1.5 updates/clk/SM) and global fp64 REDs issue at
// 0.78 lanes/clk/SM, while the path needs 128 node updates per Larmor point; only register
// accumulators keep up with the fp64 pipe (64 FMA/clk/SM).  DMMA m8n8k4 occupies that pipe for
// 16 clk per SM sub-partition (same FMA rate as DFMA) but needs one operand pair per 8 FMAs.
// One 512-thread block per SM (v2, v3) left the SM waiting at barriers and on single-warp
// dependency chains; three 256-thread (or two 384-thread) blocks with ~70-95 KB of shared memory
// each overlap one tile's geometry with another's contraction and flush.  What moved the time from
// there on was what shortens a warp's dependency chain or its wait at a barrier (phase-2 work list
// heaviest first, reciprocals for divisions, two points in flight per lane), not what trims
// instruction, shared-memory-wavefront or fp64-operation counts.
#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr int kThreads = 384;
constexpr int kCtasPerSm = 2;
constexpr int kWarps = kThreads / 32;
constexpr int kTileI = 8;     // radial cells per tile
constexpr int kTileJ = 16;    // poloidal cells per tile
constexpr int kHaloS = 2;     // ring reach in s covered by the tile, cells
constexpr int kHaloT = 4;     // ring reach in theta* covered by the tile, cells
constexpr int kCH = kTileI + 2 * kHaloS;   // cell rows held (12)
constexpr int kCW = kTileJ + 2 * kHaloT;   // cell columns held (24)
constexpr int kNH = kCH + 3;               // node rows (15)
constexpr int kNW = kCW + 3;               // node columns (27)
constexpr int kCells = kCH * kCW;          // 288
constexpr int kSegW = 12;                  // cells per walk segment
constexpr int kSegs = kCW / kSegW;         // 2
constexpr int kItems = kCH * kSegs;        // 24
constexpr int kMCap = 384;    // markers per chunk
// Larmor points per chunk, a template parameter (PCAP) of the kernel: 4 per marker slot when
// N_L <= 4 is fixed (the marker cap binds), 6 per marker slot otherwise, so that adaptive N_L (mean
// ~7 points per marker) fills the marker slots too.  The small variant leaves 30 KB more of the
// SM's 228 KB to L1.
constexpr int kPCapSmall = 1536;
constexpr int kPCapLarge = 2304;
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kNoCell = 0x1ffu;       // meta cell field of a point deposited directly
static_assert(kCW % kSegW == 0 && kSegW % 4 == 0, "segments must tile the row in groups of 4");
static_assert(kPCapSmall >= 32 * ORB_MAX_NL && kPCapLarge < 4096 && kMCap % 32 == 0 && kMCap < 2047, "caps");
static_assert(kCells < (int)kNoCell, "cell id must fit 9 bits");
static_assert(kPCapLarge * 16 < 65536 && kMCap * 64 < 65536, "perm entries hold 16-bit byte offsets");

// meta word of a point slot.  After phase 1a: marker slot << 21 | point index in the ring.
// After phase 1b: marker slot << 21 | rank inside the cell << 9 | tile-local cell.
__device__ __forceinline__ unsigned meta_marker(unsigned m) { return m >> 21; }

struct MarkerTmp {      // phase 1a -> 1b hand-over, 32 bytes
  double a, b;          // (x0, z0), or (s, theta*) when N_L = 1
  double rho;
  int n;                // N_L; bit 8 set if the marker's phi cell is not this block's slab
  int k0;               // first phi node (phi cell - 1)
};

template <int G, int PCAP>
struct Smem {
  static constexpr int kPCap = PCAP;
  static constexpr int kPermCap = PCAP + 3 * kCells;   // points + padding to batches of 4
  double tile[kNH * kNW * 8];            // [node row][node col][grid*4 + phi plane]
  double2 rec[kPCap + 1];                // (t_s, t_theta) of a Larmor point; [kPCap] = dummy
  double mtab[(kMCap + 1) * 8];          // per marker: c*wphi[0..3], c*vpar*wphi[0..3]; [kMCap] = dummy (zeros)
  union {
    MarkerTmp mtmp[kMCap];               // phases 1a-1b
    unsigned int perm[kPermCap];         // phases 1c-2: points grouped by cell, each cell padded
  };                                     // to 4; entry = point slot | marker slot << 16
  unsigned int meta[kPCap + 1];
  unsigned int count[kCells + 1];        // per-cell counts
  unsigned int cstart[kCells + 1];       // exclusive scan of the padded counts
  unsigned int row_begin[kTileI], row_off[kTileI + 1];
  int deferred[2][kWarps];
  int n_deferred[2];
  int take_deferred;
  int next_group;
  unsigned int npts, nmark, pts_end;
  int full;
  int next_item;
  int n_items;                           // row segments of this chunk that hold points
  unsigned char item_order[kItems];      // ... heaviest first
};

#ifdef ORB_PHASE_CLOCKS
#define ORB_CLK(i)                                                          \
  do {                                                                      \
    if (tid == 0) {                                                         \
      const long long now__ = clock64();                                    \
      atomicAdd(d_points + 2 + (i), (unsigned long long)(now__ - clk__));   \
      clk__ = now__;                                                        \
    }                                                                       \
    __syncwarp();                                                           \
  } while (0)
#else
#define ORB_CLK(i) do { } while (0)
#endif

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
                                                  const double* cw, const double* cwv,
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
        if (G == 2) atomicAdd(jpar + row + kk, v * cwv[d]);
      }
    }
  }
}

template <int G, int PCAP>   // G = 1: rho only; G = 2: rho and jpar; PCAP: points per chunk
__global__ void __launch_bounds__(kThreads, kCtasPerSm)
k_deposit_tile(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
               const TileBins TB, double* __restrict__ rho, double* __restrict__ jpar,
               unsigned long long* __restrict__ d_points, int tiles_i, int tiles_j) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<G, PCAP>& S = *reinterpret_cast<Smem<G, PCAP>*>(smem_raw);
  constexpr int kPCap = PCAP;
  constexpr int kPermCap = Smem<G, PCAP>::kPermCap;

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
#ifdef ORB_PHASE_CLOCKS
  long long clk__ = clock64();
#endif
  const int tj = blockIdx.x, ti = blockIdx.y, k = blockIdx.z;
  const int i_lo = ti * kTileI, j_lo = tj * kTileJ;
  const int i_hi = min(i_lo + kTileI, P.ns), j_hi = min(j_lo + kTileJ, P.nth);
  const int row_base = i_lo - kHaloS;        // radial cell (= first basis index) of cell row 0
  const int cellcol_base = j_lo - kHaloT;    // theta* cell of cell column 0 (may be < 0)

  if (tid == 0) {
    uint32_t off = 0;
    for (int r = 0; r < kTileI; ++r) {
      uint32_t b, n;
      tile_run(P, cell_start, TB, tj, ti, k, r, b, n);
      S.row_begin[r] = b;
      S.row_off[r] = off;
      off += n;
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
    // dummy point and dummy marker used to pad every cell's point list to a multiple of 4
    S.rec[kPCap] = make_double2(0.0, 0.0);
    S.meta[kPCap] = (unsigned)kMCap << 21;
#pragma unroll
    for (int d = 0; d < 8; ++d) S.mtab[kMCap * 8 + d] = 0.0;
  }
  // (the zeroing overlaps thread 0's loads of the row offsets)
  for (int x = tid; x <= kCells; x += kThreads) S.count[x] = 0;
  for (int x = tid; x < kNH * kNW * 8; x += kThreads) S.tile[x] = 0.0;
  __syncthreads();
  const uint32_t n_tile = S.row_off[kTileI];
  if (n_tile == 0) return;
  const int n_groups = (int)((n_tile + 31) / 32);

  ORB_CLK(0);   // prologue
  unsigned int my_points = 0, my_fallback = 0;
  int cur = 0;     // which deferred list is being consumed this chunk
  int chunk = 0;

  for (;;) {
    // ------------------------------------------------------------------ phase 1a: markers
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
        const double c = P.q * m.w * __drcp_rn((double)n);
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
      // the marker was binned into slab k, so k0 == k - 1 up to rounding at a cell boundary;
      // if not, its points take the direct path
      const int k_ok = have && (k0 == k - 1);

      int incl, total;
      if (P.adaptive || n_tile - (uint32_t)grp * 32u < 32u) {
        incl = n;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int t = __shfl_up_sync(kFull, incl, o);
          if (lane >= o) incl += t;
        }
        total = __shfl_sync(kFull, incl, 31);
      } else {   // fixed N_L, full group: no scan needed
        incl = (lane + 1) * P.n_fixed;
        total = 32 * P.n_fixed;
      }

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

      const unsigned int ms = mb + (unsigned)lane;
      {
        double2* e = reinterpret_cast<double2*>(S.mtab + (size_t)ms * 8);
        e[0] = make_double2(cw[0], cw[1]);
        e[1] = make_double2(cw[2], cw[3]);
        e[2] = make_double2(cw[0] * vpar, cw[1] * vpar);
        e[3] = make_double2(cw[2] * vpar, cw[3] * vpar);
        MarkerTmp t;
        t.a = ga; t.b = gb; t.rho = grho;
        t.n = n | (k_ok ? 0 : 256);
        t.k0 = k0;
        S.mtmp[ms] = t;
      }
      {
        unsigned int q = pb + (unsigned)(incl - n);
        const unsigned int hi = ms << 21;
        for (int l = 0; l < n; ++l) S.meta[q + l] = hi | (unsigned)l;
      }
    }
    __syncthreads();
    ORB_CLK(1);   // phase 1a

    // ------------------------------------------------------------------ phase 1b: Larmor points
    const unsigned int n_rec = min(S.npts, S.pts_end);
    bool any_direct = false;
#pragma unroll 2
    for (unsigned int q = tid; q < n_rec; q += kThreads) {
      const unsigned int m0 = S.meta[q];
      const unsigned int ms = meta_marker(m0);
      const int l = (int)(m0 & 0x1fu);
      const MarkerTmp mt = S.mtmp[ms];
      const int n = mt.n & 255;
      GuidingCentre g;
      g.x0 = mt.a;
      g.z0 = mt.b;
      g.rho = mt.rho;
      double s_l, ts_l;
      larmor_point(P, g, ring_entry(P, n, l), s_l, ts_l);
      if (n == 1) {   // R8: the guiding centre itself, (s, theta*) as stored
        s_l = mt.a;
        ts_l = mt.b;
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
      if (mt.n < 256 && lr >= 0 && lr < kCH && lc >= 0 && lc < kCW) {
        const unsigned int cell = (unsigned)(lr * kCW + lc);
        S.rec[q] = make_double2(t_s, t_t);
        const unsigned int rank = atomicAdd(&S.count[cell], 1u);
        S.meta[q] = (ms << 21) | (rank << 9) | cell;
      } else {
        // footprint leaves the tile (long ring, or phi rounding): direct path below
        S.rec[q] = make_double2(s_l, ts_l);
        S.meta[q] = (ms << 21) | kNoCell;
        any_direct = true;
      }
    }
    if (any_direct) {   // rare: global atomics for the points marked above (own slots only)
      for (unsigned int q = tid; q < n_rec; q += kThreads) {
        const unsigned int m0 = S.meta[q];
        if ((m0 & 0x1ffu) != kNoCell) continue;
        const unsigned int ms = meta_marker(m0);
        const double2 pt = S.rec[q];
        const double* e = S.mtab + (size_t)ms * 8;
        ++my_fallback;
        deposit_point_global<G>(P, pt.x, pt.y, S.mtmp[ms].k0, e, e + 4, rho, jpar);
      }
    }
    __syncthreads();
    ORB_CLK(2);   // phase 1b

    // ------------------------------------------------------------------ phase 1c: sort by cell
    if (wid == 0) {
      // exclusive scan of the kCells counts, each padded to a multiple of 4: 9 cells per lane
      constexpr int per = (kCells + 31) / 32;
      unsigned int loc[per];
      unsigned int sum = 0;
#pragma unroll
      for (int x = 0; x < per; ++x) {
        const int c = lane * per + x;
        loc[x] = c < kCells ? ((S.count[c] + 3u) & ~3u) : 0;
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
        if (c < kCells) S.cstart[c] = ex;
        ex += loc[x];
      }
      if (lane == 31) S.cstart[kCells] = inc;
      __syncwarp();
      // phase 2 work list: the row segments that hold points, heaviest first (longest processing
      // time first keeps the warps' finishing times close: less waiting at the barrier)
      unsigned int wgt = 0;
      if (lane < kItems) {
        const int c0 = (lane >> 1) * kCW + (lane & 1) * kSegW;
        wgt = S.cstart[c0 + kSegW] - S.cstart[c0];
      }
      int rank = 0;
#pragma unroll
      for (int j = 0; j < kItems; ++j) {
        const unsigned int wj = __shfl_sync(kFull, wgt, j);
        rank += (wj > wgt || (wj == wgt && j < lane)) ? 1 : 0;
      }
      if (lane < kItems && wgt > 0) S.item_order[rank] = (unsigned char)lane;
      const unsigned int nz = __ballot_sync(kFull, lane < kItems && wgt > 0);
      if (lane == 0) S.n_items = __popc(nz);
    } else {
      // mtmp is dead from here on: its storage becomes perm, pre-filled with the dummy point
      const unsigned int fill = ((unsigned)kPCap * 16u) | (((unsigned)kMCap * 64u) << 16);
      for (int x = tid - 32; x < kPermCap; x += kThreads - 32) S.perm[x] = fill;
    }
    __syncthreads();
    for (unsigned int q = tid; q < n_rec; q += kThreads) {
      const unsigned int m = S.meta[q];
      const unsigned int c = m & 0x1ffu;
      if (c != kNoCell) S.perm[S.cstart[c] + ((m >> 9) & 0xfffu)] = (q * 16u) | (((m >> 21) * 64u) << 16);
    }
    __syncthreads();
    ORB_CLK(3);   // phase 1c

    // ------------------------------------------------------------------ phase 2: contraction
    {
      const int g = lane >> 2, kk = lane & 3, hi = lane >> 4, a = g & 3;
      // perm entries hold byte offsets: point slot * 16 | marker slot * 64 << 16
      const char* rec_b = reinterpret_cast<const char*>(S.rec);
      const char* mt_b = reinterpret_cast<const char*>(S.mtab + g);

      for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(&S.next_item, 1);
        item = __shfl_sync(kFull, item, 0);
        if (item >= S.n_items) break;
        item = S.item_order[item];
        const int lr = item >> 1, sg = item & 1;
        const int c_first = lr * kCW + sg * kSegW;
        // node (row lr + a, column sg*kSegW + n), channels 2kk, 2kk+1
        double* pbase = S.tile + ((lr + a) * kNW + sg * kSegW) * 8 + 2 * kk;
        int idle = 4;   // cells since the last one that had points: >= 4 means all slots are zero
        // radial basis a of the row's cell: cubic in t_s (clamped ends differ from the cardinal one)
        const int irow = row_base + lr;   // points exist only where 0 <= irow < ns
        const double* tb = P.scoef + ((size_t)irow * 4 + a) * 4;
        const double q0 = __ldg(tb), q1 = __ldg(tb + 1), q2 = __ldg(tb + 2), q3 = __ldg(tb + 3);
        double c0a = 0.0, c0b = 0.0, c1a = 0.0, c1b = 0.0;

        // One batch = 4 points (lane's point: kk).  Every lane evaluates its own operands: the
        // radial weight ws_a (3 FMA) and, from y = t or 1 - t, the two cardinal theta* pieces its
        // slots need in phase U: A = y^3/6 and B = 2/3 - y^2 + y^3/2 cover all four pieces
        // (w0(t) = A(1-t), w1(t) = B(t), w2(t) = B(1-t), w3(t) = A(t)).  No shuffles.
#define ORB_BATCH(U, POS)                                                            \
        {                                                                            \
          const unsigned int pe = S.perm[POS];                                       \
          const double2 t = *reinterpret_cast<const double2*>(rec_b + (pe & 0xffffu)); \
          const double b = *reinterpret_cast<const double*>(mt_b + (pe >> 16));      \
          const double ws = fma(fma(fma(q3, t.x, q2), t.x, q1), t.x, q0);            \
          const int p1 = (hi - (U)) & 3;                                             \
          const double y = (p1 & 1) ? t.y : 1.0 - t.y;                               \
          const double y2 = y * y;                                                   \
          const double y3 = y2 * y;                                                  \
          const double wA = y3 * (1.0 / 6.0);                                        \
          const double wB = fma(y3, 0.5, (2.0 / 3.0) - y2);                          \
          const bool fa = (p1 == 0) || (p1 == 3);                                    \
          dmma884(c0a, c0b, ws * (fa ? wA : wB), b);                                 \
          dmma884(c1a, c1b, ws * (fa ? wB : wA), b);                                 \
        }

#define ORB_RETIRE(U, NCOL)                                                          \
        if (idle < 4) {                                                              \
          double* dst = pbase + (NCOL) * 8;                                          \
          if ((U) < 2) {                                                             \
            if (hi == (U)) {                                                         \
              atomicAdd(dst, c0a);                                                   \
              atomicAdd(dst + 1, c0b);                                               \
              c0a = 0.0; c0b = 0.0;                                                  \
            }                                                                        \
          } else {                                                                   \
            if (hi == (U) - 2) {                                                     \
              atomicAdd(dst, c1a);                                                   \
              atomicAdd(dst + 1, c1b);                                               \
              c1a = 0.0; c1b = 0.0;                                                  \
            }                                                                        \
          }                                                                          \
          __syncwarp();   /* the CAS loops diverge; mma.sync.aligned needs the warp whole */ \
        }

        __syncwarp();   // mma.sync.aligned below needs the whole warp converged
#pragma unroll 1
        for (int cc = 0; cc < kSegW; cc += 4) {
          if (idle >= 4 && S.cstart[c_first + cc + 4] == S.cstart[c_first + cc]) {
            idle += 4;   // four empty cells and an empty window: nothing to add or retire
            continue;
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int cell = c_first + cc + u;
            const unsigned int end = S.cstart[cell + 1];
            unsigned int pos = S.cstart[cell] + kk;
            idle = (pos < end) ? 0 : idle + 1;
#pragma unroll 2
            for (; pos < end; pos += 4) ORB_BATCH(u, pos)
            ORB_RETIRE(u, cc + u)
          }
        }
        ++idle;
        ORB_RETIRE(0, kSegW)
        ++idle;
        ORB_RETIRE(1, kSegW + 1)
        ++idle;
        ORB_RETIRE(2, kSegW + 2)
#undef ORB_RETIRE
#undef ORB_BATCH
      }
    }
#ifdef ORB_PHASE_CLOCKS
    if (tid == 0) atomicAdd(d_points + 8, (unsigned long long)(clock64() - clk__));
#endif
    __syncthreads();
    ORB_CLK(4);   // phase 2

    // ------------------------------------------------------------------ next chunk?
    const bool more = S.n_deferred[cur ^ 1] > 0 || S.next_group < n_groups;
    __syncthreads();
    if (!more) break;
    cur ^= 1;
    ++chunk;
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

  // a9: flush the tile once.  8 consecutive lanes run along the channels of a node (4 phi planes
  // = one 32-byte sector of the k-fastest grid, per grid).
  {
    const int ch = tid & 7;
    double* __restrict__ out = (ch < 4 ? rho : jpar) + wrap_index(k - 1 + (ch & 3), P.nph);
    const int64_t row_stride = (int64_t)P.nth * P.nph;
    if (G == 2 || ch < 4) {
      for (int node = tid >> 3; node < kNH * kNW; node += kThreads / 8) {
        const double v = S.tile[node * 8 + ch];
        if (v == 0.0) continue;
        const int nr = node / kNW, tc = node - nr * kNW;
        const int gi = row_base + nr;           // zero outside [0, ns + 2]: no point maps there
        int gj = cellcol_base - 1 + tc;
        while (gj < 0) gj += P.nth;
        while (gj >= P.nth) gj -= P.nth;
        atomicAdd(out + gi * row_stride + (int64_t)gj * P.nph, v);
      }
    }
  }

  ORB_CLK(5);   // flush (thread 0's share)
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

template <int G, int PCAP>
int launch(const Params& P, const Markers& M, const uint32_t* cell_start, const TileBins& TB,
           double* rho, double* jpar,
           unsigned long long* d_points, cudaStream_t st) {
  const int tiles_i = (P.ns + kTileI - 1) / kTileI;
  const int tiles_j = (P.nth + kTileJ - 1) / kTileJ;
  const dim3 blocks((unsigned)tiles_j, (unsigned)tiles_i, (unsigned)P.nph);
  const size_t smem = sizeof(Smem<G, PCAP>);
  if (cudaFuncSetAttribute(k_deposit_tile<G, PCAP>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)smem) != cudaSuccess)
    return -1;
  k_deposit_tile<G, PCAP><<<blocks, kThreads, smem, st>>>(P, M, cell_start, TB, rho, jpar, d_points,
                                                         tiles_i, tiles_j);
  return 1;
}

}  // namespace

int launch_deposit_tile(const Params& P, const Markers& M, const uint32_t* cell_start,
                        const TileBins& TB, double* rho,
                        double* jpar, unsigned long long* d_points, cudaStream_t st) {
  if (M.n == 0) return 0;
  if (!P.adaptive && P.n_fixed <= 4)
    return jpar ? launch<2, kPCapSmall>(P, M, cell_start, TB, rho, jpar, d_points, st)
                : launch<1, kPCapSmall>(P, M, cell_start, TB, rho, jpar, d_points, st);
  return jpar ? launch<2, kPCapLarge>(P, M, cell_start, TB, rho, jpar, d_points, st)
              : launch<1, kPCapLarge>(P, M, cell_start, TB, rho, jpar, d_points, st);
}

}  // namespace orb
