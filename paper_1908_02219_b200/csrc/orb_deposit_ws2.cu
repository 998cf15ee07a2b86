// Tile deposition, v6 (hot-path steps a1-a6, a8, a9) for fixed N_L <= 4: the persistent
// warp-specialised pipeline of orb_deposit_ws.cu (v5) with 16-byte point records, chunks of most of
// a tile and a third pipeline stage.  The product path for fixed N_L <= 4.
//
// What round 2's knock-out experiments on v5 showed (profiles/r02_experiments.md): what costs is
// what is paid once per chunk and row segment -- the column retire into the shared tile, the cell
// visits, the producers' barriers and scan -- and v5's 64-byte operand records limit a chunk to 256
// markers and the ring to two stages.  Here a point's record is its 16-byte in-cell coordinate
// pair (t_s, t_theta), left where the producer wrote it; the on-chip sort by cell only writes a
// 4-byte permutation entry per point, and the consumer lane evaluates its own MMA operands from
// (t_s, t_theta): one radial cubic with lane-constant coefficients (tabulated pieces of the clamped
// basis) and the two cardinal theta* pieces of its accumulator slots, y^3/6 and 2/3 - y^2 + y^3/2 at
// y = t or 1 - t.  A stage of 384 markers (rho + j_par; 512 for rho only) is 58 KB, so three
// stages fit.  Measured (cfg3 / cfg1): 14.4 / 2.9 ms against 16.4 / 3.6 ms for v5 (15.1 ms before
// the consumers' operand evaluation was trimmed to 53 instructions per pair of batches).  The chunk
// capacity was swept: 256 -> 16.6 ms, 320 -> 17.0, 384 -> 15.4 (two stages; 15.1 with three),
// 448 -> 15.7, 576 (a cfg3 tile in ONE chunk) -> 17.7: two unequal chunks per tile pipeline better
// than one (the consumers' flush then falls on a short chunk) and better than two equal ones.
//
//   producer warps (8): per round one lane = one marker (up to 2 rounds per chunk): geometry,
//        marker table, its <= 4 points -> (t_s, t_theta) record + cell | rank (shared 32-bit atomic)
//        in a scratch word; [barrier] one warp scans the padded cell counts and lists the row
//        segments, heaviest first; [barrier] every point: permutation entry at its sorted slot
//        (cells padded to batches of 4 with a dummy point of a zero marker).
//   consumer warps (8): as in v5 (row segments of 12 cells, four fixed accumulator slots, finished
//        columns parked in registers, one pipelined CAS pass per segment, one flush per tile); the
//        permutation stream is read two batches ahead, records and marker channels one ahead.
#include "orb_geom.cuh"

namespace orb {

namespace {

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
constexpr int kPPL = 4;                    // Larmor points per marker slot
#ifndef ORB_V6_STAGES
#define ORB_V6_STAGES 3
#endif
constexpr int kStages = ORB_V6_STAGES;
constexpr unsigned kFull = 0xffffffffu;
constexpr unsigned kNone = 0xffffffffu;
static_assert(kCW % kSegW == 0 && kSegW % 4 == 0, "segments must tile the row in groups of 4");
static_assert(kCells < 512, "cell id must fit 9 bits");

#ifdef ORB_PHASE_CLOCKS
#define ORB_CLK_DECL long long clk__ = clock64()
#define ORB_CLK(cond, i)                                                    \
  do {                                                                      \
    if (cond) {                                                             \
      const long long now__ = clock64();                                    \
      atomicAdd(d_points + (i), (unsigned long long)(now__ - clk__));       \
      clk__ = now__;                                                        \
    }                                                                       \
  } while (0)
#else
#define ORB_CLK_DECL do { } while (0)
#define ORB_CLK(cond, i) do { } while (0)
#endif

// ---- synchronisation primitives (PTX)
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "ORB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra ORB_DONE;\n"
      "bra ORB_WAIT;\n"
      "ORB_DONE:\n"
      "}" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

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


template <int G>
struct Shape {
#ifndef ORB_V6_PW
#define ORB_V6_PW 8
#endif
  static constexpr int kProd = ORB_V6_PW * 32;
  static constexpr int kCons = 512 - kProd;
  static constexpr int kThreads = kProd + kCons;
#ifndef ORB_V6_MCAP
#define ORB_V6_MCAP 384
#endif
#ifndef ORB_V6_MCAP1
#define ORB_V6_MCAP1 512
#endif
  static constexpr int kMCap = G == 1 ? ORB_V6_MCAP1 : ORB_V6_MCAP;   // markers per chunk
  static constexpr int kRounds = (kMCap + kProd - 1) / kProd;
  static constexpr int kPts = kMCap * kPPL;            // Larmor points per chunk (2304)
  static constexpr int kPad = kMCap;                   // dummy entries that pad cells to batches of 4
  static constexpr int kSlots = kPts + kPad;
  static constexpr int kChan = 4 * G;                  // channels per node / marker
  // a permutation entry holds two BYTE offsets: of the point record (16 bytes each) in the low
  // half, of the marker's channel row (kChan doubles each) in the high half
  static constexpr unsigned kDummy = (unsigned)(kPts * 16) | ((unsigned)(kMCap * kChan * 8) << 16);
  static_assert(kSlots % 4 == 0 && kPts * 16 < 65536 && kMCap * kChan * 8 < 65536,
                "perm entries are 16 + 16 bits");
};

struct StageInfo {
  int n_items;          // row segments with points; < 0: no more work (producers are done)
  int last;             // this chunk is the last one of its tile: flush afterwards
  int k, row_base, cellcol_base;   // the tile
  int next_item;
  unsigned char item_order[kItems];
};

template <int G>
struct Smem {
  using Sh = Shape<G>;
  alignas(16) double tile[kNH * kNW * Sh::kChan];   // [node row][node col][grid*4 + phi plane]
  struct alignas(16) Stage {
    alignas(16) double2 rec[Sh::kPts + 1];          // (t_s, t_theta) of point slot q; [kPts]: dummy
    alignas(16) double mtab[(Sh::kMCap + 1) * Sh::kChan];   // per marker: c*wphi[0..3] (, x vpar); last = zeros
    unsigned int perm[Sh::kSlots + 16];             // sorted by cell: point slot | marker slot << 16
    unsigned int cs[kCells + 1];                    // first sorted slot of the cell | points << 16
    StageInfo info;
  } st[kStages];
  unsigned int meta[Sh::kPts];                      // producers: cell | rank << 9 of point slot q
  unsigned int count[kCells];                       // producers
  unsigned long long full[kStages], empty[kStages];
};

// Direct deposition of one Larmor point given its cell and in-cell coordinates, with global
// atomics (points outside the tile's halo, or beyond a chunk's padding capacity).
template <int G>
__device__ __noinline__ void deposit_point_cell(const Params& P, int ci, double t_s, int cj,
                                                double t_t, int k0, const double* chan,
                                                double* __restrict__ rho,
                                                double* __restrict__ jpar) {
  double ws[4], wt[4];
  radial_cell_weights(P, ci, t_s, ws);
  cardinal_weights(t_t, wt);
#pragma unroll
  for (int a = 0; a < 4; ++a) {
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const double v = ws[a] * (6.0 * wt[b]);   // chan carries 1/6 (see the producer)
      const int64_t row = ((int64_t)(ci + a) * P.nth + wrap_index(cj - 1 + b, P.nth)) * (int64_t)P.nph;
#pragma unroll
      for (int d = 0; d < 4; ++d) {
        const int kk = wrap_index(k0 + d, P.nph);
        atomicAdd(rho + row + kk, v * chan[d]);
        if (G == 2) atomicAdd(jpar + row + kk, v * chan[4 + d]);
      }
    }
  }
}


// ------------------------------------------------------------------------------------ producer
template <int G>
__device__ __forceinline__ void producer(Smem<G>& S, const Params& P, const Markers& M,
                                         const uint32_t* __restrict__ cell_start, const TileBins& TB,
                                         double* __restrict__ rho, double* __restrict__ jpar,
                                         unsigned long long* __restrict__ d_points, int tiles_i,
                                         int tiles_j) {
  using Sh = Shape<G>;
  constexpr int kChan = Sh::kChan;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int n_tiles = tiles_i * tiles_j * P.nph;
  unsigned int my_points = 0, my_fallback = 0;
  unsigned int it = 0;   // chunks emitted so far (stage = it % kStages)
  ORB_CLK_DECL;

  auto load_desc = [&](int t, uint32_t& b, uint32_t& n) {
    b = 0;
    n = 0;
    if (t < n_tiles && lane < kTileI) {
      const int tj = t % tiles_j, ti = (t / tiles_j) % tiles_i, k = t / (tiles_j * tiles_i);
      tile_run(P, cell_start, TB, tj, ti, k, lane, b, n);
    }
  };
  // marker v of the tile -> global marker index (lanes hold the descriptor runs)
  // (binary search for the last run whose offset is <= v: empty runs share their offset with the
  // next one; the result is only used for v below the tile's marker count)
  auto marker_index = [&](uint32_t v, uint32_t rb, uint32_t rn, uint32_t ro) -> int64_t {
    static_assert(kTileI == 8, "three search steps");
    int r = (v >= __shfl_sync(kFull, ro, 4)) ? 4 : 0;
    r += (v >= __shfl_sync(kFull, ro, r + 2)) ? 2 : 0;
    r += (v >= __shfl_sync(kFull, ro, r + 1)) ? 1 : 0;
    (void)rn;
    return (int64_t)__shfl_sync(kFull, rb, r) + (v - __shfl_sync(kFull, ro, r));
  };

  uint32_t nb_rb, nb_rn;       // next tile's descriptor (prefetched)
  int T = blockIdx.x;
  load_desc(T, nb_rb, nb_rn);

  for (; T < n_tiles; T += gridDim.x) {
    const uint32_t rb = nb_rb, rn = nb_rn;
    load_desc(T + gridDim.x, nb_rb, nb_rn);
    uint32_t ro = rn;          // exclusive prefix of the run lengths
#pragma unroll
    for (int o = 1; o < kTileI; o <<= 1) {
      const uint32_t t = __shfl_up_sync(kFull, ro, o);
      if (lane >= o) ro += t;
    }
    const uint32_t n_tile = __shfl_sync(kFull, ro, kTileI - 1);
    ro -= rn;
    if (n_tile == 0) continue;
    const int tj = T % tiles_j, ti = (T / tiles_j) % tiles_i, k = T / (tiles_j * tiles_i);
    const int row_base = ti * kTileI - kHaloS;        // radial cell (= first basis index) of cell row 0
    const int cellcol_base = tj * kTileJ - kHaloT;    // theta* cell of cell column 0 (may be < 0)
    const uint32_t n_chunks = (n_tile + Sh::kMCap - 1) / Sh::kMCap;
    // (uniform over the tile) only tiles that reach the two end cells of the clamped radial
    // basis need the tabulated pieces on the direct path
    for (uint32_t chunk = 0; chunk < n_chunks; ++chunk) {
      const int stage = (int)(it % kStages);
      typename Smem<G>::Stage& St = S.st[stage];
      mbar_wait(&S.empty[stage], ((it / kStages) & 1u) ^ 1u);
      ORB_CLK(tid == 0, 2);
      const bool last_chunk = chunk + 1 == n_chunks;
      const uint32_t v0 = chunk * Sh::kMCap;
      const uint32_t n_here = min((uint32_t)Sh::kMCap, n_tile - v0);

      // -------------------------------------------------- phases A + B, one marker per lane and round
      MarkerData m_next;
      {
        const int64_t p0 = marker_index(v0 + (uint32_t)tid, rb, rn, ro);
        m_next.s = m_next.th = m_next.ph = m_next.vpar = m_next.mu = m_next.w = 0.0;
        if ((uint32_t)tid < n_here) m_next = load_marker(M, p0);
      }
#pragma unroll 1
      for (int r = 0; r < Sh::kRounds; ++r) {
        const uint32_t u = (uint32_t)(r * Sh::kProd + tid);     // marker slot in the chunk
        if ((uint32_t)(r * Sh::kProd) >= n_here) break;         // (uniform)
        const bool have = u < n_here;
        const MarkerData m = m_next;
        if (r + 1 < Sh::kRounds && (uint32_t)((r + 1) * Sh::kProd) < n_here) {   // (uniform) prefetch
          const int64_t pn = marker_index(v0 + u + Sh::kProd, rb, rn, ro);
          if (u + Sh::kProd < n_here) m_next = load_marker(M, pn);
        }
        if (!have) continue;
        const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
        const int un = g.n;
        my_points += (unsigned)un;
        // (1/6: the consumers evaluate 6 x the theta* pieces)
        const double c = P.q * m.w * __drcp_rn((double)un) * (1.0 / 6.0);
        double wp[4];
        const int k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
        const bool k_ok = (k0 == k - 1);
        double* chan = St.mtab + (size_t)u * kChan;
        {
          double2* e = reinterpret_cast<double2*>(chan);
          e[0] = make_double2(c * wp[0], c * wp[1]);
          e[1] = make_double2(c * wp[2], c * wp[3]);
          if (G == 2) {
            const double cv = c * m.vpar;
            e[2] = make_double2(cv * wp[0], cv * wp[1]);
            e[3] = make_double2(cv * wp[2], cv * wp[3]);
          }
        }
        // the marker's <= 4 points, four independent chains
        double psl[kPPL], ptl[kPPL], pX[kPPL], pY[kPPL];
        bool slow = false;
        const int nring = max(un, 1);
        const double ga = un == 1 ? g.s : g.x0, gb = un == 1 ? g.ts : g.z0;
#pragma unroll
        for (int j = 0; j < kPPL; ++j) {
          const int l = (j < un) ? j : 0;
          bool ok;
          larmor_point_fast(P, ga, gb, g.rho, g.ts, g.cg, g.sg, ring_entry(P, nring, l), psl[j], ptl[j],
                            pX[j], pY[j], ok);
          slow |= !ok && (j < un);
          if (!ok) ptl[j] = 4.0 * kTwoPi;   // marks the point for the slow path
        }
        if (un == 1) {   // R8: the guiding centre itself, (s, theta*) as stored
          psl[0] = ga;
          ptl[0] = gb;
        } else if (slow) {   // rare: the ring comes near the axis, full-range atan2
#pragma unroll
          for (int j = 0; j < kPPL; ++j)
            if (ptl[j] > 3.0 * kTwoPi) ptl[j] = atan2(pY[j], pX[j]);
        }
#pragma unroll
        for (int j = 0; j < kPPL; ++j) {
          const unsigned int q = u * kPPL + (unsigned)j;
          unsigned int mt = kNone;
          if (j < un) {
            const double xs = psl[j] * (double)P.ns;
            const int ci = min((int)xs, P.ns - 1);
            const double t_s = xs - (double)ci;
            double t_t;
            const int cj = periodic_cell(ptl[j], P.nth_scale, P.nth, t_t);
            const int lr = ci - row_base;
            int lc = cj - cellcol_base;
            if (lc >= P.nth) lc -= P.nth;
            if (lc < 0) lc += P.nth;
            if (k_ok && lr >= 0 && lr < kCH && lc >= 0 && lc < kCW) {
              const unsigned int cell = (unsigned)(lr * kCW + lc);
              const unsigned int rank = atomicAdd(&S.count[cell], 1u);
              St.rec[q] = make_double2(t_s, t_t);
              mt = cell | (rank << 9);
            } else {   // footprint leaves the tile (long ring, or phi rounding): direct path
              ++my_fallback;
              deposit_point_cell<G>(P, ci, t_s, cj, t_t, k0, chan, rho, jpar);
            }
          }
          S.meta[q] = mt;
        }
      }
      ORB_CLK(tid == 0, 3);
      named_bar_sync(1, Sh::kProd);
      ORB_CLK(tid == 0, 4);

      // -------------------------------------------------- phase C: scan, work list (one warp)
      if (wid == 0) {
        constexpr int per = (kCells + 31) / 32;
        unsigned int loc[per], cnt[per];
        unsigned int sum = 0;
#pragma unroll
        for (int x = 0; x < per; ++x) {
          const int c = lane * per + x;
          cnt[x] = c < kCells ? S.count[c] : 0;
          if (c < kCells) S.count[c] = 0;
          loc[x] = (cnt[x] + 3u) & ~3u;
          sum += loc[x];
        }
        unsigned int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const unsigned int t = __shfl_up_sync(kFull, inc, o);
          if (lane >= o) inc += t;
        }
        // Cells that do not fit the stage's slots keep count 0 (their points take the direct
        // path) and, like every cell after them, start where the written slots end.
        unsigned int ex = inc - sum;
        unsigned int limit = (unsigned)Sh::kSlots;
        {
          unsigned int e2 = ex;
#pragma unroll
          for (int x = 0; x < per; ++x) {
            if (loc[x] > 0 && e2 + loc[x] > (unsigned)Sh::kSlots) limit = min(limit, e2);
            e2 += loc[x];
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) limit = min(limit, __shfl_xor_sync(kFull, limit, o));
        }
#pragma unroll
        for (int x = 0; x < per; ++x) {
          const int c = lane * per + x;
          const bool fits = ex + loc[x] <= limit;
          if (c < kCells) St.cs[c] = min(ex, limit) | ((fits ? cnt[x] : 0u) << 16);
          ex += loc[x];
        }
        if (lane == 31) St.cs[kCells] = min(inc, limit);
        __syncwarp();
        unsigned int wgt = 0;
        if (lane < kItems) {
          const int c0 = (lane >> 1) * kCW + (lane & 1) * kSegW;
          wgt = (St.cs[c0 + kSegW] & 0xffffu) - (St.cs[c0] & 0xffffu);
        }
        int rank = 0;
#pragma unroll
        for (int j = 0; j < kItems; ++j) {
          const unsigned int wj = __shfl_sync(kFull, wgt, j);
          rank += (wj > wgt || (wj == wgt && j < lane)) ? 1 : 0;
        }
        if (lane < kItems && wgt > 0) St.info.item_order[rank] = (unsigned char)lane;
        const unsigned int nz = __ballot_sync(kFull, lane < kItems && wgt > 0);
        if (lane == 0) {
          St.info.n_items = __popc(nz);
          St.info.last = last_chunk ? 1 : 0;
          St.info.k = k;
          St.info.row_base = row_base;
          St.info.cellcol_base = cellcol_base;
          St.info.next_item = 0;
        }
      }
      named_bar_sync(1, Sh::kProd);
      ORB_CLK(tid == 0, 5);

      // -------------------------------------------------- phase D: permutation entries, by cell
      {
        constexpr unsigned kDummy = Sh::kDummy;
        const unsigned int n_q = n_here * kPPL;
        for (unsigned int q = (unsigned)tid; q < n_q; q += Sh::kProd) {
          const unsigned int mt = S.meta[q];
          if (mt == kNone) continue;
          const unsigned int cell = mt & 0x1ffu, rank = mt >> 9;
          const unsigned int pk = St.cs[cell];
          const unsigned int cnt = pk >> 16;
          const unsigned int u = q / kPPL;
          if (cnt == 0) {   // the chunk's padding capacity is exhausted: direct path
            const int lr = (int)cell / kCW, lc = (int)cell - lr * kCW;
            const double2 t = St.rec[q];
            ++my_fallback;
            deposit_point_cell<G>(P, row_base + lr, t.x, wrap_index(cellcol_base + lc, P.nth), t.y, k - 1,
                                  St.mtab + (size_t)u * kChan, rho, jpar);
            continue;
          }
          unsigned int p = (pk & 0xffffu) + rank;
          St.perm[p] = (q << 4) | ((u * (unsigned)(kChan * 8)) << 16);
          if (rank + 1 == cnt)   // the cell's last point pads the cell to a batch of 4
            for (++p; (p & 3u) != 0; ++p) St.perm[p] = kDummy;
        }
      }
      mbar_arrive(&S.full[stage]);
      ORB_CLK(tid == 0, 6);
      ++it;
    }
  }

  // no more work: tell the consumers
  {
    const int stage = (int)(it % kStages);
    mbar_wait(&S.empty[stage], ((it / kStages) & 1u) ^ 1u);
    if (tid == 0) S.st[stage].info.n_items = -1;
    mbar_arrive(&S.full[stage]);
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

// ------------------------------------------------------------------------------------ consumer
template <int G>
__device__ __forceinline__ void consumer(Smem<G>& S, const Params& P, double* __restrict__ rho,
                                         double* __restrict__ jpar,
                                         unsigned long long* __restrict__ d_points) {
  using Sh = Shape<G>;
  constexpr int kChan = Sh::kChan;
  const int ctid = threadIdx.x - Sh::kProd;        // 0 .. kCons-1
  const int lane = ctid & 31;
  const int g = lane >> 2, kk = lane & 3, hi = lane >> 4, a = g & 3;
  unsigned int it = 0;
  ORB_CLK_DECL;

  for (;; ++it) {
    const int stage = (int)(it % kStages);
    typename Smem<G>::Stage& St = S.st[stage];
    mbar_wait(&S.full[stage], (it / kStages) & 1u);
    ORB_CLK(ctid == 0, 8);
    const int n_items = St.info.n_items;
    if (n_items < 0) break;
    const int last = St.info.last, tk = St.info.k, row_base = St.info.row_base,
              cellcol_base = St.info.cellcol_base;
    // this lane's channel of a marker, and the point records, as byte pointers (see Shape::kDummy)
    const char* mt_b = reinterpret_cast<const char*>(St.mtab + (G == 2 ? g : (g & 3)));
    const char* rec_b = reinterpret_cast<const char*>(St.rec);
    const unsigned int* perm_l = St.perm + kk;               // this lane's point of a batch

    for (;;) {
      int item = 0;
      if (lane == 0) item = atomicAdd(&St.info.next_item, 1);
      item = __shfl_sync(kFull, item, 0);
      if (item >= n_items) break;
      item = St.info.item_order[item];
      const int lr = item >> 1, sg = item & 1;
      const int c_first = lr * kCW + sg * kSegW;
      // node (row lr + a, column sg*kSegW + n), channels 2kk, 2kk+1
      double* pbase = S.tile + ((lr + a) * kNW + sg * kSegW) * kChan + 2 * kk;
      double c0a = 0.0, c0b = 0.0, c1a = 0.0, c1b = 0.0;
      // radial piece a on this cell row: lane-constant cubic (tabulated pieces of the clamped basis;
      // the cardinal pieces away from the two end cells).  The row holds points, so it is a grid row.
      const double* tb = P.scoef + ((size_t)(row_base + lr) * 4 + a) * 4;
      const double r0 = __ldg(tb), r1 = __ldg(tb + 1), r2 = __ldg(tb + 2), r3 = __ldg(tb + 3);

      // The batches of a row segment are contiguous in the sorted order: one linear stream of
      // permutation entries, read two batches ahead; the point records and marker channels they
      // name one batch ahead, in two alternating register sets.  The stream is read up to three
      // batches beyond the segment's end: every entry of perm is valid at all times (the array is
      // initialised with the dummy entry and only ever holds valid entries).
      unsigned int pk = St.cs[c_first];
      const unsigned int* pp = perm_l + (pk & 0xffffu);
      double2 At, Bt;
      double Ab = 0.0, Bb = 0.0;
      unsigned int pe;
#define ORB_LD(S, e)                                                                  \
      S##t = *reinterpret_cast<const double2*>(rec_b + ((e) & 0xffffu));              \
      if (G == 2 || g < 4) S##b = *reinterpret_cast<const double*>(mt_b + ((e) >> 16));
      // y = t or 1 - t; the two pieces of this lane's slots are y^3/6 and 2/3 - y^2 + y^3/2, here
      // times 6 (y^3 and 4 - 6 y^2 + 3 y^3: the coefficients are instruction immediates); the
      // producer folds the 1/6 into the marker's channel values
#define ORB_MMA(S)                                                                    \
      {                                                                               \
        const double ws = fma(fma(fma(r3, S##t.x, r2), S##t.x, r1), S##t.x, r0);      \
        const double ym = S##t.y - yoff;            /* y = |ym| */                    \
        const double y2 = ym * ym;                                                    \
        const double outer = y2 * fabs(ym);                                           \
        const double mid = fma(3.0 * y2, fabs(ym) - 2.0, 4.0);                        \
        const double a0 = ws * (outer_first ? outer : mid);                           \
        const double a1 = ws * (outer_first ? mid : outer);                           \
        dmma884(c0a, c0b, a0, S##b);                                                  \
        dmma884(c1a, c1b, a1, S##b);                                                  \
      }
      pe = pp[0];
      ORB_LD(A, pe)
      pe = pp[4];

      // Column retire, deferred: stepping past cell U of a group of four finishes one node column
      // of the window.  Its two accumulators are parked in registers (t0: the column this lane's
      // first slot held, t1: the second) and all parked columns are added into the shared tile
      // in one pipelined pass after the walk.
#define ORB_PARK(U)                                                                   \
      if ((U) < 2) {                                                                  \
        if (hi == (U)) { t0a = c0a; t0b = c0b; c0a = 0.0; c0b = 0.0; }                \
      } else {                                                                        \
        if (hi == (U) - 2) { t1a = c1a; t1b = c1b; c1a = 0.0; c1b = 0.0; }            \
      }

      // node column (cell - 1 + b) lives in slot (U + b) & 3: this lane's slots hi and hi + 2 carry
      // the pieces b0 = (hi - U) & 3 and b0 ^ 2; pieces 1, 3 are evaluated at y = t, pieces 0, 2 at
      // y = 1 - t; pieces 0 and 3 are y^3/6, pieces 1 and 2 are 2/3 - y^2 + y^3/2
#define ORB_CELL(U)                                                                   \
      {                                                                               \
        int nb = (int)(((pk >> 16) + 3u) >> 2);                                       \
        pk = St.cs[c_first + cc + (U) + 1];                                           \
        const int b0 = (hi - (U)) & 3;                                                \
        const double yoff = ((U) & 1) ? yoff_odd : yoff_even;                         \
        const bool outer_first = b0 == 0 || b0 == 3;                                  \
        _Pragma("unroll 1") for (; nb >= 2; nb -= 2) {                                \
          ORB_LD(B, pe)                                                               \
          pe = pp[8];                                                                 \
          ORB_MMA(A)                                                                  \
          ORB_LD(A, pe)                                                               \
          pe = pp[12];                                                                \
          ORB_MMA(B)                                                                  \
          pp += 8;                                                                    \
        }                                                                             \
        if (nb) {                                                                     \
          ORB_LD(B, pe)                                                               \
          pe = pp[8];                                                                 \
          ORB_MMA(A)                                                                  \
          At = Bt; Ab = Bb;                                                           \
          pp += 4;                                                                    \
        }                                                                             \
        ORB_PARK(U)                                                                   \
      }

      // y = |t - yoff|: t for the odd pieces, 1 - t for the even ones (b0 = (hi - U) & 3)
      const double yoff_even = hi ? 0.0 : 1.0, yoff_odd = 1.0 - yoff_even;
      // parked columns: pair i holds node columns 4i + hi (first slot) and 4i + hi + 2 (second)
      double q0a[4], q0b[4], q1a[4], q1b[4];
      double t0a = 0.0, t0b = 0.0, t1a = 0.0, t1b = 0.0;
      __syncwarp();   // mma.sync.aligned below needs the whole warp converged
#pragma unroll 1
      for (int cc = 0; cc < kSegW; cc += 4) {
        ORB_CELL(0)
        ORB_CELL(1)
        ORB_CELL(2)
        ORB_CELL(3)
#pragma unroll
        for (int i = 0; i < 3; ++i)
          if (cc == 4 * i) {
            q0a[i] = t0a; q0b[i] = t0b; q1a[i] = t1a; q1b[i] = t1b;
          }
      }
      // the three columns beyond the last cell: 12 + hi (first slot), 14 (second slot, hi = 0)
      q0a[3] = c0a; q0b[3] = c0b;
      q1a[3] = hi == 0 ? c1a : 0.0;
      q1b[3] = hi == 0 ? c1b : 0.0;

      if (G == 2 || kk < 2) {
        unsigned long long* col0 = reinterpret_cast<unsigned long long*>(pbase + hi * kChan);
#pragma unroll
        for (int s2 = 0; s2 < 2; ++s2) {
          // four columns per pass: loads, adds and CAS of the pass are independent
          unsigned long long* ad[4];
          unsigned long long oa[4], ob[4], na[4], nb2[4];
          double va[4], vb[4];
          bool live[4];
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            ad[i] = col0 + (4 * i + 2 * s2) * kChan;
            va[i] = s2 ? q1a[i] : q0a[i];
            vb[i] = s2 ? q1b[i] : q0b[i];
            live[i] = va[i] != 0.0 || vb[i] != 0.0;
          }
#pragma unroll
          for (int i = 0; i < 4; ++i)
            if (live[i]) {
              const ulonglong2 o = *reinterpret_cast<const ulonglong2*>(ad[i]);
              oa[i] = o.x;
              ob[i] = o.y;
            }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            na[i] = (unsigned long long)__double_as_longlong(__longlong_as_double((long long)oa[i]) + va[i]);
            nb2[i] = (unsigned long long)__double_as_longlong(__longlong_as_double((long long)ob[i]) + vb[i]);
          }
          unsigned long long ga[4], gb2[4];
#pragma unroll
          for (int i = 0; i < 4; ++i)
            if (live[i]) {
              ga[i] = atomicCAS(ad[i], oa[i], na[i]);
              gb2[i] = atomicCAS(ad[i] + 1, ob[i], nb2[i]);
            }
#pragma unroll
          for (int i = 0; i < 4; ++i)
            if (live[i]) {   // rare: another warp updated the node in between
              if (ga[i] != oa[i]) atomicAdd(reinterpret_cast<double*>(ad[i]), va[i]);
              if (gb2[i] != ob[i]) atomicAdd(reinterpret_cast<double*>(ad[i] + 1), vb[i]);
            }
        }
      }
      __syncwarp();
#undef ORB_PARK
#undef ORB_CELL
#undef ORB_MMA
#undef ORB_LD
    }
    __syncwarp();
    mbar_arrive(&S.empty[stage]);
    ORB_CLK(ctid == 0, 9);

    if (last) {
      // a9: all consumers are done with the tile -> flush it once and clear it.  kChan / 2
      // consecutive lanes run along the channels of a node (4 phi planes = one 32-byte sector per
      // grid); one thread = two channels (two consecutive phi planes): 128-bit shared loads and
      // clears, the node's index arithmetic once per pair.
      named_bar_sync(2, Sh::kCons);
      constexpr int kPairs = kChan / 2;
      const int ch = 2 * (ctid % kPairs);
      double* __restrict__ out = (G == 2 && ch >= 4) ? jpar : rho;
      const int ka = wrap_index(tk - 1 + (ch & 3), P.nph), kb = wrap_index(tk + (ch & 3), P.nph);
      const int64_t row_stride = (int64_t)P.nth * P.nph;
      for (int node = ctid / kPairs; node < kNH * kNW; node += Sh::kCons / kPairs) {
        double2* cell = reinterpret_cast<double2*>(S.tile + node * kChan + ch);
        const double2 v = *cell;
        if (v.x == 0.0 && v.y == 0.0) continue;
        *cell = make_double2(0.0, 0.0);
        const int nr = node / kNW, tc = node - nr * kNW;
        const int gi = row_base + nr;           // zero outside [0, ns + 2]: no point maps there
        int gj = cellcol_base - 1 + tc;
        while (gj < 0) gj += P.nth;
        while (gj >= P.nth) gj -= P.nth;
        double* dst = out + gi * row_stride + (int64_t)gj * P.nph;
        if (v.x != 0.0) atomicAdd(dst + ka, v.x);
        if (v.y != 0.0) atomicAdd(dst + kb, v.y);
      }
      named_bar_sync(2, Sh::kCons);
      ORB_CLK(ctid == 0, 10);
    }
  }
}


template <int G>
__global__ void __launch_bounds__(Shape<G>::kThreads, 1)
k_deposit_ws2(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
              const TileBins TB, double* __restrict__ rho, double* __restrict__ jpar,
              unsigned long long* __restrict__ d_points, int tiles_i, int tiles_j) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<G>& S = *reinterpret_cast<Smem<G>*>(smem_raw);
  using Sh = Shape<G>;
  const int tid = threadIdx.x;
#ifdef ORB_POISON_SMEM
  for (size_t x = tid; x < sizeof(S) / 4; x += Sh::kThreads) reinterpret_cast<unsigned int*>(smem_raw)[x] = 0xffffffffu;
  __syncthreads();
#endif
  for (int x = tid; x < kNH * kNW * Sh::kChan; x += Sh::kThreads) S.tile[x] = 0.0;
  for (int x = tid; x < kCells; x += Sh::kThreads) S.count[x] = 0;
  for (int s = 0; s < kStages; ++s) {
    constexpr unsigned kDummy = Sh::kDummy;
    for (int x = tid; x < Sh::kSlots + 16; x += Sh::kThreads) S.st[s].perm[x] = kDummy;
    if (tid < Sh::kChan) S.st[s].mtab[Sh::kMCap * Sh::kChan + tid] = 0.0;   // the zero marker
    if (tid == 0) S.st[s].rec[Sh::kPts] = make_double2(0.0, 0.0);           // the dummy point
  }
  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) {
      mbar_init(&S.full[s], Sh::kProd);
      mbar_init(&S.empty[s], Sh::kCons);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid < Sh::kProd) {
    producer<G>(S, P, M, cell_start, TB, rho, jpar, d_points, tiles_i, tiles_j);
  } else {
    consumer<G>(S, P, rho, jpar, d_points);
  }
}

template <int G>
int launch(const Params& P, const Markers& M, const uint32_t* cell_start, const TileBins& TB,
           double* rho, double* jpar, unsigned long long* d_points, int sms, cudaStream_t st) {
  const int tiles_i = (P.ns + kTileI - 1) / kTileI;
  const int tiles_j = (P.nth + kTileJ - 1) / kTileJ;
  const int64_t n_tiles = (int64_t)tiles_i * tiles_j * P.nph;
  const int blocks = (int)(n_tiles < sms ? n_tiles : sms);
  const size_t smem = sizeof(Smem<G>);
  static_assert(sizeof(Smem<G>) <= 232448, "shared memory of one block must fit one SM");
  if (cudaFuncSetAttribute(k_deposit_ws2<G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) !=
      cudaSuccess)
    return -1;
  k_deposit_ws2<G><<<blocks, Shape<G>::kThreads, smem, st>>>(P, M, cell_start, TB, rho, jpar, d_points,
                                                            tiles_i, tiles_j);
  return 1;
}

}  // namespace

// fixed N_L <= 4 only
int launch_deposit_ws2(const Params& P, const Markers& M, const uint32_t* cell_start,
                       const TileBins& TB, double* rho, double* jpar, unsigned long long* d_points,
                       int sms, cudaStream_t st) {
  if (M.n == 0) return 0;
  return jpar ? launch<2>(P, M, cell_start, TB, rho, jpar, d_points, sms, st)
              : launch<1>(P, M, cell_start, TB, rho, jpar, d_points, sms, st);
}

}  // namespace orb
