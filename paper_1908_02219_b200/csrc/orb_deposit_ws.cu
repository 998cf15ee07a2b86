// Tile deposition, v5 (hot-path steps a1-a6, a8, a9): ONE persistent thread block per SM,
// warp-specialised.  Producer warps turn markers into sorted, ready-to-use MMA operands; consumer
// warps do nothing but operand loads, fp64 MMAs and column retires; the two sides hand chunks
// over through a two-stage ring in shared memory guarded by mbarriers, so the geometry of chunk
// i+1 overlaps the contraction of chunk i inside the SM (the fp64 pipe is the shared roof).
//
// Why (profiles/r01_final_deposit_ncu.md): v4 ran every phase on every warp
// with six block-wide barriers per chunk; it issued 34.7 warp instructions per Larmor point, 19 of
// them in the contraction, because each MMA lane re-evaluated its spline operands from (t_s,
// t_theta) -- work that costs one instruction per 4 points there and one per 32 points in a
// point-parallel phase.  Here the point-parallel producer evaluates the 4 + 4 weights of a point
// once and stores them at the point's sorted position; a consumer batch is 5 shared loads, 2 DMUL
// and 2 DMMA.
//
// Work decomposition (same tiles as v4: 1 toroidal slab x 8 radial x 16 poloidal cells, halo 2 / 4
// cells; the markers of a tile are found through the binning pass's per-cell offsets):
//
//   producer warps (PW x 32 lanes; one lane = one "unit" = up to 4 Larmor points of one marker)
//     A  marker -> guiding-centre geometry, N_L, c = q w / N_L, the marker's channel values
//        c wphi[0..3] (and x v_par) into the stage's marker table.  Fixed N_L <= 4: the lane keeps
//        its marker (no hand-over).  Otherwise the markers' units are laid out by a warp prefix sum
//        and handed over through shared memory, so that N_L = 4..32 keeps every lane busy.
//     B  the unit's points, 4 independent chains per lane: ring point -> (s_l, theta*_l) -> cell and
//        in-cell coordinates, kept in registers; a shared 32-bit atomic on the cell's counter gives
//        the point's rank in its cell.  Points whose cell leaves the tile's halo go straight to
//        global atomics (rare; counted).
//     C  (one warp) exclusive scan of the per-cell counts, each padded to a multiple of 4; the
//        list of row segments that hold points, heaviest first.
//     D  each point: 4 radial + 4 poloidal spline weights, written at the point's sorted slot as one
//        64-byte operand record (cells are padded with zero-weight records).  This is the paper's
//        "sorting Larmor points by cell" done on chip.
//   consumer warps (CW x 32 lanes) take row segments of 12 cells and walk them along theta*.  All
//        points of a cell hit the same 4 x 4 nodes x 4 phi planes x {rho, jpar}:
//            C[node(a,b)][channel] = sum_pts  ws_a(pt) wt_b(pt) * chan(marker(pt))
//        as two DMMA m8n8k4 per 4 points with register accumulators; the four node columns of the
//        window live in four fixed slots, and stepping to the next cell retires the finished column
//        into the shared tile (fp64 CAS add).  After the tile's last chunk the consumers flush the
//        tile ONCE with fp64 RED.ADD to global memory and clear it, while the producers are already
//        two chunks into the next tile.
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
constexpr int kPPL = 4;                    // Larmor points per producer lane and chunk (one unit)
constexpr int kStages = 2;
constexpr unsigned kFull = 0xffffffffu;
static_assert(kCW % kSegW == 0 && kSegW % 4 == 0, "segments must tile the row in groups of 4");
static_assert(kCells < 512, "cell id must fit 9 bits");

// Optional per-phase SM-clock sums (build with -DORB_PHASE_CLOCKS; read with orb_debug_counters):
// producers (thread 0):   [2] wait empty  [3] A + B  [4] wait B->C  [5] C + wait  [6] D
// consumers (first lane): [8] wait full   [9] items  [10] flush incl. its two barriers
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

struct MarkerTmp {      // phase A -> B hand-over (general mode), 64 bytes
  double a, b;          // (x0, z0), or (s, theta*) when N_L = 1
  double rho;
  double ts, cg, sg;    // wrapped theta* of the guiding centre, its cosine and sine
  int n;                // N_L; bit 8 set if the marker's phi cell is not this tile's slab
  int k0;               // first phi node (phi cell - 1)
  double pad_;
};

template <int G, int PW, int CW>
struct Shape {
  static constexpr int kProd = PW * 32;
  static constexpr int kCons = CW * 32;
  static constexpr int kThreads = kProd + kCons;
  static constexpr int kUnits = kProd;                 // units per chunk
  static constexpr int kPts = kUnits * kPPL;           // Larmor points per chunk
  static constexpr int kPad = (G == 2) ? 224 : 448;    // zero-weight padding slots per chunk
  static constexpr int kSlots = kPts + kPad;
  static constexpr int kMCap = kUnits;                 // marker slots per chunk
  static constexpr int kChan = 4 * G;                  // channels per node / marker
  static_assert(kSlots % 4 == 0 && kSlots < 65536, "slots");
  static_assert(kMCap * kChan * 8 < 65536, "marker byte offsets are 16-bit");
};

struct StageInfo {
  int n_items;          // row segments with points; < 0: no more work (producers are done)
  int last;             // this chunk is the last one of its tile: flush afterwards
  int k, row_base, cellcol_base;   // the tile
  int next_item;
  unsigned char item_order[kItems];
};

template <int G, int PW, int CW>
struct Smem {
  using Sh = Shape<G, PW, CW>;
  alignas(16) double tile[kNH * kNW * Sh::kChan];   // [node row][node col][grid*4 + phi plane]
  struct alignas(16) Stage {
    // operand records, one batch of 4 slots = 256 bytes: ws[slot][a] (128 B), wt[slot][b] (128 B).
    // While the stage is being built (general mode, phases A-B) its first bytes hold the
    // marker hand-over table and the unit list.
    alignas(16) double ops[Sh::kSlots * 8];
    alignas(16) double mtab[(Sh::kMCap + 1) * Sh::kChan];   // per marker: c*wphi[0..3] (, x vpar); last = zeros
    unsigned short midx[Sh::kSlots];            // byte offset of the slot's marker in mtab
    unsigned int cs[kCells + 1];                // first slot of the cell | points in the cell << 16
    StageInfo info;
  } st[kStages];
  unsigned int count[kCells];                   // producers only
  unsigned long long full[kStages], empty[kStages];
  // general-mode chunk assembly (producers only)
  int deferred[2][PW];
  int n_deferred[2];
  int take_deferred, next_group, nmark, nunits, units_end, full_flag;
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
      const double v = ws[a] * wt[b];
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
template <int G, int PW, int CW, bool SELF>
__device__ __forceinline__ void producer(Smem<G, PW, CW>& S, const Params& P, const Markers& M,
                                         const uint32_t* __restrict__ cell_start, const TileBins& TB,
                                         double* __restrict__ rho, double* __restrict__ jpar,
                                         unsigned long long* __restrict__ d_points, int tiles_i,
                                         int tiles_j) {
  using Sh = Shape<G, PW, CW>;
  constexpr int kChan = Sh::kChan;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int n_tiles = tiles_i * tiles_j * P.nph;
  unsigned int my_points = 0, my_fallback = 0;
  unsigned int it = 0;   // chunks emitted so far (stage = it % kStages)
  ORB_CLK_DECL;

  // tile descriptor, lanes 0..7: first marker and marker count of the tile's radial rows
  auto load_desc = [&](int t, uint32_t& b, uint32_t& n) {
    b = 0;
    n = 0;
    if (t < n_tiles && lane < kTileI) {
      const int tj = t % tiles_j, ti = (t / tiles_j) % tiles_i, k = t / (tiles_j * tiles_i);
      tile_run(P, cell_start, TB, tj, ti, k, lane, b, n);
    }
  };
  // marker v of the tile -> global marker index (lanes hold the descriptor rows)
  // (binary search for the last run whose offset is <= v: empty runs share their offset with the
  // next one, so the run found is the one that holds v; -1 beyond the tile's last marker)
  auto marker_index = [&](uint32_t v, uint32_t rb, uint32_t rn, uint32_t ro) -> int64_t {
    static_assert(kTileI == 8, "three search steps");
    int r = (v >= __shfl_sync(kFull, ro, 4)) ? 4 : 0;
    r += (v >= __shfl_sync(kFull, ro, r + 2)) ? 2 : 0;
    r += (v >= __shfl_sync(kFull, ro, r + 1)) ? 1 : 0;
    const uint32_t o = __shfl_sync(kFull, ro, r), n = __shfl_sync(kFull, rn, r);
    const int64_t p = (int64_t)__shfl_sync(kFull, rb, r) + (v - o);
    return (v - o < n) ? p : -1;
  };

  uint32_t nb_rb, nb_rn;       // next tile's descriptor (prefetched)
  int T = blockIdx.x;
  load_desc(T, nb_rb, nb_rn);
  MarkerData pm;               // prefetched marker of the next chunk (SELF mode)
  bool pm_valid = false;
  pm.s = pm.th = pm.ph = pm.vpar = pm.mu = pm.w = 0.0;

  for (; T < n_tiles; T += gridDim.x) {
    // ---- this tile's descriptor; prefetch the next one
    const uint32_t rb = nb_rb, rn = nb_rn;
    load_desc(T + gridDim.x, nb_rb, nb_rn);
    uint32_t ro = rn;          // exclusive prefix of the row counts
#pragma unroll
    for (int o = 1; o < kTileI; o <<= 1) {
      const uint32_t t = __shfl_up_sync(kFull, ro, o);
      if (lane >= o) ro += t;
    }
    const uint32_t n_tile = __shfl_sync(kFull, ro, kTileI - 1);
    ro -= rn;
    if (n_tile == 0) {
      pm_valid = false;
      continue;
    }
    const int tj = T % tiles_j, ti = (T / tiles_j) % tiles_i, k = T / (tiles_j * tiles_i);
    const int row_base = ti * kTileI - kHaloS;        // radial cell (= first basis index) of cell row 0
    const int cellcol_base = tj * kTileJ - kHaloT;    // theta* cell of cell column 0 (may be < 0)

    const int n_groups = (int)((n_tile + 31) / 32);
    int cur = 0;
    if (!SELF) {
      if (tid == 0) {
        S.n_deferred[0] = S.n_deferred[1] = 0;
        S.take_deferred = 0;
        S.next_group = 0;
        S.nmark = 0;
        S.nunits = 0;
        S.units_end = 0x7fffffff;
        S.full_flag = 0;
      }
      named_bar_sync(1, Sh::kProd);
    }
    const uint32_t n_chunks_self = (n_tile + Sh::kUnits - 1) / Sh::kUnits;

    for (uint32_t chunk = 0;; ++chunk) {
      const int stage = (int)(it % kStages);
      typename Smem<G, PW, CW>::Stage& St = S.st[stage];
      mbar_wait(&S.empty[stage], ((it / kStages) & 1u) ^ 1u);
      ORB_CLK(tid == 0, 2);

      // unit state: up to kPPL points of one marker, first ring index l0
      double ga = 0.0, gb = 0.0, grho = 0.0;   // (x0, z0, rho_L), or (s, theta*, -) when N_L = 1
      double gts = 0.0, gcg = 1.0, gsg = 0.0;  // theta* of the guiding centre, cos, sin
      int un = 0, l0 = 0, k0 = 0, k_ok = 0;
      unsigned int mslot = 0;
      bool last_chunk;

      if (SELF) {
        // ------------------------------------------------ phase A, one lane = one marker = one unit
        const uint32_t v = chunk * Sh::kUnits + (uint32_t)tid;
        const bool have = v < n_tile;
        last_chunk = chunk + 1 == n_chunks_self;
        MarkerData m = pm;
        if (!pm_valid) {   // (uniform over the block) no prefetch reached this chunk
          const int64_t p0 = marker_index(v, rb, rn, ro);
          if (have) m = load_marker(M, p0);
        }
        // prefetch the marker of this lane's next unit: next chunk of this tile, or first chunk
        // of the next tile (its descriptor was requested one tile ago)
        {
          int64_t np = -1;
          if (!last_chunk) {
            np = marker_index(v + Sh::kUnits, rb, rn, ro);
          } else {
            uint32_t xo = nb_rn;
#pragma unroll
            for (int o = 1; o < kTileI; o <<= 1) {
              const uint32_t t = __shfl_up_sync(kFull, xo, o);
              if (lane >= o) xo += t;
            }
            xo -= nb_rn;
            np = marker_index((uint32_t)tid, nb_rb, nb_rn, xo);
          }
          pm_valid = true;   // (np < 0: the lane has no marker there; pm is not used then)
          if (np >= 0) pm = load_marker(M, np);
        }
        mslot = (unsigned)tid;
        if (have) {
          const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
          un = g.n;
          const double c = P.q * m.w * __drcp_rn((double)un);
          double wp[4];
          k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
          k_ok = (k0 == k - 1);
          double2* e = reinterpret_cast<double2*>(St.mtab + (size_t)mslot * kChan);
          e[0] = make_double2(c * wp[0], c * wp[1]);
          e[1] = make_double2(c * wp[2], c * wp[3]);
          if (G == 2) {
            const double cv = c * m.vpar;
            e[2] = make_double2(cv * wp[0], cv * wp[1]);
            e[3] = make_double2(cv * wp[2], cv * wp[3]);
          }
          if (un == 1) {   // R8: the guiding centre itself
            ga = g.s;
            gb = g.ts;
          } else {
            ga = g.x0;
            gb = g.z0;
          }
          grho = g.rho;
          gts = g.ts;
          gcg = g.cg;
          gsg = g.sg;
          my_points += (unsigned)un;
        }
      } else {
        // ------------------------------------------------ phase A, general: markers -> unit list
        MarkerTmp* mtmp = reinterpret_cast<MarkerTmp*>(St.ops);
        unsigned int* unit_tab = reinterpret_cast<unsigned int*>(mtmp + Sh::kMCap);
        for (;;) {
          int grp = -1;
          if (lane == 0) {
            const int di = atomicAdd(&S.take_deferred, 1);
            if (di < S.n_deferred[cur]) {
              grp = S.deferred[cur][di];
            } else if (!*(volatile int*)&S.full_flag) {
              const int gi = atomicAdd(&S.next_group, 1);
              if (gi < n_groups) grp = gi;
            }
          }
          grp = __shfl_sync(kFull, grp, 0);
          if (grp < 0) break;
          const uint32_t v = (uint32_t)grp * 32u + (uint32_t)lane;
          const bool have = v < n_tile;
          const int64_t p = marker_index(v, rb, rn, ro);
          int n = 0, mk0 = 0;
          double a0 = 0.0, b0 = 0.0, r0 = 0.0, cw[4] = {0.0, 0.0, 0.0, 0.0}, vpar = 0.0;
          double mts = 0.0, mcg = 1.0, msg = 0.0;
          if (have) {
            const MarkerData m = load_marker(M, p);
            const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
            n = g.n;
            const double c = P.q * m.w * __drcp_rn((double)n);
            double wp[4];
            mk0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
#pragma unroll
            for (int d = 0; d < 4; ++d) cw[d] = c * wp[d];
            vpar = m.vpar;
            if (n == 1) {
              a0 = g.s;
              b0 = g.ts;
            } else {
              a0 = g.x0;
              b0 = g.z0;
            }
            r0 = g.rho;
            mts = g.ts;
            mcg = g.cg;
            msg = g.sg;
          }
          const int u = (n + kPPL - 1) / kPPL;
          int incl = u;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFull, incl, o);
            if (lane >= o) incl += t;
          }
          const int total = __shfl_sync(kFull, incl, 31);
          unsigned int mb = 0, ub = 0;
          int ok = 1;
          if (lane == 0) {
            mb = atomicAdd((unsigned int*)&S.nmark, 32u);
            if (mb + 32u > (unsigned)Sh::kMCap) {
              ok = 0;
            } else {
              ub = atomicAdd((unsigned int*)&S.nunits, (unsigned)total);
              if (ub + (unsigned)total > (unsigned)Sh::kUnits) {
                ok = 0;
                atomicMin(&S.units_end, (int)ub);
              }
            }
            if (!ok) {
              S.full_flag = 1;
              const int slot = atomicAdd(&S.n_deferred[cur ^ 1], 1);
              S.deferred[cur ^ 1][slot] = grp;
            }
          }
          ok = __shfl_sync(kFull, ok, 0);
          if (!ok) break;
          mb = __shfl_sync(kFull, mb, 0);
          ub = __shfl_sync(kFull, ub, 0);
          my_points += (unsigned)n;
          const unsigned int ms = mb + (unsigned)lane;
          double2* e = reinterpret_cast<double2*>(St.mtab + (size_t)ms * kChan);
          e[0] = make_double2(cw[0], cw[1]);
          e[1] = make_double2(cw[2], cw[3]);
          if (G == 2) {
            e[2] = make_double2(cw[0] * vpar, cw[1] * vpar);
            e[3] = make_double2(cw[2] * vpar, cw[3] * vpar);
          }
          MarkerTmp t;
          t.a = a0;
          t.b = b0;
          t.rho = r0;
          t.ts = mts;
          t.cg = mcg;
          t.sg = msg;
          t.pad_ = 0.0;
          t.n = n | ((have && mk0 == k - 1) ? 0 : 256);
          t.k0 = mk0;
          mtmp[ms] = t;
          const unsigned int q0 = ub + (unsigned)(incl - u);
          for (int j = 0; j < u; ++j) unit_tab[q0 + j] = ms | ((unsigned)j << 16);
        }
        named_bar_sync(1, Sh::kProd);
        last_chunk = !(S.n_deferred[cur ^ 1] > 0 || S.next_group < n_groups);
        const int n_units = min(S.nunits, S.units_end);
        if (tid < n_units) {
          const unsigned int ut = unit_tab[tid];
          mslot = ut & 0xffffu;
          const MarkerTmp t = mtmp[mslot];
          ga = t.a;
          gb = t.b;
          grho = t.rho;
          gts = t.ts;
          gcg = t.cg;
          gsg = t.sg;
          un = t.n & 255;
          k_ok = t.n < 256;
          k0 = t.k0;
          l0 = (int)(ut >> 16) * kPPL;
        }
      }

      // -------------------------------------------------- phase B: the unit's Larmor points
      double pts[kPPL], ptt[kPPL];   // in-cell coordinates
      int pcr[kPPL];                 // tile-local cell | rank in the cell << 9; -1: none;
                                     // <= -2: outside the tile, global cell -(pcr + 2)
      bool any_direct = false;
      const double* chan = St.mtab + (size_t)mslot * kChan;
      {
        // straight-line geometry of the 4 points (no branches: the chains interleave)
        double psl[kPPL], ptl[kPPL], pX[kPPL], pY[kPPL];
        bool slow = false;
        const int nring = max(un, 1);
#pragma unroll
        for (int j = 0; j < kPPL; ++j) {
          const int l = (l0 + j < un) ? l0 + j : 0;
          bool ok;
          larmor_point_fast(P, ga, gb, grho, gts, gcg, gsg, ring_entry(P, nring, l), psl[j], ptl[j],
                            pX[j], pY[j], ok);
          slow |= !ok && (l0 + j < un);
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
          pcr[j] = -1;
          const double xs = psl[j] * (double)P.ns;
          const int ci = min((int)xs, P.ns - 1);
          pts[j] = xs - (double)ci;
          const int cj = periodic_cell(ptl[j], P.nth_scale, P.nth, ptt[j]);
          const int lr = ci - row_base;
          int lc = cj - cellcol_base;
          if (lc >= P.nth) lc -= P.nth;
          if (lc < 0) lc += P.nth;
          if (l0 + j < un) {
            if (k_ok && lr >= 0 && lr < kCH && lc >= 0 && lc < kCW) {
              const unsigned int cell = (unsigned)(lr * kCW + lc);
              const unsigned int rank = atomicAdd(&S.count[cell], 1u);
              pcr[j] = (int)(cell | (rank << 9));
            } else {
              // footprint leaves the tile (long ring, or phi rounding): direct path, below
              pcr[j] = -2 - (ci * P.nth + cj);
              any_direct = true;
            }
          }
        }
      }
      if (any_direct) {   // rare: global atomics, kept out of the unrolled point loop
#pragma unroll
        for (int j = 0; j < kPPL; ++j) {
          if (pcr[j] > -2) continue;
          const int gc = -(pcr[j] + 2);
          ++my_fallback;
          deposit_point_cell<G>(P, gc / P.nth, pts[j], gc % P.nth, ptt[j], k0, chan, rho, jpar);
          pcr[j] = -1;
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
        // path) and, like every cell after them, start where the written slots end: the consumers
        // stream a row segment's slots linearly and must never run into unwritten ones.
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
        // work list: the row segments that hold points, heaviest first
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
          if (!SELF) {
            S.n_deferred[cur] = 0;
            S.take_deferred = 0;
            S.nmark = 0;
            S.nunits = 0;
            S.units_end = 0x7fffffff;
            S.full_flag = 0;
          }
        }
      }
      named_bar_sync(1, Sh::kProd);
      ORB_CLK(tid == 0, 5);

      // -------------------------------------------------- phase D: operand records, sorted by cell
      {
        char* ops_b = reinterpret_cast<char*>(St.ops);
        // (uniform over the tile) only tiles that reach the two end cells of the clamped radial
        // basis need the tabulated pieces; everywhere else the radial weights are cardinal too
        const bool edge = row_base < 2 || row_base + kCH - 1 > P.ns - 3;
        bool any_ovf = false;
#pragma unroll
        for (int j = 0; j < kPPL; ++j) {
          if (pcr[j] < 0) continue;
          const unsigned int cell = (unsigned)pcr[j] & 0x1ffu, rank = (unsigned)pcr[j] >> 9;
          const unsigned int pk = St.cs[cell];
          const unsigned int cnt = pk >> 16;
          if (cnt == 0) {   // the chunk's padding capacity is exhausted: direct path, below
            any_ovf = true;
            continue;
          }
          pcr[j] = -1;
          const int lr = (int)cell / kCW, lc = (int)cell - lr * kCW;
          unsigned int p = (pk & 0xffffu) + rank;
          double ws[4], wt[4];
          if (edge) {
            radial_cell_weights(P, row_base + lr, pts[j], ws);
          } else {
            cardinal_weights(pts[j], ws);
          }
          cardinal_weights(ptt[j], wt);
          char* rec = ops_b + (p >> 2) * 256u + (p & 3u) * 32u;
          double2* o = reinterpret_cast<double2*>(rec);
          o[0] = make_double2(ws[0], ws[1]);
          o[1] = make_double2(ws[2], ws[3]);
          // theta* weights rotated by the cell's walk phase U = column & 3, so that a consumer
          // lane finds the weight of its accumulator slot at a fixed offset: R[(b + U) & 3] = wt[b]
          double* r = reinterpret_cast<double*>(rec + 128);
          const int U = lc & 3;
          r[U] = wt[0];
          r[(U + 1) & 3] = wt[1];
          r[(U + 2) & 3] = wt[2];
          r[(U + 3) & 3] = wt[3];
          St.midx[p] = (unsigned short)(mslot * (unsigned)(kChan * 8));
          if (rank + 1 == cnt) {   // the cell's last point pads the cell to a batch of 4
            for (++p; (p & 3u) != 0; ++p) {
              double2* z = reinterpret_cast<double2*>(ops_b + (p >> 2) * 256u + (p & 3u) * 32u);
              z[0] = z[1] = z[8] = z[9] = make_double2(0.0, 0.0);
              St.midx[p] = (unsigned short)(Sh::kMCap * kChan * 8);
            }
          }
        }
        if (any_ovf) {
#pragma unroll
          for (int j = 0; j < kPPL; ++j) {
            if (pcr[j] < 0) continue;
            const int cell = pcr[j] & 0x1ff;
            const int lr = cell / kCW, lc = cell - lr * kCW;
            ++my_fallback;
            deposit_point_cell<G>(P, row_base + lr, pts[j], wrap_index(cellcol_base + lc, P.nth),
                                  ptt[j], k0, chan, rho, jpar);
          }
        }
      }
      mbar_arrive(&S.full[stage]);
      ORB_CLK(tid == 0, 6);
      ++it;
      if (!SELF) cur ^= 1;
      if (last_chunk) break;
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
template <int G, int PW, int CW>
__device__ __forceinline__ void consumer(Smem<G, PW, CW>& S, const Params& P,
                                         double* __restrict__ rho, double* __restrict__ jpar,
                                         unsigned long long* __restrict__ d_points) {
  using Sh = Shape<G, PW, CW>;
  constexpr int kChan = Sh::kChan;
  const int ctid = threadIdx.x - Sh::kProd;        // 0 .. kCons-1
  const int lane = ctid & 31;
  const int g = lane >> 2, kk = lane & 3, hi = lane >> 4, a = g & 3;
  unsigned int it = 0;
  ORB_CLK_DECL;

  for (;; ++it) {
    const int stage = (int)(it % kStages);
    typename Smem<G, PW, CW>::Stage& St = S.st[stage];
    mbar_wait(&S.full[stage], (it / kStages) & 1u);
    ORB_CLK(ctid == 0, 8);
    const int n_items = St.info.n_items;
    if (n_items < 0) break;
    const int last = St.info.last, tk = St.info.k, row_base = St.info.row_base,
              cellcol_base = St.info.cellcol_base;

    // this lane's operands of a batch (4 slots, 256 bytes): ws[kk][a], and the rotated theta*
    // weights of its two accumulator slots, R[kk][hi] and R[kk][hi + 2]
    const char* ops_b = reinterpret_cast<const char*>(St.ops) + kk * 32 + a * 8;
    const int wo0 = 128 - a * 8 + hi * 8, wo1 = wo0 + 16;
    const char* mt_b = reinterpret_cast<const char*>(St.mtab + (G == 2 ? g : (g & 3)));
    const unsigned short* midx = St.midx + kk;

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

      // The batches of a row segment are contiguous in the sorted order: one linear operand
      // stream, loaded one batch ahead of the MMAs (marker offsets two ahead), across cell
      // boundaries, in two alternating register sets (A, B) so that no operand is ever copied.
      // The stream is read up to two batches beyond the segment's end (valid shared memory: the
      // fields that follow ops / midx in the stage; the values are never used, the marker offsets
      // are clamped to the table and to 8-byte alignment).
      constexpr unsigned kMoCap = (unsigned)(Sh::kMCap * kChan * 8);   // the zero marker
      unsigned int pk = St.cs[c_first];
      const char* p = ops_b + (pk & 0xffffu) * 64u;
      const unsigned short* mi = midx + (pk & 0xffffu);
      double Aw, Ax0, Ax1, Ab = 0.0, Bw, Bx0, Bx1, Bb = 0.0;
#define ORB_LD(S, q, off)                                                             \
      S##w = *reinterpret_cast<const double*>((q));                                   \
      S##x0 = *reinterpret_cast<const double*>((q) + wo0);                            \
      S##x1 = *reinterpret_cast<const double*>((q) + wo1);                            \
      if (G == 2 || g < 4) S##b = *reinterpret_cast<const double*>(mt_b + (off));
#define ORB_MMA(S)                                                                    \
      {                                                                               \
        const double a0 = S##w * S##x0, a1 = S##w * S##x1;                            \
        dmma884(c0a, c0b, a0, S##b);                                                  \
        dmma884(c1a, c1b, a1, S##b);                                                  \
      }
      ORB_LD(A, p, min((unsigned)mi[0] & 0xfff8u, kMoCap))
      unsigned int mo = min((unsigned)mi[4] & 0xfff8u, kMoCap);

      // Column retire, deferred: stepping past cell U of a group of four finishes one node column
      // of the window.  Its two accumulators are parked in registers (t0: the column this lane's
      // first slot held, t1: the second) and all parked columns are added into the shared tile
      // in one pipelined pass after the walk -- one round of CAS latency per row segment instead
      // of two per cell.
#define ORB_PARK(U)                                                                   \
      if ((U) < 2) {                                                                  \
        if (hi == (U)) { t0a = c0a; t0b = c0b; c0a = 0.0; c0b = 0.0; }                \
      } else {                                                                        \
        if (hi == (U) - 2) { t1a = c1a; t1b = c1b; c1a = 0.0; c1b = 0.0; }            \
      }

#define ORB_CELL(U)                                                                   \
      {                                                                               \
        int nb = (int)(((pk >> 16) + 3u) >> 2);                                       \
        pk = St.cs[c_first + cc + (U) + 1];                                           \
        _Pragma("unroll 1") for (; nb >= 2; nb -= 2) {                                \
          ORB_LD(B, p + 256, mo)                                                      \
          mo = min((unsigned)mi[8] & 0xfff8u, kMoCap);                                          \
          ORB_MMA(A)                                                                  \
          ORB_LD(A, p + 512, mo)                                                      \
          mo = min((unsigned)mi[12] & 0xfff8u, kMoCap);                                         \
          ORB_MMA(B)                                                                  \
          p += 512;                                                                   \
          mi += 8;                                                                    \
        }                                                                             \
        if (nb) {                                                                     \
          ORB_LD(B, p + 256, mo)                                                      \
          mo = min((unsigned)mi[8] & 0xfff8u, kMoCap);                                          \
          ORB_MMA(A)                                                                  \
          Aw = Bw; Ax0 = Bx0; Ax1 = Bx1; Ab = Bb;                                     \
          p += 256;                                                                   \
          mi += 4;                                                                    \
        }                                                                             \
        ORB_PARK(U)                                                                   \
      }

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
      // a9: all consumers are done with the tile -> flush it once and clear it.  kChan consecutive
      // lanes run along the channels of a node (4 phi planes = one 32-byte sector per grid).
      named_bar_sync(2, Sh::kCons);
      const int ch = ctid % kChan;
      double* __restrict__ out = ((G == 2 && ch >= 4) ? jpar : rho) + wrap_index(tk - 1 + (ch & 3), P.nph);
      const int64_t row_stride = (int64_t)P.nth * P.nph;
      for (int node = ctid / kChan; node < kNH * kNW; node += Sh::kCons / kChan) {
        const double v = S.tile[node * kChan + ch];
        if (v == 0.0) continue;
        S.tile[node * kChan + ch] = 0.0;
        const int nr = node / kNW, tc = node - nr * kNW;
        const int gi = row_base + nr;           // zero outside [0, ns + 2]: no point maps there
        int gj = cellcol_base - 1 + tc;
        while (gj < 0) gj += P.nth;
        while (gj >= P.nth) gj -= P.nth;
        atomicAdd(out + gi * row_stride + (int64_t)gj * P.nph, v);
      }
      named_bar_sync(2, Sh::kCons);
      ORB_CLK(ctid == 0, 10);
    }
  }
}

template <int G, int PW, int CW, bool SELF>
__global__ void __launch_bounds__((PW + CW) * 32, 1)
k_deposit_ws(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
             const TileBins TB, double* __restrict__ rho, double* __restrict__ jpar,
             unsigned long long* __restrict__ d_points, int tiles_i, int tiles_j) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  Smem<G, PW, CW>& S = *reinterpret_cast<Smem<G, PW, CW>*>(smem_raw);
  using Sh = Shape<G, PW, CW>;
  const int tid = threadIdx.x;
#ifdef ORB_POISON_SMEM
  for (size_t x = tid; x < sizeof(S) / 4; x += Sh::kThreads) reinterpret_cast<unsigned int*>(smem_raw)[x] = 0xffffffffu;
  __syncthreads();
#endif
  for (int x = tid; x < kNH * kNW * Sh::kChan; x += Sh::kThreads) S.tile[x] = 0.0;
  for (int x = tid; x < kCells; x += Sh::kThreads) S.count[x] = 0;
  if (tid < kStages * Sh::kChan) {
    const int s = tid / Sh::kChan, d = tid % Sh::kChan;
    S.st[s].mtab[Sh::kMCap * Sh::kChan + d] = 0.0;   // the zero marker of the padding records
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
    producer<G, PW, CW, SELF>(S, P, M, cell_start, TB, rho, jpar, d_points, tiles_i, tiles_j);
  } else {
    consumer<G, PW, CW>(S, P, rho, jpar, d_points);
  }
}

template <int G, int PW, int CW, bool SELF>
int launch(const Params& P, const Markers& M, const uint32_t* cell_start, const TileBins& TB,
           double* rho, double* jpar, unsigned long long* d_points, int sms, cudaStream_t st) {
  const int tiles_i = (P.ns + kTileI - 1) / kTileI;
  const int tiles_j = (P.nth + kTileJ - 1) / kTileJ;
  const int64_t n_tiles = (int64_t)tiles_i * tiles_j * P.nph;
  const int blocks = (int)(n_tiles < sms ? n_tiles : sms);
  const size_t smem = sizeof(Smem<G, PW, CW>);
  static_assert(sizeof(Smem<G, PW, CW>) <= 232448, "shared memory of one block must fit one SM");
  if (cudaFuncSetAttribute(k_deposit_ws<G, PW, CW, SELF>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)smem) != cudaSuccess)
    return -1;
  k_deposit_ws<G, PW, CW, SELF><<<blocks, (PW + CW) * 32, smem, st>>>(P, M, cell_start, TB, rho, jpar,
                                                                      d_points, tiles_i, tiles_j);
  return 1;
}

}  // namespace

int launch_deposit_ws(const Params& P, const Markers& M, const uint32_t* cell_start,
                      const TileBins& TB, double* rho, double* jpar, unsigned long long* d_points,
                      int sms, cudaStream_t st) {
  if (M.n == 0) return 0;
#ifndef ORB_CW
#define ORB_CW 8
#endif
  constexpr int PW = 8, CW = ORB_CW;
  const bool self = !P.adaptive && P.n_fixed <= kPPL;
  if (self)
    return jpar ? launch<2, PW, CW, true>(P, M, cell_start, TB, rho, jpar, d_points, sms, st)
                : launch<1, PW, CW, true>(P, M, cell_start, TB, rho, jpar, d_points, sms, st);
  return jpar ? launch<2, PW, CW, false>(P, M, cell_start, TB, rho, jpar, d_points, sms, st)
              : launch<1, PW, CW, false>(P, M, cell_start, TB, rho, jpar, d_points, sms, st);
}

}  // namespace orb
