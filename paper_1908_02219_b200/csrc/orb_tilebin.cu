// Incremental re-binning.  PAPER.md:169-173: the bucket sort pays for
// itself on the deposit but is "the most time-consuming part" of the run; PAPER.md:235 proposes
// to "track markers leaving cells" instead of sorting from scratch.  A dense cell-sorted array
// cannot be updated in place (any insertion shifts everything behind it), so this second binning
// layout trades memory for updatability:
//
//   slack tile bins   every deposit tile (1 toroidal slab x 8 radial x 16 poloidal cells, the unit
//                     of work of the tile kernels) is cut into its 8 radial rows; bin b (1 x 16
//                     cells) owns a fixed-capacity segment rec[b * cap .. b * cap + count[b]) of
//                     64-byte marker records, in any order.  The tile kernels take a tile's markers
//                     in chunks of 256-384, run by run, so a chunk still covers a few whole radial
//                     rows, as with the dense layout.  (Measured on cfg3: whole-tile bins, whose
//                     chunks spread their Larmor points over all 288 cells of the halo window, gave
//                     30.4 ms deposits, quarter-tile bins 18.8 ms, row bins 16.5 ms = the dense
//                     layout's.)  cap ~ 1.5 x the mean occupancy + 64.
//   build             ONE pass: slot = atomicAdd(count[tile]); no histogram, no scan.
//   rebin             after the marker coordinates changed in the records (orb_markers_refresh,
//                     or a pusher writing them in place): one warp per bin re-derives each
//                     record's tile; markers that left are copied to a mover buffer and the
//                     segment is compacted (tail records fill the holes); a second kernel
//                     appends the movers to their new tiles.  Cost: one 32-byte sector per marker
//                     (s, theta*, phi) + 4 x 64 bytes per mover.
//
// Nothing downstream relies on a marker being in the RIGHT tile for correctness, only for speed
// (points outside a block's tile take the direct global path).  That makes every overflow benign:
// a full tile sends the marker to the next tile with room; a full mover buffer leaves the marker
// where it was until the next rebin.
#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr int kTileI = 8, kTileJ = 16;
constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ uint32_t tile_of(const Params& P, int tiles_i, int tiles_j, double s, double th,
                                            double ph) {
  int i = min(max((int)(s * (double)P.ns), 0), P.ns - 1);
  int j = (int)(wrap_2pi(th) * P.nth_scale);
  int k = (int)(wrap_2pi(ph) * P.nph_scale);
  j = min(max(j, 0), P.nth - 1);
  k = min(max(k, 0), P.nph - 1);
  const uint32_t tile = ((uint32_t)k * (uint32_t)tiles_i + (uint32_t)(i / kTileI)) * (uint32_t)tiles_j +
                        (uint32_t)(j / kTileJ);
  return tile * (uint32_t)kTileBinSubs + (uint32_t)((i % kTileI) / (kTileI / kTileBinSubs));
}

// claim a slot in tile t, or in the next tile with room (benign mis-binning, see the header)
__device__ __forceinline__ int64_t claim_slot(uint32_t* __restrict__ count, uint32_t t, uint32_t n_tiles,
                                              uint32_t cap) {
  for (uint32_t probe = 0; probe < n_tiles; ++probe) {
    const uint32_t slot = atomicAdd(count + t, 1u);   // counts may overshoot cap: readers clamp
    if (slot < cap) return (int64_t)t * cap + slot;
    t = t + 1 < n_tiles ? t + 1 : 0;
  }
  return -1;   // unreachable: n_tiles * cap > n
}

__device__ __forceinline__ void store_record(double* __restrict__ out, double s, double th, double ph,
                                             double vp, double mu, double w, double idx_bits) {
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(out), "d"(s), "d"(th), "d"(ph), "d"(vp)
               : "memory");
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(out + 4), "d"(mu), "d"(w),
               "d"(idx_bits), "d"(0.0)
               : "memory");
}

// Two markers per thread (one 128-bit load per array, the arrays are 16-byte aligned): the pass is
// bound by the latency of its dependent chain load -> atomic -> store, not by DRAM bandwidth
// (2.3 TB/s with one marker per thread), so more independent chains per thread is what helps.
__global__ void __launch_bounds__(256)
k_tilebin_build(const Params P, const Markers M, const TileBins T, uint32_t* __restrict__ count,
                double* __restrict__ rec, const int64_t base) {
  const int64_t p = 2 * ((int64_t)blockIdx.x * blockDim.x + threadIdx.x);
  if (p >= M.n) return;
  if (p + 1 < M.n) {
    const double2 s = __ldg(reinterpret_cast<const double2*>(M.s + p));
    const double2 th = __ldg(reinterpret_cast<const double2*>(M.th + p));
    const double2 ph = __ldg(reinterpret_cast<const double2*>(M.ph + p));
    const double2 vp = M.vpar ? __ldg(reinterpret_cast<const double2*>(M.vpar + p)) : make_double2(0.0, 0.0);
    const double2 mu = __ldg(reinterpret_cast<const double2*>(M.mu + p));
    const double2 w = __ldg(reinterpret_cast<const double2*>(M.w + p));
    const uint32_t t0 = tile_of(P, T.tiles_i, T.tiles_j, s.x, th.x, ph.x);
    const uint32_t t1 = tile_of(P, T.tiles_i, T.tiles_j, s.y, th.y, ph.y);
    const int64_t d0 = claim_slot(count, t0, T.n_tiles, T.cap);
    const int64_t d1 = claim_slot(count, t1, T.n_tiles, T.cap);
    if (d0 >= 0)
      store_record(rec + d0 * kRecDoubles, s.x, th.x, ph.x, vp.x, mu.x, w.x, __longlong_as_double((long long)(base + p)));
    if (d1 >= 0)
      store_record(rec + d1 * kRecDoubles, s.y, th.y, ph.y, vp.y, mu.y, w.y,
                   __longlong_as_double((long long)(base + p + 1)));
    return;
  }
  const double s = __ldg(M.s + p), th = __ldg(M.th + p), ph = __ldg(M.ph + p);
  const uint32_t t = tile_of(P, T.tiles_i, T.tiles_j, s, th, ph);
  const int64_t dst = claim_slot(count, t, T.n_tiles, T.cap);
  if (dst < 0) return;
  store_record(rec + dst * kRecDoubles, s, th, ph, M.vpar ? __ldg(M.vpar + p) : 0.0, __ldg(M.mu + p),
               __ldg(M.w + p), __longlong_as_double((long long)(base + p)));
}

// records <- current values of the bound arrays (by the original index kept in the record)
__global__ void __launch_bounds__(256)
k_tilebin_refresh(const Markers M, const TileBins T, const uint32_t* __restrict__ count,
                  double* __restrict__ rec) {
  const uint32_t t = blockIdx.x;
  const uint32_t n = min(__ldg(count + t), T.cap);
  for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
    double* r = rec + ((int64_t)t * T.cap + i) * kRecDoubles;
    const double ib = r[6];
    const int64_t p = (int64_t)__double_as_longlong(ib);
    store_record(r, __ldg(M.s + p), __ldg(M.th + p), __ldg(M.ph + p), M.vpar ? __ldg(M.vpar + p) : 0.0,
                 __ldg(M.mu + p), __ldg(M.w + p), ib);
  }
}

// One warp per bin: movers out, segment compacted.  counters[0] += movers extracted,
// counters[1] += movers left in place because the mover buffer was full.  The mover buffer is
// claimed once per BLOCK (one atomic on the shared counter per 8 bins, not per warp pass: with a
// counter per pass the kernel was bound by same-address atomics, 1.4 ms at 1 % movers on cfg3).
constexpr int kWarpsPerBlock = 8;
constexpr int kMaxIter = 64;    // cap <= 32 * kMaxIter records per bin

__global__ void __launch_bounds__(kWarpsPerBlock * 32)
k_tilebin_extract(const Params P, const TileBins T, uint32_t* __restrict__ count, double* __restrict__ rec,
                  double* __restrict__ movers, uint32_t mv_cap, uint32_t* __restrict__ mv_count,
                  unsigned long long* __restrict__ counters) {
  __shared__ unsigned short hole[kWarpsPerBlock][32 * kMaxIter / 2 + 32];
  __shared__ unsigned short tail[kWarpsPerBlock][32 * kMaxIter / 2 + 32];
  __shared__ uint32_t warp_movers[kWarpsPerBlock];
  __shared__ uint32_t block_base;
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t t = blockIdx.x * kWarpsPerBlock + wid;
  const bool live = t < T.n_tiles;
  const uint32_t n = live ? min(count[t], T.cap) : 0u;
  double* base = rec + (int64_t)(live ? t : 0) * T.cap * kRecDoubles;
  const int iters = (int)((n + 31) / 32);
  // pass 1: who leaves?  bit x of `gone`: record x * 32 + lane belongs to another bin
  unsigned long long gone = 0;
  uint32_t n_gone = 0;
  for (int x = 0; x < iters; ++x) {
    const uint32_t i = (uint32_t)x * 32u + (uint32_t)lane;
    if (i < n) {
      const double4 a = *reinterpret_cast<const double4*>(base + (size_t)i * kRecDoubles);
      if (tile_of(P, T.tiles_i, T.tiles_j, a.x, a.y, a.z) != t) {
        gone |= 1ull << x;
        ++n_gone;
      }
    }
  }
  uint32_t incl = n_gone;   // inclusive prefix over the lanes
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(kFull, incl, o);
    if (lane >= o) incl += v;
  }
  const uint32_t warp_total = __shfl_sync(kFull, incl, 31);
  if (lane == 0) warp_movers[wid] = warp_total;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
    for (int w = 0; w < kWarpsPerBlock; ++w) tot += warp_movers[w];
    block_base = tot ? atomicAdd(mv_count, tot) : 0u;
  }
  __syncthreads();
  if (!live || n == 0) {
    if (live && lane == 0) count[t] = 0;
    return;
  }
  if (warp_total == 0) {
    if (lane == 0) count[t] = n;
    return;
  }
  uint32_t my_slot = block_base + (incl - n_gone);
  for (int w = 0; w < wid; ++w) my_slot += warp_movers[w];
  // pass 1b: copy this lane's movers out (slot 7 <- destination bin); movers beyond the buffer's
  // capacity stay where they are (mis-binned) until the next rebin
  uint32_t n_back = 0;
  for (int x = 0; x < iters; ++x) {
    if (!((gone >> x) & 1ull)) continue;
    if (my_slot < mv_cap) {
      const uint32_t i = (uint32_t)x * 32u + (uint32_t)lane;
      const double4* r = reinterpret_cast<const double4*>(base + (size_t)i * kRecDoubles);
      const double4 a = r[0];
      double4 b = r[1];
      b.w = __longlong_as_double((long long)tile_of(P, T.tiles_i, T.tiles_j, a.x, a.y, a.z));
      double4* o = reinterpret_cast<double4*>(movers + (size_t)my_slot * kRecDoubles);
      o[0] = a;
      o[1] = b;
    } else {
      gone &= ~(1ull << x);
      ++n_back;
    }
    ++my_slot;
  }
  uint32_t tot_gone = n_gone - n_back, tot_back = n_back;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    tot_gone += __shfl_xor_sync(kFull, tot_gone, o);
    tot_back += __shfl_xor_sync(kFull, tot_back, o);
  }
  const uint32_t n_new = n - tot_gone;
  // pass 2: holes below n_new, stayers at or above n_new; equally many of both
  uint32_t nh = 0, nt = 0;
  for (int x = 0; x < iters; ++x) {
    const uint32_t i = (uint32_t)x * 32u + (uint32_t)lane;
    const bool is_gone = (gone >> x) & 1ull;
    const bool h = i < n_new && is_gone;
    const bool s = i >= n_new && i < n && !is_gone;
    const unsigned bh = __ballot_sync(kFull, h), bs = __ballot_sync(kFull, s);
    if (h) hole[wid][nh + __popc(bh & ((1u << lane) - 1u))] = (unsigned short)i;
    if (s) tail[wid][nt + __popc(bs & ((1u << lane) - 1u))] = (unsigned short)i;
    nh += __popc(bh);
    nt += __popc(bs);
  }
  __syncwarp();
  for (uint32_t q = lane; q < nh; q += 32) {
    const double4* src = reinterpret_cast<const double4*>(base + (size_t)tail[wid][q] * kRecDoubles);
    double4* dst = reinterpret_cast<double4*>(base + (size_t)hole[wid][q] * kRecDoubles);
    const double4 a = src[0], b = src[1];
    dst[0] = a;
    dst[1] = b;
  }
  if (lane == 0) {
    count[t] = n_new;
    if (tot_gone) atomicAdd(counters, (unsigned long long)tot_gone);
    if (tot_back) atomicAdd(counters + 1, (unsigned long long)tot_back);
  }
}

__global__ void __launch_bounds__(256)
k_tilebin_insert(const TileBins T, uint32_t* __restrict__ count, double* __restrict__ rec,
                 const double* __restrict__ movers, uint32_t mv_cap, const uint32_t* __restrict__ mv_count) {
  const uint32_t n = min(*mv_count, mv_cap);
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const double4* m = reinterpret_cast<const double4*>(movers + (size_t)i * kRecDoubles);
    const double4 a = m[0];
    double4 b = m[1];
    const uint32_t dest = (uint32_t)__double_as_longlong(b.w);
    b.w = 0.0;
    const int64_t dst = claim_slot(count, dest, T.n_tiles, T.cap);
    if (dst < 0) continue;
    double4* o = reinterpret_cast<double4*>(rec + dst * kRecDoubles);
    o[0] = a;
    o[1] = b;
  }
}

}  // namespace

int launch_tilebin_build(const Params& P, const Markers& M, const TileBins& T, uint32_t* count, double* rec,
                         cudaStream_t st, int64_t base, bool append) {
  if (!append &&
      cudaMemsetAsync(count, 0, (size_t)T.n_tiles * sizeof(uint32_t), st) != cudaSuccess)
    return -1;
  if (M.n == 0) return 0;
  const int64_t blocks = ((M.n + 1) / 2 + 255) / 256;
  k_tilebin_build<<<(unsigned int)blocks, 256, 0, st>>>(P, M, T, count, rec, base);
  return 1;
}

int launch_tilebin_refresh(const Markers& M, const TileBins& T, const uint32_t* count, double* rec,
                           cudaStream_t st) {
  if (M.n == 0) return 0;
  k_tilebin_refresh<<<T.n_tiles, 128, 0, st>>>(M, T, count, rec);
  return 1;
}

int launch_tilebin_rebin(const Params& P, const TileBins& T, uint32_t* count, double* rec, double* movers,
                         uint32_t mv_cap, uint32_t* mv_count, unsigned long long* counters,
                         cudaStream_t st) {
  if (T.cap > 32u * kMaxIter) return -1;
  if (cudaMemsetAsync(mv_count, 0, sizeof(uint32_t), st) != cudaSuccess) return -1;
  const unsigned int blocks = (T.n_tiles + kWarpsPerBlock - 1) / kWarpsPerBlock;
  k_tilebin_extract<<<blocks, kWarpsPerBlock * 32, 0, st>>>(P, T, count, rec, movers, mv_cap, mv_count,
                                                          counters);
  unsigned int ib = (mv_cap + 255) / 256;
  if (ib > 148u * 16u) ib = 148u * 16u;
  if (ib == 0) ib = 1;
  k_tilebin_insert<<<ib, 256, 0, st>>>(T, count, rec, movers, mv_cap, mv_count);
  return 2;
}

}  // namespace orb
