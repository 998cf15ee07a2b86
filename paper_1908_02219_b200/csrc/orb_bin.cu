// Marker binning (hot-path step a7): counting sort of the markers by the field
// cell of their guiding centre -- the bucket sort of PAPER.md:167 ("sorting of
// markers with respect to the field cells"), key order phi-major
//   key = (k_phi * ns + i_s) * ntheta + j_theta                         (R17)
// so that the markers of one toroidal cell slab and one radial row are contiguous
// along theta*.  Three passes:
//   1. count:   rank[p] = atomicAdd(count[key(p)], 1)       (integer atomics in L2)
//   2. scan:    cell_start = exclusive prefix sum of count   (3 small kernels)
//   3. scatter: record(cell_start[key(p)] + rank[p]) = marker p, as one 64-byte
//               record {s, theta*, phi, vpar, mu, w, index in bound order, 0} (two 32-byte
//               stores) so
//               that a random-order input costs 2 whole sectors per marker, not 6
//               partial ones.
// The order inside a cell is whatever the atomics gave (any order is correct, R18).
// Nothing downstream relies on the key for correctness, only for locality.
#include "orb_geom.cuh"

namespace orb {

__device__ __forceinline__ uint32_t cell_key(const Params& P, double s, double th, double ph) {
  int i = min(max((int)(s * (double)P.ns), 0), P.ns - 1);
  double ts = wrap_2pi(th);
  double ps = wrap_2pi(ph);
  int j = (int)(ts * P.nth_scale);
  int k = (int)(ps * P.nph_scale);
  j = min(max(j, 0), P.nth - 1);
  k = min(max(k, 0), P.nph - 1);
  return ((uint32_t)k * (uint32_t)P.ns + (uint32_t)i) * (uint32_t)P.nth + (uint32_t)j;
}

__global__ void __launch_bounds__(256)
k_bin_count(const Params P, const Markers M, uint32_t* __restrict__ count,
            uint32_t* __restrict__ rank) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= M.n) return;
  const uint32_t key = cell_key(P, __ldg(M.s + p), __ldg(M.th + p), __ldg(M.ph + p));
  const uint32_t r = atomicAdd(count + key, 1u);
  if (rank) rank[p] = r;
}

constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
  __shared__ uint32_t warp_sums[kScanThreads / 32];
  __shared__ uint32_t block_total;
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_sums[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    uint32_t ws = lane < kScanThreads / 32 ? warp_sums[lane] : 0;
    uint32_t wi = ws;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      uint32_t t = __shfl_up_sync(0xffffffffu, wi, o);
      if (lane >= o) wi += t;
    }
    if (lane < kScanThreads / 32) warp_sums[lane] = wi - ws;
    if (lane == 31) block_total = wi;
  }
  __syncthreads();
  const uint32_t r = inc - v + warp_sums[wid];
  if (total) *total = block_total;
  __syncthreads();
  return r;
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_reduce(const uint32_t* __restrict__ count, int64_t n, uint32_t* __restrict__ block_sums) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile;
  uint32_t sum = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    const int64_t idx = base + (int64_t)i * kScanThreads + threadIdx.x;
    if (idx < n) sum += count[idx];
  }
  uint32_t total;
  block_exclusive_scan(sum, &total);
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_block_sums(uint32_t* __restrict__ block_sums, int nb) {
  uint32_t carry = 0;
  for (int base = 0; base < nb; base += kScanThreads) {
    const int idx = base + threadIdx.x;
    const uint32_t v = idx < nb ? block_sums[idx] : 0;
    uint32_t total;
    const uint32_t ex = block_exclusive_scan(v, &total);
    if (idx < nb) block_sums[idx] = ex + carry;
    carry += total;
  }
}

// in place: count[0..n) -> exclusive offsets; count[n] = grand total
__global__ void __launch_bounds__(kScanThreads)
k_scan_apply(uint32_t* __restrict__ count, int64_t n, const uint32_t* __restrict__ block_sums) {
  const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
  uint32_t v[kScanItems];
  uint32_t sum = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    v[i] = (base + i < n) ? count[base + i] : 0;
    sum += v[i];
  }
  uint32_t total;
  uint32_t ex = block_exclusive_scan(sum, &total) + block_sums[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) count[base + i] = ex;
    ex += v[i];
  }
  if (blockIdx.x == gridDim.x - 1 && threadIdx.x == kScanThreads - 1) count[n] = ex;
}

__global__ void __launch_bounds__(256)
k_bin_scatter(const Params P, const Markers M, const uint32_t* __restrict__ cell_start,
              const uint32_t* __restrict__ rank, double* __restrict__ rec) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= M.n) return;
  const double s = __ldg(M.s + p), th = __ldg(M.th + p), ph = __ldg(M.ph + p);
  const uint32_t key = cell_key(P, s, th, ph);
  const int64_t dst = (int64_t)__ldg(cell_start + key) + rank[p];
  // two 256-bit stores = two whole 32-byte sectors per marker: a partial-sector write that
  // misses in L2 makes it fetch the sector from DRAM first (measured: +3.8 GB of reads on cfg3
  // with four 16-byte stores, +6.6 GB with 48-byte records)
  double* out = rec + dst * kRecDoubles;
  const double vp = M.vpar ? __ldg(M.vpar + p) : 0.0;
  const double mu = __ldg(M.mu + p), w = __ldg(M.w + p);
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(out), "d"(s), "d"(th), "d"(ph), "d"(vp)
               : "memory");
  // slot 6: the marker's index in bound order (bit pattern), for results that go back to the
  // caller's order (orb_gather)
  asm volatile("st.global.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(out + 4), "d"(mu), "d"(w),
               "d"(__longlong_as_double((long long)p)), "d"(0.0)
               : "memory");
}

// exclusive scan in place: count[0..n) -> offsets, count[n] = total; block_sums: n / 4096 + 2 words
int launch_scan(uint32_t* count, int64_t n, uint32_t* block_sums, cudaStream_t st) {
  const int nb = (int)((n + kScanTile - 1) / kScanTile);
  if (nb == 0) return 0;
  k_scan_reduce<<<nb, kScanThreads, 0, st>>>(count, n, block_sums);
  k_scan_block_sums<<<1, kScanThreads, 0, st>>>(block_sums, nb);
  k_scan_apply<<<nb, kScanThreads, 0, st>>>(count, n, block_sums);
  return 3;
}

int launch_bin(const Params& P, const Markers& M, const BinScratch& B, bool presorted,
               cudaStream_t st) {
  int launches = 0;
  const int64_t nc = B.ncells;
  if (cudaMemsetAsync(B.cell_start, 0, (size_t)(nc + 1) * sizeof(uint32_t), st) != cudaSuccess)
    return -1;
  if (M.n > 0) {
    const int64_t blocks = (M.n + 255) / 256;
    k_bin_count<<<(unsigned int)blocks, 256, 0, st>>>(P, M, B.cell_start,
                                                      presorted ? nullptr : B.rank);
    ++launches;
  }
  launches += launch_scan(B.cell_start, nc, B.block_sums, st);
  if (!presorted && M.n > 0) {
    const int64_t blocks = (M.n + 255) / 256;
    k_bin_scatter<<<(unsigned int)blocks, 256, 0, st>>>(P, M, B.cell_start, B.rank, B.rec);
    ++launches;
  }
  return launches;
}

}  // namespace orb
