// C ABI of liborb_b200 (include/orb.h): handle, scratch ownership, argument
// checks, launches.  No arithmetic of the method lives here.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>
#include <vector>

#include "orb_internal.h"

using namespace orb;

// orb_deposit_host pipelines the markers in this many slices: the host->device copy of slice
// i+1 overlaps binning and deposition of slice i (the call is PCIe-bound: 48 B per marker)
constexpr int kHostSlices = 8;
// ... and deposits them in this many groups of slices: group k ends after slice kHostGroupEnd[k].
// A deposit over all tiles costs ~5.5 ms + 9.6 ms x (fraction of the markers) on cfg3, so few groups;
// measured e2e ms per call on cfg3: {6, 8} 71.5, {7, 8} 78.1, one deposit per slice 73.5,
// 16 slices {12, 16} 71.5, {13, 16} 74.6 (profiles/r02_experiments.md section 7).
constexpr int kHostGroups = 2;
constexpr int kHostGroupEnd[kHostGroups] = {6, kHostSlices};

struct orb_grid {
  orb_grid_desc_t desc;
  int64_t ncells;
  int64_t nnodes;

  // bound markers (borrowed) and binning state
  Markers bound;
  uint32_t bind_flags;
  bool have_bind;
  bool binned;

  // scratch (owned)
  BinScratch bin;
  int64_t bin_capacity;      // markers the rank/rec buffers can hold
  double* scoef;             // device table of the radial spline pieces (ns*16 doubles)
  double2* ring;             // device ring table
  double ring_alpha0;
  bool ring_valid;
  unsigned long long* d_points;
  cudaEvent_t dep_event;     // recorded after the last deposit (orb_last_points waits on it)
  bool dep_event_valid;
  int sms;                   // multiprocessors of the device

  // slack tile bins (ORB_MARKERS_TILE_BINS; orb_tilebin.cu), owned
  bool tile_mode;            // the current binding uses them
  TileBins tb;               // geometry of the bins; tb.count aliases tb_count
  uint32_t* tb_count;
  int64_t tb_count_capacity; // tiles
  double* tb_rec;
  int64_t tb_rec_capacity;   // records
  double* tb_movers;
  int64_t tb_mv_capacity;    // records
  uint32_t* tb_mv_count;
  unsigned long long* tb_counters;   // [0] movers of the last rebin, [1] movers left in place

  RingScratch ringdata;      // Larmor ring data (orb_ring_reserve; orb_cellowner.cu), owned

  // orb_deposit_host staging (owned)
  double* hbuf[6];
  int64_t hbuf_capacity;
  double* hgrid[2];
  cudaStream_t hstream[2];   // orb_deposit_host: [0] copies, [1] kernels
  cudaEvent_t hevent[kHostSlices];
  bool keep_counters;        // internal: next deposit adds to the point counters

  int64_t launches;
  char err[512];
};

namespace {

struct DeviceGuard {
  int prev;
  bool ok;
  explicit DeviceGuard(int dev) : prev(-1), ok(false) {
    if (cudaGetDevice(&prev) != cudaSuccess) { prev = -1; }
    ok = (cudaSetDevice(dev) == cudaSuccess);
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

int fail(orb_grid* g, int code, const char* what, cudaError_t ce = cudaSuccess) {
  if (g) {
    if (ce != cudaSuccess)
      snprintf(g->err, sizeof(g->err), "%s: %s (%s)", orb_strerror(code), what,
               cudaGetErrorString(ce));
    else
      snprintf(g->err, sizeof(g->err), "%s: %s", orb_strerror(code), what);
  }
  return code;
}

#define ORB_CUDA(g, call)                                           \
  do {                                                              \
    cudaError_t ce__ = (call);                                      \
    if (ce__ != cudaSuccess) {                                      \
      cudaGetLastError();                                           \
      return fail((g), ce__ == cudaErrorMemoryAllocation ? ORB_E_NOMEM : ORB_E_CUDA, #call, ce__); \
    }                                                               \
  } while (0)

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

Params make_params(const orb_grid* g, const orb_nl_policy_t* pol) {
  Params P;
  P.ns = g->desc.ns;
  P.nth = g->desc.ntheta;
  P.nph = g->desc.nphi;
  P.theta_map = g->desc.theta_map;
  P.eps = g->desc.a / g->desc.r0;
  P.b0 = g->desc.b0;
  P.inv_b0 = 1.0 / g->desc.b0;
  P.rho_star = g->desc.rho_star;
  P.q = g->desc.q;
  P.nth_scale = (double)g->desc.ntheta / kTwoPi;
  P.nph_scale = (double)g->desc.nphi / kTwoPi;
  P.adaptive = 0;
  P.n_fixed = 1;
  P.n_max = 1;
  P.rho_ref = 1.0;
  P.inv_rho_ref = 1.0;
  if (pol) {
    P.adaptive = pol->mode == ORB_NL_ADAPTIVE;
    P.n_fixed = pol->n_fixed;
    P.n_max = P.adaptive ? pol->n_max : pol->n_fixed;
    P.rho_ref = P.adaptive ? pol->rho_ref : 1.0;
    P.inv_rho_ref = 1.0 / P.rho_ref;
  }
  P.ring = g->ring;
  P.scoef = g->scoef;
  return P;
}

int check_policy(orb_grid* g, const orb_nl_policy_t* pol) {
  if (!pol) return fail(g, ORB_E_INVAL, "policy is NULL");
  if (pol->mode != ORB_NL_FIXED && pol->mode != ORB_NL_ADAPTIVE)
    return fail(g, ORB_E_INVAL, "policy.mode");
  if (pol->n_fixed < 1 || pol->n_fixed > ORB_MAX_NL)
    return fail(g, ORB_E_INVAL, "policy.n_fixed out of [1, ORB_MAX_NL]");
  if (pol->mode == ORB_NL_ADAPTIVE) {
    if (pol->n_max < pol->n_fixed || pol->n_max > ORB_MAX_NL)
      return fail(g, ORB_E_INVAL, "policy.n_max out of [n_fixed, ORB_MAX_NL]");
    if (!(pol->rho_ref > 0.0) || !isfinite(pol->rho_ref))
      return fail(g, ORB_E_INVAL, "policy.rho_ref must be > 0");
  }
  if (!isfinite(pol->alpha0)) return fail(g, ORB_E_INVAL, "policy.alpha0");
  return ORB_OK;
}

// (cos, sin)(alpha0 + 2 pi l / N) for N = 1..ORB_MAX_NL, l < N; entry at N(N-1)/2 + l.  Built by a
// one-block kernel on the caller's stream (no host synchronisation, capturable in a CUDA graph).
int upload_ring(orb_grid* g, double alpha0, cudaStream_t st) {
  if (g->ring_valid && g->ring_alpha0 == alpha0) return ORB_OK;
  int l = launch_ring_table(g->ring, alpha0, st);
  if (l < 0) return fail(g, ORB_E_CUDA, "ring table launch", cudaGetLastError());
  g->launches += l;
  g->ring_alpha0 = alpha0;
  g->ring_valid = true;
  return ORB_OK;
}

void free_bin(orb_grid* g) {
  cudaFree(g->bin.rank);
  cudaFree(g->bin.rec);
  g->bin.rank = nullptr;
  g->bin.rec = nullptr;
  g->bin_capacity = 0;
}

// marker-proportional scratch (rank + binned records); called from orb_markers_bind / orb_reserve
// only, so that orb_markers_bin and orb_deposit never allocate (cudaMalloc synchronises)
int ensure_bin_scratch(orb_grid* g, int64_t n) {
  if (n > g->bin_capacity) {
    free_bin(g);
    ORB_CUDA(g, cudaMalloc(&g->bin.rank, (size_t)n * sizeof(uint32_t)));
    if (cudaMalloc(&g->bin.rec, (size_t)n * kRecDoubles * sizeof(double)) != cudaSuccess) {
      cudaGetLastError();
      free_bin(g);
      return fail(g, ORB_E_NOMEM, "binned-record scratch");
    }
    g->bin_capacity = n;
  }
  return ORB_OK;
}

void free_ringdata(orb_grid* g) {
  cudaFree(g->ringdata.off);
  cudaFree(g->ringdata.cell_start);
  cudaFree(g->ringdata.block_sums);
  cudaFree(g->ringdata.ring);
  cudaFree(g->ringdata.sorted);
  memset(&g->ringdata, 0, sizeof(g->ringdata));
}

void free_tilebins(orb_grid* g) {
  cudaFree(g->tb_count);
  cudaFree(g->tb_rec);
  cudaFree(g->tb_movers);
  cudaFree(g->tb_mv_count);
  cudaFree(g->tb_counters);
  g->tb_count = nullptr;
  g->tb_rec = nullptr;
  g->tb_movers = nullptr;
  g->tb_mv_count = nullptr;
  g->tb_counters = nullptr;
  g->tb_count_capacity = g->tb_rec_capacity = g->tb_mv_capacity = 0;
}

// geometry and scratch of the slack tile bins for n markers (called from orb_markers_bind)
int ensure_tilebins(orb_grid* g, int64_t n) {
  TileBins T;
  T.tiles_i = (g->desc.ns + 7) / 8;
  T.tiles_j = (g->desc.ntheta + 15) / 16;
  const int64_t n_tiles = (int64_t)T.tiles_i * T.tiles_j * g->desc.nphi * kTileBinSubs;   // bins
  if (n_tiles >= ((int64_t)1 << 31)) return fail(g, ORB_E_INVAL, "too many tiles");
  T.n_tiles = (uint32_t)n_tiles;
  const int64_t mean = (n + n_tiles - 1) / n_tiles;
  int64_t cap = (mean + mean / 2 + 64 + 7) & ~(int64_t)7;   // occupied bins hold ~1.25 x the mean
  if (cap > 2048) cap = 2048;   // one warp compacts a bin with a 64-bit mask per lane
  if (mean + mean / 4 > cap)
    return fail(g, ORB_E_INVAL, "ORB_MARKERS_TILE_BINS: more than 1638 markers per bin (one radial row of a tile) on average");
  if (n_tiles * cap >= ((int64_t)1 << 32)) return fail(g, ORB_E_INVAL, "tile bins exceed 2^32 records");
  T.cap = (uint32_t)cap;
  T.count = nullptr;
  const int64_t mv = n / 2 + 1024;
  if (n_tiles > g->tb_count_capacity || n_tiles * cap > g->tb_rec_capacity || mv > g->tb_mv_capacity) {
    free_tilebins(g);
    if (cudaMalloc(&g->tb_count, (size_t)n_tiles * sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&g->tb_rec, (size_t)(n_tiles * cap) * kRecDoubles * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&g->tb_movers, (size_t)mv * kRecDoubles * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&g->tb_mv_count, sizeof(uint32_t)) != cudaSuccess ||
        cudaMalloc(&g->tb_counters, 2 * sizeof(unsigned long long)) != cudaSuccess ||
        cudaMemset(g->tb_counters, 0, 2 * sizeof(unsigned long long)) != cudaSuccess) {
      cudaGetLastError();
      free_tilebins(g);
      return fail(g, ORB_E_NOMEM, "slack tile bins");
    }
    g->tb_count_capacity = n_tiles;
    g->tb_rec_capacity = n_tiles * cap;
    g->tb_mv_capacity = mv;
  }
  T.count = g->tb_count;
  g->tb = T;
  return ORB_OK;
}

int do_bin(orb_grid* g, cudaStream_t st) {
  if (g->tile_mode) {
    Params P = make_params(g, nullptr);
    Markers M = g->bound;
    M.rec = nullptr;
    int l = launch_tilebin_build(P, M, g->tb, g->tb_count, g->tb_rec, st);
    if (l < 0) return fail(g, ORB_E_CUDA, "tile-bin build launch", cudaGetLastError());
    g->launches += l;
    ORB_CUDA(g, cudaGetLastError());
    g->binned = true;
    return ORB_OK;
  }
  const bool presorted = (g->bind_flags & ORB_MARKERS_SORTED) != 0;
  if (!presorted && g->bound.n > g->bin_capacity)
    return fail(g, ORB_E_STATE, "binning scratch missing (bind allocates it)");
  Params P = make_params(g, nullptr);
  Markers M = g->bound;
  M.rec = nullptr;
  int l = launch_bin(P, M, g->bin, presorted, st);
  if (l < 0) return fail(g, ORB_E_CUDA, "binning launch", cudaGetLastError());
  g->launches += l;
  ORB_CUDA(g, cudaGetLastError());
  g->binned = true;
  return ORB_OK;
}

// host wait for the last deposit enqueued on this handle
cudaError_t wait_deposit(orb_grid* g) {
  return g->dep_event_valid ? cudaEventSynchronize(g->dep_event) : cudaDeviceSynchronize();
}

}  // namespace

extern "C" {

int orb_version(void) { return ORB_VERSION; }

const char* orb_strerror(int code) {
  switch (code) {
    case ORB_OK: return "ok";
    case ORB_E_INVAL: return "invalid argument";
    case ORB_E_STATE: return "invalid call order";
    case ORB_E_NOMEM: return "out of device memory";
    case ORB_E_CUDA: return "CUDA error";
    default: return "unknown status";
  }
}

const char* orb_last_error(const orb_grid_t* g) { return g ? g->err : ""; }

int orb_grid_create(const orb_grid_desc_t* d, orb_grid_t** out) {
  if (!d || !out) return ORB_E_INVAL;
  if (d->ns < 4 || d->ntheta < 4 || d->nphi < 4) return ORB_E_INVAL;
  if (!(d->r0 > 0.0) || !(d->a > 0.0) || !(d->a < d->r0) || !(d->b0 > 0.0)) return ORB_E_INVAL;
  if (!(d->rho_star >= 0.0) || !isfinite(d->rho_star) || !isfinite(d->q)) return ORB_E_INVAL;
  if (d->theta_map != 0 && d->theta_map != 1) return ORB_E_INVAL;
  const int64_t ncells = (int64_t)d->ns * d->ntheta * d->nphi;
  const int64_t nnodes = (int64_t)(d->ns + 3) * d->ntheta * d->nphi;
  if (ncells >= (int64_t)1 << 31) return ORB_E_INVAL;
  // launch-grid limits of the tile kernels (65535 blocks along y and z)
  if (d->nphi > 65535 || (d->ns + 7) / 8 > 65535) return ORB_E_INVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || d->device < 0 || d->device >= ndev) {
    cudaGetLastError();
    return ORB_E_CUDA;
  }
  DeviceGuard dg(d->device);
  if (!dg.ok) return ORB_E_CUDA;
  orb_grid* g = new (std::nothrow) orb_grid();
  if (!g) return ORB_E_NOMEM;
  memset(g, 0, sizeof(*g));
  g->desc = *d;
  g->ncells = ncells;
  g->nnodes = nnodes;
  g->bin.ncells = ncells;
  const int total = ORB_MAX_NL * (ORB_MAX_NL + 1) / 2;
  std::vector<double> table;
  build_radial_table(d->ns, table);
  if (cudaMalloc(&g->scoef, table.size() * sizeof(double)) != cudaSuccess ||
      cudaMemcpy(g->scoef, table.data(), table.size() * sizeof(double), cudaMemcpyHostToDevice) !=
          cudaSuccess ||
      cudaMalloc(&g->ring, total * sizeof(double2)) != cudaSuccess ||
      cudaMalloc(&g->d_points, kCounters * sizeof(unsigned long long)) != cudaSuccess ||
      cudaMemset(g->d_points, 0, kCounters * sizeof(unsigned long long)) != cudaSuccess ||
      cudaMalloc(&g->bin.cell_start, (size_t)(ncells + 1) * sizeof(uint32_t)) != cudaSuccess ||
      cudaMalloc(&g->bin.block_sums, (size_t)((ncells + 4095) / 4096 + 1) * sizeof(uint32_t)) !=
          cudaSuccess ||
      cudaEventCreateWithFlags(&g->dep_event, cudaEventDisableTiming) != cudaSuccess ||
      cudaDeviceGetAttribute(&g->sms, cudaDevAttrMultiProcessorCount, d->device) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(g->scoef);
    cudaFree(g->ring);
    cudaFree(g->d_points);
    cudaFree(g->bin.cell_start);
    cudaFree(g->bin.block_sums);
    if (g->dep_event) cudaEventDestroy(g->dep_event);
    delete g;
    return ORB_E_CUDA;
  }
  *out = g;
  return ORB_OK;
}

int orb_grid_destroy(orb_grid_t* g) {
  if (!g) return ORB_OK;
  DeviceGuard dg(g->desc.device);
  cudaDeviceSynchronize();
  free_bin(g);
  free_tilebins(g);
  free_ringdata(g);
  cudaFree(g->bin.cell_start);
  cudaFree(g->bin.block_sums);
  cudaFree(g->scoef);
  cudaFree(g->ring);
  cudaFree(g->d_points);
  for (int i = 0; i < 6; ++i) cudaFree(g->hbuf[i]);
  cudaFree(g->hgrid[0]);
  cudaFree(g->hgrid[1]);
  for (int i = 0; i < 2; ++i)
    if (g->hstream[i]) cudaStreamDestroy(g->hstream[i]);
  for (int i = 0; i < kHostSlices; ++i)
    if (g->hevent[i]) cudaEventDestroy(g->hevent[i]);
  if (g->dep_event) cudaEventDestroy(g->dep_event);
  cudaGetLastError();
  delete g;
  return ORB_OK;
}

int orb_spline_table_radial(int32_t ns, double* out) {
  if (ns < 4 || !out) return ORB_E_INVAL;
  std::vector<double> table;
  build_radial_table(ns, table);
  memcpy(out, table.data(), table.size() * sizeof(double));
  return ORB_OK;
}

int orb_grid_shape(const orb_grid_t* g, int64_t dims[3]) {
  if (!g || !dims) return ORB_E_INVAL;
  dims[0] = g->desc.ns + 3;
  dims[1] = g->desc.ntheta;
  dims[2] = g->desc.nphi;
  return ORB_OK;
}

int orb_markers_bind(orb_grid_t* g, int64_t n, const double* s, const double* theta,
                     const double* phi, const double* vpar, const double* mu, const double* w,
                     uint32_t flags) {
  if (!g) return ORB_E_INVAL;
  if (n < 0) return fail(g, ORB_E_INVAL, "n < 0");
  if (n >= ((int64_t)1 << 32) - 1) return fail(g, ORB_E_INVAL, "n too large");
  if (flags & ~(ORB_MARKERS_SORTED | ORB_MARKERS_TILE_BINS)) return fail(g, ORB_E_INVAL, "unknown bind flag");
  if ((flags & ORB_MARKERS_SORTED) && (flags & ORB_MARKERS_TILE_BINS))
    return fail(g, ORB_E_INVAL, "ORB_MARKERS_SORTED and ORB_MARKERS_TILE_BINS exclude each other");
  if (n > 0 && (!s || !theta || !phi || !mu || !w)) return fail(g, ORB_E_INVAL, "NULL marker array");
  if (!aligned16(s) || !aligned16(theta) || !aligned16(phi) || !aligned16(vpar) ||
      !aligned16(mu) || !aligned16(w))
    return fail(g, ORB_E_INVAL, "marker arrays must be 16-byte aligned");
  if (flags & ORB_MARKERS_TILE_BINS) {
    DeviceGuard dg(g->desc.device);
    if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
    int rc = ensure_tilebins(g, n);
    if (rc != ORB_OK) return rc;
  } else if (!(flags & ORB_MARKERS_SORTED) && n > g->bin_capacity) {
    DeviceGuard dg(g->desc.device);
    if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
    int rc = ensure_bin_scratch(g, n);
    if (rc != ORB_OK) return rc;
  }
  g->tile_mode = (flags & ORB_MARKERS_TILE_BINS) != 0;
  g->bound.s = s;
  g->bound.th = theta;
  g->bound.ph = phi;
  g->bound.vpar = vpar;
  g->bound.mu = mu;
  g->bound.w = w;
  g->bound.rec = nullptr;
  g->bound.n = n;
  g->bind_flags = flags;
  g->have_bind = true;
  g->binned = false;
  g->err[0] = 0;
  return ORB_OK;
}

int orb_reserve(orb_grid_t* g, int64_t n) {
  if (!g) return ORB_E_INVAL;
  if (n < 0 || n >= ((int64_t)1 << 32) - 1) return fail(g, ORB_E_INVAL, "n out of range");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  return ensure_bin_scratch(g, n);
}

int orb_ring_reserve(orb_grid_t* g, int64_t n_markers, int64_t n_points) {
  if (!g) return ORB_E_INVAL;
  if (n_markers < 0 || n_points < 0 || n_markers >= ((int64_t)1 << 32) - 1 ||
      n_points >= ((int64_t)1 << 32) - 1)
    return fail(g, ORB_E_INVAL, "orb_ring_reserve: counts out of range");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  if (n_markers == 0 && n_points == 0) {   // release the scratch
    free_ringdata(g);
    return ORB_OK;
  }
  if (n_markers <= g->ringdata.markers && n_points <= g->ringdata.capacity) return ORB_OK;
  free_ringdata(g);
  RingScratch R;
  memset(&R, 0, sizeof(R));
  const int64_t widest = n_markers > g->ncells ? n_markers : g->ncells;
  const size_t pts = (size_t)(n_points > 0 ? n_points : 1) * 6 * sizeof(double);
  if (cudaMalloc(&R.off, (size_t)(n_markers + 1) * sizeof(uint32_t)) != cudaSuccess ||
      cudaMalloc(&R.cell_start, (size_t)(g->ncells + 1) * sizeof(uint32_t)) != cudaSuccess ||
      cudaMalloc(&R.block_sums, (size_t)(widest / 4096 + 2) * sizeof(uint32_t)) != cudaSuccess ||
      cudaMalloc(&R.ring, pts) != cudaSuccess || cudaMalloc(&R.sorted, pts) != cudaSuccess) {
    cudaGetLastError();
    g->ringdata = R;
    free_ringdata(g);
    return fail(g, ORB_E_NOMEM, "Larmor ring data");
  }
  R.capacity = n_points;
  R.markers = n_markers;
  g->ringdata = R;
  return ORB_OK;
}

int orb_markers_bin(orb_grid_t* g, void* stream) {
  if (!g) return ORB_E_INVAL;
  if (!g->have_bind) return fail(g, ORB_E_STATE, "orb_markers_bin before orb_markers_bind");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  return do_bin(g, static_cast<cudaStream_t>(stream));
}

int orb_deposit(orb_grid_t* g, double* rho, double* jpar, const orb_nl_policy_t* pol,
                void* stream) {
  if (!g) return ORB_E_INVAL;
  if (!rho) return fail(g, ORB_E_INVAL, "rho is NULL");
  if (!aligned16(rho) || !aligned16(jpar)) return fail(g, ORB_E_INVAL, "grids must be 16-byte aligned");
  int rc = check_policy(g, pol);
  if (rc != ORB_OK) return rc;
  if (!g->have_bind) return fail(g, ORB_E_STATE, "orb_deposit before orb_markers_bind");
  if (jpar && !g->bound.vpar && g->bound.n > 0)
    return fail(g, ORB_E_INVAL, "jpar requested but markers were bound without vpar");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  cudaStream_t st = static_cast<cudaStream_t>(stream);

  rc = upload_ring(g, pol->alpha0, st);
  if (rc != ORB_OK) return rc;
  const bool ring_algo = (pol->flags & ORB_DEPOSIT_ALGO_RING_DATA) != 0;
  if (ring_algo && (!g->ringdata.off || g->bound.n > g->ringdata.markers))
    return fail(g, ORB_E_STATE, "ORB_DEPOSIT_ALGO_RING_DATA needs orb_ring_reserve for the bound markers");
  const bool atomic_algo = (pol->flags & ORB_DEPOSIT_ALGO_ATOMIC) != 0;
  const bool tile_v4 = (pol->flags & ORB_DEPOSIT_ALGO_TILE_V4) != 0;
  const bool tile_v5 = (pol->flags & ORB_DEPOSIT_ALGO_TILE_WS) != 0;
  const bool no_bin = (pol->flags & ORB_DEPOSIT_NO_BIN) != 0;
  if (!no_bin && !atomic_algo && !ring_algo && !g->binned) {
    rc = do_bin(g, st);
    if (rc != ORB_OK) return rc;
  }
  if (pol->flags & ORB_DEPOSIT_ZERO_FIRST) {
    ORB_CUDA(g, cudaMemsetAsync(rho, 0, (size_t)g->nnodes * sizeof(double), st));
    if (jpar) ORB_CUDA(g, cudaMemsetAsync(jpar, 0, (size_t)g->nnodes * sizeof(double), st));
  }
  if (!g->keep_counters)
    ORB_CUDA(g, cudaMemsetAsync(g->d_points, 0, kCounters * sizeof(unsigned long long), st));

  Params P = make_params(g, pol);
  Markers M = g->bound;
  const bool use_binned = g->binned && !no_bin;
  const bool presorted = (g->bind_flags & ORB_MARKERS_SORTED) != 0;
  if (use_binned && !presorted) M.rec = g->tile_mode ? g->tb_rec : g->bin.rec;
  TileBins TB = g->tb;
  if (!g->tile_mode) TB.count = nullptr;
  int l;
  if (ring_algo) {
    M.rec = nullptr;   // the Larmor ring data are built from the bound arrays; no marker binning
    l = launch_deposit_ringdata(P, M, g->ringdata, rho, jpar, g->d_points, st);
  } else if (atomic_algo || !use_binned) {
    l = launch_deposit_atomic(P, M, rho, jpar, g->d_points, st);
  } else if (tile_v4 || (!tile_v5 && (P.adaptive || P.n_fixed > 4))) {
    // N_L > 4 or adaptive: the one-block-per-tile kernel, whose point slots are filled by a
    // prefix sum over the markers, keeps its lanes busier than the persistent kernels'
    // unit hand-over (measured: cfg2 5.5 vs 7.5 ms, cfg4 70 vs 111 ms)
    l = launch_deposit_tile(P, M, g->bin.cell_start, TB, rho, jpar, g->d_points, st);
  } else if (tile_v5 || P.n_fixed == 1) {
    // N_L = 1 (drift-kinetic species): one point per marker slot; the 256-marker chunks of the first
    // persistent kernel are faster there (single_node electrons: 2.65 vs 3.19 ms)
    l = launch_deposit_ws(P, M, g->bin.cell_start, TB, rho, jpar, g->d_points, g->sms, st);
  } else {
    // fixed N_L = 2..4: the persistent kernel with whole-tile-sized chunks (cfg3 14.4 vs 16.4 ms,
    // cfg1 2.9 vs 3.6 ms against ORB_DEPOSIT_ALGO_TILE_WS)
    l = launch_deposit_ws2(P, M, g->bin.cell_start, TB, rho, jpar, g->d_points, g->sms, st);
  }
  if (l < 0) return fail(g, ORB_E_CUDA, "deposit launch", cudaGetLastError());
  g->launches += l;
  ORB_CUDA(g, cudaGetLastError());
  // orb_last_points waits on this event; an event cannot be waited on from the host while its
  // stream is being captured into a graph, so then the device-wide wait is used instead
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) cudaGetLastError();
  if (cap == cudaStreamCaptureStatusNone) {
    ORB_CUDA(g, cudaEventRecord(g->dep_event, st));
    g->dep_event_valid = true;
  } else {
    g->dep_event_valid = false;
  }
  return ORB_OK;
}

int orb_gather(orb_grid_t* g, int32_t n_fields, const double* const* fields, double* const* out,
               const orb_nl_policy_t* pol, void* stream) {
  if (!g) return ORB_E_INVAL;
  if (n_fields < 1 || n_fields > ORB_MAX_FIELDS) return fail(g, ORB_E_INVAL, "n_fields out of [1, ORB_MAX_FIELDS]");
  if (!fields || !out) return fail(g, ORB_E_INVAL, "fields / out is NULL");
  int rc = check_policy(g, pol);
  if (rc != ORB_OK) return rc;
  if (!g->have_bind) return fail(g, ORB_E_STATE, "orb_gather before orb_markers_bind");
  for (int f = 0; f < n_fields; ++f) {
    if (!fields[f] || (!out[f] && g->bound.n > 0)) return fail(g, ORB_E_INVAL, "NULL field / out pointer");
    if (!aligned16(fields[f])) return fail(g, ORB_E_INVAL, "fields must be 16-byte aligned");
  }
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  rc = upload_ring(g, pol->alpha0, st);
  if (rc != ORB_OK) return rc;
  const bool direct = (pol->flags & (ORB_DEPOSIT_NO_BIN | ORB_DEPOSIT_ALGO_ATOMIC)) != 0;
  if (!direct && !g->binned) {
    rc = do_bin(g, st);
    if (rc != ORB_OK) return rc;
  }
  ORB_CUDA(g, cudaMemsetAsync(g->d_points, 0, kCounters * sizeof(unsigned long long), st));
  Params P = make_params(g, pol);
  Markers M = g->bound;
  const bool presorted = (g->bind_flags & ORB_MARKERS_SORTED) != 0;
  if (!direct && !presorted) M.rec = g->tile_mode ? g->tb_rec : g->bin.rec;
  TileBins TB = g->tb;
  if (!g->tile_mode) TB.count = nullptr;
  int l = launch_gather(P, M, g->bin.cell_start, TB, n_fields, fields, out, g->d_points, !direct, st);
  if (l < 0) return fail(g, ORB_E_CUDA, "gather launch", cudaGetLastError());
  g->launches += l;
  ORB_CUDA(g, cudaGetLastError());
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) cudaGetLastError();
  if (cap == cudaStreamCaptureStatusNone) {
    ORB_CUDA(g, cudaEventRecord(g->dep_event, st));
    g->dep_event_valid = true;
  } else {
    g->dep_event_valid = false;
  }
  return ORB_OK;
}

int orb_grid_zero(orb_grid_t* g, double* rho, double* jpar, void* stream) {
  if (!g) return ORB_E_INVAL;
  if (!rho) return fail(g, ORB_E_INVAL, "rho is NULL");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  ORB_CUDA(g, cudaMemsetAsync(rho, 0, (size_t)g->nnodes * sizeof(double), st));
  if (jpar) ORB_CUDA(g, cudaMemsetAsync(jpar, 0, (size_t)g->nnodes * sizeof(double), st));
  return ORB_OK;
}

int orb_last_points(orb_grid_t* g, int64_t* n_points) {
  if (!g || !n_points) return ORB_E_INVAL;
  DeviceGuard dg(g->desc.device);
  unsigned long long v = 0;
  ORB_CUDA(g, wait_deposit(g));
  ORB_CUDA(g, cudaMemcpy(&v, g->d_points, sizeof(v), cudaMemcpyDeviceToHost));
  *n_points = (int64_t)v;
  return ORB_OK;
}

int orb_last_fallback_points(orb_grid_t* g, int64_t* n_points) {
  if (!g || !n_points) return ORB_E_INVAL;
  DeviceGuard dg(g->desc.device);
  unsigned long long v = 0;
  ORB_CUDA(g, wait_deposit(g));
  ORB_CUDA(g, cudaMemcpy(&v, g->d_points + 1, sizeof(v), cudaMemcpyDeviceToHost));
  *n_points = (int64_t)v;
  return ORB_OK;
}

int orb_debug_counters(orb_grid_t* g, uint64_t out[16]) {
  if (!g || !out) return ORB_E_INVAL;
  DeviceGuard dg(g->desc.device);
  ORB_CUDA(g, wait_deposit(g));
  ORB_CUDA(g, cudaMemcpy(out, g->d_points, kCounters * sizeof(unsigned long long),
                         cudaMemcpyDeviceToHost));
  return ORB_OK;
}

int orb_debug_binned(orb_grid_t* g, double* rec_host, uint32_t* cell_start_host,
                     int32_t* rec_doubles) {
  if (!g || !cell_start_host || !rec_doubles) return ORB_E_INVAL;
  if (!g->have_bind || !g->binned || g->tile_mode)
    return fail(g, ORB_E_STATE, "orb_debug_binned needs markers binned in the dense layout");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  ORB_CUDA(g, cudaDeviceSynchronize());
  ORB_CUDA(g, cudaMemcpy(cell_start_host, g->bin.cell_start,
                         (size_t)(g->ncells + 1) * sizeof(uint32_t), cudaMemcpyDeviceToHost));
  const bool presorted = (g->bind_flags & ORB_MARKERS_SORTED) != 0;
  *rec_doubles = presorted ? 0 : kRecDoubles;
  if (!presorted && rec_host && g->bound.n > 0)
    ORB_CUDA(g, cudaMemcpy(rec_host, g->bin.rec, (size_t)g->bound.n * kRecDoubles * sizeof(double),
                           cudaMemcpyDeviceToHost));
  return ORB_OK;
}

int orb_markers_refresh(orb_grid_t* g, void* stream) {
  if (!g) return ORB_E_INVAL;
  if (!g->have_bind || !g->tile_mode || !g->binned)
    return fail(g, ORB_E_STATE, "orb_markers_refresh needs binned ORB_MARKERS_TILE_BINS markers");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  Markers M = g->bound;
  M.rec = nullptr;
  int l = launch_tilebin_refresh(M, g->tb, g->tb_count, g->tb_rec, static_cast<cudaStream_t>(stream));
  if (l < 0) return fail(g, ORB_E_CUDA, "refresh launch", cudaGetLastError());
  g->launches += l;
  ORB_CUDA(g, cudaGetLastError());
  return ORB_OK;
}

int orb_markers_rebin(orb_grid_t* g, void* stream) {
  if (!g) return ORB_E_INVAL;
  if (!g->have_bind || !g->tile_mode || !g->binned)
    return fail(g, ORB_E_STATE, "orb_markers_rebin needs binned ORB_MARKERS_TILE_BINS markers");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  ORB_CUDA(g, cudaMemsetAsync(g->tb_counters, 0, 2 * sizeof(unsigned long long), st));
  Params P = make_params(g, nullptr);
  int l = launch_tilebin_rebin(P, g->tb, g->tb_count, g->tb_rec, g->tb_movers, (uint32_t)g->tb_mv_capacity,
                               g->tb_mv_count, g->tb_counters, st);
  if (l < 0) return fail(g, ORB_E_CUDA, "rebin launch", cudaGetLastError());
  g->launches += l;
  ORB_CUDA(g, cudaGetLastError());
  return ORB_OK;
}

int orb_last_moved(orb_grid_t* g, int64_t* n_moved, int64_t* n_left_in_place) {
  if (!g || !n_moved) return ORB_E_INVAL;
  if (!g->tile_mode || !g->tb_counters) return fail(g, ORB_E_STATE, "no slack tile bins");
  DeviceGuard dg(g->desc.device);
  unsigned long long v[2] = {0, 0};
  ORB_CUDA(g, cudaDeviceSynchronize());
  ORB_CUDA(g, cudaMemcpy(v, g->tb_counters, sizeof(v), cudaMemcpyDeviceToHost));
  *n_moved = (int64_t)v[0];
  if (n_left_in_place) *n_left_in_place = (int64_t)v[1];
  return ORB_OK;
}

int orb_markers_layout(const orb_grid_t* g, orb_marker_layout_t* out) {
  if (!g || !out) return ORB_E_INVAL;
  if (!g->have_bind || !g->tile_mode) return ORB_E_STATE;
  out->records = g->tb_rec;
  out->count = g->tb_count;
  out->record_doubles = kRecDoubles;
  out->capacity = g->tb.cap;
  out->n_bins = g->tb.n_tiles;
  out->tiles_s = g->tb.tiles_i;
  out->tiles_theta = g->tb.tiles_j;
  return ORB_OK;
}

int orb_debug_tilebins(orb_grid_t* g, double* rec_host, uint32_t* count_host) {
  if (!g || !rec_host || !count_host) return ORB_E_INVAL;
  if (!g->have_bind || !g->tile_mode || !g->binned) return fail(g, ORB_E_STATE, "no binned slack tile bins");
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  ORB_CUDA(g, cudaDeviceSynchronize());
  ORB_CUDA(g, cudaMemcpy(count_host, g->tb_count, (size_t)g->tb.n_tiles * sizeof(uint32_t),
                         cudaMemcpyDeviceToHost));
  int64_t off = 0;
  for (uint32_t t = 0; t < g->tb.n_tiles; ++t) {
    const uint32_t c = count_host[t] < g->tb.cap ? count_host[t] : g->tb.cap;
    count_host[t] = c;
    if (c == 0) continue;
    if (off + c > g->bound.n) return fail(g, ORB_E_STATE, "tile counts exceed the bound marker count");
    ORB_CUDA(g, cudaMemcpy(rec_host + off * kRecDoubles, g->tb_rec + (size_t)t * g->tb.cap * kRecDoubles,
                           (size_t)c * kRecDoubles * sizeof(double), cudaMemcpyDeviceToHost));
    off += c;
  }
  return ORB_OK;
}

int orb_launch_count(const orb_grid_t* g, int64_t* n) {
  if (!g || !n) return ORB_E_INVAL;
  *n = g->launches;
  return ORB_OK;
}

int orb_deposit_host(orb_grid_t* g, int64_t n, const double* s, const double* theta,
                     const double* phi, const double* vpar, const double* mu, const double* w,
                     double* rho_host, double* jpar_host, const orb_nl_policy_t* pol,
                     int64_t* n_points, int64_t* h2d_bytes, int64_t* d2h_bytes) {
  if (!g) return ORB_E_INVAL;
  if (n < 0 || !rho_host) return fail(g, ORB_E_INVAL, "n < 0 or rho_host NULL");
  if (n > 0 && (!s || !theta || !phi || !mu || !w)) return fail(g, ORB_E_INVAL, "NULL marker array");
  if (jpar_host && !vpar && n > 0) return fail(g, ORB_E_INVAL, "jpar_host needs vpar");
  int rc = check_policy(g, pol);
  if (rc != ORB_OK) return rc;
  DeviceGuard dg(g->desc.device);
  if (!dg.ok) return fail(g, ORB_E_CUDA, "cudaSetDevice");
  if (n > g->hbuf_capacity) {
    for (int i = 0; i < 6; ++i) {
      cudaFree(g->hbuf[i]);
      g->hbuf[i] = nullptr;
    }
    g->hbuf_capacity = 0;
    for (int i = 0; i < 6; ++i) ORB_CUDA(g, cudaMalloc(&g->hbuf[i], (size_t)n * sizeof(double)));
    g->hbuf_capacity = n;
  }
  for (int i = 0; i < 2; ++i)
    if (!g->hgrid[i]) ORB_CUDA(g, cudaMalloc(&g->hgrid[i], (size_t)g->nnodes * sizeof(double)));
  for (int i = 0; i < 2; ++i)
    if (!g->hstream[i]) ORB_CUDA(g, cudaStreamCreateWithFlags(&g->hstream[i], cudaStreamNonBlocking));
  for (int i = 0; i < kHostSlices; ++i)
    if (!g->hevent[i]) ORB_CUDA(g, cudaEventCreateWithFlags(&g->hevent[i], cudaEventDisableTiming));
  const double* src[6] = {s, theta, phi, vpar, mu, w};
  int64_t up = 0, down = 0;
  cudaStream_t s_copy = g->hstream[0], st = g->hstream[1];
  double* rho_d = g->hgrid[0];
  double* jpar_d = jpar_host ? g->hgrid[1] : nullptr;
  // slices of even length keep every slice pointer 16-byte aligned
  const int n_slices = n >= ((int64_t)1 << 22) ? kHostSlices : 1;
  const int64_t per = ((n + n_slices - 1) / n_slices + 1) & ~(int64_t)1;
  if (n == 0) {
    rc = orb_grid_zero(g, rho_d, jpar_d, st);
    if (rc != ORB_OK) return rc;
    ORB_CUDA(g, cudaMemsetAsync(g->d_points, 0, kCounters * sizeof(unsigned long long), st));
  }
  // The whole device copy is bound once with slack tile bins sized for all n markers.  Each slice
  // is APPENDED to the bins as soon as its copy has landed (the one-pass build claims bin slots
  // with atomics, so it does not care in how many launches the markers come); the deposit kernel
  // runs once per GROUP of slices, so a tile is zeroed, walked and flushed kHostGroups times per
  // call, not once per slice.  The first group's deposit overlaps the copies of the last slices.
  // (The algorithms that read the bound arrays themselves — ORB_DEPOSIT_NO_BIN, _ALGO_ATOMIC,
  // _ALGO_RING_DATA — have no per-tile cost and are run slice by slice.)
  const bool by_slice =
      (pol->flags & (ORB_DEPOSIT_NO_BIN | ORB_DEPOSIT_ALGO_ATOMIC | ORB_DEPOSIT_ALGO_RING_DATA)) != 0;
  if (n > 0 && !by_slice) {
    rc = orb_markers_bind(g, n, g->hbuf[0], g->hbuf[1], g->hbuf[2], vpar ? g->hbuf[3] : nullptr,
                          g->hbuf[4], g->hbuf[5], ORB_MARKERS_TILE_BINS);
    if (rc != ORB_OK) return rc;
  }
  const Params Pb = make_params(g, nullptr);
  bool first_of_group = true, first_group = true;
  for (int i = 0; i < n_slices && n > 0; ++i) {
    const int64_t off = i * per;
    const int64_t len = (off + per <= n ? per : n - off);
    if (len <= 0) break;
    for (int f = 0; f < 6; ++f) {
      if (!src[f]) continue;
      ORB_CUDA(g, cudaMemcpyAsync(g->hbuf[f] + off, src[f] + off, (size_t)len * sizeof(double),
                                  cudaMemcpyHostToDevice, s_copy));
      up += len * (int64_t)sizeof(double);
    }
    ORB_CUDA(g, cudaEventRecord(g->hevent[i], s_copy));
    ORB_CUDA(g, cudaStreamWaitEvent(st, g->hevent[i], 0));
    if (by_slice) {
      rc = orb_markers_bind(g, len, g->hbuf[0] + off, g->hbuf[1] + off, g->hbuf[2] + off,
                            vpar ? g->hbuf[3] + off : nullptr, g->hbuf[4] + off, g->hbuf[5] + off, 0);
      if (rc != ORB_OK) return rc;
      orb_nl_policy_t p2 = *pol;
      if (i == 0) p2.flags |= ORB_DEPOSIT_ZERO_FIRST; else p2.flags &= ~ORB_DEPOSIT_ZERO_FIRST;
      g->keep_counters = i > 0;
      rc = orb_deposit(g, rho_d, jpar_d, &p2, st);
      g->keep_counters = false;
      if (rc != ORB_OK) return rc;
      continue;
    }
    Markers M = g->bound;
    M.s += off;
    M.th += off;
    M.ph += off;
    if (M.vpar) M.vpar += off;
    M.mu += off;
    M.w += off;
    M.rec = nullptr;
    M.n = len;
    int l = launch_tilebin_build(Pb, M, g->tb, g->tb_count, g->tb_rec, st, off, !first_of_group);
    if (l < 0) return fail(g, ORB_E_CUDA, "tile-bin build launch", cudaGetLastError());
    g->launches += l;
    first_of_group = false;
    const bool last = off + len >= n;
    bool group_end = last;
    for (int k = 0; k < kHostGroups; ++k) group_end = group_end || (i + 1 == kHostGroupEnd[k]);
    if (!group_end) continue;
    orb_nl_policy_t p2 = *pol;
    if (first_group) p2.flags |= ORB_DEPOSIT_ZERO_FIRST; else p2.flags &= ~ORB_DEPOSIT_ZERO_FIRST;
    g->keep_counters = !first_group;
    g->binned = true;          // the bins hold exactly this group's markers
    rc = orb_deposit(g, rho_d, jpar_d, &p2, st);
    g->keep_counters = false;
    g->binned = false;
    if (rc != ORB_OK) return rc;
    first_group = false;
    first_of_group = true;
  }
  ORB_CUDA(g, cudaMemcpyAsync(rho_host, rho_d, (size_t)g->nnodes * sizeof(double),
                              cudaMemcpyDeviceToHost, st));
  down += g->nnodes * (int64_t)sizeof(double);
  if (jpar_host) {
    ORB_CUDA(g, cudaMemcpyAsync(jpar_host, jpar_d, (size_t)g->nnodes * sizeof(double),
                                cudaMemcpyDeviceToHost, st));
    down += g->nnodes * (int64_t)sizeof(double);
  }
  ORB_CUDA(g, cudaStreamSynchronize(st));
  // the handle stays bound to the whole device copy, not binned (the bins hold the last group)
  if (n == 0 || by_slice) {
    rc = orb_markers_bind(g, n, g->hbuf[0], g->hbuf[1], g->hbuf[2], vpar ? g->hbuf[3] : nullptr,
                          g->hbuf[4], g->hbuf[5], 0);
    if (rc != ORB_OK) return rc;
  }
  if (n_points) {
    unsigned long long v = 0;
    ORB_CUDA(g, cudaMemcpy(&v, g->d_points, sizeof(v), cudaMemcpyDeviceToHost));
    *n_points = (int64_t)v;
  }
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = down;
  return ORB_OK;
}

}  // extern "C"
