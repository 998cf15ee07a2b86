// Internal declarations shared by the translation units of liborb_b200.
// Not part of the public ABI (see include/orb.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "orb.h"

namespace orb {

constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr int kCounters = 16;    // device counters: [0] Larmor points, [1] direct-path points, [2..] debug
// binned marker record: s, theta*, phi, vpar, mu, w, the marker's index in bound order (an
// integer bit pattern) + 1 double of padding.  64 bytes = two whole
// 32-byte sectors, so the random-order scatter of the counting sort never leaves a partially
// written sector for DRAM to read back (48-byte records cost 6.6 GB of fill reads on cfg3).
constexpr int kRecDoubles = 8;

// Everything a kernel needs to know about grid, geometry, species and N_L policy.
// Passed by value as a kernel parameter.
struct Params {
  int ns, nth, nph;      // cells
  int theta_map;
  double eps;            // a / r0
  double b0, inv_b0;
  double rho_star;
  double q;
  double nth_scale;      // ntheta / 2pi
  double nph_scale;      // nphi / 2pi
  // N_L policy
  int adaptive;
  int n_fixed;           // N_L, or n_min when adaptive
  int n_max;
  double rho_ref, inv_rho_ref;
  // ring table: entry (N, l) at N*(N-1)/2 + l holds (cos, sin)(alpha0 + 2 pi l / N), N = 1..ORB_MAX_NL
  const double2* ring;
  // radial spline pieces: scoef[(c*4 + a)*4 + d] = coefficient of t^d of basis c+a on cell c
  // (orb_spline_table.cu)
  const double* scoef;
};

// Bound markers: either the caller's SoA arrays (in bound order) or the library's
// binned array-of-records scratch (rec != nullptr), 6 doubles per marker.
struct Markers {
  const double* s;
  const double* th;
  const double* ph;
  const double* vpar;   // may be nullptr
  const double* mu;
  const double* w;
  const double* rec;    // binned records, or nullptr
  int64_t n;
};

// Slack tile bins (orb_tilebin.cu, NEXT-2): tile t = (k * tiles_i + ti) * tiles_j + tj is cut into
// kTileBinSubs bins of 8 / kTileBinSubs radial rows; bin b = t * kTileBinSubs + sub owns the records
// [b * cap, b * cap + min(count[b], cap)) of Markers::rec.  count == nullptr: the dense cell-sorted
// layout of orb_bin.cu (per-cell offsets) is in use instead.
constexpr int kTileBinSubs = 8;
struct TileBins {
  const uint32_t* count;
  uint32_t cap, n_tiles;   // n_tiles: number of BINS (tiles * kTileBinSubs)
  int tiles_i, tiles_j;
};

// ---- kernels' host-side launchers (each returns the number of kernels it launched, <0 on error)
int launch_deposit_atomic(const Params& P, const Markers& M, double* rho, double* jpar,
                          unsigned long long* d_points, cudaStream_t st);

struct BinScratch {
  uint32_t* rank;        // n
  uint32_t* cell_start;  // ncells + 1 (counts during pass 1, exclusive offsets afterwards)
  uint32_t* block_sums;  // scan scratch
  double* rec;           // n * kRecDoubles
  int64_t ncells;
};
int launch_bin(const Params& P, const Markers& M, const BinScratch& B, bool presorted,
               cudaStream_t st);

int launch_deposit_tile(const Params& P, const Markers& M, const uint32_t* cell_start,
                        const TileBins& TB, double* rho, double* jpar, unsigned long long* d_points,
                        cudaStream_t st);

// v5: one persistent, warp-specialised block per SM (orb_deposit_ws.cu); sms = multiprocessors
int launch_deposit_ws(const Params& P, const Markers& M, const uint32_t* cell_start,
                      const TileBins& TB, double* rho, double* jpar, unsigned long long* d_points,
                      int sms, cudaStream_t st);

// get fields + gyroaverage (orb_gather.cu); fields / out: host arrays of n_fields device pointers
int launch_gather(const Params& P, const Markers& M, const uint32_t* cell_start, const TileBins& TB,
                  int n_fields,
                  const double* const* fields, double* const* out, unsigned long long* d_points,
                  bool tiled, cudaStream_t st);

// slack tile bins: one-pass build, refresh of the records from the bound arrays, incremental rebin
// base = index of M's first marker in the bound arrays (kept in each record); append = add to the
// bins as they stand instead of emptying them first (orb_deposit_host bins slice by slice)
int launch_tilebin_build(const Params& P, const Markers& M, const TileBins& T, uint32_t* count, double* rec,
                         cudaStream_t st, int64_t base = 0, bool append = false);
int launch_tilebin_refresh(const Markers& M, const TileBins& T, const uint32_t* count, double* rec,
                           cudaStream_t st);
int launch_tilebin_rebin(const Params& P, const TileBins& T, uint32_t* count, double* rec, double* movers,
                         uint32_t mv_cap, uint32_t* mv_count, unsigned long long* counters,
                         cudaStream_t st);

// Materialised Larmor ring data + cell-owner deposition (orb_cellowner.cu, NEXT-3)
struct RingScratch {
  uint32_t* off;         // markers + 1: N_L per marker -> first point slot of the marker
  uint32_t* cell_start;  // ncells + 1: Larmor points per cell -> offsets
  uint32_t* block_sums;  // scan scratch for both
  double* ring;          // capacity * 6 doubles, marker order
  double* sorted;        // capacity * 6 doubles, cell order
  int64_t capacity;      // Larmor points the two arrays hold
  int64_t markers;       // markers off[] can hold
};
int launch_deposit_ringdata(const Params& P, const Markers& M, const RingScratch& R, double* rho,
                            double* jpar, unsigned long long* d_points, cudaStream_t st);

// v6: v5's pipeline with whole-tile chunks and 16-byte point records (orb_deposit_ws2.cu); fixed N_L <= 4
int launch_deposit_ws2(const Params& P, const Markers& M, const uint32_t* cell_start,
                       const TileBins& TB, double* rho, double* jpar, unsigned long long* d_points,
                       int sms, cudaStream_t st);

// ring table (cos, sin)(alpha0 + 2 pi l / N), built on the device (orb_ring.cu)
int launch_ring_table(double2* ring, double alpha0, cudaStream_t st);

// host: polynomial pieces of the clamped radial cubic B-splines, ns*16 doubles
void build_radial_table(int ns, std::vector<double>& out);

}  // namespace orb
