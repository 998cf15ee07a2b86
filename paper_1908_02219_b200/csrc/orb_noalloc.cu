// orb_deposit_noalloc: the one entry point of the library that allocates NOTHING, for callers
// that cannot call cudaMalloc at all (code under CUDA graph capture, tight serving loops, harnesses
// that forbid it) and therefore cannot create an orb_grid_t handle either.
//
// It is a variant of the global-atomics deposition kernel (orb_deposit_atomic.cu; PAPER.md:97,
// hot-path steps a1-a6 + a8 with one fp64 reduction per node update), which needs three pieces of
// scratch besides its inputs and outputs: the Larmor-ring table (a4), the polynomial pieces of the
// clamped radial splines (a6) and the point counter.  The handle-based path keeps them in memory
// that orb_grid_create allocates; here they live in ONE file-scope device array of fixed size,
// which every GPU that loads the library holds until the process exits:
//
//   g_noalloc_scratch : kScratchBytes = 139 776 bytes (136.5 KiB)
//     [0, 128)          16 counters ([0] = sum of N_L of the call)
//     [256, 8704)       ring table, ORB_MAX_NL (ORB_MAX_NL + 1) / 2 entries (cos, sin)
//     [8704, 139776)    radial pieces, ORB_NOALLOC_MAX_NS cells x 16 coefficients
//
// so the radial resolution is limited to ns <= ORB_NOALLOC_MAX_NS (1024); the marker count is not
// limited by the scratch.  Both tables are rebuilt ON THE DEVICE by a small kernel at the start of
// every call (ns and alpha0 may change from call to call, and the array keeps whatever the last
// call left), and the counters are cleared: nothing is carried from one call to the next.  All
// calls on a device share the array, so two calls that overlap on the GPU (different streams, or
// graphs replayed concurrently) RACE on it; calls on one stream are ordered and safe.
//
// In host code the array's name is only a host-side stand-in for the device symbol: its device
// address is fetched once per device with cudaGetSymbolAddress (that device current) and that
// pointer is what the kernels receive.
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "orb_geom.cuh"

namespace orb {

namespace {

constexpr int kRingEntries = ORB_MAX_NL * (ORB_MAX_NL + 1) / 2;                  // 528
constexpr size_t kOffCounters = 0;
constexpr size_t kOffRing = 256;
constexpr size_t kOffScoef = kOffRing + (size_t)kRingEntries * sizeof(double2);  // 8704
constexpr size_t kScratchBytes = kOffScoef + (size_t)ORB_NOALLOC_MAX_NS * 16 * sizeof(double);
static_assert(kOffScoef % 256 == 0, "the radial table starts on a 256-byte boundary");
static_assert(kCounters * sizeof(unsigned long long) <= kOffRing, "counters overlap the ring table");

static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned char* g_scratch_ptr[kMaxDevices];   // device address of g_noalloc_scratch, per device

// knot m of the clamped cubic knot vector {0,0,0,0, 1, ..., ns-1, ns,ns,ns,ns}
__device__ __forceinline__ double knot_of(int m, int ns) {
  return (double)min(max(m - 3, 0), ns);
}

// Fills the two tables of the scratch for this call: thread e < 528 writes ring entry e
// ((cos, sin)(alpha0 + 2 pi l / N) at N (N - 1) / 2 + l, R7); thread c < ns writes the 16
// coefficients of radial cell c: basis c + a on cell c as a cubic in t = s ns - c, from the
// Cox-de Boor recursion run on polynomial coefficients (R11), in the layout of
// Params::scoef.
__global__ void __launch_bounds__(256)
k_noalloc_tables(unsigned char* __restrict__ scratch, int ns, double alpha0) {
  const int x = blockIdx.x * blockDim.x + threadIdx.x;
  if (x < kRingEntries) {
    int n = (int)((1.0 + sqrt(1.0 + 8.0 * (double)x)) * 0.5);
    while (n * (n - 1) / 2 > x) --n;
    while (n * (n + 1) / 2 <= x) ++n;
    const int l = x - n * (n - 1) / 2;
    double sn, cs;
    sincos(alpha0 + kTwoPi * (double)l / (double)n, &sn, &cs);
    reinterpret_cast<double2*>(scratch + kOffRing)[x] = make_double2(cs, sn);
  }
  if (x >= ns) return;
  const int c = x, span = c + 3;
  double N[4][4], nx[4][4];   // N[j][d]: coefficient of t^d of N_{span-p+j, p}
#pragma unroll
  for (int j = 0; j < 4; ++j)
#pragma unroll
    for (int d = 0; d < 4; ++d) N[j][d] = 0.0;
  N[0][0] = 1.0;
#pragma unroll
  for (int p = 1; p <= 3; ++p) {
#pragma unroll
    for (int j = 0; j < 4; ++j) {
#pragma unroll
      for (int d = 0; d < 4; ++d) nx[j][d] = 0.0;
      if (j > p) continue;
      const int i = span - p + j;
      if (j >= 1) {   // (x - T_i) / (T_{i+p} - T_i) N_{i,p-1}
        const double den = knot_of(i + p, ns) - knot_of(i, ns);
        if (den > 0.0) {
          const double al = ((double)c - knot_of(i, ns)) / den, be = 1.0 / den;
          nx[j][0] += al * N[j - 1][0];
#pragma unroll
          for (int d = 1; d < 4; ++d) nx[j][d] += al * N[j - 1][d] + be * N[j - 1][d - 1];
        }
      }
      if (j <= p - 1) {   // (T_{i+p+1} - x) / (T_{i+p+1} - T_{i+1}) N_{i+1,p-1}
        const double den = knot_of(i + p + 1, ns) - knot_of(i + 1, ns);
        if (den > 0.0) {
          const double al = (knot_of(i + p + 1, ns) - (double)c) / den, be = -1.0 / den;
          nx[j][0] += al * N[j][0];
#pragma unroll
          for (int d = 1; d < 4; ++d) nx[j][d] += al * N[j][d] + be * N[j][d - 1];
        }
      }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
      for (int d = 0; d < 4; ++d) N[j][d] = nx[j][d];
  }
  double* out = reinterpret_cast<double*>(scratch + kOffScoef) + (size_t)c * 16;
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int d = 0; d < 4; ++d) out[a * 4 + d] = N[a][d];
}

// The deposition itself: one thread per marker, every node update a hardware fp64 reduction in
// L2 (the kernel of orb_deposit_atomic.cu), with the ring table, the radial pieces and the point
// counter taken from the scratch array whose device address is passed in.
__global__ void __launch_bounds__(256)
k_deposit_noalloc(Params P, const Markers M, double* __restrict__ rho, double* __restrict__ jpar,
                  unsigned char* __restrict__ scratch) {
  P.ring = reinterpret_cast<const double2*>(scratch + kOffRing);
  P.scoef = reinterpret_cast<const double*>(scratch + kOffScoef);
  unsigned long long* counters = reinterpret_cast<unsigned long long*>(scratch + kOffCounters);
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned int my_points = 0;
  if (p < M.n) {
    const MarkerData m = load_marker(M, p);
    const GuidingCentre g = guiding_centre(P, m.s, m.th, m.mu);
    const int n = g.n;
    my_points = (unsigned int)n;
    const double c = P.q * m.w / (double)n;
    const double cj = c * m.vpar;
    double wp[4];
    const int k0 = periodic_weights(wrap_2pi(m.ph), P.nph_scale, P.nph, wp);
    int kk[4];
    double cw[4], cjw[4];
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      kk[d] = wrap_index(k0 + d, P.nph);
      cw[d] = c * wp[d];
      cjw[d] = cj * wp[d];
    }
    for (int l = 0; l < n; ++l) {
      double s_l = g.s, ts_l = g.ts;   // R8: N_L = 1 is the guiding centre itself
      if (n > 1) larmor_point(P, g, ring_entry(P, n, l), s_l, ts_l);
      double ws[4], wt[4];
      const int i0 = radial_weights(P, s_l, ws);
      const int j0 = periodic_weights(ts_l, P.nth_scale, P.nth, wt);
#pragma unroll
      for (int a = 0; a < 4; ++a) {
#pragma unroll
        for (int b = 0; b < 4; ++b) {
          const double v = ws[a] * wt[b];
          const int64_t row =
              ((int64_t)(i0 + a) * P.nth + wrap_index(j0 + b, P.nth)) * (int64_t)P.nph;
#pragma unroll
          for (int d = 0; d < 4; ++d) {
            atomicAdd(rho + row + kk[d], v * cw[d]);
            if (jpar) atomicAdd(jpar + row + kk[d], v * cjw[d]);
          }
        }
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) my_points += __shfl_down_sync(0xffffffffu, my_points, o);
  if ((threadIdx.x & 31) == 0 && my_points) atomicAdd(counters, (unsigned long long)my_points);
}

int refuse(char* errbuf, int32_t errbuf_len, int code, const char* fmt, ...) {
  if (errbuf && errbuf_len > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
    va_end(ap);
  }
  return code;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

}  // namespace orb

using namespace orb;

extern "C" int orb_deposit_noalloc(const orb_grid_desc_t* d, int64_t n, const double* s,
                                   const double* theta, const double* phi, const double* vpar,
                                   const double* mu, const double* w, double* rho, double* jpar,
                                   const orb_nl_policy_t* pol, void* stream, int64_t* n_points,
                                   char* errbuf, int32_t errbuf_len) {
  if (errbuf && errbuf_len > 0) errbuf[0] = 0;
  // ---- argument checks: nothing below touches the device before they have passed
  if (!d || !pol) return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: desc or policy is NULL");
  if (d->ns < 4 || d->ntheta < 4 || d->nphi < 4)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: ns, ntheta, nphi must be >= 4");
  if (d->ns > ORB_NOALLOC_MAX_NS)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL,
                  "orb_deposit_noalloc: ns = %d exceeds ORB_NOALLOC_MAX_NS = %d (the static scratch "
                  "holds the radial spline pieces of that many cells); use orb_grid_create + "
                  "orb_deposit for larger grids",
                  (int)d->ns, (int)ORB_NOALLOC_MAX_NS);
  if ((int64_t)d->ns * d->ntheta * d->nphi >= (int64_t)1 << 31)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: more than 2^31 - 1 cells");
  if (!(d->r0 > 0.0) || !(d->a > 0.0) || !(d->a < d->r0) || !(d->b0 > 0.0) || !(d->rho_star >= 0.0) ||
      !isfinite(d->rho_star) || !isfinite(d->q) || (d->theta_map != 0 && d->theta_map != 1))
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: invalid grid descriptor");
  if (d->device < 0 || d->device >= kMaxDevices)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: device out of [0, %d)", kMaxDevices);
  if (pol->mode != ORB_NL_FIXED && pol->mode != ORB_NL_ADAPTIVE)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: policy.mode");
  if (pol->n_fixed < 1 || pol->n_fixed > ORB_MAX_NL)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: policy.n_fixed out of [1, ORB_MAX_NL]");
  if (pol->mode == ORB_NL_ADAPTIVE &&
      (pol->n_max < pol->n_fixed || pol->n_max > ORB_MAX_NL || !(pol->rho_ref > 0.0) || !isfinite(pol->rho_ref)))
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: policy.n_max / policy.rho_ref");
  if (!isfinite(pol->alpha0)) return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: policy.alpha0");
  if (pol->flags & ~(uint32_t)ORB_DEPOSIT_ZERO_FIRST)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL,
                  "orb_deposit_noalloc: only ORB_DEPOSIT_ZERO_FIRST is accepted in policy.flags");
  if (n < 0 || n >= ((int64_t)1 << 32) - 1)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: n out of range");
  if (!rho) return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: rho is NULL");
  if (n > 0 && (!s || !theta || !phi || !mu || !w))
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: NULL marker array");
  if (jpar && !vpar && n > 0)
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: jpar needs vpar");
  if (!aligned16(s) || !aligned16(theta) || !aligned16(phi) || !aligned16(vpar) || !aligned16(mu) ||
      !aligned16(w) || !aligned16(rho) || !aligned16(jpar))
    return refuse(errbuf, errbuf_len, ORB_E_INVAL, "orb_deposit_noalloc: arrays must be 16-byte aligned");

  // ---- the device, and once per device the address of the scratch array on it
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) {
    cudaGetLastError();
    prev = -1;
  }
  cudaError_t ce = cudaSetDevice(d->device);
  if (ce != cudaSuccess) {
    cudaGetLastError();
    return refuse(errbuf, errbuf_len, ORB_E_CUDA, "orb_deposit_noalloc: cudaSetDevice(%d): %s", (int)d->device,
                  cudaGetErrorString(ce));
  }
  struct Restore {
    int prev;
    ~Restore() {
      if (prev >= 0) cudaSetDevice(prev);
    }
  } restore{prev};
  unsigned char* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ptr[d->device]) {
      void* ptr = nullptr;
      ce = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);   // d->device is current
      if (ce != cudaSuccess || !ptr) {
        cudaGetLastError();
        return refuse(errbuf, errbuf_len, ORB_E_CUDA, "orb_deposit_noalloc: cudaGetSymbolAddress: %s",
                      cudaGetErrorString(ce));
      }
      g_scratch_ptr[d->device] = static_cast<unsigned char*>(ptr);
    }
    scratch = g_scratch_ptr[d->device];
  }

  cudaStream_t st = static_cast<cudaStream_t>(stream);
#define ORB_NA(call)                                                                         \
  do {                                                                                       \
    ce = (call);                                                                             \
    if (ce != cudaSuccess) {                                                                 \
      cudaGetLastError();                                                                    \
      return refuse(errbuf, errbuf_len, ORB_E_CUDA, "orb_deposit_noalloc: %s: %s", #call,    \
                    cudaGetErrorString(ce));                                                 \
    }                                                                                        \
  } while (0)

  // ---- this call's scratch contents: counters cleared, both tables rebuilt for (ns, alpha0)
  ORB_NA(cudaMemsetAsync(scratch + kOffCounters, 0, kCounters * sizeof(unsigned long long), st));
  {
    const int items = d->ns > kRingEntries ? d->ns : kRingEntries;
    k_noalloc_tables<<<(items + 255) / 256, 256, 0, st>>>(scratch, d->ns, pol->alpha0);
    ORB_NA(cudaGetLastError());
  }
  const int64_t nnodes = (int64_t)(d->ns + 3) * d->ntheta * d->nphi;
  if (pol->flags & ORB_DEPOSIT_ZERO_FIRST) {
    ORB_NA(cudaMemsetAsync(rho, 0, (size_t)nnodes * sizeof(double), st));
    if (jpar) ORB_NA(cudaMemsetAsync(jpar, 0, (size_t)nnodes * sizeof(double), st));
  }
  if (n > 0) {
    Params P;
    P.ns = d->ns;
    P.nth = d->ntheta;
    P.nph = d->nphi;
    P.theta_map = d->theta_map;
    P.eps = d->a / d->r0;
    P.b0 = d->b0;
    P.inv_b0 = 1.0 / d->b0;
    P.rho_star = d->rho_star;
    P.q = d->q;
    P.nth_scale = (double)d->ntheta / kTwoPi;
    P.nph_scale = (double)d->nphi / kTwoPi;
    P.adaptive = pol->mode == ORB_NL_ADAPTIVE;
    P.n_fixed = pol->n_fixed;
    P.n_max = P.adaptive ? pol->n_max : pol->n_fixed;
    P.rho_ref = P.adaptive ? pol->rho_ref : 1.0;
    P.inv_rho_ref = 1.0 / P.rho_ref;
    P.ring = nullptr;    // the kernel takes both tables from the scratch pointer
    P.scoef = nullptr;
    Markers M;
    M.s = s;
    M.th = theta;
    M.ph = phi;
    M.vpar = vpar;
    M.mu = mu;
    M.w = w;
    M.rec = nullptr;
    M.n = n;
    const int64_t blocks = (n + 255) / 256;
    k_deposit_noalloc<<<(unsigned int)blocks, 256, 0, st>>>(P, M, rho, jpar, scratch);
    ORB_NA(cudaGetLastError());
  }
  if (n_points) {   // optional and synchronous: waits for `stream`, copies 8 bytes back
    unsigned long long v = 0;
    ORB_NA(cudaMemcpyAsync(&v, scratch + kOffCounters, sizeof(v), cudaMemcpyDeviceToHost, st));
    ORB_NA(cudaStreamSynchronize(st));
    *n_points = (int64_t)v;
  }
#undef ORB_NA
  return ORB_OK;
}
