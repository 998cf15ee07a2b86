/*
 * orb.h -- C ABI of liborb_b200: gyro-averaged charge and parallel-current
 * deposition of delta-f markers onto a 3-D cubic B-spline grid, on one NVIDIA
 * B200 (sm_100a).  Plain C; callers need no CUDA header.
 *
 * What is computed (citations are lines of arxiv 1908.02219 as extracted in
 * PAPER.md; "R<n>" are the readings listed in DESIGN.md where the paper is
 * silent):
 *
 *   rho [i,j,k] += sum_p (q w_p        / N_L(p)) sum_l Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p)
 *   jpar[i,j,k] += sum_p (q w_p vpar_p / N_L(p)) sum_l Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p)
 *
 *   - markers are structure-of-arrays in magnetic coordinates (s, theta*, phi)
 *     (PAPER.md:21, 39); fields are 3-D finite-element cubic B-splines
 *     (PAPER.md:19, 39): clamped (open knot vector) in s, periodic in theta*, phi;
 *   - every marker is expanded into N_L Larmor points on a ring of radius
 *     rho_L = rho* sqrt(2 mu / B) in the poloidal plane at the marker's phi
 *     (R5-R7), N_L fixed or proportional to the ring size
 *     (R9);
 *   - geometry: concentric circular flux surfaces R = R0 + a s cos(theta),
 *     Z = a s sin(theta), B = B0 / (1 + (a/R0) s cos(theta)), theta* the
 *     straight-field-line angle tan(theta* / 2) = sqrt((1-e)/(1+e)) tan(theta/2),
 *     e = (a/R0) s (R1-R3);
 *   - a point that leaves the plasma (s_l > 1) is deposited at s_l = 1 (R11);
 *   - "deposit" without sorting loops over markers and the finite elements they
 *     touch with atomic accumulation; with sorting, markers are
 *     first bucket-sorted by field cell.  Both are offered here.
 *
 * Conventions common to all calls
 *   - every call returns ORB_OK (0) or a negative orb_status code; nothing
 *     throws, aborts or prints.  orb_strerror() gives a static description;
 *     orb_last_error() the detailed message of the last failing call on a handle.
 *   - "device pointer" = memory of the CUDA device given in the descriptor
 *     (e.g. torch.Tensor.data_ptr()); "host pointer" = ordinary host memory.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *     Calls that take a stream only enqueue work on it; they neither synchronise
 *     the host nor allocate, so a sequence orb_markers_bin / orb_grid_zero /
 *     orb_deposit can be captured into a CUDA graph.  A handle keeps state between
 *     calls (binned order, ring table, counters): issue the calls of one handle to
 *     ONE stream, or order the streams yourself (events) -- the library does not.
 *   - there is no CPU fallback: without a usable CUDA device orb_grid_create
 *     fails with ORB_E_CUDA.
 */
#ifndef ORB_H_
#define ORB_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ORB_VERSION 100
#define ORB_MAX_NL 32 /* largest number of Larmor points per marker */
#define ORB_MAX_FIELDS 8 /* fields per orb_gather call */

typedef enum {
  ORB_OK = 0,
  ORB_E_INVAL = -1, /* bad argument: NULL, n < 0, ns/ntheta/nphi < 4, a >= r0, N_L out of
                       [1, ORB_MAX_NL], n_max < n_min, pointer not 16-byte aligned        */
  ORB_E_STATE = -2, /* call order: deposit/bin before bind                              */
  ORB_E_NOMEM = -3, /* scratch allocation failed                                        */
  ORB_E_CUDA = -4   /* CUDA runtime / launch error (see orb_last_error)                 */
} orb_status;

typedef struct orb_grid orb_grid_t; /* opaque; owned by the library */

/* Grid + geometry + species.  Sizes are in CELLS; the deposited arrays have
 * (ns+3) x ntheta x nphi NODES (basis functions): the clamped cubic basis in s
 * has ns+3 functions, the periodic ones one per cell (R11). */
typedef struct {
  int32_t ns, ntheta, nphi; /* >= 4 each                                                  */
  double r0, a, b0;         /* major radius, minor radius (a < r0), field on axis (R1,R2) */
  double rho_star;          /* thermal Larmor radius / a  (>= 0)  (R6)                    */
  double q;                 /* species charge                                             */
  int32_t theta_map;        /* 1: theta* is the straight-field-line angle (R3, default);
                               0: theta* == geometric theta                               */
  int32_t device;           /* CUDA device ordinal                                        */
} orb_grid_desc_t;

enum { ORB_NL_FIXED = 0, ORB_NL_ADAPTIVE = 1 };

/* flags of orb_nl_policy_t.flags */
#define ORB_DEPOSIT_ZERO_FIRST 0x1u  /* zero rho/jpar on the stream before adding              */
#define ORB_DEPOSIT_NO_BIN 0x2u      /* never bin: deposit markers in the order they are bound  */
#define ORB_DEPOSIT_ALGO_ATOMIC 0x4u /* use the one-thread-per-marker global-atomics kernel
                                        (the GPU algorithm of) instead of the
                                        shared-memory tile kernel                              */
#define ORB_DEPOSIT_ALGO_TILE_V4 0x8u /* force the one-block-per-tile kernel (all warps run all
                                        phases; several blocks per SM)                          */
#define ORB_DEPOSIT_ALGO_TILE_WS 0x10u /* force the first persistent warp-specialised kernel (64-byte
                                        operand records, chunks of 256 markers); kept for
                                        comparison.  By default the library picks by N_L policy:
                                        the persistent kernel with 16-byte point records and
                                        whole-tile-sized chunks (orb_deposit_ws2.cu) for fixed
                                        N_L = 2..4, this one for N_L = 1, the one-block-per-tile
                                        kernel for larger or adaptive N_L.                        */
#define ORB_DEPOSIT_ALGO_TILE_WS2 0x40u /* (no effect: names the default for fixed N_L = 2..4)     */
#define ORB_DEPOSIT_ALGO_RING_DATA 0x20u /* the paper's own organisation, as a
                                        measured alternative: materialise the Larmor ring data in
                                        device memory, bucket-sort the Larmor POINTS by field
                                        cell, then loop over cells with the points of a cell in
                                        the inner loop.  Needs orb_ring_reserve; uses the bound
                                        arrays directly (no marker binning).                     */

/* Number of Larmor points per marker (R7-R9):
 *   FIXED:    N_L = n_fixed
 *   ADAPTIVE: N_L = min(n_max, n_fixed * max(1, ceil(rho_L / rho_ref)))
 * N_L = 1 deposits the guiding centre itself (R8).  Gyro-phases are
 * alpha_l = alpha0 + 2 pi l / N_L measured from +R towards +Z. */
typedef struct {
  int32_t mode;    /* ORB_NL_FIXED | ORB_NL_ADAPTIVE                                      */
  int32_t n_fixed; /* FIXED: N_L.  ADAPTIVE: n_min.   1..ORB_MAX_NL                       */
  int32_t n_max;   /* ADAPTIVE: cap, n_fixed..ORB_MAX_NL (ignored when FIXED)             */
  uint32_t flags;  /* ORB_DEPOSIT_*                                                       */
  double rho_ref;  /* ADAPTIVE: reference radius in units of a (> 0)                      */
  double alpha0;   /* gyro-phase of point 0, radians                                      */
} orb_nl_policy_t;

/* flags of orb_markers_bind */
#define ORB_MARKERS_SORTED 0x1u /* markers are already sorted by guiding-centre cell key
                                   (k_phi*ns + i_s)*ntheta + j_theta (non-decreasing; R17);
                                   binning then only locates the cell boundaries            */

#define ORB_MARKERS_TILE_BINS 0x2u /* bin into slack tile bins (one fixed-capacity segment of records
                                     per 1 x 16 cells and toroidal slab -- one radial row of a
                                     deposit tile; ~2.5x the dense layout's memory): built in ONE
                                     pass (no histogram, no scan) and refreshed incrementally with
                                     orb_markers_rebin.  Excludes
                                     ORB_MARKERS_SORTED.  At most ~1300 markers per bin on average. */

/* Creates a handle for one grid on desc->device and allocates nothing that
 * scales with the marker count yet.  *out is written only on success. */
int orb_grid_create(const orb_grid_desc_t *desc, orb_grid_t **out);

/* Frees the handle and all scratch.  Synchronises the device.  NULL is accepted. */
int orb_grid_destroy(orb_grid_t *g);

/* dims = (ns+3, ntheta, nphi): shape of rho / jpar, C order, k_phi fastest:
 * index = (i_s*ntheta + j_theta)*nphi + k_phi  (R14). */
int orb_grid_shape(const orb_grid_t *g, int64_t dims[3]);

/* Binds n markers given as six DEVICE arrays of n doubles (structure of arrays,
 * PAPER.md:21): s in [0,1], theta* and phi any finite angle in radians (wrapped to
 * [0,2pi)), parallel velocity, magnetic moment mu >= 0, weight.  Pointers are
 * BORROWED: no copy is made; they must stay valid and unmodified until the next
 * bind or destroy, and the library never writes to them.  vpar may be NULL if
 * jpar will always be NULL.  Pointers must be 16-byte aligned.  Marker VALUES are
 * not validated; s outside [0,1] is treated as the nearest bound (R11).  Any
 * previous binning is discarded.  n = 0 is legal.
 * Unless ORB_MARKERS_SORTED is given, bind makes sure the binning scratch (68 bytes
 * per marker) can hold n markers; growing it allocates device memory, which
 * synchronises the device -- call orb_reserve first to keep bind allocation-free. */
int orb_markers_bind(orb_grid_t *g, int64_t n, const double *s, const double *theta,
                     const double *phi, const double *vpar, const double *mu, const double *w,
                     uint32_t flags);

/* Pre-allocates the marker-proportional scratch for up to n markers (ORB_E_NOMEM if the
 * device cannot hold it).  Optional: orb_markers_bind grows it on demand. */
int orb_reserve(orb_grid_t *g, int64_t n);

/* Reserves the scratch of ORB_DEPOSIT_ALGO_RING_DATA: Larmor ring data for up to n_points Larmor
 * points (2 x 48 bytes each: in marker order and sorted by cell) of up to n_markers markers.
 * Allocates (synchronises); call it outside timed / captured regions; (0, 0) frees the scratch.
 * Points beyond n_points are
 * still deposited (directly, with global atomics) and counted by orb_last_fallback_points. */
int orb_ring_reserve(orb_grid_t *g, int64_t n_markers, int64_t n_points);

/* Runs (or refreshes) the binning pass alone on `stream`, so that it can be timed
 * apart from the deposit (BASELINE.json config 4; the bucket sort of PAPER.md:167):
 * counting sort of the bound markers by guiding-centre cell into library-owned
 * scratch.  For ORB_MARKERS_SORTED bindings only the per-cell offsets are built.
 * Asynchronous; never allocates. */
int orb_markers_bin(orb_grid_t *g, void *stream);

/* Adds the charge density into rho and, if jpar != NULL, the parallel current
 * into jpar (DEVICE arrays of orb_grid_shape doubles, owned by the caller).
 * Asynchronous on `stream`.  Bins first if the markers are not binned yet, unless
 * ORB_DEPOSIT_NO_BIN or ORB_DEPOSIT_ALGO_ATOMIC is set.  The result is the plain
 * sum above up to fp64 summation order (atomic ordering is the only source of
 * run-to-run difference). */
int orb_deposit(orb_grid_t *g, double *rho, double *jpar, const orb_nl_policy_t *policy,
                void *stream);

/* Get fields + gyroaverage -- the transpose of orb_deposit (stage 3 of the PIC step, "the
 * interpolation of the field at particle positions"; with the Larmor ring data it
 * is 'get fields' at the Larmor points followed by 'gyroaveraging' back to the guiding centre,
 * PAPER.md:73, 89; the paper's largest GPU win).  For every bound marker p and
 * field f (reading R20 of DESIGN.md: the paper prints no formula):
 *
 *   out[f][p] = (1 / N_L(p)) sum_l sum_{i,j,k} fields[f][i,j,k] Ls_i(s_pl) Lt_j(ts_pl) Lp_k(phi_p)
 *
 * with the ring, the map and the cubic B-splines of orb_deposit, so that for any field F
 *   sum_nodes rho[n] F[n] = q sum_p w_p out[p]      (adjointness; rho from orb_deposit).
 * fields / out: HOST arrays of n_fields (1..ORB_MAX_FIELDS) DEVICE pointers; fields[f] has
 * orb_grid_shape doubles (layout of rho, 16-byte aligned, only read); out[f] has n doubles and is
 * written in BOUND marker order whatever the binning did (owned by the caller; the pointer
 * arrays themselves are read during the call only).  The marker weights and vpar are not used.
 * Asynchronous on `stream`; bins first if the markers are not binned yet (never allocates);
 * ORB_DEPOSIT_NO_BIN or ORB_DEPOSIT_ALGO_ATOMIC in policy->flags select the one-thread-per-marker
 * kernel that reads the grid directly, in bound order.  orb_last_points / orb_last_fallback_points
 * then refer to this call.  Field gradients are not formed. */
int orb_gather(orb_grid_t *g, int32_t n_fields, const double *const *fields, double *const *out,
               const orb_nl_policy_t *policy, void *stream);

/* ---- Incremental re-binning.  PAPER.md:169-173: the bucket sort is "the most
 * time-consuming part" and cancels the gain it brings to the deposit; PAPER.md:235 proposes to
 * track the markers that leave their cell instead of sorting from scratch.  For markers bound with
 * ORB_MARKERS_TILE_BINS the library keeps its binned copy in slack tile bins: orb_markers_bin
 * builds them in ONE pass; after the markers have moved, orb_markers_rebin relocates only those that
 * left their tile.  The binned records are the data the deposit and gather kernels read, so the
 * new coordinates must reach them first: either orb_markers_refresh (copies the current values of
 * the six bound arrays into the records) or a pusher that updates the records in place
 * (orb_markers_layout).  Deposits are then identical to those after a fresh orb_markers_bin up
 * to summation order; a marker that ends in a neighbouring tile (full tile, full mover buffer) only
 * costs speed.  All three calls are asynchronous on `stream` and never allocate. */

/* records <- current values of the bound arrays (every marker; 64-byte record writes). */
int orb_markers_refresh(orb_grid_t *g, void *stream);

/* Re-derives every record's bin from its (s, theta*, phi); moves the records that left their bin
 * (one 32-byte read per marker + 256 bytes per mover).  ORB_E_STATE unless the markers are bound with
 * ORB_MARKERS_TILE_BINS and binned. */
int orb_markers_rebin(orb_grid_t *g, void *stream);

/* Markers moved by the last orb_markers_rebin, and (optional) movers left in place because the
 * mover buffer (n/2 records) was full -- they move at the next rebin.  Synchronises the device. */
int orb_last_moved(orb_grid_t *g, int64_t *n_moved, int64_t *n_left_in_place);

/* Where the binned records live, for a pusher that updates them in place (DEVICE pointers, owned by
 * the library, valid until the next bind/destroy): record r of bin b is records[(b*capacity + r) *
 * record_doubles + {0: s, 1: theta*, 2: phi, 3: vpar, 4: mu, 5: w, 6: index in bound order (int64
 * bits), 7: 0}], r < min(count[b], capacity);
 * bin b = ((k_phi*tiles_s + i_s/8)*tiles_theta + j_theta/16)*8 + i_s%8, n_bins of them. */
typedef struct {
  double *records;
  const uint32_t *count;
  int32_t record_doubles;
  uint32_t capacity, n_bins;
  int32_t tiles_s, tiles_theta;
} orb_marker_layout_t;
int orb_markers_layout(const orb_grid_t *g, orb_marker_layout_t *out);

/* Zeroes rho and, if not NULL, jpar (DEVICE arrays of orb_grid_shape doubles) on `stream`
 * (two cudaMemsetAsync; no kernel).  Equivalent to ORB_DEPOSIT_ZERO_FIRST, offered as a call of
 * its own so that a harness can time the deposit kernels apart from the zeroing. */
int orb_grid_zero(orb_grid_t *g, double *rho, double *jpar, void *stream);

/* Sum of N_L over the markers of the last orb_deposit on this handle.
 * Waits for that deposit only (an event recorded on its stream; if the deposit was
 * captured into a CUDA graph, for the whole device) and copies 8 bytes back. */
int orb_last_points(orb_grid_t *g, int64_t *n_points);

/* Of those, the Larmor points of the last orb_deposit whose 4x4 (s, theta*) footprint left the
 * shared-memory tile of their block and were deposited with global atomics instead (a
 * performance diagnostic; 0 for the global-atomics algorithm).  Synchronises like
 * orb_last_points. */
int orb_last_fallback_points(orb_grid_t *g, int64_t *n_points);

/* End-to-end convenience for callers whose data lives on the HOST: copies the six
 * marker arrays (host pointers, n doubles each; vpar may be NULL iff jpar_host is
 * NULL) to library-owned device buffers, binds, deposits into zeroed device grids
 * and copies rho (and jpar) back into the host arrays, which are OVERWRITTEN.
 * Above 2^22 markers the work is pipelined on two library-owned streams: the markers travel in
 * 8 slices; each slice is appended to the slack tile bins (ORB_MARKERS_TILE_BINS layout, sized for
 * all n markers) as soon as its copy has landed, and the deposit kernel runs once per GROUP of
 * slices (6 + 2), so that a tile is visited twice per call, not once per slice; the first group's
 * deposit overlaps the last two copies (the call is bound by the host link: 48 B per marker).
 * With ORB_DEPOSIT_NO_BIN, _ALGO_ATOMIC or _ALGO_RING_DATA every slice is deposited on its own.
 * Use pinned host memory for the overlap to happen.
 * Synchronous.  Leaves the handle bound to the library's own device copies (not binned).
 * h2d_bytes / d2h_bytes (optional) receive the bytes moved. */
int orb_deposit_host(orb_grid_t *g, int64_t n, const double *s, const double *theta,
                     const double *phi, const double *vpar, const double *mu, const double *w,
                     double *rho_host, double *jpar_host, const orb_nl_policy_t *policy,
                     int64_t *n_points, int64_t *h2d_bytes, int64_t *d2h_bytes);

/* Number of kernel launches the library has enqueued on this handle so far
 * (memsets and copies not counted). */
int orb_launch_count(const orb_grid_t *g, int64_t *n_launches);

/* ------------------------------------------------------------------------------------------
 * Harness and diagnostic calls.  NOT part of the product path: nothing above needs them; they
 * exist so that tests and bench.py can look inside (binned order, per-phase clocks, spline
 * table) and measure the fp64 roof of the device the bench runs on.  All are synchronous.
 * ------------------------------------------------------------------------------------------ */

/* Diagnostic: the 16 device counters of the last orb_deposit.  out[0] = Larmor points,
 * out[1] = points deposited directly; out[2..15] = per-phase SM clock sums of the tile kernel
 * (block-thread 0), non-zero only in a library built with -DORB_PHASE_CLOCKS.  Synchronises. */
int orb_debug_counters(orb_grid_t *g, uint64_t out[16]);

/* Diagnostic: copies the result of the last binning pass to the HOST (bucket sort of
 * PAPER.md:167; R17, R18).  cell_start_host (ncells + 1 uint32, ncells = ns*ntheta*nphi):
 * exclusive offsets per guiding-centre cell in key order (k_phi*ns + i_s)*ntheta + j_theta.
 * *rec_doubles receives the record stride in doubles (8: s, theta*, phi, vpar, mu, w, the
 * marker's index in bound order as a 64-bit integer bit pattern, 0) and
 * rec_host (n * 8 doubles, may be NULL) the binned records -- or 0 and nothing if the markers
 * were bound with ORB_MARKERS_SORTED (then the bound order IS the binned order).
 * ORB_E_STATE if the markers are not binned.  Synchronises the device. */
int orb_debug_binned(orb_grid_t *g, double *rec_host, uint32_t *cell_start_host,
                     int32_t *rec_doubles);

/* Diagnostic, slack tile bins: count_host (n_bins uint32) and the records of all bins, bin by
 * bin, packed into rec_host (n * 8 doubles).  Meant for small cases (one copy per bin). */
int orb_debug_tilebins(orb_grid_t *g, double *rec_host, uint32_t *count_host);

/* Host-only diagnostic, no device needed: the polynomial pieces of the clamped (open knot
 * vector) radial cubic B-splines that the tile kernel evaluates (R11).
 * out (HOST, ns*16 doubles): out[(c*4 + a)*4 + d] = coefficient of t^d, t = s*ns - c in [0,1),
 * of basis function c+a on radial cell c.  ORB_E_INVAL if ns < 4 or out is NULL. */
int orb_spline_table_radial(int32_t ns, double *out);

/* Harness aid, not part of the hot path: measures the fp64 FMA rate of `device` (8 independent
 * DFMA chains per thread, 4 x 512 threads per SM, one timed launch after a warm-up) and writes it
 * as TFLOP/s (2 flop per FMA).  The deposition is bound by the fp64 pipe, so this is the roof
 * bench.py reports `roofline_alu` against.  Synchronous; takes a few milliseconds. */
int orb_probe_dfma(int32_t device, double *tflops);

/* ---- Allocation-free deposit, for callers that cannot call cudaMalloc at all (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it) and so cannot hold an orb_grid_t.
 * The definition of orb_deposit (same ring, map, splines and N_L policy),
 * computed by a variant of the one-thread-per-marker global-atomics kernel whose scratch (Larmor
 * ring table, radial spline pieces, point counter) lives in ONE file-scope device array of
 * 139 776 bytes (csrc/orb_noalloc.cu) that every GPU loading the library holds until exit.
 * Limit: desc->ns <= ORB_NOALLOC_MAX_NS, else ORB_E_INVAL with the reason in errbuf; the marker
 * count is not limited.  The call makes no cudaMalloc / cudaFree and calls no allocating routine:
 * it clears the counter, rebuilds both tables on the device for this call's (ns, alpha0), and
 * launches the deposit, all on `stream`.
 *   desc                 grid, geometry, species, device (as for orb_grid_create; only read)
 *   n; s .. w            DEVICE marker arrays of n doubles, 16-byte aligned, only read; vpar may
 *                        be NULL iff jpar is NULL
 *   rho, jpar            DEVICE grids of (ns + 3) * ntheta * nphi doubles (layout of
 *                        orb_grid_shape), 16-byte aligned, ADDED to; jpar may be NULL
 *   policy               N_L policy; of the flags only ORB_DEPOSIT_ZERO_FIRST is accepted
 *   n_points             NULL: the call is asynchronous.  Otherwise (HOST pointer) the call waits
 *                        for `stream` and returns the sum of N_L (not under graph capture)
 *   errbuf, errbuf_len   optional HOST buffer that receives the message of a failing call
 * All calls on a device SHARE the scratch array, which keeps the last call's contents: calls on
 * one stream are ordered and safe; calls that overlap on the GPU (other streams, concurrently
 * replayed graphs) race on it and must be serialised by the caller.
 * Speed: that of ORB_DEPOSIT_ALGO_ATOMIC (about 10x slower than the tile kernels on cfg3). */
#define ORB_NOALLOC_MAX_NS 1024
int orb_deposit_noalloc(const orb_grid_desc_t *desc, int64_t n, const double *s,
                        const double *theta, const double *phi, const double *vpar,
                        const double *mu, const double *w, double *rho, double *jpar,
                        const orb_nl_policy_t *policy, void *stream, int64_t *n_points,
                        char *errbuf, int32_t errbuf_len);

/* ------------------------------------------------------------------------------------------ */

/* Static text for a status code. */
const char *orb_strerror(int code);

/* Detailed message of the last failing call on g (includes cudaGetErrorString);
 * "" if none.  The pointer stays valid until the next call on g. */
const char *orb_last_error(const orb_grid_t *g);

int orb_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ORB_H_ */
