/*
 * tpc.h -- C ABI of the B200-native TPC sector track finding (libtpc_b200.so).
 *
 * Method: PAPER.md:27-30 (section 2: hits carry a time, seeding "scales the time to z linearly using the
 * average drift velocity" and "assumes all tracks are primaries coming from the origin"; a first preliminary
 * Kalman fit is used to find the full track) and PAPER.md:37-41 (section 3: Cellular-Automaton seeding handles
 * the combinatorial part, then single-hypothesis Kalman track following, linear in the event size).
 * The paper names the steps only; their exact definition (S0..S6, readings A1..A33, tunables table T) is in
 * DESIGN.md section 4 and is what every entry point below computes.  Every step runs in hand-written CUDA
 * kernels for sm_100a; there is no CPU fallback: without a CUDA device tpc_create returns TPC_E_CUDA.
 *
 * Conventions
 *  - All functions return 0 (TPC_OK) or a negative tpc_status; no exception or abort crosses this boundary.
 *    tpc_last_error gives a human-readable message for the last failure on that context.
 *  - "host or device" pointers are classified with cudaPointerGetAttributes.  Input arrays are COPIED (the
 *    caller keeps ownership; host memory -- pageable or pinned -- may be freed or overwritten as soon as the load call
 *    returns, device memory once the context's stream has reached the copy).  Output arrays are LIBRARY-OWNED and stay valid until the next tpc_find_tracks*,
 *    tpc_clear or tpc_destroy on the same context.
 *  - A context is not thread-safe; different contexts are independent.  All device work of a context is issued
 *    on one CUDA stream (tpc_set_stream; default: the legacy default stream).
 *  - Units: cm, microseconds, Tesla, GeV/c.  Frames: per-sector local frame, x along the sector centre line (pad
 *    rows at x = row_x[r]), y along the pads, z along the drift: z = z_max - vdrift * t (S0).
 */
#ifndef TPC_B200_TPC_H_
#define TPC_B200_TPC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tpc_ctx tpc_ctx;

typedef enum {
  TPC_OK = 0,
  TPC_E_ARG = -1,      /* bad argument (null pointer, out-of-range sector/row, n < 0, non-increasing row_x, non-finite Bz/vdrift, unknown parameter) */
  TPC_E_STATE = -2,    /* call not allowed in this state (tpc_set_param after the first load, debug getter before tpc_find_tracks, ...) */
  TPC_E_NOMEM = -3,    /* host or device allocation failed */
  TPC_E_CUDA = -4,     /* CUDA runtime error (includes: no CUDA device) */
  TPC_E_CAPACITY = -5  /* a fixed-width field would overflow (more than 2^24 tracklets, more than 2^31-1 clusters in one (sector,row), n_rows > 255) */
} tpc_status;

/* Geometry of the detector as the tracker sees it (the TPC, its sectors and pad rows).  Copied by tpc_create. */
typedef struct {
  int32_t n_sectors;      /* e.g. 36 = 18 per side; sectors are independent units of the path */
  int32_t n_rows;         /* pad rows per sector, 3..255 (configs: 152) */
  const float* row_x;     /* HOST pointer, n_rows local-x positions of the pad rows, cm, strictly increasing, > 0 */
  float sector_dphi;      /* opening angle of a sector, rad (20 deg) */
  float z_max;            /* drift length, cm (250) */
  float t_frame;          /* us; 0 => triggered event (z-windows projected from the origin); > 0 => continuous time frame of this length (shift-invariant z search, reading A6) */
  float sigma_y, sigma_z; /* cm; measurement errors used by the Kalman filter (0.1, 0.15) */
} tpc_geometry;

/* Result of tpc_find_tracks / tpc_find_tracks_device: per track the 5-parameter state, covariance, chi2/NDF and cluster indices.
 * Arrays are host memory for tpc_find_tracks and device memory for tpc_find_tracks_device; library-owned in both cases.
 * Track order: ascending tracklet index = ascending (sector, start row, start position in the sorted row). */
typedef struct {
  int64_t n_tracks, n_cluster_refs;
  const int32_t* sector;    /* [n_tracks] */
  const float* x;           /* [n_tracks] local x of the state = row_x of the innermost cluster used by the fit */
  const float* par;         /* [n_tracks][5]  y, z, sin(phi), dz/ds, q/pT   (cm, cm, -, -, c/GeV); z is the S0-scaled z */
  const float* cov;         /* [n_tracks][15] lower triangle, row-major: (0,0)(1,0)(1,1)(2,0)(2,1)(2,2)... */
  const float* chi2;        /* [n_tracks] chi2 of the inward fit of the tracklet */
  const int32_t* ndf;       /* [n_tracks] 2 * (clusters in the fit) - 5 */
  const int32_t* tracklet;  /* [n_tracks] index of the tracklet (= start hit) the track comes from */
  const int64_t* cl_begin;  /* [n_tracks+1] offsets into cl_row / cl_index */
  const int32_t* cl_row;    /* [n_cluster_refs] pad row, ascending within a track */
  const int32_t* cl_index;  /* [n_cluster_refs] index into the caller's arrays of that (sector,row) as passed to tpc_load_clusters */
} tpc_tracks;

/* Result of tpc_refit_tracks: S7 of DESIGN.md section 4 ("first preliminary fit ... improve the
 * z-estimation"; readings A37, A38).  One entry per track of the last tpc_find_tracks* call, same order.  Arrays are library-owned,
 * host memory (device_result = 0) or device memory (device_result = 1), valid until the next call on the context. */
typedef struct {
  int64_t n_tracks;
  const int32_t* n;         /* [n_tracks] clusters used by the inward pass (= owned clusters unless a transport failed) */
  const int32_t* ndf;       /* [n_tracks] 2*n - 5 */
  const float*   x;         /* [n_tracks] local x of the refitted state (row of the innermost cluster used) */
  const float*   par;       /* [n_tracks][5]  y, z, sin(phi), dz/ds, q/pT after the refit over the owned clusters */
  const float*   cov;       /* [n_tracks][15] lower triangle, row-major */
  const float*   chi2;      /* [n_tracks] chi2 of the inward pass */
  const float*   z0;        /* [n_tracks] scaled z of the track at the beam line (x = y = 0), cm */
  const float*   t0;        /* [n_tracks] collision time estimate -z0 / vdrift, us (about 0 for a triggered primary) */
  float ms_refit;           /* device time of K7 (CUDA events on the context's stream), ms */
} tpc_refit;

/* Result of tpc_mark_clusters: S8 of DESIGN.md section 4 ("The tracker forms tubes of 1.5 cm
 * around each track, and marks unattached clusters as adjacent to the tube of the track with the highest transverse momentum it lies
 * in"; reading A40).  One entry per loaded cluster, in the caller's order: units (sector*n_rows+row) ascending, inside a unit the index
 * in the arrays passed to tpc_load_clusters*.  Library-owned, host (device_result = 0) or device memory, valid until the next call. */
typedef struct {
  int64_t n_clusters;
  const int32_t* status;    /* [n_clusters] 0 = in no tube, 1 = attached (in the cluster list of a track), 2 = adjacent */
  const int32_t* track;     /* [n_clusters] track of the last tpc_find_tracks* call it is attached / adjacent to, -1 for status 0 */
  float ms_mark;            /* device time of K8 (CUDA events on the context's stream), ms */
} tpc_cluster_marks;

/* Result of tpc_merge_tracks: S9 of DESIGN.md section 4 ("Locally, e. g. at the TPC sector
 * boundaries, there are still some improvements to be done"; the matching rule is this build's reading A41, the paper prints none): for every track of the last tpc_find_tracks* call the track that continues it in the neighbouring sector and
 * the track it continues.  Library-owned, host (device_result = 0) or device memory, valid until the next call on the context. */
typedef struct {
  int64_t n_tracks;
  const int32_t* next;      /* [n_tracks] index of the continuing segment in the neighbouring sector, -1 = none */
  const int32_t* prev;      /* [n_tracks] index of the segment this track continues, -1 = none */
  float ms_merge;           /* device time of K9 (CUDA events on the context's stream), ms */
} tpc_merges;

/* Result of tpc_find_loopers: S10 of DESIGN.md section 4 (SURVEY.md section 8(f).3 "recognise returning legs / extra turns"
 * "looping tracks", "secondary legs of looping tracks below 200 MeV/c"; reading A46 -- the paper prints no rule): the tracks
 * of one sector that are successive turns of one looping particle (same circle in the pad plane, displaced along z by whole pitches).
 * One entry per track of the last tpc_find_tracks* call.  Library-owned, host (device_result = 0) or device memory. */
typedef struct {
  int64_t n_tracks;
  const int32_t* prev;      /* [n_tracks] the track that is an earlier turn of the same particle (the nearest one found), -1 = none */
  const int32_t* root;      /* [n_tracks] first turn of the group (the track itself if it follows nobody) */
  const int32_t* turn;      /* [n_tracks] number of turns after the root (0 for a root) */
  float ms_loopers;         /* device time of K10 (CUDA events on the context's stream), ms */
} tpc_loopers;

/* Per-step device times of the last tpc_find_tracks* call (CUDA events on the context's stream), ms. */
typedef struct {
  float ms_upload;          /* host staging -> device (0 if the clusters were already device-resident) */
  float ms_grid;            /* K1: S0 + S1 */
  float ms_neighbours;      /* K2: S2 */
  float ms_clean_start;     /* K3: S3 + S4 (clean, flag, scan, compact) */
  float ms_tracklets;       /* K5: S5 */
  float ms_selector;        /* K6: S6 (owner keys, count, scan, emit) */
  float ms_download;        /* device -> host copy of the tracks (0 for tpc_find_tracks_device) */
  float ms_total;           /* first event to last event */
  int64_t n_clusters, n_bins, n_start_hits, n_tracklets_kept, n_tracks, n_cluster_refs;
  int64_t launches;         /* number of kernels of this library launched by the call */
  int64_t n_propagations, n_updates, n_pickups;   /* S5 work counters: helix transports, Kalman updates, grid pick-ups */
} tpc_timings;

/* One (sector,row) of the S1 grid, host copies (library-owned), for parity tests. */
typedef struct {
  int32_t n, ny, nz;
  float y_lo, z_lo, inv_s;
  const float* yz;          /* [n][2] sorted (y, z) */
  const int32_t* perm;      /* [n] sorted position -> index in the caller's arrays */
  const int32_t* bin_start; /* [ny*nz+1] */
} tpc_grid_view;

/* All tracklets of the last call (S5 output before selection), host copies (library-owned). rowhit is [n_rows][n_tracklets]
 * (row-major over rows), -1 = no cluster; entries outside [first_row, last_row] are -1. */
typedef struct {
  int64_t n_tracklets;
  const int32_t* sector; const int32_t* start_row; const int32_t* n_hits; const int32_t* first_row; const int32_t* last_row;
  const float* chi2; const float* x; const float* par; const float* cov;
  const int32_t* rowhit;
} tpc_tracklet_view;

/* Create a context: copies the geometry, computes the per-row constant tables, selects the current CUDA
 * device.  bz_tesla: uniform solenoid field along z; vdrift_cm_per_us: average drift velocity used by S0. */
int tpc_create(const tpc_geometry* geometry, float bz_tesla, float vdrift_cm_per_us, tpc_ctx** out);

/* Tunables of DESIGN.md table T by name: wy wz dzdx_max wz0 cut2 min_seed c0_y c0_z c0_sinphi c0_dzds c0_qpt s_max n_sigma
 * w_max max_gap edge_margin min_hits grid_scale, plus debug_keep (1 = keep pre-cleaning link tables for tpc_debug_get_links) and
 * link_skip (default 0; 1 = S2', the gap-tolerant seeding variant of SURVEY.md section 8(f).2: a cluster without an accepted pair on
 * the adjacent rows may link over one missing row; changes the result; skip_cut2 = cut2 of the pairs that
 * skip a row, default 1.75 = cut2, 0.4375 keeps the efficiency of the default path), bridge_rows / bridge_min /
 * bridge_rescue (seed-bridging variants, readings A39 / A39c; ignored with link_skip), and
 * pinned_async (default 0; 1 = a PINNED host source of tpc_load_clusters* is read by DMA on the context's stream AFTER the load call
 * has returned: the caller then keeps those buffers untouched until the next tpc_find_tracks* on the context returns.  With 0 the
 * load call returns only when the library has read its inputs, as the conventions above state).
 * Only before the first load after tpc_create / tpc_clear. */
int tpc_set_param(tpc_ctx*, const char* name, double value);

/* CUDA stream (cudaStream_t as void*) on which all device work of this context is issued, e.g.
 * torch.cuda.current_stream().cuda_stream.  NULL = default stream. */
int tpc_set_stream(tpc_ctx*, void* cuda_stream);

/* Load the clusters of one pad row of one sector: pad_y (cm), time (us) and charge fp32 arrays of length n, host or device
 * (all three of the same kind).  charge is accepted for interface completeness and never read on this path (may be NULL).
 * A second load for the same (sector,row) replaces the first; any order; a (sector,row) never loaded is empty.  No kernel is
 * launched here: the arrays are staged (pinned host arena, one H2D copy at tpc_find_tracks; device arrays: one D2D copy). */
int tpc_load_clusters(tpc_ctx*, int sector, int row, const float* pad_y, const float* time, const float* charge, int n);

/* Same for a whole event / time frame in one call: unit_off is a HOST array of n_sectors*n_rows+1 ascending offsets
 * (unit = sector*n_rows+row) into pad_y / time / charge (host or device).  Replaces everything loaded before. */
int tpc_load_clusters_batch(tpc_ctx*, const int64_t* unit_off, const float* pad_y, const float* time, const float* charge);

/* Run S0..S6 on everything loaded.  out: host arrays (see tpc_tracks). */
int tpc_find_tracks(tpc_ctx*, tpc_tracks* out);
/* Same, but the result arrays stay in device memory (only the two counts are read back). */
int tpc_find_tracks_device(tpc_ctx*, tpc_tracks* out);

/* S7: refit every track of the last tpc_find_tracks* call over the clusters it owns and estimate its collision time.
 * Errors: TPC_E_ARG (null), TPC_E_STATE (no completed tpc_find_tracks* call on this context), TPC_E_NOMEM, TPC_E_CUDA. */
int tpc_refit_tracks(tpc_ctx*, int device_result, tpc_refit* out);

/* S8: attachment status of every cluster with respect to the tracks of the last tpc_find_tracks* call; tube_cm > 0 (the paper: 1.5).
 * Errors: TPC_E_ARG (null, tube_cm not > 0 or not finite), TPC_E_STATE (no completed tpc_find_tracks* call), TPC_E_NOMEM, TPC_E_CUDA. */
int tpc_mark_clusters(tpc_ctx*, float tube_cm, int device_result, tpc_cluster_marks* out);

/* S9: match track segments across sector boundaries (tunables merge_edge, merge_rows, merge_dy, merge_dz, merge_ds, merge_dt).
 * Errors: TPC_E_ARG (null), TPC_E_STATE (no completed tpc_find_tracks* call), TPC_E_NOMEM, TPC_E_CUDA. */
int tpc_merge_tracks(tpc_ctx*, int device_result, tpc_merges* out);

/* S10: group the tracks of the last tpc_find_tracks* call that are turns of one looping particle (tunables loop_qmin [c/GeV, 5 = 200
 * MeV/c], loop_dy, loop_ds, loop_dt, loop_dq, loop_pmin, loop_frac, loop_nmax [1..255]).
 * Errors: TPC_E_ARG (null), TPC_E_STATE (no completed tpc_find_tracks* call), TPC_E_NOMEM, TPC_E_CUDA. */
int tpc_find_loopers(tpc_ctx*, int device_result, tpc_loopers* out);

/* S10 for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): the
 * same kernels and the same result as tpc_find_loopers (reading A46; "secondary legs of looping tracks
 * below 200 MeV/c"), but the call allocates NOTHING -- no cudaMalloc / cudaFree, no growth of a library buffer -- and does not
 * synchronise: the four launches are queued on the context's stream and the call returns.
 * Inputs (DEVICE memory, caller-owned, read on the stream): sector [n_tracks] in ascending order (as tpc_find_tracks* returns them,
 * each in 0 .. n_sectors-1), x [n_tracks], par [n_tracks][5] (y, z, sin phi, dz/ds, q/pT) -- e.g. the arrays of tpc_find_tracks_device.
 * Outputs (DEVICE memory, caller-owned, n_tracks int32 each): prev = previous turn of the same particle (-1 none), root = first turn
 * of the group, turn = turns after the root.  Valid once the stream has reached the end of the call's work.
 * Scratch: one file-scope static __device__ array of the library (2 MiB + 8 KiB; every GPU that loads the library holds it until the
 * process exits), which bounds the size: n_tracks <= TPC_NOALLOC_MAX_TRACKS and n_sectors <= 1022.  ALL calls on a device share that
 * array, whichever context or stream they use: calls whose work overlaps on the GPU (two streams, or two contexts on different
 * streams) race on it and give undefined results -- keep them on one stream or order them with events.  The array keeps the previous
 * call's contents; the per-sector counters in it, the only words that must start at zero, are zeroed by the first kernel of every call,
 * and no other word is read before the same call has written it.
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress, no allocation); make one call before a
 * graph capture begins.  The current CUDA device must be the one the context was created on.
 * Needs no preceding tpc_find_tracks*: field, s_max and the loop_* tunables are taken from the context.
 * Errors: TPC_E_ARG (null context / array, negative n_tracks, an array that is not device memory), TPC_E_CAPACITY (n_tracks or
 * n_sectors beyond the limit: nothing is launched), TPC_E_STATE (another device is current), TPC_E_CUDA.  n_tracks = 0 is a no-op. */
#define TPC_NOALLOC_MAX_TRACKS 262144
int tpc_find_loopers_noalloc(tpc_ctx*, int64_t n_tracks, const int32_t* d_sector, const float* d_x, const float* d_par,
                             int32_t* d_prev, int32_t* d_root, int32_t* d_turn);

/* Forget the clusters and results, keep geometry, parameters and buffers (one call per event / time frame). */
int tpc_clear(tpc_ctx*);
void tpc_destroy(tpc_ctx*);
const char* tpc_last_error(const tpc_ctx*);   /* never NULL; ctx may be NULL (message of the last failed tpc_create) */

int tpc_get_timings(tpc_ctx*, tpc_timings* out);

/* Measurement utility for bench.py ("builder measures an FMA-loop peak"): fp32 fused-multiply-add throughput of
 * the device at the clocks of the moment, in TFLOP/s (2 flops per FMA; 8 independent chains per thread, 2048 threads per SM).  It is
 * the denominator of the roofline of the ALU-bound kernels; not part of the tracking path. */
int tpc_measure_fp32_peak(tpc_ctx*, float* tflops);

/* Parity / debug exports of the last tpc_find_tracks* call (host copies, library-owned, valid until the next call on the context). */
int tpc_debug_get_grid(tpc_ctx*, int sector, int row, tpc_grid_view* out);
/* cleaned = 0: S2 tables (needs debug_keep = 1), 1: after S3.  up/dn: [n] positions in the sorted order of row+1 / row-1, -1 = none. */
int tpc_debug_get_links(tpc_ctx*, int sector, int row, int cleaned, const int32_t** up, const int32_t** dn, int32_t* n);
/* Row distance of the links returned by the LAST tpc_debug_get_links call: 1 for a link to the adjacent row, 2 for a link that skips
 * a row (only with tpc_set_param("link_skip", 1): S2' of DESIGN.md reading A45), 0 where there is no link.  [n] entries each. */
int tpc_debug_get_link_rows(tpc_ctx*, const int8_t** up_k, const int8_t** dn_k, int32_t* n);
/* start hits in list order: unit = sector*n_rows+row and sorted position. */
int tpc_debug_get_start_hits(tpc_ctx*, const int32_t** unit, const int32_t** pos, int64_t* n);
int tpc_debug_get_tracklets(tpc_ctx*, tpc_tracklet_view* out);

/* Version of the ABI (incremented on incompatible change). */
int tpc_abi_version(void);
/* 1 if this library was built with -DTPC_CHECKED (libtpc_b200_checked.so: every data-dependent gather / scatter index in the kernels is
 * bounds-checked and a failure makes tpc_find_tracks* return TPC_E_CUDA), 0 for the product build. */
int tpc_checked_build(void);

#ifdef __cplusplus
}
#endif
#endif /* TPC_B200_TPC_H_ */
