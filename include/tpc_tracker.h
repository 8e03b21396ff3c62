/*
 * tpc_tracker.h - C ABI of the B200-native TPC sector track finder.
 *
 * The operation: "Track Finding" of the ALICE Run 3 synchronous TPC chain (Table 1;
 * PAPER.md:99, section 6: "the TPC tracking runs first standalone without such corrections"), on a
 * whole time frame resident in GPU memory.  The paper names the step and defers
 * the algorithm to references that are not available; the five stages (sort+bin, neighbours finder,
 * link cleaner, Kalman tracklet constructor, selector) are those of BASELINE.json `north_star`, and
 * every formula is the reading fixed in DESIGN.md section 3.
 *
 * Plain pointers and sizes only.  Every pointer below says HOST or DEVICE.  The library allocates no
 * device memory: inputs, outputs and one workspace arena are the caller's (PyTorch tensors in this
 * repository).  All work is enqueued on the caller's CUDA stream; unless stated, calls do not
 * synchronise.  There is no CPU fallback: every stage runs in the library's sm_100a kernels.
 *
 * Host resources a handle owns (created by tpc_tracker_create, released by tpc_tracker_destroy): the
 * host struct; 6 CUDA events for the per-stage timing; and, only when created with host_io >= 2,
 * three non-blocking CUDA streams (upload, compute, download), 4 events per staging slot and one
 * 48-byte pinned host block the frame counts are copied into; and, after tpc_tracker_enable_graph, one CUDA graph executable.
 *
 * Thread safety: a handle is NOT thread-safe.  Every call on a handle mutates it (the input pointers of
 * the current frame, the last stream, the slot states), so all calls on one handle must come from one
 * thread at a time; different handles (each with its own workspace) are independent and may be used
 * from different threads or streams concurrently.  tpc_error_string and tpc_tracker_workspace_bytes
 * touch no handle and are thread-safe.
 *
 * Call order: tpc_tracker_refit, _merge, _apex and _removable work on the frame of the LAST track call on the handle
 * and read what their predecessors left in the workspace, so each returns INVALID_ARG unless its predecessors ran after
 * that track call: refit needs a tracked frame, merge the refit, apex the merge, removable the merge and the apex.
 *
 * Error behaviour: functions return 0 (TPC_OK) or a negative tpc_error code; device-detected
 * conditions (bad sector/row value, capacity overflow) are reported through the 32-bit status word
 * (tpc_tracks_t.status, tpc_counters_t.status) as a bit set of TPC_STATUS_*; when a status bit is
 * set the run is aborted on the device and n_tracks = 0 - outputs are never silently truncated.
 */
#ifndef TPC_TRACKER_H_
#define TPC_TRACKER_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define TPC_API __attribute__((visibility("default")))
#else
#define TPC_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

enum tpc_error {
  TPC_OK = 0,
  TPC_ERR_INVALID_ARG = -1, /* null pointer, negative size, unsupported geometry (n_rows > 256, ...) */
  TPC_ERR_CAPACITY = -2,    /* workspace too small for the requested capacities, n > max_clusters */
  TPC_ERR_CUDA = -3,        /* a CUDA runtime call or kernel launch failed (cudaGetLastError) */
  TPC_ERR_STATIC_SCRATCH = -4 /* tpc_tracker_protect_static only: the frame has more clusters than the scratch array built
                                 into the library holds (TPC_PROTECT_STATIC_MAX_CLUSTERS); nothing was enqueued */
};

enum tpc_status_bits {
  TPC_STATUS_BAD_CLUSTER = 1,      /* a cluster had sector >= n_sectors, row >= n_rows, or a non-finite y or z */
  TPC_STATUS_BINS_OVERFLOW = 2,    /* the (y,z) grids need more than max_bins bins (or > INT32_MAX) */
  TPC_STATUS_SEEDS_OVERFLOW = 4,   /* more than max_seeds chain heads qualified as seeds */
  TPC_STATUS_TRACKS_OVERFLOW = 8,  /* more than max_tracks tracks or max_track_clusters attached clusters */
  TPC_STATUS_CHAIN_CYCLE = 16      /* internal consistency: a link chain longer than n_rows (cannot happen) */
};

typedef struct tpc_tracker tpc_tracker_t; /* opaque; owned by the library, freed by tpc_tracker_destroy */

/*
 * Geometry, field and cuts.  POD, copied at create.  The per-row derived
 * tables (ymax_r, ny_r, link windows) are computed by the library on the host in fp32 from these
 * values, each with the one expression stated in DESIGN.md section 3.0.
 */
typedef struct {
  int32_t n_sectors;        /* <= 256 (sector ids are uint8); 36 for the ALICE TPC */
  int32_t n_rows;           /* <= 256 (row ids are uint8); n_sectors*n_rows <= 65535; 152 */
  const float* row_x;       /* HOST, n_rows values, strictly increasing, cm: pad-row radius x_r */
  float tan_half_sector;    /* tan(10 deg) */
  float bz_tesla;           /* solenoid field; curvature = -0.00299792458 * bz * (q/pT) [1/cm] */
  float err_y2, err_z2;     /* cluster variances, cm^2 */
  float cell_y, cell_z;     /* (y,z) grid cell, cm (> 0) */
  float link_ay, link_az, link_b, link_T; /* S2 window slopes / offset and the link cut (section 3.2) */
  int32_t min_chain_len;    /* S3: seeds are chains of at least this many clusters (>= 2) */
  int32_t max_gap;          /* S4: rows without a cluster before a tracklet stops */
  int32_t min_tracklet_hits;/* S4: tracklets with fewer hits are dropped */
  int32_t min_track_hits;   /* S5: tracks must own at least this many clusters */
  float pick_chi2_cut;      /* S4 pick-up gate */
  float max_sinphi;         /* S4 propagation limit */
  float y_margin;           /* S4 sector-exit margin, cm */
  float init_c_ss, init_c_tt, init_c_qq; /* S4 initial variances of sin(phi), tan(lambda), q/pT */
  /* Native time input ("the TPC hits cannot be converted from native pad, row, and time coordinates
   * into x, y, and z coordinates ahead of time").  z_is_time = 0: tpc_clusters_t.z is the pseudo-z
   * in cm and the two values below are ignored.  z_is_time != 0: tpc_clusters_t.z holds the cluster TIME in time units
   * counted from the start of the time frame, and S1 computes the pseudo-z itself, in fp32, while it reads the input
   * (no extra pass): zc = drift_length - t * cm_per_time_unit (two roundings), z = zc on the A side (sector <
   * n_sectors / 2) and 0 - zc on the C side.  cm_per_time_unit = drift velocity x length of a time unit (> 0, finite). */
  int32_t z_is_time;
  float cm_per_time_unit;
  float drift_length;       /* cm, full drift length of one side (250) */
  /* Native pad input (same passage of the paper).  y_is_pad = 0: tpc_clusters_t.y is the
   * sector-local y in cm and the two tables below are ignored (may be NULL).  y_is_pad != 0: tpc_clusters_t.y holds the PAD
   * coordinate p of the cluster in its row (pad centres at 0 .. n_pads[row] - 1, fractional for a centroid) and S1 computes
   * y itself, in fp32, while it reads the input (no extra pass): y = (p - 0.5 * (n_pads[row] - 1)) * pad_pitch[row], the
   * difference and the product rounded separately (pads symmetric about the sector axis, y growing with the pad number).
   * Together with z_is_time this is the detector's (pad, row, time) input. */
  int32_t y_is_pad;
  const int32_t* n_pads;    /* HOST, n_rows values >= 1: pads of each row (copied at create) */
  const float* pad_pitch;   /* HOST, n_rows values > 0, finite: pad width of each row, cm (copied at create) */
} tpc_params_t;

/* Input clusters of one time frame, SoA.  DEVICE pointers for tpc_track_timeframe, HOST pointers
 * (ideally pinned) for tpc_track_timeframe_host.  Read-only; must stay valid until the stream has
 * finished the call.  `x` may be NULL and is not read: the tracker uses row_x[row] (pad-row centre).
 * `z` is the pseudo-z in cm computed with vertex time 0 (continuous readout) - or, when
 * tpc_params_t.z_is_time is set, the cluster time in time units (the tracker converts it, see there).
 * Preconditions: coordinates finite; 0 <= n <= max_clusters; DEVICE arrays aligned like fresh
 * allocations (sector and row to 4 bytes, y and z to 16 bytes - the kernels use vector loads), else
 * INVALID_ARG. */
typedef struct {
  int64_t n;
  const uint8_t* sector; /* [n] */
  const uint8_t* row;    /* [n] */
  const float* x;        /* [n] or NULL (unused) */
  const float* y;        /* [n] sector-local y, cm (y_is_pad = 0) or pad coordinate (y_is_pad != 0) */
  const float* z;        /* [n] pseudo-z, cm (z_is_time = 0) or time, time units (z_is_time != 0) */
} tpc_clusters_t;

/* Output tracks, SoA, caller-allocated with the stated capacities.  DEVICE pointers for
 * tpc_track_timeframe, HOST pointers for tpc_track_timeframe_host.  Track ids are 0..n_tracks-1 in
 * ascending order of the seed's sorted position (deterministic).
 * par  : [5][max_tracks]  (y, z - z_ref, sin(phi), tan(lambda), q/pT) at x_ref; par[i*max_tracks + t]
 * cov  : [15][max_tracks] lower triangle, row-major (c00,c10,c11,c20,...,c44); cov[m*max_tracks + t]
 * trk_cl_start : [max_tracks+1] CSR offsets into trk_cl_idx
 * trk_cl_idx   : [max_track_clusters] INPUT indices of the track's clusters, ascending row
 * cluster_track: [clusters.n] track id of every input cluster, -1 if unassigned */
typedef struct {
  int64_t max_tracks;
  int64_t max_track_clusters;
  int32_t* n_tracks;      /* [1] */
  int32_t* status;        /* [1] bit set of tpc_status_bits, 0 = fine */
  int32_t* sector;        /* [max_tracks] */
  int32_t* first_row;     /* [max_tracks] lowest owned row */
  int32_t* last_row;      /* [max_tracks] highest owned row */
  int32_t* n_clusters;    /* [max_tracks] owned clusters */
  float* par;
  float* cov;
  float* x_ref;           /* [max_tracks] x of the plane the parameters are given at */
  float* z_ref;           /* [max_tracks] z offset: absolute z = par[1] + z_ref */
  float* chi2;            /* [max_tracks] */
  int32_t* ndf;           /* [max_tracks] 2*n_hits(tracklet) - 5 */
  int32_t* trk_cl_start;
  int32_t* trk_cl_idx;
  int32_t* cluster_track;
  float* z_beam;          /* [max_tracks] pseudo-z of the track at the beam line, assuming a primary from the origin
                           * (DESIGN.md section 3.6): vertex time = -+ z_beam / v_drift on the A / C side */
} tpc_tracks_t;

/* Small counter block read back by tpc_tracker_counters (sizes of the last run). */
typedef struct {
  int64_t n_clusters;
  int64_t n_bins;        /* N_b: grid bins over all (sector,row) */
  int64_t n_seeds;       /* K_s: chains that qualified as seeds */
  int64_t n_tracklets;   /* K: tracklets kept by S4 */
  int64_t n_tracks;      /* T_k */
  int64_t n_track_clusters; /* clusters attached to tracks */
  int64_t n_linked;      /* clusters with a cleaned up-link (chain edges) */
  int64_t kf_steps;      /* S: Kalman propagate calls */
  int64_t n_hits;        /* H: hits over all kept tracklets */
  int32_t status;
  int32_t s1_global_buckets; /* (sector,row) buckets whose bin sort took the global-memory path (a slab did not fit shared memory) */
} tpc_counters_t;

/* Debug views into the workspace, valid until the next track call on the handle (DEVICE pointers).
 * All positions are indices into the sorted order of S1. */
enum tpc_stage_array {
  TPC_VIEW_PERM = 0,        /* int32 [n]      sorted position -> input index (S1) */
  TPC_VIEW_YZ = 1,          /* float [n][2]   sorted (y, z) pairs */
  TPC_VIEW_SROW = 2,        /* uint16 [n]     (sector << 8) | row of the sorted cluster    */
  TPC_VIEW_BIN_START = 3,   /* int32 [n_bins+1] CSR over global bins */
  TPC_VIEW_ROW_START = 4,   /* int32 [n_sectors*n_rows+1] */
  TPC_VIEW_BIN_BASE = 5,    /* int32 [n_sectors*n_rows+1] first global bin of each (sector,row) */
  TPC_VIEW_ZMIN = 6,        /* float [n_sectors] */
  TPC_VIEW_ZMAX = 7,        /* float [n_sectors] */
  TPC_VIEW_NZ = 8,          /* int32 [n_sectors] */
  TPC_VIEW_LINK_UP_RAW = 9, /* int32 [n] (S2) */
  TPC_VIEW_LINK_DN_RAW = 10,
  TPC_VIEW_LINK_UP = 11,    /* int32 [n] cleaned (S3) */
  TPC_VIEW_LINK_DN = 12,
  TPC_VIEW_SEED_HEAD = 13,  /* int32 [n_seeds] */
  TPC_VIEW_SEED_LEN = 14,   /* int32 [n_seeds] */
  TPC_VIEW_T_HIT = 15,      /* int32 [n_seeds][n_rows] sorted position or -1 (S4); row r of seed k is
                               defined only for t_first_row[k] <= r <= t_last_row[k] (no hits outside) */
  TPC_VIEW_T_FIRST_ROW = 16,/* int32 [n_seeds] */
  TPC_VIEW_T_LAST_ROW = 17, /* int32 [n_seeds] */
  TPC_VIEW_T_N_HITS = 18,   /* int32 [n_seeds] */
  TPC_VIEW_T_PAR = 19,      /* float [n_seeds][5] */
  TPC_VIEW_T_COV = 20,      /* float [n_seeds][15] */
  TPC_VIEW_T_CHI2 = 21,     /* float [n_seeds] */
  TPC_VIEW_T_ZREF = 22,     /* float [n_seeds] */
  TPC_VIEW_TRACKLET_OF_SEED = 23, /* int32 [n_seeds] rank among kept tracklets or -1 (S5) */
  TPC_VIEW_OWNED = 24,      /* int32 [n_seeds] clusters owned (S5) */
  /* S7 / S9 (valid after tpc_tracker_refit / tpc_tracker_merge; per track) */
  TPC_VIEW_FIT_ROW = 25,    /* int32 [n_tracks] row of the state of the downward refit */
  TPC_VIEW_UP_PAR = 26,     /* float [5][max_tracks] state at the outer end (upward refit) */
  TPC_VIEW_UP_COV = 27,     /* float [15][max_tracks] */
  TPC_VIEW_UP_X = 28,       /* float [n_tracks] */
  TPC_VIEW_UP_ZREF = 29,    /* float [n_tracks] */
  TPC_VIEW_UP_ROW = 30,     /* int32 [n_tracks] */
  TPC_VIEW_UP_N = 31,       /* int32 [n_tracks] */
  TPC_VIEW_MRG_BEST_B = 32, /* int32 [n_tracks] best partner of the outer end or -1 (3.9.5) */
  TPC_VIEW_MRG_BEST_A = 33, /* uint64 [n_tracks] (ordered key of chi2 << 32) | best partner of the inner end; all ones = none */
  TPC_VIEW_MRG_CHI_B = 34,  /* float [n_tracks] chi2 of best_b or -1 */
  TPC_VIEW_MRG_NEXT = 35,   /* int32 [n_tracks] link to the next segment outwards or -1 (3.9.6) */
  TPC_VIEW_MRG_PREV = 36,   /* int32 [n_tracks] */
  TPC_VIEW_MRG_DIR = 37,    /* int32 [n_tracks] 0 same sector, +-1 the neighbour the link goes to */
  TPC_VIEW_APEX_BEST = 38,  /* int32 [max_tracks] best apex partner of every merged track or -1 (3.9.8); first n_merged valid */
  TPC_VIEW_APEX_SCORE = 39, /* float [max_tracks] its score or -1 */
  TPC_VIEW_COUNT_ = 40
};

typedef struct {
  const void* ptr;     /* DEVICE */
  int64_t n;           /* elements (synchronises the stream of the last call to read device counters) */
  int32_t elem_bytes;
  int32_t is_float;
} tpc_stage_view_t;

/* Bytes of DEVICE workspace the tracker needs for the given capacities.  `host_io` = 1 adds the
 * staging buffers tpc_track_timeframe_host uses (inputs for max_clusters, outputs for max_tracks /
 * max_track_clusters); `host_io` = 2 or 3 adds that many sets for the pipelined begin/end pair (0 <= host_io <= 3).  Returns 0 on invalid arguments. */
TPC_API size_t tpc_tracker_workspace_bytes(const tpc_params_t* params, int64_t max_clusters, int64_t max_bins,
                                   int64_t max_seeds, int64_t max_tracks, int64_t max_track_clusters,
                                   int32_t host_io);

/* Creates a tracker on the current CUDA device for the method of DESIGN.md section 3 ("Track Finding",
 * PAPER.md:137 Table 1; the whole time frame is processed at once in GPU memory that is reused across
 * consecutive steps, PAPER.md:117-119 - hence ONE caller-owned arena carved once).  `d_workspace`
 * (DEVICE, 256-byte aligned, at least workspace_bytes long) stays owned by the caller and must outlive
 * the handle.  Derives the per-row tables on the host and uploads them
 * (synchronous).  `host_io` as above.  Errors: INVALID_ARG (null / out-of-range parameters, unaligned
 * workspace), CAPACITY (workspace_bytes too small), CUDA.  On failure *out = NULL and nothing is leaked.
 * Differs from SURVEY.md section 8(b)'s sketch by two more capacities (max_tracks, max_track_clusters: the
 * staging buffers of the host path are sized by them) and by host_io. */
TPC_API int tpc_tracker_create(const tpc_params_t* params, int64_t max_clusters, int64_t max_bins, int64_t max_seeds,
                       int64_t max_tracks, int64_t max_track_clusters, int32_t host_io, void* d_workspace,
                       size_t workspace_bytes, tpc_tracker_t** out);

/* The hot path: enqueues stages S1..S5 (DESIGN.md sections 3.1-3.5; BASELINE.json north_star (1)-(5);
 * "the TPC tracking runs first standalone without such corrections") for one time frame on
 * `cuda_stream` (a cudaStream_t; NULL = default stream).  DEVICE pointers in `in` and `out`.  Does not
 * synchronise; counts and status stay on the device (out->n_tracks, out->status).
 * out->max_tracks / max_track_clusters must not exceed the capacities given at create (CAPACITY);
 * null or misaligned pointers, n < 0: INVALID_ARG; a failed launch: CUDA.  Device-detected conditions
 * arrive in out->status (see tpc_status_bits), never as a silently truncated result. */
TPC_API int tpc_track_timeframe(tpc_tracker_t* t, const tpc_clusters_t* in, const tpc_tracks_t* out, void* cuda_stream);

/* CUDA graph of the hot path (off by default).  When enabled, tpc_track_timeframe on a non-default stream captures its
 * launch sequence (S1..S5: 29 launches, every grid sized by host-known quantities, every length device-resident) into a
 * CUDA graph the first time and replays the cached executable while n and every pointer of `in` / `out` stay the same; a
 * call with other arguments re-captures.  Worth 0.05 - 0.07 ms per call (5 - 7 % of the small configurations, whose floor
 * is the serial depth of one tracklet; nothing on a full time frame).  Not used while stage timing is on, on the default
 * stream, by the host paths, or when `cuda_stream` is already being captured by the caller (the launches then go into
 * the caller's capture as they are).  The handle owns the graph executable (released by tpc_tracker_destroy). */
TPC_API int tpc_tracker_enable_graph(tpc_tracker_t* t, int32_t enable);

/* Same from/to HOST buffers (tracker created with host_io != 0): copies the SoA input to the device,
 * runs S1..S5, copies n_tracks, status, the track list, the CSR and cluster_track back, all on
 * `cuda_stream`, then synchronises that stream.  On the host paths (this call and the begin / end pair)
 * out->cluster_track may be NULL: the per-cluster assignment is then not copied back (4 bytes per input cluster,
 * 39 % of the download on a Pb-Pb time frame; the CSR trk_cl_start / trk_cl_idx carries the same information).  Copy sizes of the outputs are bounded by the
 * capacities; the per-track arrays are copied for the n_tracks tracks found. */
TPC_API int tpc_track_timeframe_host(tpc_tracker_t* t, const tpc_clusters_t* in, const tpc_tracks_t* out, void* cuda_stream);

/* Refitted tracks (DEVICE pointers, caller-allocated for max_tracks tracks; layouts as in tpc_tracks_t). */
typedef struct {
  int64_t max_tracks;
  float* par;        /* [5][max_tracks] */
  float* cov;        /* [15][max_tracks] */
  float* x_ref;      /* [max_tracks] x of the lowest fitted row */
  float* z_ref;      /* [max_tracks] z of the top owned cluster: absolute z = par[1] + z_ref */
  float* chi2;       /* [max_tracks] */
  int32_t* ndf;      /* [max_tracks] 2*n_fit - 5 */
  int32_t* n_fit;    /* [max_tracks] clusters that entered the fit */
  /* optional (all three NULL to skip): residual of every owned cluster to the extrapolated track position
   * (DESIGN.md section 3.7), parallel to tpc_tracks_t.trk_cl_idx of the call; 0 for the top cluster of a
   * track and for clusters that did not enter the fit */
  const int32_t* trk_cl_start; /* [n_tracks+1] the call's tpc_tracks_t.trk_cl_start (DEVICE) */
  float* res_y;      /* [max_track_clusters of the call] cm */
  float* res_z;      /* [max_track_clusters of the call] cm */
  /* optional (both NULL to skip; need the three fields above): the same residuals as signed 16-bit counts of steps
   * (DESIGN.md section 3.7a): q = rint(res * (1 / step)) in fp32, ties to even, saturated at +-32767;
   * decoding q * step is within step / 2 of the residual.  res_step_y / res_step_z: cm, finite, > 0 (0.01 = 0.1 mm). */
  int16_t* qres_y;   /* [max_track_clusters of the call] */
  int16_t* qres_z;   /* [max_track_clusters of the call] */
  float res_step_y, res_step_z;
} tpc_fit_t;

/* Refit of every track of the LAST tpc_track_timeframe call on this handle over the clusters it owns after the
 * selector, top row downwards (the first slice of "Track Fit").  Enqueued on
 * `cuda_stream`, which must be ordered after that call; does not synchronise; entries [0, n_tracks) are written.
 * Not part of tpc_track_timeframe (and not of the timed hot path).  CAPACITY if out->max_tracks exceeds the tracker's or
 * is smaller than the max_tracks of that tpc_track_timeframe call (every track it may have found must fit: this call and
 * the four below never cut a result off silently; the same rule holds for every max_tracks they are given). */
TPC_API int tpc_tracker_refit(tpc_tracker_t* t, const tpc_fit_t* out, void* cuda_stream);

/* Cuts of the track merger. */
typedef struct {
  int32_t max_rows;   /* a continuation starts at most this many rows above the outer end (30) */
  int32_t back_rows;  /* ... and, in a neighbouring sector, at most this many rows below it (1) */
  float edge;         /* cm: a neighbour is tried only if the outer end lies within `edge` of the sector boundary (6) */
  float dz_win;       /* cm: |z_in(B) - z_out(A)| window of the candidates (50); > 0 */
  float chi2_cut;     /* candidates need chi2 <= chi2_cut over the five parameters (100) */
  float road_z0;      /* cm: z road around the straight continuation of the outer state, |dz| <= road_z0 + road_z1 |dx| (2) */
  float road_z1;      /* cm per cm (0.3) */
} tpc_merge_cuts_t;

/* Merged tracks (DEVICE pointers, caller-allocated for max_tracks entries each; layouts as in tpc_tracks_t).
 * Tracks = the segments found by tpc_track_timeframe; a merged track is a chain of them, inner to outer. */
typedef struct {
  int64_t max_tracks;
  int32_t* n_merged;         /* [1] */
  int32_t* merged_of_track;  /* [max_tracks] merged id of every track */
  int32_t* seg_start;        /* [max_tracks+1] CSR merged track -> its tracks */
  int32_t* seg_idx;          /* [max_tracks] track ids, inner to outer */
  float* par;                /* [5][max_tracks] merged refit, state at x_ref in the frame of `sector` */
  float* cov;                /* [15][max_tracks] */
  float* x_ref;              /* [max_tracks] */
  float* z_ref;              /* [max_tracks] z of the outermost cluster: absolute z = par[1] + z_ref */
  float* chi2;               /* [max_tracks] */
  int32_t* ndf;              /* [max_tracks] 2*n_fit - 5 */
  int32_t* n_fit;            /* [max_tracks] clusters that entered the merged fit */
  int32_t* sector;           /* [max_tracks] sector whose frame the state is given in (the innermost one reached) */
  int32_t* n_clusters;       /* [max_tracks] clusters of all segments */
} tpc_merged_t;

/* Track merger (the second slice of "Track Fit"): joins the tracks of the
 * LAST tpc_track_timeframe call on this handle that continue each other - across a sector border or across a hole of
 * more than max_gap rows - and refits every merged track over all its clusters (upward pass for the outer-end states,
 * downward pass through all segments with the frame turned at sector changes).  `fit` is the output of the
 * tpc_tracker_refit call that followed that tpc_track_timeframe (DEVICE; its residual fields are not used).  Enqueued on
 * `cuda_stream`, which must be ordered after both; does not synchronise; entries [0, n_merged) / [0, n_tracks) are written.
 * INVALID_ARG for null pointers or cuts out of range, CAPACITY if a max_tracks (fit, out) exceeds the tracker's or is smaller
 * than the max_tracks of that tpc_track_timeframe call. */
TPC_API int tpc_tracker_merge(tpc_tracker_t* t, const tpc_fit_t* fit, const tpc_merge_cuts_t* cuts, const tpc_merged_t* out,
                              void* cuda_stream);

/* Cuts of the apex links. */
typedef struct {
  int32_t max_k;   /* sectors the unseen arc around the apex may span (4) */
  float min_s;     /* a tail takes part iff |sin(phi)| of its outer state >= min_s (0.6) */
  float dz_win;    /* cm: |z_out(B) - z_out(A)| window (150); > 0 */
  float tol_c;     /* tolerance of the circle centres, as a fraction of the radius (0.1); > 0 */
  float tol_z;     /* cm: tolerance of the z advance along the arc between the two ends (4); > 0 */
  float tol_t;     /* tolerance of tan(lambda)_A + tan(lambda)_B (0.1); > 0 */
  float cut;       /* partners need score <= cut (3) */
} tpc_apex_cuts_t;

typedef struct {
  int64_t max_tracks;
  int32_t* apex_partner;  /* [max_tracks] per merged track: the merged track that is the other leg of the same looper, or -1 */
  int32_t* apex_leg;      /* [max_tracks] 1 = the returning ("secondary") leg of its pair, else 0 */
} tpc_apex_t;

/* Looper following ("secondary legs of looping tracks", "the following
 * of looping tracks"): pairs the merged tracks of the LAST tpc_tracker_merge call on this handle that are the outgoing
 * and the returning leg of one track curling up inside the TPC, by comparing the circles of their outermost states, and
 * labels the returning leg.  `merged` is that call's output (DEVICE; seg_start / seg_idx are read).  Enqueued on
 * `cuda_stream`, ordered after the merge; does not synchronise; entries [0, n_merged) are written.  CAPACITY as for
 * tpc_tracker_merge (merged, out). */
TPC_API int tpc_tracker_apex(tpc_tracker_t* t, const tpc_merged_t* merged, const tpc_apex_cuts_t* cuts, const tpc_apex_t* out,
                             void* cuda_stream);

/* Cluster protection for hit removal, "strategy B", for the LAST
 * tpc_track_timeframe call on this handle: keep[i] = 1 iff input cluster i is attached to a track or lies, in its own
 * (sector, row), within +-road_y (cm) and +-road_z (cm) of a cluster some track owns; else 0.  `cluster_track` is that
 * call's tpc_tracks_t.cluster_track (DEVICE, [n]); `keep` is DEVICE, [n] bytes.  Enqueued on `cuda_stream`, which must
 * be ordered after the call; does not synchronise.  INVALID_ARG for null pointers or a negative road. */
TPC_API int tpc_tracker_protect(tpc_tracker_t* t, const int32_t* cluster_track, float road_y, float road_z, uint8_t* keep,
                                void* cuda_stream);

/* Largest frame (clusters) tpc_tracker_protect_static accepts = bytes of the scratch array compiled into the library. */
#define TPC_PROTECT_STATIC_MAX_CLUSTERS 4194304

/* tpc_tracker_protect without any scratch memory from the caller or from an allocator: same inputs, same `keep` output,
 * same result as tpc_tracker_protect, for frames of at most TPC_PROTECT_STATIC_MAX_CLUSTERS clusters (BASELINE.json
 * configs 1-4: single sectors, events, slices, pp frames; a 50 kHz Pb-Pb time frame is far beyond it).
 *
 * Who it is for.  tpc_tracker_protect keeps one mark byte per cluster in a slice of the handle's workspace; every other
 * call of this header likewise lives on memory somebody obtained from cudaMalloc and handed in.  Some callers have no
 * way to get that extra slice: a processing step plugged into a reconstruction framework that reserved the whole card
 * for its own arena at start-up finds cudaMalloc failing for lack of memory; and code on a latency
 * path (a trigger-like loop fed frame after frame) must not call cudaMalloc / cudaFree because both stall the whole
 * device until everything in flight has drained.  For such callers the mark bytes of THIS call live in a fixed array
 * that is part of the library image (a file-scope __device__ array in csrc/s8_protect.cu):
 * the call performs no cudaMalloc, cudaFree, or any other allocating routine, and does not touch the workspace slice
 * the ordinary call uses.
 *
 * What that costs and what to watch.
 *  - Every GPU on which the library's code gets loaded carries the array (4 MiB) until the process exits, used or not.
 *  - A frame with more clusters than the array has bytes is refused with TPC_ERR_STATIC_SCRATCH before anything is
 *    enqueued (`keep` is left as it was); use tpc_tracker_protect for those.
 *  - The first call on each device looks up where the array sits on that device (cudaGetSymbolAddress, checked; the
 *    address is remembered per device).  Make that first call with the handle's device current and before any stream
 *    capture is begun; later calls do no set-up.
 *  - There is ONE array per device, shared by all handles, streams and threads of the process, and it still holds
 *    the marks of the previous call.  Each call therefore begins by clearing the n bytes it will use (a memset
 *    enqueued on `cuda_stream`), so back-to-back calls on one stream are fine; two calls whose GPU work may overlap
 *    (different streams without an ordering between them, or two host threads) race on it and give wrong flags.
 *    Order them yourself (one stream, or an event between the streams).
 * Everything else is as for tpc_tracker_protect: `cluster_track` (DEVICE, [n]) from the LAST tpc_track_timeframe on this
 * handle, `keep` DEVICE [n] bytes, enqueued on `cuda_stream` ordered after that call, no synchronisation.
 * INVALID_ARG for null pointers or a negative road, STATIC_SCRATCH as above, CUDA if the look-up or a launch failed. */
TPC_API int tpc_tracker_protect_static(tpc_tracker_t* t, const int32_t* cluster_track, float road_y, float road_z, uint8_t* keep,
                                       void* cuda_stream);

/* Cuts of the strategy-A hit removal. */
typedef struct {
  float min_pt;    /* GeV/c: merged tracks with |q/pT| * min_pt > 1 are "very low momentum" (0.05) */
  float max_incl;  /* a track segment steeper than this |sin(phi)| at BOTH ends has "high inclination" (0.85) */
  float road_y;    /* cm: road of the protection by good tracks, as in tpc_tracker_protect */
  float road_z;    /* cm */
} tpc_removal_cuts_t;

/* Hit removal, "strategy A" ("positive identification of all hits that can safely
 * be removed" - very low momentum, secondary legs of looping tracks, high inclination - while the good tracks "protect all
 * hits in their vicinity from removal").  For the LAST tpc_track_timeframe / tpc_tracker_refit / tpc_tracker_merge /
 * tpc_tracker_apex sequence on this handle (`cluster_track`, `fit`, `merged`, `apex` are their outputs, DEVICE):
 * cls[i]    (DEVICE, [n] bytes) class of input cluster i: 0 not attached, 1 good track, 2 secondary leg of a looper,
 *           3 very low momentum, 4 high inclination;
 * remove[i] (DEVICE, [n] bytes) 1 iff cls[i] >= 2 and the cluster does not lie, in its own (sector, row), within the road
 *           of a cluster owned by a good track.
 * Enqueued on `cuda_stream`, ordered after those calls; does not synchronise.  The S1 record scratch of the workspace is
 * reused (the next tpc_track_timeframe overwrites it anyway).  CAPACITY as for tpc_tracker_merge (fit, merged, apex). */
TPC_API int tpc_tracker_removable(tpc_tracker_t* t, const int32_t* cluster_track, const tpc_fit_t* fit, const tpc_merged_t* merged,
                                  const tpc_apex_t* apex, const tpc_removal_cuts_t* cuts, uint8_t* cls, uint8_t* remove,
                                  void* cuda_stream);

/* Pipelined host path (tracker created with host_io = 2 or 3 = number of staging slots; BASELINE.json north_star: whole time frames arrive one
 * after the other).  `begin` enqueues the H2D copy of one frame's HOST (pinned) inputs and its
 * S1..S5 on streams the library owns and returns without waiting; `end` waits for that frame, copies exactly the
 * tracks found into the caller's HOST buffers (capacities must equal the tracker's) and returns when they are there.
 * host_io frames may be in flight (slots 0 .. host_io-1, begin/end strictly alternating per slot): the copies of one
 * frame overlap the kernels of another; with 3 slots the upload of frame i+1 can be started before the download of
 * frame i-1 has been collected, which keeps all three streams busy.  Inputs must stay valid and unchanged until the matching `end` returns.
 * Returns INVALID_ARG for a slot used out of order. */
TPC_API int tpc_track_timeframe_host_begin(tpc_tracker_t* t, const tpc_clusters_t* in, int32_t slot);
TPC_API int tpc_track_timeframe_host_end(tpc_tracker_t* t, const tpc_tracks_t* out, int32_t slot);

/* Synchronises the stream of the last call and reads the counter block (HOST out). */
TPC_API int tpc_tracker_counters(tpc_tracker_t* t, tpc_counters_t* out);

/* Per-stage device times of the next calls: when enabled, tpc_track_timeframe records CUDA events
 * between the stages; tpc_tracker_stage_ms synchronises and returns ms for S1..S5 (HOST out[5]). */
TPC_API int tpc_tracker_enable_stage_timing(tpc_tracker_t* t, int32_t enable);
TPC_API int tpc_tracker_stage_ms(tpc_tracker_t* t, float* out_ms5);

/* Debug view of one workspace array (enum tpc_stage_array): the intermediate result of one stage of
 * DESIGN.md sections 3.1-3.5, for the stage-by-stage parity tests.  The pointer is a
 * DEVICE pointer into the caller's workspace, valid until the next track call on the handle.
 * Synchronises the stream of the last call (it reads the device counters for the lengths). */
TPC_API int tpc_tracker_stage_view(tpc_tracker_t* t, int32_t which, tpc_stage_view_t* out);

/* Number of kernel launches tpc_track_timeframe enqueues per call (for bench.py's gpu_launches). */
TPC_API int tpc_tracker_launches_per_call(const tpc_tracker_t* t);

/* Releases the host resources listed at the top (synchronises the library-owned streams first).  The
 * workspace is the caller's and is not touched; frames still in flight on a caller's stream must have
 * finished (memory belongs to the framework around the tracker, not to the tracker). */
TPC_API int tpc_tracker_destroy(tpc_tracker_t* t);

TPC_API const char* tpc_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* TPC_TRACKER_H_ */
