/*
 * tpcca.h -- C-ABI of the B200-native per-sector TPC track finder (arXiv 1811.11481).
 *
 * The operation: PAPER.md:49-51 (section 2) -- for each of the 36 TPC sectors, a cellular automaton
 * links hit triplets that lie close to a straight line, consecutive links are concatenated into
 * seeds, each seed is fitted with a (simplified) Kalman filter, extrapolated through the TPC picking
 * up adjacent hits without following multiple hypotheses, and refitted; PAPER.md:65-68 (outward,
 * then inward through the seed with outlier rejection); PAPER.md:71 (final refit inward, outward,
 * inward); PAPER.md:93 (cluster time already scaled linearly to z, arbitrarily long TPC);
 * PAPER.md:121 (fp32).  Every constant the paper leaves open is a field of tpcca_params with the
 * default of DESIGN.md Table A.
 *
 * Conventions: plain pointers and sizes, no framework types.  "device" = CUDA device memory of the
 * current device, "host" = ordinary host memory.  The library never allocates or frees device
 * memory: all scratch lives in the caller-provided workspace.  All entry points return 0 on success
 * or a negative tpcca_status; tpcca_last_error() describes the last failure of the calling thread.
 * There is no CPU fallback: without a CUDA device tpcca_init fails.
 *
 * Streams: all calls on one handle share the handle's workspace, so the library runs them on the GPU in the order they were
 * made even if each is given a different stream (every enqueueing call makes its stream wait for an event recorded at the end
 * of the previous call on the handle; free when the stream is the same).  Calls on one handle from several host threads at
 * once are not supported; different handles are independent.
 */
#ifndef TPCCA_H
#define TPCCA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tpcca_handle tpcca_handle;

enum tpcca_status {
  TPCCA_OK = 0,
  TPCCA_ERR_ARGUMENT = -1, /* null / misaligned pointer, n > max_clusters, offsets not monotone ... */
  TPCCA_ERR_NOT_INIT = -2,
  TPCCA_ERR_CUDA = -3      /* a CUDA runtime call or kernel launch failed */
};

/* device-side status bits (tpcca_out_header.status) */
enum {
  TPCCA_STAT_TRACKLET_OVERFLOW = 1, /* more start hits than max_tracklets: highest ids dropped */
  TPCCA_STAT_TRACK_OVERFLOW = 2,    /* more tracks than max_tracks: highest ids dropped */
  TPCCA_STAT_BAD_CLUSTER = 4,       /* a cluster with row outside [0,n_rows) or a non-finite y / z was ignored */
  TPCCA_STAT_BIN_OVERFLOW = 8,      /* internal grid capacity hit (never with the default sizing) */
  TPCCA_STAT_CHAIN_TRUNCATED = 16   /* tpcca_merge / tpcca_fit_legs: a chain of more than 24 sector segments was fitted over its
                                       first 24 only (impossible with the default cuts: every segment gains >= 8 rows of 152);
                                       reported in the header of that call and of the later calls on the same frame */
};

/* Geometry (152 pad rows; 36 trapezoidal sectors). */
typedef struct {
  int32_t n_sectors;     /* 1..64; 36 for the full TPC (0-17 side A, 18-35 side C) */
  int32_t n_rows;        /* 2..256; 152 */
  const float* row_x;    /* host, n_rows, cm, strictly increasing; copied by tpcca_init */
  float tan_half_angle;  /* tan(10 deg): a row spans |y| <= x*tan_half_angle */
} tpcca_geometry;

/* Parameters.  Physics fields follow DESIGN.md Table A (A1-A13); grid_* only shape the search
 * acceleration structure and never change a result. */
typedef struct {
  float sigma_y, sigma_z;                   /* cluster errors, cm */
  float nbr_dydx, nbr_dzdx;                 /* neighbour window slope per cm of row distance */
  float nbr_margin_y, nbr_margin_z;         /* neighbour window margins, cm */
  float triplet_cut;                        /* max straight-line triplet cost */
  float cov0[5];                            /* initial / reset covariance diagonal */
  float pick_cut, reject_cut;               /* 2-dof distance cuts: pick-up, seed-hit rejection */
  int32_t max_gap;                          /* consecutive rows without hit before stopping */
  float edge_margin, max_sinphi;
  int32_t min_seed_hits, min_tracklet_hits, min_track_hits;
  float qual_scale;
  float grid_bin_y, grid_bin_z_min;         /* cm */
  float grid_bins_per_cluster;              /* target bins per cluster in a row slice, <= 4 */
  int64_t max_clusters;                     /* capacity per call, <= 4e8 (32-bit positions and bin ids) */
  int32_t max_tracklets, max_tracks;
  void* workspace;                          /* device, >= tpcca_workspace_bytes(), 256-byte aligned; caller-owned */
  size_t workspace_bytes;
} tpcca_params;

/* Input cluster, sector-local coordinates: x along the sector axis (must equal row_x[row]), y across,
 * z along the drift.  16 bytes, read as one float4. */
typedef struct { float x, y, z; int32_t row; } tpcca_cluster;

/* Output: header followed by max_tracks records. */
typedef struct { int32_t n_tracks, n_tracklets, n_start_hits, status; } tpcca_out_header; /* 16 B */
typedef struct {
  int32_t sector, first_row, last_row, n_hits;
  float x, y, z, sinphi, dzds, qpt;         /* state at x = row_x[first_row] (innermost hit) */
  float cov[15];                            /* lower triangle of cov(y, z, sinphi, dzds, qpt) */
  float chi2;                               /* of the last (inward) refit pass */
  int32_t ndf;                              /* 2*n_hits-5, or -1 if the refit transport failed */
  int32_t pad[5];
} tpcca_track_rec;                          /* 128 B */

/* Fill *p with the defaults of DESIGN.md Table A (capacities 0, workspace NULL). */
void tpcca_default_params(tpcca_params* p);

/* Bytes of device workspace needed for the capacities in *p (workspace fields ignored).  0 on bad arguments. */
size_t tpcca_workspace_bytes(const tpcca_geometry* g, const tpcca_params* p);

/* Create a tracker on the current CUDA device.  Host-only work plus one small upload (row_x).
 * Returns NULL on error (see tpcca_last_error). */
tpcca_handle* tpcca_init(const tpcca_geometry* g, float bz_tesla, const tpcca_params* p);

/* Track one time frame: steps (a)-(g) of DESIGN.md for all sectors, enqueued on `stream`; returns
 * without waiting.  clusters: device, n records, clusters of sector s at
 * [sector_offsets[s], sector_offsets[s+1]) in any order, 16-byte aligned.  sector_offsets: HOST,
 * n_sectors+1 entries, CSR, read before return.  stream: a cudaStream_t (NULL = default stream).
 * out_tracks: device, sizeof(header) + max_tracks*128 bytes; tracks in canonical order.
 * out_hit_assignment: device, n int32 in input order, track id or -1.
 * n == 0 is valid (header all zero).  Capacity overflow sets header.status and truncates; nothing is
 * ever written out of bounds. */
int tpcca_track(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* sector_offsets,
                void* stream, void* out_tracks, int32_t* out_hit_assignment);

/* Same, end to end from HOST buffers (pinned for best speed): copies clusters host->device into the
 * workspace, tracks, copies header, tracks and assignment device->host and waits for them.
 * out_tracks: host, sizeof(header) + max_tracks*128 bytes (only n_tracks records are written).
 * Equivalent to tpcca_track_host_async + tpcca_wait; refused while async frames are in flight. */
int tpcca_track_host(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* sector_offsets,
                     void* stream, void* out_tracks, int32_t* out_hit_assignment);

/* Pipelined host call ("processing two events concurrently on one GPU"; PAPER.md:177 host<->GPU
 * transfers).  Same arguments as tpcca_track_host; returns after ENQUEUEING the host->device copy (internal copy
 * stream), the kernels (`stream`) and the device->host copy of header and assignment (second internal stream).  At
 * most TWO frames may be in flight per handle (two staging slots inside the one workspace): while the kernels of
 * frame k run, the input of frame k+1 is uploaded and the results of frame k-1 are downloaded.  The host buffers
 * of a frame must stay valid and untouched until its tpcca_wait returns.  Returns TPCCA_ERR_ARGUMENT if two frames
 * are already in flight. */
int tpcca_track_host_async(tpcca_handle* h, const tpcca_cluster* clusters, int64_t n, const int32_t* sector_offsets,
                           void* stream, void* out_tracks, int32_t* out_hit_assignment);

/* Blocks until the OLDEST frame submitted with tpcca_track_host_async is complete: its header and assignment have
 * arrived, then its n_tracks track records are copied (third internal stream) -- frames complete in submission
 * order.  TPCCA_ERR_ARGUMENT if no frame is in flight. */
int tpcca_wait(tpcca_handle* h);

/* Intermediates of the last tpcca_track on this handle, translated to INPUT-index space so that they
 * can be compared with an independent implementation.  dst: device.  Enqueued on `stream`. */
enum tpcca_intermediate {
  TPCCA_LINK_UP_RAW = 0,    /* int32[n]  (b) before cleaning */
  TPCCA_LINK_DOWN_RAW = 1,  /* int32[n] */
  TPCCA_LINK_UP = 2,        /* int32[n]  (c) mutual links only */
  TPCCA_LINK_DOWN = 3,      /* int32[n] */
  TPCCA_START_HITS = 4,     /* int32[n_start_hits], canonical order = tracklet ids */
  TPCCA_TRACKLET_ROW_HITS = 5, /* int32[n_start_hits][n_rows], -1 = no hit (void tracklets: all -1) */
  TPCCA_TRACKLET_INTS = 6,  /* int32[n_start_hits][4]: valid, first_row, last_row, n_hits */
  TPCCA_TRACKLET_FLOATS = 7,/* float[n_start_hits][8]: x, y, z-z_ref, sinphi, dzds, qpt, chi2, z_ref */
  TPCCA_TRACK_TRACKLET = 8, /* int32[n_tracks]: tracklet id of each track */
  TPCCA_TRACK_OUTER = 9,    /* float[n_tracks][24]: outer end of each track (state after the outward refit pass):
                               x, y, z, sinphi, dzds, qpt, cov[15], 3 unused */
  TPCCA_SHARED = 10,        /* int32[n]: 1 if the cluster was also collected by the tracklet of another accepted track */
  TPCCA_MERGE_LINK_NEXT = 11 /* int32[n_tracks]: after tpcca_merge, the sector track this one continues into, or -1 */
};
/* dst_device: 16-byte aligned, `bytes` long.  The call reads the live counts of the last frame (it synchronises
 * `stream`) and returns TPCCA_ERR_ARGUMENT, writing nothing, if `bytes` is smaller than the table. */
int tpcca_get_intermediate(tpcca_handle* h, int what, void* dst_device, size_t bytes, void* stream);

/* Debugging aid: the i-th array carved out of the workspace (byte offset from params.workspace, bytes in use; arrays start
 * on 256-byte boundaries, so the bytes between the end of one and the start of the next are never touched by a correct
 * kernel -- tests fill the workspace with a pattern and check those gaps afterwards).  TPCCA_ERR_ARGUMENT past the last. */
int tpcca_debug_workspace_layout(tpcca_handle* h, int i, size_t* offset, size_t* bytes);

/* Debugging aid: with on != 0 every tpcca_track on this handle synchronises after each stage and names the stage
 * that faulted in tpcca_last_error().  Off by default; never use it in a timed run. */
int tpcca_set_debug(tpcca_handle* h, int on);

/* ---- Sector-segment merger and final fit ("The second phase merges the track segments found in the
 * individual sectors and performs the final track fit with the full Kalman filter"; :69 outlier rejection by predicted
 * chi2; :70 enlarged errors for shared clusters; :71 three passes, Table B). */
typedef struct {
  float merge_chi2_cut;        /* match: sum over the 5 parameters of diff^2 / (var_A + var_B) */
  float merge_dz_max;          /* cm, |z_B - z_A| between the two ends */
  float merge_edge_dist;       /* cm, the outer end must lie this close to the sector's side */
  int32_t merge_row_back, merge_row_fwd; /* first_row(B) - last_row(A) in [-back, fwd] */
  float fit_reject_cut;        /* 2-dof predicted distance above which a hit is left out of a pass of the final fit */
  float shared_err_scale;      /* sigma_y, sigma_z multiplier of shared clusters in the final fit */
  int32_t ring;                /* sectors per z side closing the ring (18); 0: no neighbours, nothing merges; 1 and values
                                  above 64 are refused (a sector would be its own neighbour) */
} tpcca_merge_params;
void tpcca_default_merge_params(tpcca_merge_params* p);

/* Merge the sector tracks of the LAST tpcca_track / tpcca_track_host* on this handle and fit the merged tracks; enqueued
 * on `stream` (the stream of that call, or one ordered after it), returns without waiting.  The out_tracks buffer of that
 * call must still be valid and unchanged (it is read); everything else lives in the workspace.
 * out_merged: device, 16-byte aligned, sizeof(tpcca_out_header) + max_tracks * 128 bytes: header {n_tracks = merged
 *   tracks, n_tracklets = links, n_start_hits = merged fits that failed (ndf = -1), status}, then one tpcca_track_rec per
 *   merged track in the order of their innermost segments' track ids: sector / first_row / state of the innermost
 *   segment's frame, last_row of the outermost, n_hits of all segments, pad = {segments, outermost sector, hits rejected
 *   in the last pass (-1: the fit failed, ndf = -1 and the state is the innermost segment's own fit), shared hits,
 *   innermost sector-track id}.
 * out_track_merged: device, max_tracks int32: merged track of every sector track (compose with out_hit_assignment). */
int tpcca_merge(tpcca_handle* h, const tpcca_merge_params* mp, void* stream, void* out_merged, int32_t* out_track_merged);

/* ---- z / time estimate of the tracks of a time frame ("After the Kalman fit of the initial seed, the
 * position of closest approach to the beam line is computed and assumed as z-position (and thus time) of the primary
 * vertex"; :109 refined after the merge; :119 "In case clusters of a fully merged secondary track are outside the real
 * TPC volume, the track is shifted inside").  For every sector track of the last tpcca_track and,
 * if out_merged is not NULL, every merged track of the last tpcca_merge: z of the helix at its closest approach to
 * the beam line (z_dca), the shift that brings all its clusters inside the drift volume of their side
 * (z_shift = z_dca clamped; side A: 0 <= z - shift <= z_max, side C mirrored), the collision time
 * t0_us = side * z_shift / vdrift, and the signed transverse distance of closest approach (dca_xy).
 * out_sector / out_merged: device, max_tracks records of 16 bytes, 16-byte aligned.  Enqueued on `stream`. */
typedef struct { float z_dca, z_shift, t0_us, dca_xy; } tpcca_time_rec;
int tpcca_estimate_time(tpcca_handle* h, float vdrift_cm_per_us, float z_max_cm, void* stream,
                        tpcca_time_rec* out_sector, tpcca_time_rec* out_merged);

/* ---- Legs of low-pT loopers and cluster tags ("additional legs of looping tracks do not point to the vertex
 * ... special low-pT track merging"; :157 clusters to remove for the compression factor: "very low-pT looping tracks below
 * 50 MeV/c, additional legs of tracks below 200 MeV/c, and track segments with high inclination angle"; DESIGN.md section 14,
 * Table D).  Two merged tracks that are consecutive legs of one helix (same circle in the sector plane, opposite fitted
 * curvature, z consistent with the arc between them) are linked: outer end to outer end over the turning point, inner end
 * to inner end through the region below the first pad row (the looper passes the beam line and comes out again one
 * pitch further in z); clusters are tagged for removal. */
typedef struct {
  float leg_min_qpt;          /* (GeV/c)^-1: only ends with |q/pT| >= this are candidates */
  float leg_min_sinphi;       /* and |sin(phi)| >= this at an outer end */
  float leg_inner_min_sinphi; /* ... at an inner end */
  float leg_apex_margin;      /* cm: outer ends only, the turning point xc + R must lie below row_x[last] + margin */
  int32_t leg_max_sector_gap; /* outer: the partner's end lies 0..gap sectors AHEAD in the turning sense */
  int32_t leg_inner_max_sector_gap; /* inner: at most this many sectors away, either way round */
  float leg_max_turn;         /* rad, < pi: turning angle between two outer ends */
  float leg_inner_max_turn;   /* rad, < 2 pi: turning angle between two inner ends */
  float leg_centre_frac, leg_centre_abs; /* centre distance <= frac * mean radius + abs (cm) */
  float leg_radius_frac;      /* |R_A - R_B| <= frac * mean radius */
  float leg_dz_max;           /* cm: z_B - z_A - mean slope * arc */
  float leg_dzds_tol;         /* |dzds_A + dzds_B| (the legs are fitted in opposite senses) */
  float tag_qpt_low;          /* TAG_LOW_PT: |q/pT| of the merged track above this (20 = 50 MeV/c) */
  float tag_qpt_leg;          /* TAG_EXTRA_LEG: additional leg with |q/pT| above this (5 = 200 MeV/c) */
  float tag_sinphi;           /* TAG_HIGH_INCLINATION: local |sin(phi)| above this */
  int32_t ring;               /* sectors per z side closing the ring (18); 0: partners in the same sector only; 1 and > 64 refused */
} tpcca_leg_params;
void tpcca_default_leg_params(tpcca_leg_params* p);
enum { TPCCA_TAG_LOW_PT = 1, TPCCA_TAG_EXTRA_LEG = 2, TPCCA_TAG_HIGH_INCLINATION = 4 };
typedef struct {
  int32_t n_links_outer, n_links_inner, n_tag_low_pt, n_tag_extra_leg, n_tag_high_inclination, pad[3];
} tpcca_leg_summary; /* 32 B */

/* Link legs and tag clusters for the merged tracks of the LAST tpcca_merge on this handle (whose outputs, and those of the
 * tpcca_track before it, must still be valid and unchanged); enqueued on `stream`, returns without waiting.
 * out_leg_partner: device, max_tracks int32: merged track joined at the outer turning point, or -1 (mutual).
 * out_leg_partner_inner: device, max_tracks int32: merged track joined through the inner region, or -1 (mutual).
 * out_leg_first: device, max_tracks bytes: 1 = first (or only) leg of its chain -- no linked neighbour has its inner end
 *   at a smaller |z| --, 0 = additional leg.
 * out_cluster_tags: device, n bytes in INPUT order (n of the last tpcca_track): TPCCA_TAG_* bits, 0 for clusters on no track.
 * out_summary: device, 16-byte aligned, 32 bytes: links per kind and tagged clusters per bit.
 * TPCCA_ERR_ARGUMENT without a preceding tpcca_merge, for null / misaligned pointers or parameters out of range
 * (leg_max_turn must be < pi, leg_inner_max_turn < 2 pi, thresholds and tolerances > 0). */
int tpcca_find_legs(tpcca_handle* h, const tpcca_leg_params* lp, void* stream, int32_t* out_leg_partner,
                    int32_t* out_leg_partner_inner, uint8_t* out_leg_first, uint8_t* out_cluster_tags,
                    tpcca_leg_summary* out_summary);

/* ---- One fit through both legs of a turn ("the refit was tuned to enable arbitrary rotations for following the
 * full helix", Table E).  For every pair of merged tracks joined at an outer turning point by the
 * last tpcca_find_legs, a three-pass Kalman fit over the hits of BOTH legs in trajectory order; the frame of the filter is
 * turned in sector steps so that the track always points roughly along its x axis, and a hit seen from a turned frame
 * enters with the error sigma_y * |cos(beta) + sin(beta) tan(phi)|. */
typedef struct {
  float fit_rot_sinphi;    /* turn the frame one sector step while |sin(phi)| exceeds this */
  float fit_step_sinphi;   /* a transport never takes |sin(phi)| beyond this: it stops there and the frame is turned */
  float fit_min_d;         /* hits whose pad row runs nearly along the track (|D| below this) are not used */
  float fit_reject_cut;    /* 2-dof predicted distance above which a hit is left out of a pass */
  float shared_err_scale;  /* sigma_y, sigma_z multiplier of shared clusters */
  int32_t ring;            /* sectors per z side closing the ring; must be even (18) for the report in the first leg's frame */
} tpcca_leg_fit_params;
void tpcca_default_leg_fit_params(tpcca_leg_fit_params* p);

/* Fit the pairs of the LAST tpcca_find_legs on this handle (whose out_leg_partner, and the outputs of the tpcca_merge and
 * tpcca_track before it, must still be valid and unchanged); enqueued on `stream`, returns without waiting.
 * out_fits: device, 16-byte aligned, sizeof(tpcca_out_header) + max_tracks * 128 bytes: header {n_tracks = pairs,
 *   n_tracklets = fits that failed (ndf = -1), n_start_hits = 0, status}, then one tpcca_track_rec per pair in the order
 *   of the pair's lower merged id: state at the innermost hit of the FIRST leg (smaller |z| of the inner end), in that
 *   leg's innermost sector frame, direction outward -- comparable with the leg's own merged record --, first_row = its
 *   row, last_row = the row of the other leg's innermost hit, n_hits of both legs, ndf = 2 * used - 5,
 *   pad = {first leg, other leg, hits not used in the last pass (-1: failed), frame turns, 0}.
 * TPCCA_ERR_ARGUMENT without a preceding tpcca_find_legs, for null / misaligned pointers or parameters out of range. */
int tpcca_fit_legs(tpcca_handle* h, const tpcca_leg_fit_params* fp, void* stream, void* out_fits);

/* Per-stage device times, averaged over the tpcca_track calls (at most the last 32) made since profiling
 * was switched on (CUDA events recorded on each call's stream; synchronises those events).  ms: host float[TPCCA_N_STAGES]. */
enum { TPCCA_STAGE_GRID = 0, TPCCA_STAGE_NEIGHBOURS, TPCCA_STAGE_CLEAN_START, TPCCA_STAGE_TRACKLETS,
       TPCCA_STAGE_SELECT, TPCCA_STAGE_REFIT, TPCCA_N_STAGES };
int tpcca_set_profiling(tpcca_handle* h, int on);  /* 0 off, 1 stage events, 2 stage + per-kernel events */
int tpcca_get_stage_ms(tpcca_handle* h, float* ms);

/* Device time of the main kernels of the LAST tpcca_track made with profiling level 2 (two CUDA events around each
 * launch on the call's stream; synchronises them).  ms: host float[TPCCA_N_KERNELS]. */
enum tpcca_kernel_id { TPCCA_K_SLICE_SCATTER = 0, TPCCA_K_SLICE_SORT, TPCCA_K_NEIGHBOURS, TPCCA_K_CLEAN, TPCCA_K_TL_E1,
                       TPCCA_K_TL_E2, TPCCA_K_TL_E3A, TPCCA_K_TL_E3B, TPCCA_K_WEIGHTS, TPCCA_K_SELECT_OWN, TPCCA_K_ASSIGN,
                       TPCCA_K_REFIT, TPCCA_N_KERNELS };
int tpcca_get_kernel_ms(tpcca_handle* h, float* ms);

/* Device-side work counters of the last tpcca_track (synchronises `stream`): host int64[TPCCA_N_WORK]. */
enum { TPCCA_WORK_N_BINS = 0,      /* grid bins of the frame */
       TPCCA_WORK_ROW_STEPS,       /* Kalman row steps (transport attempts) taken by the tracklet constructor */
       TPCCA_WORK_SEARCHES,        /* pick-up searches (grid look-ups) by the tracklet constructor */
       TPCCA_WORK_TRACK_HITS,      /* hits owned by accepted tracks */
       TPCCA_WORK_TRACKLET_HITS,   /* hits of all valid tracklets (one weight atomic each) */
       TPCCA_WORK_STEPS_E1, TPCCA_WORK_STEPS_E2, TPCCA_WORK_STEPS_E3A, TPCCA_WORK_STEPS_E3B, /* row steps per constructor kernel */
       TPCCA_N_WORK };
int tpcca_get_stats(tpcca_handle* h, int64_t* stats, void* stream);

/* Kernels launched by the last tpcca_track / tpcca_track_host on this handle. */
int tpcca_last_launch_count(tpcca_handle* h);

/* ---- Link cleaner and start-hit finder that allocates nothing and needs no workspace (steps (c) and (d): PAPER.md:49, a
 * link between neighbouring rows is kept only if both ends agree, and the hits where a chain of links begins are collected;
 * DESIGN.md O3 / O4).
 *
 * For whom: callers that cannot obtain device memory at run time and therefore have no workspace to pass to tpcca_init --
 * a component inside a process whose framework took all GPU memory for its own allocator at start-up, a monitoring task
 * inspecting the links of a frame it does not own, or code in a real-time loop where cudaMalloc / cudaFree would
 * synchronise the device under the frames being tracked on other streams.  This call makes no cudaMalloc, cudaFree or
 * other allocating call: the scratch of its compaction (one counter and one int32 per 1024 clusters) is a fixed array
 * built into the library image, 131,328 bytes of device memory that every GPU loading the library holds until the process
 * exits.  Hence the hard limit n <= TPCCA_STATIC_MAX_CLUSTERS; a larger n returns TPCCA_ERR_ARGUMENT (text in
 * tpcca_last_error) and nothing is written.
 *
 * link_up_raw / link_down_raw: device, int32[n], links before cleaning in any index space of [0, n), -1 (or any value
 *   outside [0, n)) = no link -- e.g. TPCCA_LINK_UP_RAW / TPCCA_LINK_DOWN_RAW of tpcca_get_intermediate.
 * out_link_up / out_link_down: device, int32[n]: the link where the partner points back, else -1.  Must not overlap the
 *   inputs or each other.
 * out_start_hits: device, int32[n] capacity: the clusters with an up link and no down link after cleaning, in ASCENDING
 *   index (tpcca_track orders them by sector, row, z, y instead: same set, different order).
 * out_n_start: device, one int32: how many.   All pointers 4-byte aligned; the caller owns every buffer.
 * stream: a cudaStream_t of the CURRENT device; the work is enqueued and the call returns without waiting.
 *
 * Sharing: there is ONE scratch array per GPU and every call uses it, whatever the stream or thread.  Two calls on the same
 * GPU that could run at the same time race on it and give wrong start hits: keep them on one stream, or order them with
 * events.  Calls on different GPUs are independent.  The array keeps the previous call's contents; the one word that must
 * be zero is cleared on `stream` at the start of every call.
 * First call on a device: it looks up the device address of the array (cudaGetSymbolAddress, with that device current) and
 * remembers it; this may load the CUDA module.  Make that first call during set-up, before any stream capture is begun.
 * n == 0 is valid (*out_n_start = 0).  Returns 0, TPCCA_ERR_ARGUMENT or TPCCA_ERR_CUDA. */
#define TPCCA_STATIC_MAX_CLUSTERS 33554432LL /* 2^25 */
int tpcca_clean_links_static(const int32_t* link_up_raw, const int32_t* link_down_raw, int64_t n, void* stream,
                             int32_t* out_link_up, int32_t* out_link_down, int32_t* out_start_hits, int32_t* out_n_start);

const char* tpcca_last_error(void);
void tpcca_free(tpcca_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* TPCCA_H */
