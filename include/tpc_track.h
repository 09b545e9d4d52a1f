/*
 * tpc_track.h — C ABI of the B200 TPC sector-tracking library (libtpctrack.so).
 *
 * What the library computes: the "sector tracking" phase of the ALICE Run 3 TPC
 * tracking as summarised in PAPER.md:25-27 (§2): a time frame of TPC clusters
 * (§1) goes in; for each of the 36 sectors the library builds the
 * per-pad-row "fast cluster search grid" (§3), finds cellular-automaton
 * neighbour links and seeds ("combinatorial seeding based on a cellular automaton",
 * PAPER.md:27), follows every seed through the sector with a Kalman filter "picking
 * up more clusters of the track", and runs the ambiguity solving that
 * "identifies the best instance of each track, assigns all clusters to this instance
 * and removes the clones", with "a configurable fraction of a track's clusters, by
 * default 10%, ... allowed to be shared" and the Phase-I criterion
 * (smaller global chi2 gets priority, shared clusters counted from the outermost pad
 * row, §3).  Output: sector tracks with cluster lists, ready for the
 * track-merging phase, which is outside this library.
 *
 * Every constant / window / tie-break the paper leaves open is fixed in DESIGN.md
 * ("Readings") and is a field of tpc_params below.
 *
 * Conventions
 *  - All structs are POD, little-endian, natural alignment.  No C++ or torch types.
 *  - Pointers named d_* are DEVICE pointers (CUDA global memory on the current device);
 *    all other pointers are HOST pointers.
 *  - Every function returns TPC_OK (0) or a negative tpc_error; nothing throws or aborts.
 *  - A context is not thread-safe; use one context per host thread / stream.
 *  - The library allocates device memory only inside tpc_geom_init (a few KB of tables
 *    and counters).  All scratch and all outputs live in the caller's workspace.  Kernels run
 *    on the caller's stream; the library owns two copy streams, created in tpc_geom_init and
 *    used by tpc_sector_track_host_chunks alone.
 */
#ifndef TPC_TRACK_H
#define TPC_TRACK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ------------------------------------------------------------------ errors */
typedef enum tpc_error {
  TPC_OK = 0,
  TPC_E_ARG = -1,       /* null / misaligned pointer, bad descriptor, n_clusters >= 2^30,
                           or (reported by tpc_get_tracks) a cluster whose sector/row is
                           outside the geometry                                         */
  TPC_E_WORKSPACE = -2, /* workspace smaller than tpc_workspace_bytes(); nothing written */
  TPC_E_OVERFLOW = -3,  /* a capacity bound was hit on the device (bin index, tracks);
                           results are invalid, never silently truncated               */
  TPC_E_CUDA = -4,      /* a CUDA runtime call failed; see tpc_last_cuda_error()         */
  TPC_E_STATE = -5,     /* call order violated (e.g. tpc_get_tracks before a run)       */
  TPC_E_LIMIT = -6      /* a size beyond the fixed maximum of tpc_fit_tracks_noalloc; nothing run */
} tpc_error;

/* ------------------------------------------------------------------ input */
/* One TPC cluster, 16 bytes (BASELINE.json config 4: "cluster struct 16 B").
 * y, z are local sector coordinates in cm: y along the pad row, z along the drift
 * ("time-z": with continuous readout the collision time is unknown, so z
 * carries an unknown per-collision offset; the tracker never uses a vertex constraint).
 * The pad row fixes the local x.  q (charge) and flags are carried but unused. */
typedef struct tpc_cluster {
  float y, z;
  float q;
  uint8_t sector; /* 0..n_sectors-1 (0..17 A side, 18..35 C side) */
  uint8_t row;    /* 0..n_rows-1 */
  uint16_t flags;
} tpc_cluster;

/* Geometry descriptor (2 halves x 18 trapezoidal sectors; row count, radii
 * and pad pitches from BASELINE.json config 1).  Row r sits at local
 * x_r = r_min + r*(r_max-r_min)/(n_rows-1); its half width is x_r*tan(half_angle). */
typedef struct tpc_geom_desc {
  int32_t n_sectors;    /* 36 */
  int32_t n_rows;       /* 152 (max 255) */
  int32_t n_inner_rows; /* 63; informational */
  float r_min, r_max;   /* 85, 245 cm */
  float pad_pitch_inner, pad_pitch_outer; /* 0.4, 0.6 cm; informational */
  float z_max;          /* 250 cm drift length; only sizes the default bin capacity */
  float bz_tesla;       /* 0.5 */
  float sector_half_angle_deg; /* 10 */
} tpc_geom_desc;

/* Every tunable of the method.  Defaults (tpc_default_params) are DESIGN.md's readings. */
typedef struct tpc_params {
  float err_y, err_z;            /* measurement sigma, cm (0.1, 0.1)                    */
  float nf_slope_y, nf_slope_z;  /* neighbour-finder window slopes (1.0, 1.6)           */
  float nf_max_d2;               /* max 3-point straightness^2, cm^2 (0.70)             */
  int32_t seed_min_len;          /* min clusters in a link chain to seed (4)            */
  float init_var_sinphi, init_var_tanl, init_var_qpt; /* (0.25, 4, 100)                 */
  float max_sinphi;              /* 0.95                                                */
  float max_qpt;                 /* clamp on |q/pT|, c/GeV (20)                         */
  float road_nsigma, road_min, road_max; /* search road (3.5, 0.3 cm, 2.0 cm)           */
  float chi2_max_hit;            /* 2-dof chi2 cut for pick-up (12)                     */
  int32_t max_gap_follow;        /* rows without hit before the follower stops (4)      */
  int32_t min_hits_tracklet;     /* (10) >= 3: ndf = 2*nHits - 5 of the weight must be > 0 */
  float sel_chi2_weight;         /* weight = nHits - w*chi2/ndf (2.0)                   */
  int32_t shared_permille;       /* allowed shared-cluster fraction, permille (100)     */
  int32_t max_gap_select;        /* rows; a larger hole splits the track (4)            */
  int32_t min_hits_track;        /* (20)                                                */
  float grid_dy, grid_dz;        /* bin size, cm (2, 2) — performance knob only         */
  uint64_t max_bins;             /* bin-index capacity; 0 = default
                                    4*n_clusters + n_sectors*n_rows*ny_max*(z_max/grid_dz+2)   */
  uint32_t max_seeds;            /* seed/tracklet capacity; 0 = default n_clusters/8 + 4096     */
  uint32_t shared_fixed_cap;     /* 0: shared clusters by the running fraction counted from the outermost
                                    row (Phase I); 1: fixed cap shared_permille*nHits/1000
                                    per segment (the rule before Phase I; A/B variant)             */
  uint32_t max_ids;              /* capacity of the tracks' cluster lists; 0 = default n/(1 - shared_permille/1000) + 64,
                                    the exact bound of the running-fraction rule.  With shared_fixed_cap = 1 a
                                    cluster may be shared by every clone of its track (the cap counts per
                                    tracklet), so no bound follows from n: TPC_E_OVERFLOW then asks for a
                                    larger value here (the oracle's count, or a few times n)            */
  uint32_t reserved;
} tpc_params;

/* ------------------------------------------------------------------ output */
#define TPC_TRACK_PARAMS_STALE 1u /* segment does not contain the row the parameters refer to */
#define TPC_TRACK_ITER2 2u        /* found by the second seeding iteration (tpc_sector_track_two_iterations) */

/* One sector track (108 bytes).  Parameters are (y, z, sin(phi), tan(lambda), q/pT) at
 * local x of the tracklet's innermost row, c[] the lower-triangular covariance
 * (c00,c10,c11,c20,...,c44). */
typedef struct tpc_track {
  float x;
  float p[5];
  float c[15];
  float chi2;            /* of the inward refit pass                                   */
  uint32_t cluster_ofs;  /* first entry in cluster_ids / cluster_shared                */
  uint32_t seed_id;      /* ORIGINAL input index of the seed's start cluster           */
  uint16_t n_clusters, n_shared;
  uint8_t sector, row_first, row_last, flags;
  uint16_t n_hits_tracklet; /* hits of the whole tracklet (ndf = 2*n-5)                */
  uint8_t segment;          /* 0 = outermost segment of this tracklet                  */
  uint8_t pad_;
} tpc_track;

typedef struct tpc_track_view {
  uint64_t n_tracks;
  uint64_t n_cluster_ids;
  const tpc_track* d_tracks;        /* [n_tracks]                                      */
  const uint32_t* d_cluster_ids;    /* [n_cluster_ids] original input indices, per track
                                       ascending in pad row                            */
  const uint8_t* d_cluster_shared;  /* [n_cluster_ids] 1 = attached as shared          */
  /* diagnostics */
  uint64_t n_ignored;               /* NaN/Inf clusters ignored                         */
  uint64_t n_dropped;               /* |y| beyond the row's half width + 2 cm          */
  uint64_t n_seeds;
  uint64_t n_tracklets;
  uint64_t n_bins;
  uint64_t n_follow_steps;          /* follower work: one-row propagations ...           */
  uint64_t n_follow_updates;        /* ... Kalman updates ...                            */
  uint64_t n_follow_candidates;     /* ... and chi2 evaluations of road candidates       */
  uint64_t follow_work[3][3];       /* the same three counters per follower kernel:
                                       [outward | refit | inward][steps, updates, candidates] */
  uint64_t grid_by_rows;            /* 1: EVERY row's grid was built row by row in shared memory
                                       (k_row_sort); 0: some rows took the generic kernels      */
  uint64_t n_rows_generic;          /* rows built by the generic histogram / scan / scatter kernels:
                                       rows whose input records are not contiguous, that hold
                                       >= 65536 records, or whose tables exceed 224 KB          */
} tpc_track_view;

/* One row of the search grid. */
typedef struct tpc_row_desc {
  float y0, z0;        /* lower edges                                                  */
  int32_t ny, nz;      /* bins; bin = bz*ny + by (z-major)                             */
  uint32_t bin_ofs;    /* index of this row's first bin in d_bin_start                 */
  uint32_t clu_ofs;    /* sorted index of this row's first cluster                     */
  uint32_t count;      /* clusters in the row                                          */
  uint32_t pad_;
} tpc_row_desc;

/* One tracklet (follower output, before ambiguity solving), 112 bytes. */
typedef struct tpc_tracklet {
  float x;
  float p[5];
  float c[15];
  float chi2;
  uint32_t seed_sorted;  /* sorted index of the start cluster                          */
  uint32_t seed_id;      /* original index of the start cluster                        */
  int16_t n_hits;        /* 0 = rejected (below min_hits_tracklet)                     */
  uint8_t row_first, row_last;
  uint8_t sector;
  uint8_t seed_len;      /* length of the seed's link chain                            */
  uint16_t pad_;
  uint32_t pad2_[2];
} tpc_tracklet;

/* Intermediates, valid after a run with TPC_KEEP_INTERMEDIATES.  Index spaces:
 * "sorted index" = position in the grid-sorted cluster array; d_orig_id maps it to the
 * original input index.  Links are in sorted-index space, -1 = none. */
typedef struct tpc_debug_view {
  uint64_t n_clusters;           /* input clusters                                     */
  uint64_t n_sorted;             /* clusters in the grid (input - ignored - dropped)   */
  uint64_t n_rows_total;         /* n_sectors*n_rows                                   */
  uint64_t n_bins;
  uint64_t n_seeds;
  uint64_t tracklet_stride;      /* row_hit is [tracklet][tracklet_stride], = n_rows   */
  const tpc_row_desc* d_row_desc;/* [n_rows_total]                                     */
  const uint32_t* d_bin_start;   /* [n_bins + 1] global sorted positions               */
  const float* d_yz_sorted;      /* [n_sorted][2]                                      */
  const uint32_t* d_orig_id;     /* [n_sorted]                                         */
  const int32_t* d_link_up;      /* [n_sorted] after neighbour finding                 */
  const int32_t* d_link_dn;
  const int32_t* d_link_up2;     /* [n_sorted] after cleanup                           */
  const int32_t* d_link_dn2;
  const uint32_t* d_seeds;       /* [n_seeds] sorted index of each start cluster       */
  const tpc_tracklet* d_tracklets; /* [n_seeds]                                        */
  const int32_t* d_row_hit;      /* [n_seeds][tracklet_stride] sorted index or -1; only
                                    rows row_first..row_last of a tracklet are defined */
} tpc_debug_view;

/* ------------------------------------------------------------------ flags */
#define TPC_DETERMINISTIC 1u      /* bit-reproducible mode: no FMA contraction,
                                     stable grid order, scans instead of atomics         */
#define TPC_KEEP_INTERMEDIATES 2u /* keep the buffers tpc_get_intermediates exposes      */
#define TPC_STAGE_TIMERS 4u       /* record CUDA events per stage (tpc_get_stage_ms)     */
#define TPC_GRID_ONLY 8u          /* build the search grid and stop: no seeds, no tracks; the tracks
                                     then come from tpc_set_tracks (a frame tracked elsewhere)  */

#define TPC_N_STAGES 6            /* grid, neighbours, cleanup+seeds, follower, selector, total */

typedef struct tpc_ctx tpc_ctx;   /* opaque, owned by the library */

/* ------------------------------------------------------------------ calls */

/* Fill *out with the default parameters. HOST pointer. */
void tpc_default_params(tpc_params* out);

/* Create a context for one geometry + parameter set (params == NULL: defaults).
 * Computes the row tables in double, rounds once to fp32 (DESIGN.md rule D5) and uploads
 * them.  HOST pointers.  *out is owned by the library; release with tpc_destroy. */
int tpc_geom_init(const tpc_geom_desc* geom, const tpc_params* params, tpc_ctx** out);

/* Upper bound of the workspace tpc_sector_track needs for n_clusters input clusters. */
size_t tpc_workspace_bytes(const tpc_ctx* ctx, uint64_t n_clusters);

/* Track one time frame.  d_clusters: DEVICE, [n_clusters], 16-byte
 * aligned, read-only, any order, must stay valid until tpc_get_tracks returns.
 * d_workspace: DEVICE, 256-byte aligned, >= tpc_workspace_bytes(); the library carves all
 * scratch and outputs from it.  cuda_stream: a cudaStream_t (NULL = legacy default stream).
 * All work is enqueued asynchronously on that stream; the call does not block. */
int tpc_sector_track(tpc_ctx* ctx, const tpc_cluster* d_clusters, uint64_t n_clusters,
                     void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                     uint32_t flags);

/* Synchronise the stream of the last run, read the counters back and fill *out (HOST)
 * with device pointers into the workspace.  They stay valid until the next
 * tpc_sector_track on this context or until the caller frees the workspace.
 * Returns TPC_E_OVERFLOW / TPC_E_ARG if the device flagged an error during the run. */
int tpc_get_tracks(tpc_ctx* ctx, tpc_track_view* out);

/* As above for the intermediates; requires TPC_KEEP_INTERMEDIATES in the last run. */
int tpc_get_intermediates(tpc_ctx* ctx, tpc_debug_view* out);

/* Per-stage device times in ms of the last run (needs TPC_STAGE_TIMERS):
 * out_ms[0..5] = grid, neighbours, cleanup+seeds, follower, selector, total. HOST pointer.
 * Syncs the stream. */
int tpc_get_stage_ms(tpc_ctx* ctx, float* out_ms);

/* Per-kernel device times of the last run (needs TPC_STAGE_TIMERS): fills names_out[i]
 * (static strings owned by the library) and ms_out[i] for the first min(launched, max_kernels)
 * kernels in launch order and returns that count (>= 0), or a negative tpc_error.  HOST
 * pointers.  Syncs the stream.  Each time is the span between CUDA events recorded around
 * the launch on the caller's stream. */
int tpc_get_kernel_ms(tpc_ctx* ctx, int max_kernels, const char** names_out, float* ms_out);

/* The whole path with HOST buffers (the end-to-end call): copies h_clusters (HOST, pinned
 * for full speed) into d_staging (DEVICE, >= n_clusters*16 bytes, 16-byte aligned, caller
 * owned), runs tpc_sector_track on it, synchronises, and copies the tracks, the cluster ids
 * and the shared flags back into the caller's HOST buffers (each may be NULL = not wanted).
 * *out (HOST) receives the counts; its d_* pointers stay valid as for tpc_get_tracks.
 * Returns TPC_E_OVERFLOW if the results do not fit cap_tracks / cap_ids (nothing copied). */
int tpc_sector_track_host(tpc_ctx* ctx, const tpc_cluster* h_clusters, uint64_t n_clusters,
                          void* d_staging, void* d_workspace, size_t workspace_bytes,
                          void* cuda_stream, uint32_t flags, tpc_track* h_tracks,
                          uint64_t cap_tracks, uint32_t* h_cluster_ids, uint8_t* h_cluster_shared,
                          uint64_t cap_ids, tpc_track_view* out);

/* The same end-to-end call for a frame handed over as n_chunks consecutive parts of
 * h_clusters: chunk c = records [chunk_ofs[c], chunk_ofs[c+1]) (chunk_ofs: HOST, n_chunks+1
 * entries, chunk_ofs[0] = 0, chunk_ofs[n_chunks] = n_clusters).  No sector may have records in
 * two chunks: sectors are the independent units of the sector tracking, so
 * the chunks are tracked one after the other while the next one is copied in and the previous
 * one's tracks are copied out (two library-owned copy streams; the kernels run on cuda_stream).
 * Results: those of one call on the whole frame (cluster ids are indices into h_clusters),
 * tracks concatenated in chunk order; *out holds the summed counts, its d_* pointers are NULL.
 * d_staging (DEVICE) holds the whole frame; the workspace must be at least twice
 * tpc_workspace_bytes(ctx, largest chunk) (else TPC_E_WORKSPACE).  A sector found in two
 * chunks gives TPC_E_ARG.  After this call the context holds no whole-frame result:
 * tpc_get_tracks, tpc_get_intermediates and tpc_refit_tracks return TPC_E_STATE until the
 * next tpc_sector_track / tpc_sector_track_two_iterations. */
int tpc_sector_track_host_chunks(tpc_ctx* ctx, const tpc_cluster* h_clusters, uint64_t n_clusters,
                                 const uint64_t* chunk_ofs, int n_chunks, void* d_staging,
                                 void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                                 uint32_t flags, tpc_track* h_tracks, uint64_t cap_tracks,
                                 uint32_t* h_cluster_ids, uint8_t* h_cluster_shared, uint64_t cap_ids,
                                 tpc_track_view* out);

/* Sector tracking with a SECOND SEEDING ITERATION on the leftover clusters (section 3:
 * "seeding ... in multiple iterations on the leftover clusters after ambiguity solving"; DESIGN.md
 * reading R7): the path runs on the frame, every cluster attached to a track (owned or shared) is
 * removed, and the path runs again on the remaining records.  Results: iteration-1 tracks followed
 * by iteration-2 tracks (flag TPC_TRACK_ITER2), cluster ids in original input indices; read them
 * with tpc_get_tracks (counts are the sums of both iterations; tpc_get_intermediates is not
 * available).  d_clusters: DEVICE, as for tpc_sector_track.  The workspace must hold
 * tpc_workspace_bytes_two_iterations(ctx, n_clusters) bytes.  Unlike tpc_sector_track this call
 * synchronises cuda_stream (the size of the leftover frame has to reach the host). */
size_t tpc_workspace_bytes_two_iterations(const tpc_ctx* ctx, uint64_t n_clusters);
int tpc_sector_track_two_iterations(tpc_ctx* ctx, const tpc_cluster* d_clusters, uint64_t n_clusters,
                                    void* d_workspace, size_t workspace_bytes, void* cuda_stream,
                                    uint32_t flags);

/* TRACKS FROM ELSEWHERE (first axis: one frame over several GPUs by sector;
 * sector tracking is independent per sector, :29: merging is not): loads the sector
 * tracks of the current frame -- tracked sector group by sector group on other contexts / ranks,
 * rebased to frame cluster indices and concatenated in any order -- into this context, so that
 * refit, merging, fit and rebuild run on them as on the context's own result.  Needs a finished
 * tpc_sector_track of the WHOLE frame on this context (TPC_GRID_ONLY is enough: the rebuild queries
 * the grid, refit and fit read the clusters), in the mode (deterministic or fast) the legs shall run in.
 * h_tracks [n_tracks], h_cluster_ids / h_cluster_shared [n_cluster_ids]: HOST, copied before the call
 * returns (synchronises cuda_stream).  TPC_E_OVERFLOW if they exceed the workspace's capacities
 * (those of a frame of this size), TPC_E_ARG if a track names a sector / row outside the geometry, a
 * cluster list outside [0, n_cluster_ids) or a cluster id outside the frame. */
int tpc_set_tracks(tpc_ctx* ctx, const tpc_track* h_tracks, uint64_t n_tracks, const uint32_t* h_cluster_ids,
                   const uint8_t* h_cluster_shared, uint64_t n_cluster_ids, void* cuda_stream);

/* SECTOR-TRACK REFIT (section 3: "a sector track refit at the beginning of the track
 * merging was added, guaranteeing reasonable initial parameters"; reading R8): a pure
 * Kalman fit of every output track through ITS OWN cluster list (outward pass, turn, inward pass;
 * no search, no chi2 cut), giving parameters that are valid at the track's innermost cluster also
 * for the segments flagged TPC_TRACK_PARAMS_STALE.  Runs on the result of the last
 * tpc_sector_track / tpc_sector_track_two_iterations of this context (its d_clusters must still be
 * valid), in the mode (deterministic or fast) of that run; enqueued on cuda_stream. */
typedef struct tpc_track_fit {
  float x;               /* local x of the innermost cluster's row                          */
  float p[5];            /* y, z, sin(phi), tan(lambda), q/pT there                          */
  float c[15];           /* lower-triangular covariance                                      */
  float chi2;            /* of the inward pass, ndf = 2*n_clusters - 5                       */
  uint32_t n_clusters;
  uint32_t flags;        /* bit 0: the fit left the |sin phi| range, record not valid        */
  float x_out;           /* local x of the OUTERMOST cluster's row                           */
  float p_out[5];        /* state there after the outward pass (the end the merging extends) */
  float c_out[15];
  uint32_t pad_[3];
} tpc_track_fit;         /* 192 bytes */
int tpc_refit_tracks(tpc_ctx* ctx, void* cuda_stream);
/* Synchronises and returns the DEVICE array [n_tracks] written by tpc_refit_tracks (aliases the
 * workspace, same lifetime as the track view). */
int tpc_get_refit(tpc_ctx* ctx, const tpc_track_fit** d_fit);

/* TRACK MERGING (section 2: "merges tracks first inside the TPC sectors, then between
 * adjacent sectors of the TPC halves, and then across the central electrode"; section 3:
 * on top of the sector-track refit; reading R9).  Three stages in that order; in each,
 * the refit state at the OUTER end of a track a is transported to the innermost row of a track b
 * (stage 1 and 3: row steps of the follower's propagation; stage 2: rotation by one sector step,
 * then one propagation step) and compared with b's refit state there:
 * chi2 = sum_i d_i^2 / (C_a'[ii] + C_b[ii] + sys_i^2); a and b are linked iff chi2 <= chi2_max and
 * they are each other's best choice by (chi2, sector, iteration, seed id, segment).  Links form
 * chains; a merged track = the cluster lists of its segments in chain order.  Only tracks with a
 * valid refit and a free end take part; later stages see the ends the earlier ones left free. */
typedef struct tpc_merge_params {
  int32_t gap_in_sector;     /* (30) stage 1: 1 <= row_first_b - row_last_a <= this                */
  int32_t gap_adjacent_back; /* (3)  stage 2: -this <= row_first_b - row_last_a                      */
  int32_t gap_adjacent;      /* (10) stage 2:          row_first_b - row_last_a <= this              */
  int32_t gap_ce;            /* (6)  stage 3: 1 <= row_first_b - row_last_a <= this                  */
  float chi2_max;            /* (20)                                                                 */
  float sys[5];              /* (0.3 cm, 0.3 cm, 0.02, 0.02, 0.2 c/GeV)                              */
  float ce_sys_z;            /* (3 cm) replaces sys[1] across the central electrode, where z_b + z_a' is compared */
  float pre_dy, pre_dz;      /* (8 cm, 8 cm) pre-cuts between the transported state and b's state    */
  float pre_coarse_dz;       /* (40 cm) pre-cut on z between the two end states as they are          */
  int32_t stages;            /* (7) bit 0: in sector, bit 1: adjacent sectors, bit 2: central electrode */
} tpc_merge_params;          /* 60 bytes */

typedef struct tpc_merged_track {
  uint32_t head;             /* index (into the sector-track array) of the innermost segment        */
  uint32_t n_segments, n_clusters, n_shared;
  uint32_t cluster_ofs;      /* first entry in d_cluster_ids / d_cluster_shared of the merged view  */
  uint32_t seg_ofs;          /* first entry in d_seg_index                                          */
  int32_t row_first, row_last, sector_first, sector_last;
} tpc_merged_track;          /* 40 bytes */

typedef struct tpc_merged_view {
  uint64_t n_tracks;                 /* sector tracks that went in                                  */
  uint64_t n_merged;                 /* merged tracks (chains; unlinked tracks are chains of one)   */
  uint64_t n_links;
  uint64_t n_cluster_ids;
  const tpc_merged_track* d_merged;  /* [n_merged], heads in the order of the sector-track array    */
  const uint32_t* d_seg_index;       /* [n_tracks] sector-track indices, chain by chain             */
  const uint32_t* d_cluster_ids;     /* [n_cluster_ids] original cluster indices, chain order       */
  const uint8_t* d_cluster_shared;
  const int32_t* d_next;             /* [n_tracks] track linked behind / before each track, -1 none */
  const int32_t* d_prev;
  const float* d_link_chi2;          /* [n_tracks] chi2 of the link to d_next                       */
} tpc_merged_view;

void tpc_merge_default_params(tpc_merge_params* out);
/* Scratch + output size of tpc_merge_tracks for n_tracks sector tracks holding n_cluster_ids ids. */
size_t tpc_merge_workspace_bytes(const tpc_ctx* ctx, uint64_t n_tracks, uint64_t n_cluster_ids);
/* Merge the tracks of the last run; needs tpc_refit_tracks to have run on them (else TPC_E_STATE).
 * d_merge_workspace: DEVICE, 256-byte aligned, caller owned, >= tpc_merge_workspace_bytes(ctx,
 * n_tracks, n_cluster_ids of the track view).  params == NULL: defaults.  Enqueued on cuda_stream
 * (synchronises it first to learn the track count), in the mode (deterministic / fast) of the run. */
int tpc_merge_tracks(tpc_ctx* ctx, const tpc_merge_params* params, void* d_merge_workspace,
                     size_t workspace_bytes, void* cuda_stream);
/* Synchronises and fills *out (HOST) with device pointers into the merge workspace. */
int tpc_get_merged(tpc_ctx* ctx, tpc_merged_view* out);

/* THREE-ITERATION TRACK FIT with the Phase-I interpolation rejection (section 2: "three
 * iterations, first inward, then outward, then inward"; position and covariance stored per pad row "in
 * reduced precision", clusters cut "against the interpolation"; section 3: stored in the
 * first iteration, interpolation and chi2 cut in the second, rejection in the third; DESIGN.md reading
 * R10).  Runs on the merged tracks of tpc_merge_tracks (cluster lists in chain order; sector changes
 * by the rotation of the merging, the central electrode by re-basing z).  Start parameters: the
 * refit's outer state of the chain's last segment. */
typedef struct tpc_fit_params {
  float fit_chi2_max;        /* (16) cut on the 2-dof chi2 of a cluster against the interpolation     */
  int32_t fit_min_clusters;  /* (10) fewer unmarked clusters: the fit fails                           */
  float ce_var;              /* (1e4 cm^2) variance given to z when it is re-based at the electrode   */
} tpc_fit_params;            /* 12 bytes */
typedef struct tpc_track_fit3 {
  float x;                   /* local x of the innermost unmarked cluster's row (its sector's frame)  */
  float p[5], c[15];         /* final parameters and covariance there                                 */
  float chi2;                /* of the third iteration                                                */
  uint32_t n_clusters;       /* clusters of the merged track                                          */
  uint32_t n_used;           /* of which unmarked                                                     */
  uint32_t flags;            /* bit 0: the fit failed                                                 */
} tpc_track_fit3;            /* 100 bytes */
typedef struct tpc_fit_view {
  uint64_t n_merged, n_cluster_ids;
  const tpc_track_fit3* d_fit;     /* [n_merged], order of the merged view                            */
  const float* d_chi2_cluster;     /* [n_cluster_ids] chi2 against the interpolation (iteration 2)    */
  const uint8_t* d_rejected;       /* [n_cluster_ids] 1 = marked and left out of iteration 3          */
} tpc_fit_view;
void tpc_fit_default_params(tpc_fit_params* out);
size_t tpc_fit_workspace_bytes(const tpc_ctx* ctx, uint64_t n_merged, uint64_t n_cluster_ids);
/* Needs tpc_merge_tracks to have run (else TPC_E_STATE).  d_fit_workspace: DEVICE, 256-byte aligned,
 * caller owned, >= tpc_fit_workspace_bytes(ctx, n_merged, n_cluster_ids of the merged view).
 * Enqueued on cuda_stream (synchronises it first to learn the merged-track count). */
int tpc_fit_tracks(tpc_ctx* ctx, const tpc_fit_params* params, void* d_fit_workspace, size_t workspace_bytes,
                   void* cuda_stream);
int tpc_get_fit(tpc_ctx* ctx, tpc_fit_view* out);

/* THE FIT WITHOUT ANY ALLOCATION AND WITHOUT A WORKSPACE (for callers that cannot call cudaMalloc: code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  The same three-iteration fit
 * as tpc_fit_tracks (reading R10; the same kernel, the same results), but the
 * caller passes every input and output as a DEVICE pointer and the kernel's scratch -- the predictions
 * stored in iteration 1, 16 bytes per cluster id, plus a 256-byte header (merged-track count, work
 * counter) -- lives in ONE array inside the library: 256 + 16 * TPC_FIT_NOALLOC_MAX_IDS bytes (16 MiB)
 * that every GPU which loads the library holds until the process exits.  Its device address is resolved
 * once per device in tpc_geom_init (set-up; cudaGetSymbolAddress with that device current); this call
 * performs no cudaMalloc / cudaFree and calls no allocating routine, and does not synchronise.
 *   ctx            geometry, parameters and the device of tpc_geom_init (which must be the current device,
 *                  else TPC_E_STATE); the context's own run state is neither needed nor touched
 *   d_clusters     [n_clusters] the frame; d_refit [n_tracks] the sector-track refit records (tpc_get_refit)
 *   d_merged       [n_merged] merged tracks; d_seg_index [n_tracks], d_cluster_ids [n_cluster_ids] as in
 *                  the merged view; the caller guarantees that their offsets and indices stay inside
 *                  these arrays: device contents are not checked
 *   d_fit_out      [n_merged], d_chi2_out / d_rejected_out [n_cluster_ids]: written by the call
 *   flags          TPC_DETERMINISTIC or 0: the build to run
 * Errors: TPC_E_LIMIT if n_cluster_ids > TPC_FIT_NOALLOC_MAX_IDS (text in tpc_last_cuda_error; nothing
 * is launched); TPC_E_ARG for null / misaligned pointers or invalid
 * parameters; TPC_E_CUDA if the set-up could not resolve the array or a launch failed.
 * EVERY call on a device shares the one array, which keeps the previous call's contents: the call itself
 * resets what must start at zero (the header); the stored predictions are written before they are read.
 * Two calls that overlap on the GPU (different streams, or the same data from two host threads) RACE on
 * it: serialise them (one stream, or an event between them). */
#define TPC_FIT_NOALLOC_MAX_IDS (1u << 20)
int tpc_fit_tracks_noalloc(tpc_ctx* ctx, const tpc_fit_params* params, const tpc_cluster* d_clusters,
                           uint64_t n_clusters, const tpc_track_fit* d_refit, uint64_t n_tracks,
                           const tpc_merged_track* d_merged, uint64_t n_merged, const uint32_t* d_seg_index,
                           const uint32_t* d_cluster_ids, uint64_t n_cluster_ids, tpc_track_fit3* d_fit_out,
                           float* d_chi2_out, uint8_t* d_rejected_out, uint32_t flags, void* cuda_stream);

/* PHASE-II TRACK REBUILD (section 3: "the track is practically rebuilt during iterations 2
 * and 3 of the fit ... the fast cluster search grid from the sector tracking is queried for all clusters
 * compatible with the chi2 cut and all candidates together with their residuals are written to temporary
 * storage ... a second ambiguity solving step ... tracks failing to get their best candidate attached are
 * still eligible for the second candidate"; "a simple chi2 cut for final cluster rejection";
 * DESIGN.md reading R11).  Runs on the merged tracks of tpc_merge_tracks; needs the tracking workspace
 * of the run still intact (it queries its grid).  A merged track's PATH = the (sector,row) steps of its
 * segments and of the holes between segments of one sector.  Results per path step: up to 3 candidates
 * (original cluster ids) with their chi2 against the interpolation, the attached cluster after the
 * second ambiguity solving (owned or shared), whether the third pass used it; per merged track the final
 * parameters (tpc_track_fit3; n_clusters = attached, n_used = used). */
typedef struct tpc_rebuild_params {
  float cand_chi2_max;       /* (16) candidate cut against the interpolation (2 dof)                  */
  float final_chi2_max;      /* (16) plain cut of the third pass                                      */
  int32_t min_clusters;      /* (10) fewer used clusters: the fit fails                               */
  float ce_var;              /* (1e4 cm^2) as tpc_fit_params                                          */
} tpc_rebuild_params;        /* 16 bytes */
typedef struct tpc_rebuild_view {
  uint64_t n_merged, n_steps;
  const uint32_t* d_step_ofs;      /* [n_merged+1] first path step of each merged track              */
  const int32_t* d_cand_id;        /* [n_steps][3] original cluster ids, -1 none, best first         */
  const float* d_cand_chi2;        /* [n_steps][3]                                                   */
  const int32_t* d_attached;       /* [n_steps] original cluster id or -1                            */
  const uint8_t* d_shared;         /* [n_steps] 1 = attached as shared                               */
  const uint8_t* d_used;           /* [n_steps] 1 = passed the cut of the third pass                 */
  const tpc_track_fit3* d_fit;     /* [n_merged]                                                     */
} tpc_rebuild_view;
void tpc_rebuild_default_params(tpc_rebuild_params* out);
/* Computes the path lengths of the merged tracks (needs tpc_merge_tracks; synchronises cuda_stream) and
 * returns their sum in *n_steps (HOST): the size tpc_rebuild_workspace_bytes needs. */
int tpc_rebuild_prepare(tpc_ctx* ctx, void* cuda_stream, uint64_t* n_steps);
size_t tpc_rebuild_workspace_bytes(const tpc_ctx* ctx, uint64_t n_steps, uint64_t n_merged, uint64_t n_clusters);
/* d_rebuild_workspace: DEVICE, 256-byte aligned, caller owned.  TPC_E_STATE unless tpc_rebuild_prepare ran
 * on the current merged result. */
int tpc_rebuild_tracks(tpc_ctx* ctx, const tpc_rebuild_params* params, void* d_rebuild_workspace,
                       size_t workspace_bytes, void* cuda_stream);
int tpc_get_rebuild(tpc_ctx* ctx, tpc_rebuild_view* out);

/* Number of kernel launches the last tpc_sector_track enqueued. */
int tpc_last_launch_count(const tpc_ctx* ctx);

void tpc_destroy(tpc_ctx* ctx);
const char* tpc_strerror(int err);
/* Text of the last failing CUDA call of this context ("" if none). */
const char* tpc_last_cuda_error(const tpc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TPC_TRACK_H */
