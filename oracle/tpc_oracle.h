/*
 * tpc_oracle.h — C interface of the CPU ORACLE of the TPC sector tracking.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or constant generator with the CUDA path under paper_2601_20569_b200/csrc: the
 * structs below are the oracle's own definitions (the parameter list of the method is the
 * same list on both sides because it IS the method's parameter list).
 *
 * What it computes: the sector tracking of PAPER.md:25-27 (section 2) with the Phase-I
 * ambiguity criterion of PAPER.md:57 (section 3) and the search grid of PAPER.md:59,
 * step by step in the order of DESIGN.md "Readings" R0..R6:
 *   R0 geometry tables, R1 grid, R2 neighbour finder, R3 link cleanup, R4 seeds,
 *   R5 Kalman track following, R6 ambiguity solving.
 * Plain single-threaded loops per sector (sectors may be spread over threads for the timed
 * baseline; the result does not depend on that).  fp32 arithmetic, only + - * / sqrt, built
 * with -ffp-contract=off (rule D1).  All results are expressed in ORIGINAL input indices
 * (rule D3).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): closed-form geometry, exact-helix
 * propagation, finite-difference Jacobian, Kalman update == weighted least squares,
 * unit-width pulls, brute-force neighbour search, grid invariants + brute-force window
 * queries, link/seed invariants, selector invariants and constructed cases; the follower's road
 * search by hand-computed cases on a radial straight track and a brute-force linear scan of every
 * search (test_oracle_road_search.py); merging (test_oracle_merging.py) and the three-iteration fit
 * (test_oracle_trackfit.py) by exact geometry, textbook least squares and hand-built cases.  Each
 * group is mutation-checked.
 * Parity unpinned: absolute efficiency / clone / fake values (the paper's Fig. 2 is an
 * image that is not in PAPER.md and is ALICE MC); only sanity floors are tested.
 */
#ifndef TPC_ORACLE_H
#define TPC_ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_cluster { /* 16 bytes, the input record (BASELINE.json config 4) */
  float y, z, q;
  uint8_t sector, row;
  uint16_t flags;
} orc_cluster;

typedef struct orc_geom {
  int32_t n_sectors, n_rows, n_inner_rows;
  float r_min, r_max, pad_pitch_inner, pad_pitch_outer, z_max, bz_tesla, sector_half_angle_deg;
} orc_geom;

typedef struct orc_params {
  float err_y, err_z;
  float nf_slope_y, nf_slope_z, nf_max_d2;
  int32_t seed_min_len;
  float init_var_sinphi, init_var_tanl, init_var_qpt;
  float max_sinphi, max_qpt;
  float road_nsigma, road_min, road_max;
  float chi2_max_hit;
  int32_t max_gap_follow, min_hits_tracklet;
  float sel_chi2_weight;
  int32_t shared_permille, max_gap_select, min_hits_track;
  float grid_dy, grid_dz;
  int32_t shared_fixed_cap; /* 0: running fraction from the outermost row (Phase I); 1: fixed cap
                               floor(shared_permille * nHits / 1000) per segment (the rule before Phase I) */
} orc_params;

typedef struct orc_row_desc {
  float y0, z0;
  int32_t ny, nz;
  uint32_t bin_ofs, clu_ofs, count, pad_;
} orc_row_desc;

typedef struct orc_seed {
  uint32_t start_id; /* original index of the start hit */
  int32_t len;       /* clusters in the link chain */
  int32_t sector, row;
} orc_seed;

typedef struct orc_tracklet {
  float x, p[5], c[15], chi2;
  uint32_t seed_id;
  int32_t n_hits; /* 0 = rejected (below min_hits_tracklet or broken) */
  int32_t row_first, row_last, sector, seed_len;
} orc_tracklet;

typedef struct orc_track {
  float x, p[5], c[15], chi2;
  uint32_t cluster_ofs, seed_id;
  int32_t n_clusters, n_shared;
  int32_t sector, row_first, row_last, flags; /* flags bit0 = PARAMS_STALE */
  int32_t n_hits_tracklet, segment;
} orc_track;

/* One road search of the follower (R5.3 / R5.6), recorded for the pins only (orc_set_trace):
 * the PREDICTED state on the row, whether the row was searched (|y| <= ylim_r), the best
 * candidate found (original id, -1 none), its chi2 and whether it was accepted. */
typedef struct orc_trace_rec {
  int32_t seed, row, dir, searched;
  float y, z, c00, c10, c11, chi2;
  int32_t picked_id, accepted;
} orc_trace_rec;

typedef struct orc_result orc_result;

void orc_default_params(orc_params* p);

/* Run the whole path on sectors [sector_lo, sector_hi) of the frame.  n_threads > 1 spreads
 * sectors over std::threads (same result).  Returns NULL on a bad argument. */
orc_result* orc_run(const orc_cluster* clusters, uint64_t n, const orc_geom* g, const orc_params* p,
                    int sector_lo, int sector_hi, int n_threads);
void orc_free(orc_result* r);

/* sizes: out[0]=n_rows_total out[1]=n_bins out[2]=n_sorted out[3]=n_seeds out[4]=n_tracks
 * out[5]=n_cluster_ids out[6]=n_ignored out[7]=n_dropped out[8]=n_bad (sector/row outside geometry)
 * out[9]=n_tracklets (n_hits>0) */
void orc_sizes(const orc_result* r, uint64_t out[10]);
/* road-search trace (pins only): orc_set_trace(1) before orc_run (single-threaded use), then
 * orc_trace_size / orc_fetch_trace; the trace is observation only, no result depends on it */
void orc_set_trace(int on);
uint64_t orc_trace_size(const orc_result* r);
void orc_fetch_trace(const orc_result* r, orc_trace_rec* out);
/* stage wall times in seconds: grid, neighbours, cleanup+seeds, follower, selector */
void orc_stage_seconds(const orc_result* r, double out[5]);
/* copy-out; any pointer may be NULL.  Links are indexed by ORIGINAL cluster index and hold
 * original indices (-1 none); entries of clusters outside [sector_lo,sector_hi) are -1. */
void orc_fetch_grid(const orc_result* r, orc_row_desc* rows, uint32_t* bin_start, uint32_t* sorted_ids);
void orc_fetch_links(const orc_result* r, int32_t* up, int32_t* dn, int32_t* up2, int32_t* dn2);
void orc_fetch_seeds(const orc_result* r, orc_seed* seeds);
void orc_fetch_tracklets(const orc_result* r, orc_tracklet* t, int32_t* row_hit /*[n_seeds][n_rows]*/);
void orc_fetch_tracks(const orc_result* r, orc_track* t, uint32_t* cluster_ids, uint8_t* shared);

/* ---- single-step entry points for the pins (float = the path's type, double = same
 * statements instantiated in double) ---- */
/* tables: x[n_rows], ymax[n_rows]; consts[0]=dx_row consts[1]=cfield (curvature per q/pT) */
void orc_geom_tables(const orc_geom* g, float* x, float* ymax, float* consts);
/* state = y,z,s,t,q,c[15] (20 values). returns 1 if propagated, 0 if the leg ends */
int orc_propagate_f(float* state, float dx, float cfield, float max_sinphi, float* jac6);
int orc_propagate_d(double* state, double dx, double cfield, double max_sinphi, double* jac6);
/* returns chi2 of the hit; *stop = 1 if |sin phi| left the range */
float orc_update_f(float* state, float ym, float zm, float vy, float vz, float max_sinphi, float max_qpt, int* stop);
double orc_update_d(double* state, double ym, double zm, double vy, double vz, double max_sinphi, double max_qpt, int* stop);
/* Kalman fit of a given hit list (truth association) exactly as steps R5.1/R5.2/R5.4/R5.5 do
 * (up pass over the hits, turn, refit down).  rows[] ascending, consecutive or with gaps.
 * out_state = 20 floats at rows[0]; returns chi2 of the down pass or -1 if the leg stopped. */
float orc_fit_hits(const orc_geom* g, const orc_params* p, const int32_t* rows, const float* y,
                   const float* z, int n, float* out_state);
/* R8 sector-track refit: pure Kalman fit of a given cluster list (rows strictly ascending, holes
 * allowed; outward pass, turn, inward pass; no search, no chi2 cut).  out_state = x, p[5], c[15], n
 * at rows[0], then x_out, p_out[5], c_out[15] = the state after the outward pass at rows[n-1]
 * (43 floats); returns the chi2 of the inward pass or -1 if the fit left |sin phi|. */
float orc_refit_hits(const orc_geom* g, const orc_params* p, const int32_t* rows, const float* y,
                     const float* z, int n, float* out_state);
/* selector on hand-made tracklets: row_hit[n_tracklets][n_rows] (cluster ids or -1),
 * n_hits/chi2/seed_id per tracklet.  Results via orc_fetch_tracks. */
orc_result* orc_select_only(const orc_geom* g, const orc_params* p, uint64_t n_clusters, int n_tracklets,
                            const int32_t* row_hit, const int32_t* n_hits, const float* chi2,
                            const uint32_t* seed_id);

/* ---- R9 track merging (tpc_merge_oracle.cpp; section 2, section 3) ---- */
typedef struct orc_merge_params {
  int32_t gap_in_sector;     /* (30) stage 1: 1 <= row_first_b - row_last_a <= this                  */
  int32_t gap_adjacent_back; /* (3)  stage 2: -this <= row_first_b - row_last_a                        */
  int32_t gap_adjacent;      /* (10) stage 2:          row_first_b - row_last_a <= this                */
  int32_t gap_ce;            /* (6)  stage 3: 1 <= row_first_b - row_last_a <= this                    */
  float chi2_max;            /* (20) match cut on the 5-parameter chi2                                 */
  float sys[5];              /* (0.3 cm, 0.3 cm, 0.02, 0.02, 0.2 c/GeV) added in quadrature per parameter */
  float ce_sys_z;            /* (3 cm) replaces sys[1] across the central electrode                   */
  float pre_dy, pre_dz;      /* (8 cm, 8 cm) pre-cuts on y and z between the transported state and b's     */
  float pre_coarse_dz;       /* (40 cm) pre-cut on z between the two end states as they are               */
  int32_t stages;            /* (7) bit 0: in sector, bit 1: adjacent sectors, bit 2: central electrode */
} orc_merge_params;

typedef struct orc_merge_track { /* one sector track as the merging sees it */
  int32_t sector, row_first, row_last, valid; /* valid = 0: refit failed, takes no part */
  uint32_t seed_id;
  int32_t segment, iter;                       /* iter = 1 for tracks of the second seeding iteration */
  float p_in[5], c_in[15];                     /* R8 state at the innermost cluster's row  */
  float p_out[5], c_out[15];                   /* R8 state after the outward pass at the outermost cluster's row */
} orc_merge_track;

void orc_merge_default_params(orc_merge_params* m);
/* next[k] / prev[k] = track linked behind / before track k (-1 none), link_chi2[k] = chi2 of the
 * link k -> next[k] (may be NULL).  Returns the number of links or -1. */
int orc_merge_links(const orc_geom* g, const orc_params* p, const orc_merge_params* m, const orc_merge_track* t,
                    int32_t n, int32_t* next, int32_t* prev, float* link_chi2);
/* rotation of a state (y,z,s,t,q,c[15]) at local *x into the neighbouring sector's frame
 * (sign +1: the sector with the next higher azimuth); returns 0 if |sin phi| leaves the range */
int orc_merge_rotate(const orc_geom* g, float* state20, float* x, int sign, float max_sinphi);

/* ---- R10 three-iteration track fit with interpolation rejection (tpc_fit_oracle.cpp;
 * PAPER.md:31,37 section 2, section 3) ---- */
typedef struct orc_fit_params {
  float fit_chi2_max;       /* (16) cut on the 2-dof chi2 of a cluster against the interpolation   */
  int32_t fit_min_clusters; /* (10) fewer unmarked clusters: the fit fails                         */
  float ce_var;             /* (1e4 cm^2) variance given to z when it is re-based at the electrode */
} orc_fit_params;
void orc_fit_default_params(orc_fit_params* f);
/* IEEE binary16 round-to-nearest-even conversions ("reduced precision" of the stored predictions) */
uint16_t orc_float_to_half(float f);
float orc_half_to_float(uint16_t h);
/* One track: n clusters in chain order (sector, row, y, z), start_stq = (sin phi, tan lambda, q/pT) at
 * the outermost cluster.  out_state = x, p[5], c[15] at the innermost unmarked cluster's row;
 * chi2_cluster[n] = interpolation chi2 of iteration 2; rejected[n] = 1 where marked; *n_used =
 * unmarked clusters.  Returns the chi2 of iteration 3, or -1 if the fit failed. */
float orc_fit_track(const orc_geom* g, const orc_params* p, const orc_fit_params* f, const int32_t* sector,
                    const int32_t* row, const float* y, const float* z, int n, const float* start_stq,
                    float* out_state, float* chi2_cluster, uint8_t* rejected, int32_t* n_used);

/* ---- R11 Phase-II track rebuild (tpc_rebuild_oracle.cpp; section 3) ---- */
#define ORC_RB_NCAND 3 /* candidates kept per (track, path step) */
typedef struct orc_rebuild_params {
  float cand_chi2_max;   /* (16) a cluster is a candidate if its chi2 against the interpolation is below */
  float final_chi2_max;  /* (16) plain cut of the third iteration                                       */
  int32_t min_clusters;  /* (10) fewer used clusters: the fit fails                                     */
  float ce_var;          /* (1e4 cm^2) as orc_fit_params                                                */
} orc_rebuild_params;
typedef struct orc_rb_segment { int32_t sector, row_first, row_last; } orc_rb_segment;
void orc_rebuild_default_params(orc_rebuild_params* r);
/* number of (sector,row) steps on the path of a chain of segments */
int64_t orc_rebuild_path_len(const orc_rb_segment* seg, int32_t n_seg);
/* Phase II for ALL merged tracks of a frame (the second ambiguity solving couples them).  Per merged
 * track m: segments segs[seg_ofs[m]..seg_ofs[m+1]), original clusters cluster_ids[clu_ofs[m]..) in chain
 * order, start (s,t,q), valid flag, a unique 64-bit id for exact ties, path steps [step_ofs[m],
 * step_ofs[m+1]).  Outputs per step: up to ORC_RB_NCAND candidates (original ids, -1 none) with their
 * chi2, the attached cluster (-1 none), shared / used flags; per track: x,p[5],c[15] (21 floats) at the
 * innermost used cluster, chi2 of pass 3, attached / used counts, flags (1 = failed).
 * Returns 0, -1 bad argument, -2 inconsistent offsets. */
int orc_rebuild(const orc_geom* g, const orc_params* p, const orc_rebuild_params* r, const orc_cluster* clusters,
                uint64_t n_clusters, int32_t n_merged, const int32_t* seg_ofs, const orc_rb_segment* segs,
                const int64_t* clu_ofs, const uint32_t* cluster_ids, const float* start_stq, const uint8_t* valid,
                const uint64_t* key_id, const int64_t* step_ofs, int32_t* cand_id, float* cand_chi2,
                int32_t* attached, uint8_t* shared, uint8_t* used, float* fit, float* chi2, int32_t* n_attached,
                int32_t* n_used, uint8_t* flags);

#ifdef __cplusplus
}
#endif
#endif
