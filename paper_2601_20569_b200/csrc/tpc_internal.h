// tpc_internal.h — internal types shared by the host API (tpc_api.cu) and the two builds of
// the kernel translation unit (tpc_kernels.cu compiled once with -DTPC_DET=1 --fmad=false as
// namespace tpc_det, once with -DTPC_DET=0 --fmad=true as namespace tpc_fast).
// Product code: nothing here is used by, or uses, the oracle.
#ifndef TPC_INTERNAL_H
#define TPC_INTERNAL_H

#include <cuda_runtime.h>
#include <stdint.h>

#include "tpc_track.h"

#define TPC_MAX_ROWS 256

// Per-context constants, resident in device global memory (DESIGN.md rule D5: tables are
// computed in double on the host and rounded once to fp32).
struct TpcConst {
  int32_t n_sectors, n_rows;
  float dx_row;   // row pitch (r_max-r_min)/(n_rows-1)
  float cfield;   // signed curvature per unit q/pT: -0.00299792458*Bz
  float inv_dy, inv_dz;
  float vy, vz;   // err_y^2, err_z^2
  float wy, wz;   // neighbour windows nf_slope_*dx_row
  tpc_params P;
  float x[TPC_MAX_ROWS];
  float ylim[TPC_MAX_ROWS];  // ymax_r + 2 cm
  int32_t ny[TPC_MAX_ROWS];
};

// error bits raised on the device
#define TPC_DEVERR_BAD_CLUSTER 1u   // sector/row outside the geometry -> TPC_E_ARG
#define TPC_DEVERR_BINS 2u          // bin index capacity            -> TPC_E_OVERFLOW
#define TPC_DEVERR_SEEDS 4u         // seed capacity                 -> TPC_E_OVERFLOW
#define TPC_DEVERR_TRACKS 8u        // track / cluster-id capacity   -> TPC_E_OVERFLOW
#define TPC_DEVERR_CHUNKS 16u       // a sector has records in two chunks of a chunked frame -> TPC_E_ARG

struct TpcCounters {
  uint32_t n_sorted, n_ignored, n_dropped, n_bad;
  uint32_t n_bins, n_tiles, n_seeds, n_tracklets;
  uint32_t n_tracks, n_ids, error;
  uint32_t grid_rows;   // 1: every row's input records are contiguous and fit k_row_sort (the per-row grid build)
  uint32_t n_rows_generic;   // rows built by the generic histogram / scan / scatter kernels instead
  uint32_t refit_next;       // chunk counter of the sector-track refit
  // work counters of the follower (roofline numerators): propagation steps, Kalman updates,
  // chi2 evaluations of road candidates
  unsigned long long follow_work[3][3];  // [kernel up/refit/down][steps, updates, candidates]
  // work queues of the three follower kernels (next unclaimed seed)
  uint32_t follow_next[3], pad_;
};

// per (sector,row) statistics of pass 1
struct TpcRowStat {
  uint32_t zmin_key, zmax_key;  // order-preserving uint image of the float
  uint32_t count;               // clusters kept in the grid
  uint32_t n_all;               // input records carrying this (sector,row), kept or not
  uint32_t first, last;         // lowest / highest input index among them
  uint32_t pad_[2];
};

#ifndef TPC_NF_TILE
#define TPC_NF_TILE 256  // clusters per neighbour-finder tile (one CTA)
#endif

// Per-row grid build (k_row_sort): one CTA per (sector,row); the row's bin counters and its
// permutation live in shared memory (16-bit entries).
#define TPC_RS_THREADS 1024
#define TPC_RS_SMEM_BYTES (224 * 1024)   // dynamic shared memory per CTA
#ifndef TPC_RS_BATCH
#ifndef TPC_RS_BATCH
#define TPC_RS_BATCH 4                   // records requested together per thread (C4: 3.08 ms; 6: 3.16, 8: 3.12)
#endif
#endif

// Seeds are handed to the follower / selector ordered by (sector, z-slab, row): tracklets that
// run at the same time then touch the same z-range of every row, which keeps their random
// accesses (grid, owner words) inside L2.  A slab is 1/TPC_SEED_SLABS of a row's z-bins.
#ifndef TPC_SEED_GROUP
#define TPC_SEED_GROUP 1    // z-slabs interleaved row by row in the seed list (must divide TPC_SEED_SLABS)
#endif
#ifndef TPC_SEED_SLABS
#define TPC_SEED_SLABS 64
#endif

// All device buffers of one run (pointers into the caller's workspace, or ctx-owned).
struct TpcBuffers {
  const tpc_cluster* clusters;
  uint32_t n;            // input clusters
  uint32_t n_sr;         // n_sectors*n_rows
  uint32_t n_sectors, n_rows;
  uint32_t id_base;      // added to every original index (chunked frames: position of the chunk in the frame)
  uint32_t chunk_tag;    // 0: whole frame; else 1 + chunk number (sector_seen check)
  uint32_t* sector_seen; // [n_sectors] tag of the chunk that brought records of the sector (ctx-owned)
  uint64_t max_bins;
  uint32_t max_seeds, max_tracks, max_ids;
  uint32_t scan_blocks;  // capacity of scan_partials
  const TpcConst* K;
  TpcCounters* cnt;
  TpcRowStat* row_stat;   // [n_sr]
  tpc_row_desc* row_desc; // [n_sr]
  uint32_t* tile_ofs;     // [n_sr+1] first neighbour-finder tile of each row
  uint16_t* tile_sr;      // [n/TPC_NF_TILE + n_sr + 1] (sector,row) of each neighbour-finder tile
  uint32_t* slot;         // [n] rank of the cluster inside its bin, 0xFFFFFFFF = not in the grid
  uint32_t* bin_start;    // [max_bins+1]
  float2* yz;             // [n] sorted
  uint32_t* orig_id;      // [n] sorted
  int32_t* link_up;       // [n]
  int32_t* link_dn;
  int32_t* link_up2;
  int32_t* link_dn2;
  uint8_t* seed_len;      // [n] chain length if the cluster is a start hit of a seed, else 0
  uint32_t* scan_partials;// [scan_blocks+1]
  uint32_t* item_cnt;     // [n_sr][TPC_SEED_SLABS] seeds per (sector,row,z-slab)
  int32_t* item_delta;    // [n_sr][TPC_SEED_SLABS] list position in (sector,slab,row) order minus rank in sorted order
  uint32_t* seeds;        // [max_seeds] sorted index of start hits, in (sector, z-slab, row, sorted index) order
  uint16_t* seed_sr;      // [max_seeds] sector*n_rows+row of each start hit
  uint4* turn;            // [max_seeds][2] state at the outermost hit (y,z,sin phi,tan lambda | q/pT,row,-,-)
  tpc_tracklet* tracklets;// [max_seeds]
  int32_t* row_hit;       // [max_seeds][n_rows]
  unsigned long long* owner;     // [n]
  unsigned long long* tl_key;    // [max_seeds]
  uint32_t* tl_mask;      // [max_seeds][2][TPC_MAX_ROWS/32] rows with a hit | rows whose hit is owned
  uint32_t* trk_mask;     // [max_tracks][2][TPC_MAX_ROWS/32] accepted rows | shared rows of each track
  uint32_t* trk_sd;       // [max_tracks] tracklet of each track
  uint32_t* seg_cnt;      // [max_seeds+1] tracks per tracklet -> exclusive scan
  uint32_t* id_cnt;       // [max_seeds+1] cluster ids per tracklet -> exclusive scan
  tpc_track* tracks;      // [max_tracks]
  uint32_t* cluster_ids;  // [max_ids]
  uint8_t* cluster_shared;// [max_ids]
  tpc_track_fit* track_fit;// [max_tracks] sector-track refit (R8)
  // compact copy of the tracks' clusters in the order of cluster_ids (written by the refit's outward pass;
  // nullptr: the kernels gather the 16-byte records of the frame by original index instead)
  float2* trk_yz;         // [max_ids] (y, z)
  uint16_t* trk_sr;       // [max_ids] sector << 8 | row
};

// Buffers of the track merging (R9), pointers into the caller's merge workspace.
#define TPC_MG_CAND 4
struct TpcMergeBuffers {
  tpc_merge_params P;
  uint32_t n_tracks, n_ids, n_rows, n_cells;
  float inv_w;            // 1 / width of a z slab of the end grid (= 1 / pre_dz)
  float ca, sa;           // cos / sin of one sector step (tables: double, rounded once)
  uint32_t* cell_start;   // [n_cells+1] inner ends per (sector, first row, z slab) -> exclusive scan
  uint32_t* cell_cursor;  // [n_cells]
  uint32_t* partials;     // scan scratch
  float* ends;            // [n_tracks][16] compact inner-end records in cell order
  int32_t* next; int32_t* prev; float* link_chi2;                  // [n_tracks]
  int32_t* best_out; uint32_t* best_out_chi; uint32_t* best_in_chi; unsigned long long* best_in_key;
  uint2* cand; uint32_t* cand_cnt;   // [n_tracks][TPC_MG_CAND] accepted candidates (partner, chi2 bits) of the stage's pass 1; their number
  uint32_t* head_ofs; uint32_t* seg_ofs; uint32_t* clu_ofs; uint32_t* seg_dst;   // [n_tracks]
  tpc_merged_track* merged;  // [n_tracks]
  uint32_t* seg_index;       // [n_tracks]
  uint32_t* ids; uint8_t* shared;   // [n_ids]
  float2* yz; uint16_t* sr;         // [n_ids] compact copy of the merged lists' clusters (nullptr: gather)
  uint32_t* counters;        // [4] n_merged, n_links, n_ids out, n_steps (R11 paths)
  uint32_t* path_ofs;        // [n_tracks+1] first path step of every merged track (R11), exclusive scan
};

// Buffers of the three-iteration track fit (R10), pointers into the caller's fit workspace.
struct TpcFitBuffers {
  tpc_fit_params P;
  float ca, sa;
  uint4* stored;           // [n_ids] predictions of iteration 1: halves (ry, rz | c00, c10 | c11, -)
  float* chi2_cluster;     // [n_ids]
  uint8_t* rejected;       // [n_ids]
  tpc_track_fit3* fit;     // [n_merged]
  uint32_t* work;          // [4] chunk counter
};

// Buffers of the Phase-II rebuild (R11), pointers into the caller's rebuild workspace.
#define TPC_RB_NCAND 3
struct TpcRebuildBuffers {
  tpc_rebuild_params P;
  float ca, sa;
  uint32_t n_merged, n_steps, n_clusters;
  const uint32_t* step_ofs;    // [n_merged+1] (= merge workspace path_ofs)
  uint4* stored;               // [n_steps] pass-1 prediction: y, z (fp32), halves C00|C10, C11 | bit 16 of .w: the
                               // step holds an original cluster; after pass 2 the region holds the loser lists
  int32_t* cand_id;            // [n_steps][3] original cluster ids, -1 none
  float* cand_chi2;            // [n_steps][3]
  int32_t* attached;           // [n_steps]
  uint8_t* shared; uint8_t* used;   // [n_steps]
  uint32_t* step_track;        // [n_steps] merged track of the step
  uint32_t* Qkey;              // [n_merged] orderable weight
  unsigned long long* tkey;    // [n_merged] 64-bit id of the track (that of its head segment)
  uint8_t* alive;              // [n_merged]
  float* stq2;                 // [n_merged][3] (s,t,q) after pass 2
  uint32_t* list_n;            // [8] lengths of the three loser lists; [4] chunk counter of pass 1+2
  unsigned long long* best;    // [n_clusters] Q key << 32 | round tag << 30 | (0x3FFFFFFF - merged track) of the best proposer; 0 none
  unsigned long long* bestId;  // [n_clusters] least 64-bit track id among proposers of equal weight (ties only)
  tpc_track_fit3* fit;         // [n_merged]
};

#define TPC_MAX_KERNELS 32
struct TpcStageEvents {
  cudaEvent_t ev[TPC_N_STAGES];  // boundaries: start, after grid, nf, seeds, follower, selector
  cudaEvent_t kev[TPC_MAX_KERNELS + 1];  // kev[0] before the first kernel, kev[i+1] after kernel i
  const char* kname[TPC_MAX_KERNELS];
  int n_kernels;
  bool enabled;
};

namespace tpc_det {
int run_rebuild_paths(const TpcBuffers& B, const TpcMergeBuffers& M, cudaStream_t stream, int n_sm);
int run_rebuild(const TpcBuffers& B, const TpcConst* host_const, const TpcMergeBuffers& M, const TpcRebuildBuffers& Rb, cudaStream_t stream, int n_sm);
int run_fit3(const TpcBuffers& B, const TpcConst* host_const, const TpcMergeBuffers& M, const TpcFitBuffers& T, uint32_t n_merged, cudaStream_t stream, int n_sm);
int run_merge(const TpcBuffers& B, const TpcConst* host_const, const TpcMergeBuffers& M, cudaStream_t stream, int n_sm);
int run_refit(const TpcBuffers& B, const TpcConst* host_const, uint32_t n_tracks, cudaStream_t stream, int n_sm);
int run_pipeline(const TpcBuffers& B, const TpcConst* host_const, cudaStream_t stream, uint32_t flags, TpcStageEvents& E, int n_sm);
}
namespace tpc_fast {
int run_rebuild_paths(const TpcBuffers& B, const TpcMergeBuffers& M, cudaStream_t stream, int n_sm);
int run_rebuild(const TpcBuffers& B, const TpcConst* host_const, const TpcMergeBuffers& M, const TpcRebuildBuffers& Rb, cudaStream_t stream, int n_sm);
int run_fit3(const TpcBuffers& B, const TpcConst* host_const, const TpcMergeBuffers& M, const TpcFitBuffers& T, uint32_t n_merged, cudaStream_t stream, int n_sm);
int run_merge(const TpcBuffers& B, const TpcConst* host_const, const TpcMergeBuffers& M, cudaStream_t stream, int n_sm);
int run_refit(const TpcBuffers& B, const TpcConst* host_const, uint32_t n_tracks, cudaStream_t stream, int n_sm);
int run_pipeline(const TpcBuffers& B, const TpcConst* host_const, cudaStream_t stream, uint32_t flags, TpcStageEvents& E, int n_sm);
}

#endif
