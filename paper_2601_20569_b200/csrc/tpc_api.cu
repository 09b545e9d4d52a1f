// tpc_api.cu — the C ABI of include/tpc_track.h: context, workspace carving, stream handling.
// Host code only; all arithmetic of the method runs in the kernels of tpc_kernels.cu.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "tpc_internal.h"

struct tpc_ctx {
  tpc_geom_desc geom;
  tpc_params params;
  TpcConst hconst;
  TpcConst* d_const = nullptr;
  TpcCounters* d_cnt = nullptr;
  TpcRowStat* d_row_stat = nullptr;
  TpcCounters* h_cnt = nullptr;  // pinned
  uint32_t* d_sector_seen = nullptr;
  // chunked host call: copy-in / copy-out streams and their events (ping-pong)
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
  TpcStageEvents events;
  int n_sm = 148;
  int device = 0;
  // last run
  bool ran = false;
  bool synced = false;
  TpcBuffers buf;
  cudaStream_t stream = nullptr;
  uint32_t flags = 0;
  int launches = 0;
  uint64_t n_bins_cap = 0;
  bool refit_done = false;     // tpc_refit_tracks ran on the current result
  bool merged = false;         // tpc_merge_tracks ran on the current result
  bool fitted = false;         // tpc_fit_tracks ran on the current merged result
  bool rb_prepared = false, rebuilt = false;   // tpc_rebuild_prepare / tpc_rebuild_tracks ran on it
  uint64_t rb_n_steps = 0;
  TpcRebuildBuffers rbuf;
  TpcMergeBuffers mbuf;
  TpcFitBuffers fbuf;
  uint32_t fit_n_merged = 0, fit_n_ids = 0;
  uint32_t* h_mcnt = nullptr;  // pinned: merge counters
  void* noalloc_scratch = nullptr;   // device address of g_fit_noalloc_scratch on this context's device (set-up)
  char noalloc_err[128] = {0};       // why it could not be resolved
  char cuda_err[256] = {0};
};

// ---- scratch of tpc_fit_tracks_noalloc: ONE array inside the library, held by every GPU that loads it.
// Layout: [0,16) counters (word 0: merged-track count), [16,32) work counter of the kernel, [256, ...) the
// predictions stored in iteration 1 (16 bytes per cluster id).  In HOST code the name below is a
// stand-in, not a device address: the address comes from cudaGetSymbolAddress, once per device, at
// set-up (noalloc_setup, called by tpc_geom_init with that device current).
#define TPC_FIT_NOALLOC_HDR 256
static __device__ __align__(256) unsigned char g_fit_noalloc_scratch[TPC_FIT_NOALLOC_HDR + 16ull * TPC_FIT_NOALLOC_MAX_IDS];

// (device code of this file names the array directly)
__global__ void k_fit_noalloc_header(uint32_t n_merged) {
  uint32_t* h = reinterpret_cast<uint32_t*>(g_fit_noalloc_scratch);
  if (threadIdx.x < 8) h[threadIdx.x] = threadIdx.x == 0 ? n_merged : 0u;
}

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

#define TPC_NOALLOC_MAX_DEVICES 64
std::mutex g_noalloc_mutex;
void* g_noalloc_ptr[TPC_NOALLOC_MAX_DEVICES] = {nullptr};
bool g_noalloc_done[TPC_NOALLOC_MAX_DEVICES] = {false};
cudaError_t g_noalloc_rc[TPC_NOALLOC_MAX_DEVICES] = {cudaSuccess};

// Once per device, with that device current.  Never fatal for the caller: a failure is reported by
// tpc_fit_tracks_noalloc alone.
void noalloc_setup(tpc_ctx* c) {
  c->noalloc_scratch = nullptr;
  if (c->device < 0 || c->device >= TPC_NOALLOC_MAX_DEVICES) {
    std::snprintf(c->noalloc_err, sizeof(c->noalloc_err), "device ordinal %d beyond %d", c->device, TPC_NOALLOC_MAX_DEVICES);
    return;
  }
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  if (!g_noalloc_done[c->device]) {
    void* p = nullptr;
    g_noalloc_rc[c->device] = cudaGetSymbolAddress(&p, g_fit_noalloc_scratch);
    g_noalloc_ptr[c->device] = g_noalloc_rc[c->device] == cudaSuccess ? p : nullptr;
    g_noalloc_done[c->device] = true;
    if (g_noalloc_rc[c->device] != cudaSuccess) (void)cudaGetLastError();
  }
  c->noalloc_scratch = g_noalloc_ptr[c->device];
  if (!c->noalloc_scratch)
    std::snprintf(c->noalloc_err, sizeof(c->noalloc_err), "cudaGetSymbolAddress: %s", cudaGetErrorString(g_noalloc_rc[c->device]));
}

int set_cuda_err(tpc_ctx* c, cudaError_t e, const char* what) {
  if (c) std::snprintf(c->cuda_err, sizeof(c->cuda_err), "%s: %s", what, cudaGetErrorString(e));
  return TPC_E_CUDA;
}

struct Capacities {
  uint64_t max_bins;
  uint32_t max_seeds, max_tracks, max_ids, scan_blocks;
};

Capacities capacities(const tpc_ctx* c, uint64_t n) {
  Capacities k;
  const tpc_params& P = c->params;
  int ny_max = 1;
  for (int r = 0; r < c->geom.n_rows; ++r) ny_max = c->hconst.ny[r] > ny_max ? c->hconst.ny[r] : ny_max;
  uint64_t bins = P.max_bins;
  if (bins == 0)
    bins = 4 * n + (uint64_t)c->geom.n_sectors * c->geom.n_rows * ny_max *
                       ((uint64_t)std::ceil(c->geom.z_max / P.grid_dz) + 2);
  if (bins > 0xFFFFFFF0ull) bins = 0xFFFFFFF0ull;
  k.max_bins = bins;
  // seeds per cluster measured on the five workloads: 1/19 (C2, C3, C4), 1/23 (C5); the default leaves
  // a third of headroom (was n/8: 18 GB of row_hit for the C4 frame); beyond it: TPC_E_OVERFLOW, set max_seeds
  uint64_t seeds = P.max_seeds ? P.max_seeds : n / 12 + 4096;
  seeds = align_up(seeds, 64);
  k.max_seeds = (uint32_t)seeds;
  const uint64_t ids = P.max_ids ? (uint64_t)P.max_ids : n * 1000 / (1000 - (uint64_t)P.shared_permille) + 64;
  k.max_ids = (uint32_t)(ids > 0xFFFFFFF0ull ? 0xFFFFFFF0ull : ids);
  k.max_tracks = (uint32_t)(k.max_ids / (uint32_t)(P.min_hits_track > 0 ? P.min_hits_track : 1) + 1);
  const uint64_t b1 = (n + 1023) / 1024 + 2, b2 = 2 * ((seeds + 255) / 256 + 2);
  k.scan_blocks = (uint32_t)(b1 > b2 ? b1 : b2);
  return k;
}

// Carve the workspace.  base == nullptr: only the size is computed.
size_t carve(const tpc_ctx* c, uint64_t n, char* base, TpcBuffers* B) {
  const Capacities k = capacities(c, n);
  const uint32_t n_sr = (uint32_t)(c->geom.n_sectors * c->geom.n_rows);
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* p = base ? base + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  };
  TpcBuffers b;
  std::memset(&b, 0, sizeof(b));
  b.n = (uint32_t)n;
  b.n_sr = n_sr;
  b.n_sectors = (uint32_t)c->geom.n_sectors;
  b.n_rows = (uint32_t)c->geom.n_rows;
  b.max_bins = k.max_bins;
  b.max_seeds = k.max_seeds;
  b.max_tracks = k.max_tracks;
  b.max_ids = k.max_ids;
  b.scan_blocks = k.scan_blocks;
  b.row_desc = (tpc_row_desc*)take(sizeof(tpc_row_desc) * n_sr);
  b.tile_ofs = (uint32_t*)take(4 * (size_t)(n_sr + 1));
  b.tile_sr = (uint16_t*)take(2 * (size_t)(n / TPC_NF_TILE + n_sr + 1));
  b.slot = (uint32_t*)take(4 * n);
  b.bin_start = (uint32_t*)take(4 * (k.max_bins + 4));
  b.yz = (float2*)take(8 * n);
  b.orig_id = (uint32_t*)take(4 * n);
  b.link_up = (int32_t*)take(4 * n);
  b.link_dn = (int32_t*)take(4 * n);
  b.link_up2 = (int32_t*)take(4 * n);
  b.link_dn2 = (int32_t*)take(4 * n);
  b.seed_len = (uint8_t*)take(n);
  b.scan_partials = (uint32_t*)take(4 * (size_t)(k.scan_blocks + 2));
  b.item_cnt = (uint32_t*)take(4 * (size_t)n_sr * TPC_SEED_SLABS);
  b.item_delta = (int32_t*)take(4 * (size_t)n_sr * TPC_SEED_SLABS);
  b.seeds = (uint32_t*)take(4 * (size_t)k.max_seeds);
  b.seed_sr = (uint16_t*)take(2 * (size_t)k.max_seeds);
  b.turn = (uint4*)take(32 * (size_t)k.max_seeds);
  b.tracklets = (tpc_tracklet*)take(sizeof(tpc_tracklet) * (size_t)k.max_seeds);
  b.row_hit = (int32_t*)take(4 * (size_t)c->geom.n_rows * k.max_seeds);
  b.owner = (unsigned long long*)take(8 * n);
  b.tl_key = (unsigned long long*)take(8 * (size_t)k.max_seeds);
  b.tl_mask = (uint32_t*)take(4 * (size_t)(2 * (TPC_MAX_ROWS / 32)) * k.max_seeds);
  b.trk_mask = (uint32_t*)take(4 * (size_t)(2 * (TPC_MAX_ROWS / 32)) * k.max_tracks);
  b.trk_sd = (uint32_t*)take(4 * (size_t)k.max_tracks);
  b.seg_cnt = (uint32_t*)take(4 * (size_t)(k.max_seeds + 1));
  b.id_cnt = (uint32_t*)take(4 * (size_t)(k.max_seeds + 1));
  b.tracks = (tpc_track*)take(sizeof(tpc_track) * (size_t)k.max_tracks);
  b.cluster_ids = (uint32_t*)take(4 * (size_t)k.max_ids);
  b.cluster_shared = (uint8_t*)take((size_t)k.max_ids);
  b.track_fit = (tpc_track_fit*)take(sizeof(tpc_track_fit) * (size_t)k.max_tracks);
  if (B) *B = b;
  return off;
}

}  // namespace

extern "C" {

void tpc_default_params(tpc_params* p) {
  std::memset(p, 0, sizeof(*p));
  p->err_y = 0.1f; p->err_z = 0.1f;
  p->nf_slope_y = 1.0f; p->nf_slope_z = 1.6f; p->nf_max_d2 = 0.70f;
  p->seed_min_len = 4;
  p->init_var_sinphi = 0.25f; p->init_var_tanl = 4.0f; p->init_var_qpt = 100.0f;
  p->max_sinphi = 0.95f; p->max_qpt = 20.0f;
  p->road_nsigma = 3.5f; p->road_min = 0.3f; p->road_max = 2.0f;
  p->chi2_max_hit = 12.0f;
  p->max_gap_follow = 4; p->min_hits_tracklet = 10;
  p->sel_chi2_weight = 2.0f;
  p->shared_permille = 100; p->max_gap_select = 4; p->min_hits_track = 20;
  p->grid_dy = 2.0f; p->grid_dz = 2.0f;
  p->max_bins = 0; p->max_seeds = 0;
  p->max_ids = 0; p->reserved = 0;
}

int tpc_geom_init(const tpc_geom_desc* geom, const tpc_params* params, tpc_ctx** out) {
  if (!geom || !out) return TPC_E_ARG;
  *out = nullptr;
  if (geom->n_sectors < 1 || geom->n_sectors > 256 || geom->n_rows < 3 || geom->n_rows > 255 ||
      !(geom->r_max > geom->r_min) || !(geom->r_min > 0.f) || !(geom->sector_half_angle_deg > 0.f) ||
      !(geom->sector_half_angle_deg < 90.f) || !(geom->z_max > 0.f))
    return TPC_E_ARG;
  tpc_params P;
  if (params) P = *params; else tpc_default_params(&P);
  if (!(P.grid_dy > 0.f) || !(P.grid_dz > 0.f) || P.shared_permille < 0 || P.shared_permille > 500 ||
      P.seed_min_len < 2 || P.seed_min_len > 255 || P.min_hits_track < 1 ||
      P.min_hits_tracklet < 3 ||   // ndf = 2*nHits - 5 of the selection weight (R6.1) must be positive
      !(P.err_y > 0.f) || !(P.err_z > 0.f) || !(P.max_sinphi > 0.f) || !(P.max_sinphi < 1.f) ||
      P.max_gap_follow < 0 || P.max_gap_select < 0)
    return TPC_E_ARG;
  tpc_ctx* c = new (std::nothrow) tpc_ctx();
  if (!c) return TPC_E_ARG;
  c->geom = *geom;
  c->params = P;
  // R0 tables in double, rounded once to fp32 (rule D5)
  TpcConst& K = c->hconst;
  std::memset(&K, 0, sizeof(K));
  K.n_sectors = geom->n_sectors;
  K.n_rows = geom->n_rows;
  const double pitch = ((double)geom->r_max - (double)geom->r_min) / (double)(geom->n_rows - 1);
  const double th = std::tan((double)geom->sector_half_angle_deg * (3.14159265358979323846 / 180.0));
  for (int r = 0; r < geom->n_rows; ++r) {
    const double xr = (double)geom->r_min + r * pitch;
    const double ym = xr * th;
    K.x[r] = (float)xr;
    K.ylim[r] = (float)(ym + 2.0);
    const int ny = (int)std::ceil(2.0 * (ym + 2.0) / (double)P.grid_dy);
    K.ny[r] = ny < 1 ? 1 : ny;
  }
  K.dx_row = (float)pitch;
  K.cfield = (float)(-0.00299792458 * (double)geom->bz_tesla);
  K.inv_dy = 1.0f / P.grid_dy;
  K.inv_dz = 1.0f / P.grid_dz;
  K.vy = P.err_y * P.err_y;
  K.vz = P.err_z * P.err_z;
  K.wy = P.nf_slope_y * K.dx_row;
  K.wz = P.nf_slope_z * K.dx_row;
  K.P = P;
  cudaError_t e;
  const uint32_t n_sr = (uint32_t)(geom->n_sectors * geom->n_rows);
  if ((e = cudaGetDevice(&c->device)) != cudaSuccess ||
      (e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device)) != cudaSuccess ||
      (e = cudaMalloc(&c->d_const, sizeof(TpcConst))) != cudaSuccess ||
      (e = cudaMalloc(&c->d_cnt, sizeof(TpcCounters))) != cudaSuccess ||
      (e = cudaMalloc(&c->d_row_stat, sizeof(TpcRowStat) * n_sr)) != cudaSuccess ||
      (e = cudaMallocHost(&c->h_cnt, sizeof(TpcCounters))) != cudaSuccess ||
      (e = cudaMallocHost(&c->h_mcnt, 4 * sizeof(uint32_t))) != cudaSuccess ||
      (e = cudaMalloc(&c->d_sector_seen, sizeof(uint32_t) * (size_t)geom->n_sectors)) != cudaSuccess ||
      (e = cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking)) != cudaSuccess ||
      (e = cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking)) != cudaSuccess ||
      (e = cudaMemcpy(c->d_const, &K, sizeof(TpcConst), cudaMemcpyHostToDevice)) != cudaSuccess) {
    std::fprintf(stderr, "tpc_geom_init: %s\n", cudaGetErrorString(e));
    tpc_destroy(c);
    return TPC_E_CUDA;
  }
  noalloc_setup(c);   // (address of the library's static scratch on this device; see tpc_fit_tracks_noalloc)
  c->events.enabled = false;
  c->events.n_kernels = 0;
  for (int i = 0; i < TPC_N_STAGES; ++i) c->events.ev[i] = nullptr;
  for (int i = 0; i <= TPC_MAX_KERNELS; ++i) c->events.kev[i] = nullptr;
  for (int i = 0; i < TPC_N_STAGES; ++i) {
    if ((e = cudaEventCreate(&c->events.ev[i])) != cudaSuccess) {
      tpc_destroy(c);
      return TPC_E_CUDA;
    }
  }
  for (int i = 0; i <= TPC_MAX_KERNELS; ++i) {
    if ((e = cudaEventCreate(&c->events.kev[i])) != cudaSuccess) {
      tpc_destroy(c);
      return TPC_E_CUDA;
    }
  }
  for (int i = 0; i < 2; ++i) {
    if ((e = cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming)) != cudaSuccess ||
        (e = cudaEventCreateWithFlags(&c->ev_out[i], cudaEventDisableTiming)) != cudaSuccess) {
      tpc_destroy(c);
      return TPC_E_CUDA;
    }
  }
  *out = c;
  return TPC_OK;
}

size_t tpc_workspace_bytes(const tpc_ctx* ctx, uint64_t n_clusters) {
  if (!ctx || n_clusters >= (1ull << 30)) return 0;
  return carve(ctx, n_clusters, nullptr, nullptr);
}

static int enqueue_track(tpc_ctx* ctx, const tpc_cluster* d_clusters, uint64_t n_clusters, void* d_workspace,
                         size_t workspace_bytes, void* cuda_stream, uint32_t flags, uint32_t id_base, uint32_t chunk_tag) {
  if (!ctx || !d_workspace || (!d_clusters && n_clusters) || n_clusters >= (1ull << 30)) return TPC_E_ARG;
  if (((uintptr_t)d_clusters & 15u) || ((uintptr_t)d_workspace & 255u)) return TPC_E_ARG;
  TpcBuffers B;
  const size_t need = carve(ctx, n_clusters, (char*)d_workspace, &B);
  if (workspace_bytes < need) return TPC_E_WORKSPACE;
  B.clusters = d_clusters;
  B.K = ctx->d_const;
  B.cnt = ctx->d_cnt;
  B.row_stat = ctx->d_row_stat;
  B.id_base = id_base;
  B.chunk_tag = chunk_tag;
  B.sector_seen = ctx->d_sector_seen;
  ctx->buf = B;
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->flags = flags;
  ctx->ran = false;
  ctx->synced = false;
  ctx->refit_done = false;
  ctx->merged = false;
  ctx->fitted = false;
  ctx->rb_prepared = false; ctx->rebuilt = false;
  ctx->events.enabled = (flags & TPC_STAGE_TIMERS) != 0;
  (void)cudaGetLastError();
  const int launches = (flags & TPC_DETERMINISTIC)
                           ? tpc_det::run_pipeline(B, &ctx->hconst, ctx->stream, flags, ctx->events, ctx->n_sm)
                           : tpc_fast::run_pipeline(B, &ctx->hconst, ctx->stream, flags, ctx->events, ctx->n_sm);
  if (launches < 0) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch");
  cudaError_t e = cudaMemcpyAsync(ctx->h_cnt, ctx->d_cnt, sizeof(TpcCounters), cudaMemcpyDeviceToHost, ctx->stream);
  if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(counters)");
  ctx->launches = launches;
  ctx->ran = true;
  return TPC_OK;
}

int tpc_sector_track(tpc_ctx* ctx, const tpc_cluster* d_clusters, uint64_t n_clusters, void* d_workspace,
                     size_t workspace_bytes, void* cuda_stream, uint32_t flags) {
  return enqueue_track(ctx, d_clusters, n_clusters, d_workspace, workspace_bytes, cuda_stream, flags, 0u, 0u);
}

static int sync_run(tpc_ctx* ctx) {
  if (!ctx) return TPC_E_ARG;
  if (!ctx->ran) return TPC_E_STATE;
  if (!ctx->synced) {
    cudaError_t e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaStreamSynchronize");
    ctx->synced = true;
  }
  return TPC_OK;
}

static int device_status(const tpc_ctx* ctx) {
  const uint32_t err = ctx->h_cnt->error;
  if (err & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS | TPC_DEVERR_TRACKS)) return TPC_E_OVERFLOW;
  if (err & (TPC_DEVERR_BAD_CLUSTER | TPC_DEVERR_CHUNKS)) return TPC_E_ARG;
  return TPC_OK;
}

int tpc_get_tracks(tpc_ctx* ctx, tpc_track_view* out) {
  if (!out) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  const TpcCounters& c = *ctx->h_cnt;
  std::memset(out, 0, sizeof(*out));
  rc = device_status(ctx);
  const bool valid = rc != TPC_E_OVERFLOW;
  out->n_tracks = valid ? c.n_tracks : 0;
  out->n_cluster_ids = valid ? c.n_ids : 0;
  out->d_tracks = ctx->buf.tracks;
  out->d_cluster_ids = ctx->buf.cluster_ids;
  out->d_cluster_shared = ctx->buf.cluster_shared;
  out->n_ignored = c.n_ignored;
  out->n_dropped = c.n_dropped;
  out->n_seeds = c.n_seeds;
  out->n_tracklets = c.n_tracklets;
  out->n_bins = c.n_bins;
  for (int a = 0; a < 3; ++a) {
    out->n_follow_steps += c.follow_work[a][0];
    out->n_follow_updates += c.follow_work[a][1];
    out->n_follow_candidates += c.follow_work[a][2];
    for (int b = 0; b < 3; ++b) out->follow_work[a][b] = c.follow_work[a][b];
  }
  out->grid_by_rows = c.grid_rows;
  out->n_rows_generic = c.n_rows_generic;
  return rc;
}

int tpc_get_intermediates(tpc_ctx* ctx, tpc_debug_view* out) {
  if (!out) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!(ctx->flags & TPC_KEEP_INTERMEDIATES)) return TPC_E_STATE;
  const TpcCounters& c = *ctx->h_cnt;
  const TpcBuffers& B = ctx->buf;
  std::memset(out, 0, sizeof(*out));
  out->n_clusters = B.n;
  out->n_sorted = c.n_sorted;
  out->n_rows_total = B.n_sr;
  out->n_bins = c.n_bins;
  out->n_seeds = c.n_seeds;
  out->tracklet_stride = (uint64_t)ctx->geom.n_rows;
  out->d_row_desc = B.row_desc;
  out->d_bin_start = B.bin_start;
  out->d_yz_sorted = (const float*)B.yz;
  out->d_orig_id = B.orig_id;
  out->d_link_up = B.link_up;
  out->d_link_dn = B.link_dn;
  out->d_link_up2 = B.link_up2;
  out->d_link_dn2 = B.link_dn2;
  out->d_seeds = B.seeds;
  out->d_tracklets = B.tracklets;
  out->d_row_hit = B.row_hit;
  return device_status(ctx);
}

int tpc_get_stage_ms(tpc_ctx* ctx, float* out_ms) {
  if (!out_ms) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!(ctx->flags & TPC_STAGE_TIMERS)) return TPC_E_STATE;
  for (int i = 0; i < TPC_N_STAGES - 1; ++i) {
    cudaError_t e = cudaEventElapsedTime(&out_ms[i], ctx->events.ev[i], ctx->events.ev[i + 1]);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaEventElapsedTime");
  }
  cudaError_t e = cudaEventElapsedTime(&out_ms[TPC_N_STAGES - 1], ctx->events.ev[0], ctx->events.ev[TPC_N_STAGES - 1]);
  if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaEventElapsedTime");
  return TPC_OK;
}

int tpc_get_kernel_ms(tpc_ctx* ctx, int max_kernels, const char** names_out, float* ms_out) {
  if (!names_out || !ms_out || max_kernels < 0) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!(ctx->flags & TPC_STAGE_TIMERS)) return TPC_E_STATE;
  const int n = ctx->events.n_kernels < max_kernels ? ctx->events.n_kernels : max_kernels;
  for (int i = 0; i < n; ++i) {
    names_out[i] = ctx->events.kname[i];
    cudaError_t e = cudaEventElapsedTime(&ms_out[i], ctx->events.kev[i], ctx->events.kev[i + 1]);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaEventElapsedTime");
  }
  return n;
}

int tpc_sector_track_host(tpc_ctx* ctx, const tpc_cluster* h_clusters, uint64_t n_clusters, void* d_staging,
                          void* d_workspace, size_t workspace_bytes, void* cuda_stream, uint32_t flags,
                          tpc_track* h_tracks, uint64_t cap_tracks, uint32_t* h_cluster_ids,
                          uint8_t* h_cluster_shared, uint64_t cap_ids, tpc_track_view* out) {
  if (!ctx || !out || (!h_clusters && n_clusters) || (!d_staging && n_clusters)) return TPC_E_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e;
  if (n_clusters) {
    e = cudaMemcpyAsync(d_staging, h_clusters, n_clusters * sizeof(tpc_cluster), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(clusters)");
  }
  int rc = tpc_sector_track(ctx, (const tpc_cluster*)d_staging, n_clusters, d_workspace, workspace_bytes,
                            cuda_stream, flags);
  if (rc != TPC_OK) return rc;
  rc = tpc_get_tracks(ctx, out);  // syncs; counts are needed to size the copies back
  if (rc != TPC_OK) return rc;
  if (out->n_tracks > cap_tracks || out->n_cluster_ids > cap_ids) return TPC_E_OVERFLOW;
  if (h_tracks && out->n_tracks) {
    e = cudaMemcpyAsync(h_tracks, out->d_tracks, out->n_tracks * sizeof(tpc_track), cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(tracks)");
  }
  if (h_cluster_ids && out->n_cluster_ids) {
    e = cudaMemcpyAsync(h_cluster_ids, out->d_cluster_ids, out->n_cluster_ids * 4, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(cluster ids)");
  }
  if (h_cluster_shared && out->n_cluster_ids) {
    e = cudaMemcpyAsync(h_cluster_shared, out->d_cluster_shared, out->n_cluster_ids, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(shared flags)");
  }
  e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaStreamSynchronize");
  return TPC_OK;
}

// cluster_ofs of a chunk's tracks refers to the chunk's own id list: shift it to the frame's
__global__ void k_shift_tracks(tpc_track* tracks, uint32_t n, uint32_t ids_base) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) tracks[i].cluster_ofs += ids_base;
}

int tpc_sector_track_host_chunks(tpc_ctx* ctx, const tpc_cluster* h_clusters, uint64_t n_clusters,
                                 const uint64_t* chunk_ofs, int n_chunks, void* d_staging, void* d_workspace,
                                 size_t workspace_bytes, void* cuda_stream, uint32_t flags, tpc_track* h_tracks,
                                 uint64_t cap_tracks, uint32_t* h_cluster_ids, uint8_t* h_cluster_shared,
                                 uint64_t cap_ids, tpc_track_view* out) {
  if (!ctx || !out || !chunk_ofs || n_chunks < 1 || (!h_clusters && n_clusters) || (!d_staging && n_clusters) ||
      !d_workspace || n_clusters >= (1ull << 30))
    return TPC_E_ARG;
  if (chunk_ofs[0] != 0 || chunk_ofs[n_chunks] != n_clusters) return TPC_E_ARG;
  uint64_t n_max = 0;
  for (int c = 0; c < n_chunks; ++c) {
    if (chunk_ofs[c + 1] < chunk_ofs[c]) return TPC_E_ARG;
    const uint64_t nc = chunk_ofs[c + 1] - chunk_ofs[c];
    n_max = nc > n_max ? nc : n_max;
  }
  // two workspaces, used alternately: the results of chunk c are read back while chunk c+1 runs
  const size_t ws_one = align_up(carve(ctx, n_max, nullptr, nullptr), 256);
  if (((uintptr_t)d_workspace & 255u) || workspace_bytes < 2 * ws_one) return TPC_E_WORKSPACE;
  char* ws[2] = {(char*)d_workspace, (char*)d_workspace + ws_one};
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e;
  std::memset(out, 0, sizeof(*out));
  if ((e = cudaMemsetAsync(ctx->d_sector_seen, 0, sizeof(uint32_t) * (size_t)ctx->geom.n_sectors, st)) != cudaSuccess)
    return set_cuda_err(ctx, e, "cudaMemsetAsync(sector_seen)");
  // the copy streams start after whatever the caller has enqueued on `st`
  if ((e = cudaEventRecord(ctx->ev_done[0], st)) != cudaSuccess) return set_cuda_err(ctx, e, "cudaEventRecord");
  if ((e = cudaStreamWaitEvent(ctx->s_in, ctx->ev_done[0], 0)) != cudaSuccess ||
      (e = cudaStreamWaitEvent(ctx->s_out, ctx->ev_done[0], 0)) != cudaSuccess)
    return set_cuda_err(ctx, e, "cudaStreamWaitEvent");
  auto copy_in = [&](int c) -> cudaError_t {
    const uint64_t o = chunk_ofs[c], nc = chunk_ofs[c + 1] - o;
    if (nc) {
      cudaError_t ee = cudaMemcpyAsync((tpc_cluster*)d_staging + o, h_clusters + o, nc * sizeof(tpc_cluster),
                                       cudaMemcpyHostToDevice, ctx->s_in);
      if (ee != cudaSuccess) return ee;
    }
    return cudaEventRecord(ctx->ev_in[c & 1], ctx->s_in);
  };
  if ((e = copy_in(0)) != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(clusters)");
  uint64_t n_tracks = 0, n_ids = 0;
  int launches = 0;
  for (int c = 0; c < n_chunks; ++c) {
    const uint64_t o = chunk_ofs[c], nc = chunk_ofs[c + 1] - o;
    e = cudaStreamWaitEvent(st, ctx->ev_in[c & 1], 0);                // chunk c is on the device
    if (e == cudaSuccess && c >= 2) e = cudaStreamWaitEvent(st, ctx->ev_out[c & 1], 0);   // workspace c&1 has been read back
    if (e != cudaSuccess) { cudaDeviceSynchronize(); ctx->ran = false; return set_cuda_err(ctx, e, "cudaStreamWaitEvent"); }
    int rc = enqueue_track(ctx, (const tpc_cluster*)d_staging + o, nc, ws[c & 1], ws_one, cuda_stream, flags,
                           (uint32_t)o, (uint32_t)c + 1u);
    if (rc != TPC_OK) { cudaDeviceSynchronize(); return rc; }
    launches += ctx->launches;
    if (c + 1 < n_chunks) {   // next chunk's copy-in runs behind this chunk's kernels
      if ((e = copy_in(c + 1)) != cudaSuccess) { cudaDeviceSynchronize(); return set_cuda_err(ctx, e, "cudaMemcpyAsync(clusters)"); }
    }
    tpc_track_view v;
    rc = tpc_get_tracks(ctx, &v);                                     // syncs `st`: counts of chunk c
    if (rc != TPC_OK) { cudaDeviceSynchronize(); return rc; }
    if (n_tracks + v.n_tracks > cap_tracks || n_ids + v.n_cluster_ids > cap_ids) { cudaDeviceSynchronize(); return TPC_E_OVERFLOW; }
    // every CUDA call of the hand-over is checked: a failure drains the streams and is reported,
    // never a partly filled result with TPC_OK
    e = cudaSuccess;
    if (v.n_tracks) {
      k_shift_tracks<<<(unsigned)((v.n_tracks + 255) / 256), 256, 0, st>>>((tpc_track*)v.d_tracks, (uint32_t)v.n_tracks, (uint32_t)n_ids);
      e = cudaPeekAtLastError();
    }
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_done[c & 1], st);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(ctx->s_out, ctx->ev_done[c & 1], 0);
    if (e == cudaSuccess && h_tracks && v.n_tracks)
      e = cudaMemcpyAsync(h_tracks + n_tracks, v.d_tracks, v.n_tracks * sizeof(tpc_track), cudaMemcpyDeviceToHost, ctx->s_out);
    if (e == cudaSuccess && h_cluster_ids && v.n_cluster_ids)
      e = cudaMemcpyAsync(h_cluster_ids + n_ids, v.d_cluster_ids, v.n_cluster_ids * 4, cudaMemcpyDeviceToHost, ctx->s_out);
    if (e == cudaSuccess && h_cluster_shared && v.n_cluster_ids)
      e = cudaMemcpyAsync(h_cluster_shared + n_ids, v.d_cluster_shared, v.n_cluster_ids, cudaMemcpyDeviceToHost, ctx->s_out);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->ev_out[c & 1], ctx->s_out);
    if (e != cudaSuccess) { cudaDeviceSynchronize(); ctx->ran = false; return set_cuda_err(ctx, e, "chunk hand-over"); }
    n_tracks += v.n_tracks; n_ids += v.n_cluster_ids;
    out->n_ignored += v.n_ignored; out->n_dropped += v.n_dropped; out->n_seeds += v.n_seeds;
    out->n_tracklets += v.n_tracklets; out->n_bins += v.n_bins;
    out->n_follow_steps += v.n_follow_steps; out->n_follow_updates += v.n_follow_updates;
    out->n_follow_candidates += v.n_follow_candidates;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) out->follow_work[a][b] += v.follow_work[a][b];
    out->grid_by_rows = (c == 0) ? v.grid_by_rows : (out->grid_by_rows & v.grid_by_rows);
    out->n_rows_generic += v.n_rows_generic;
  }
  if ((e = cudaStreamSynchronize(ctx->s_out)) != cudaSuccess) return set_cuda_err(ctx, e, "cudaStreamSynchronize(copy-out)");
  if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return set_cuda_err(ctx, e, "cudaStreamSynchronize");
  out->n_tracks = n_tracks;
  out->n_cluster_ids = n_ids;
  ctx->launches = launches;
  // the context's buffers describe the LAST chunk only: tpc_get_tracks / tpc_get_intermediates /
  // tpc_refit_tracks after a chunked call return TPC_E_STATE instead of a partial answer
  ctx->ran = false;
  return TPC_OK;
}

// ---------------------------------------------------------------- second seeding iteration (R7)
// used[i] = 1 for every cluster attached to an iteration-1 track
__global__ void k_mark_used(const uint32_t* __restrict__ ids, uint32_t n_ids, uint8_t* __restrict__ used) {
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n_ids; j += gridDim.x * blockDim.x) used[ids[j]] = 1;
}
// stable compaction of the unused records: per-block counts, one-CTA scan, write
__global__ void __launch_bounds__(1024) k_left_count(const uint8_t* __restrict__ used, uint32_t n, uint32_t* partials) {
  const uint32_t i = blockIdx.x * 1024u + threadIdx.x;
  const int c = __syncthreads_count(i < n && !used[i]);
  if (threadIdx.x == 0) partials[blockIdx.x] = (uint32_t)c;
}
__global__ void __launch_bounds__(1024) k_left_scan(uint32_t* partials, uint32_t n_blocks, uint32_t* total) {
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t s_chunk;
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t carry = 0;
  for (uint32_t b0 = 0; b0 < n_blocks; b0 += 1024) {
    const uint32_t b = b0 + threadIdx.x;
    const uint32_t v = b < n_blocks ? partials[b] : 0u;
    uint32_t inc = v;
    for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if ((int)lane >= d) inc += t; }
    if (lane == 31) wsum[w] = inc;
    __syncthreads();
    if (w == 0) {
      const uint32_t x = wsum[lane];
      uint32_t xi = x;
      for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, xi, d); if ((int)lane >= d) xi += t; }
      wsum[lane] = xi - x;
      if (lane == 31) s_chunk = xi;
    }
    __syncthreads();
    if (b < n_blocks) partials[b] = carry + wsum[w] + inc - v;
    carry += s_chunk;
    __syncthreads();
  }
  if (threadIdx.x == 0) *total = carry;
}
__global__ void __launch_bounds__(1024) k_left_write(const uint8_t* __restrict__ used, const tpc_cluster* __restrict__ in,
                                                     uint32_t n, const uint32_t* __restrict__ partials,
                                                     uint32_t* __restrict__ map, tpc_cluster* __restrict__ left) {
  __shared__ uint32_t wsum[32];
  const uint32_t i = blockIdx.x * 1024u + threadIdx.x;
  const bool keep = i < n && !used[i];
  const uint32_t m = __ballot_sync(0xffffffffu, keep);
  const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) wsum[w] = (uint32_t)__popc(m);
  __syncthreads();
  if (w == 0) {
    const uint32_t v = wsum[lane];
    uint32_t inc = v;
    for (int d = 1; d < 32; d <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d); if ((int)lane >= d) inc += t; }
    wsum[lane] = inc - v;
  }
  __syncthreads();
  if (keep) {
    const uint32_t pos = partials[blockIdx.x] + wsum[w] + (uint32_t)__popc(m & ((1u << lane) - 1u));
    map[pos] = i;
    left[pos] = in[i];
  }
}
// iteration-2 results behind the iteration-1 results, in original cluster indices
__global__ void k_append_iter2(tpc_track* __restrict__ t1, uint32_t n_t1, const tpc_track* __restrict__ t2, uint32_t n_t2,
                               uint32_t* __restrict__ ids1, uint8_t* __restrict__ sh1, uint32_t n_i1,
                               const uint32_t* __restrict__ ids2, const uint8_t* __restrict__ sh2, uint32_t n_i2,
                               const uint32_t* __restrict__ map) {
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n_t2; j += stride) {
    tpc_track t = t2[j];
    t.seed_id = map[t.seed_id];
    t.cluster_ofs += n_i1;
    t.flags |= TPC_TRACK_ITER2;
    t1[n_t1 + j] = t;
  }
  for (uint32_t j = blockIdx.x * blockDim.x + threadIdx.x; j < n_i2; j += stride) {
    ids1[n_i1 + j] = map[ids2[j]];
    sh1[n_i1 + j] = sh2[j];
  }
}

namespace {
struct Iter2Layout { size_t ws_one, used, map, left, partials, total; uint32_t n_blocks; };
Iter2Layout iter2_layout(const tpc_ctx* c, uint64_t n) {
  Iter2Layout L;
  L.ws_one = align_up(carve(c, n, nullptr, nullptr), 256);
  L.n_blocks = (uint32_t)((n + 1023) / 1024);
  size_t off = 2 * L.ws_one;
  L.used = off; off = align_up(off + n, 256);
  L.map = off; off = align_up(off + 4 * n, 256);
  L.left = off; off = align_up(off + 16 * n, 256);
  L.partials = off; off = align_up(off + 4 * ((size_t)L.n_blocks + 2), 256);
  L.total = off;
  return L;
}
}  // namespace

size_t tpc_workspace_bytes_two_iterations(const tpc_ctx* ctx, uint64_t n_clusters) {
  if (!ctx || n_clusters >= (1ull << 30)) return 0;
  return iter2_layout(ctx, n_clusters).total;
}

int tpc_sector_track_two_iterations(tpc_ctx* ctx, const tpc_cluster* d_clusters, uint64_t n_clusters, void* d_workspace,
                                    size_t workspace_bytes, void* cuda_stream, uint32_t flags) {
  if (!ctx || !d_workspace || (!d_clusters && n_clusters) || n_clusters >= (1ull << 30)) return TPC_E_ARG;
  if (((uintptr_t)d_workspace & 255u)) return TPC_E_ARG;
  const Iter2Layout L = iter2_layout(ctx, n_clusters);
  if (workspace_bytes < L.total) return TPC_E_WORKSPACE;
  char* base = (char*)d_workspace;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const uint32_t n = (uint32_t)n_clusters;
  flags &= ~(uint32_t)TPC_KEEP_INTERMEDIATES;
  // ---- iteration 1 (R1..R6)
  int rc = enqueue_track(ctx, d_clusters, n_clusters, base, L.ws_one, cuda_stream, flags, 0u, 0u);
  if (rc != TPC_OK) return rc;
  tpc_track_view v1;
  rc = tpc_get_tracks(ctx, &v1);
  if (rc != TPC_OK) return rc;
  const TpcBuffers B1 = ctx->buf;
  const TpcCounters c1 = *ctx->h_cnt;
  const int launches1 = ctx->launches;
  // ---- R7.1 / R7.2: leftover frame
  uint8_t* used = (uint8_t*)(base + L.used);
  uint32_t* map = (uint32_t*)(base + L.map);
  tpc_cluster* left = (tpc_cluster*)(base + L.left);
  uint32_t* partials = (uint32_t*)(base + L.partials);
  uint32_t* d_total = partials + L.n_blocks;
  cudaError_t e;
  if ((e = cudaMemsetAsync(used, 0, n_clusters, st)) != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemsetAsync(used)");
  uint32_t n_left = 0;
  if (n) {
    if (c1.n_ids) k_mark_used<<<ctx->n_sm * 8, 256, 0, st>>>(B1.cluster_ids, c1.n_ids, used);
    k_left_count<<<L.n_blocks, 1024, 0, st>>>(used, n, partials);
    k_left_scan<<<1, 1024, 0, st>>>(partials, L.n_blocks, d_total);
    k_left_write<<<L.n_blocks, 1024, 0, st>>>(used, d_clusters, n, partials, map, left);
    if ((e = cudaMemcpyAsync(&n_left, d_total, 4, cudaMemcpyDeviceToHost, st)) != cudaSuccess ||
        (e = cudaStreamSynchronize(st)) != cudaSuccess)
      return set_cuda_err(ctx, e, "leftover frame");
  }
  // ---- R7.3: the path on the leftover frame
  rc = enqueue_track(ctx, left, n_left, base + L.ws_one, L.ws_one, cuda_stream, flags, 0u, 0u);
  if (rc != TPC_OK) return rc;
  tpc_track_view v2;
  rc = tpc_get_tracks(ctx, &v2);
  if (rc != TPC_OK) return rc;
  const TpcCounters c2 = *ctx->h_cnt;
  // ---- R7.4: append in original indices
  if ((uint64_t)c1.n_tracks + c2.n_tracks > B1.max_tracks || (uint64_t)c1.n_ids + c2.n_ids > B1.max_ids) return TPC_E_OVERFLOW;
  if (c2.n_tracks || c2.n_ids) {
    k_append_iter2<<<ctx->n_sm * 8, 256, 0, st>>>(B1.tracks, c1.n_tracks, ctx->buf.tracks, c2.n_tracks, B1.cluster_ids,
                                                  B1.cluster_shared, c1.n_ids, ctx->buf.cluster_ids,
                                                  ctx->buf.cluster_shared, c2.n_ids, map);
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return set_cuda_err(ctx, e, "append");
  }
  // the context now describes the combined result (tpc_get_tracks reads it)
  TpcCounters c = c1;
  c.n_tracks += c2.n_tracks; c.n_ids += c2.n_ids; c.n_seeds += c2.n_seeds; c.n_tracklets += c2.n_tracklets;
  c.n_bins += c2.n_bins; c.error |= c2.error;
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) c.follow_work[a][b] += c2.follow_work[a][b];
  *ctx->h_cnt = c;
  ctx->buf = B1;
  ctx->flags = flags;
  ctx->launches = launches1 + ctx->launches + 5;
  ctx->ran = true;
  ctx->synced = true;
  ctx->refit_done = false;
  ctx->merged = false; ctx->fitted = false; ctx->rb_prepared = false; ctx->rebuilt = false;
  return TPC_OK;
}

int tpc_set_tracks(tpc_ctx* ctx, const tpc_track* h_tracks, uint64_t n_tracks, const uint32_t* h_ids,
                   const uint8_t* h_shared, uint64_t n_ids, void* cuda_stream) {
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  rc = device_status(ctx);
  if (rc != TPC_OK) return rc;
  if ((n_tracks && !h_tracks) || (n_ids && (!h_ids || !h_shared))) return TPC_E_ARG;
  const TpcBuffers& B = ctx->buf;
  if (B.id_base != 0u) return TPC_E_STATE;   // (the context holds one chunk of a chunked host call)
  if (n_tracks > B.max_tracks || n_ids > B.max_ids) return TPC_E_OVERFLOW;
  for (uint64_t i = 0; i < n_tracks; ++i) {
    const tpc_track& t = h_tracks[i];
    if ((int)t.sector >= ctx->geom.n_sectors || t.row_first > t.row_last || (int)t.row_last >= ctx->geom.n_rows ||
        (uint64_t)t.cluster_ofs + t.n_clusters > n_ids)
      return TPC_E_ARG;
  }
  for (uint64_t i = 0; i < n_ids; ++i)
    if (h_ids[i] >= B.n) return TPC_E_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaSuccess;
  if (n_tracks) e = cudaMemcpyAsync(B.tracks, h_tracks, sizeof(tpc_track) * n_tracks, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess && n_ids) e = cudaMemcpyAsync(B.cluster_ids, h_ids, 4 * n_ids, cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess && n_ids) e = cudaMemcpyAsync(B.cluster_shared, h_shared, n_ids, cudaMemcpyHostToDevice, st);
  ctx->h_cnt->n_tracks = (uint32_t)n_tracks;
  ctx->h_cnt->n_ids = (uint32_t)n_ids;
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(&ctx->d_cnt->n_tracks, &ctx->h_cnt->n_tracks, 2 * sizeof(uint32_t), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(tracks)");
  ctx->stream = st;
  ctx->refit_done = false;
  ctx->merged = false; ctx->fitted = false; ctx->rb_prepared = false; ctx->rebuilt = false;
  return TPC_OK;
}

int tpc_refit_tracks(tpc_ctx* ctx, void* cuda_stream) {
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  rc = device_status(ctx);
  if (rc == TPC_E_OVERFLOW) return rc;
  const uint32_t n_tracks = ctx->h_cnt->n_tracks;
  // The compact copy of the tracks' clusters (tpc_internal.h) goes where the tracklets' row -> hit table
  // was: dead after the selection, unless the caller asked to keep the intermediates.
  ctx->buf.trk_yz = nullptr; ctx->buf.trk_sr = nullptr;
  {
    const size_t have = 4 * (size_t)ctx->geom.n_rows * ctx->buf.max_seeds;
    const size_t yz_bytes = align_up(8 * (size_t)ctx->buf.max_ids, 256), sr_bytes = 2 * (size_t)ctx->buf.max_ids;
    if (!(ctx->flags & TPC_KEEP_INTERMEDIATES) && ctx->buf.row_hit && yz_bytes + sr_bytes <= have) {
      ctx->buf.trk_yz = reinterpret_cast<float2*>(ctx->buf.row_hit);
      ctx->buf.trk_sr = reinterpret_cast<uint16_t*>(reinterpret_cast<char*>(ctx->buf.row_hit) + yz_bytes);
    }
  }
  (void)cudaGetLastError();
  const int l = (ctx->flags & TPC_DETERMINISTIC)
                    ? tpc_det::run_refit(ctx->buf, &ctx->hconst, n_tracks, (cudaStream_t)cuda_stream, ctx->n_sm)
                    : tpc_fast::run_refit(ctx->buf, &ctx->hconst, n_tracks, (cudaStream_t)cuda_stream, ctx->n_sm);
  if (l < 0) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch (refit)");
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->synced = false;
  ctx->refit_done = true;
  ctx->merged = false; ctx->fitted = false; ctx->rb_prepared = false; ctx->rebuilt = false;
  return TPC_OK;
}

int tpc_get_refit(tpc_ctx* ctx, const tpc_track_fit** d_fit) {
  if (!d_fit) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  *d_fit = ctx->buf.track_fit;
  return TPC_OK;
}

// ---------------------------------------------------------------- track merging (R9)
namespace {
size_t carve_merge(const tpc_ctx* c, uint64_t n_tracks, uint64_t n_ids, char* base, TpcMergeBuffers* M) {
  const uint32_t n_cells = (uint32_t)c->geom.n_sectors * (uint32_t)c->geom.n_rows * 1024u;   // TPC_MG_ZB slabs
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* p = base ? base + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  };
  TpcMergeBuffers m;
  std::memset(&m, 0, sizeof(m));
  m.n_tracks = (uint32_t)n_tracks; m.n_ids = (uint32_t)n_ids; m.n_rows = (uint32_t)c->geom.n_rows; m.n_cells = n_cells;
  const size_t nt = n_tracks + 1;
  const size_t n_part = (std::max<size_t>(n_cells + 1, nt) + 1023) / 1024 + 2;
  m.cell_start = (uint32_t*)take(4 * ((size_t)n_cells + 1));
  m.cell_cursor = (uint32_t*)take(4 * (size_t)n_cells);
  m.partials = (uint32_t*)take(4 * n_part);
  m.ends = (float*)take(64 * nt);
  m.next = (int32_t*)take(4 * nt); m.prev = (int32_t*)take(4 * nt); m.link_chi2 = (float*)take(4 * nt);
  m.best_out = (int32_t*)take(4 * nt); m.best_out_chi = (uint32_t*)take(4 * nt); m.best_in_chi = (uint32_t*)take(4 * nt);
  m.best_in_key = (unsigned long long*)take(8 * nt);
  m.cand = (uint2*)take(8 * (size_t)TPC_MG_CAND * nt); m.cand_cnt = (uint32_t*)take(4 * nt);
  m.head_ofs = (uint32_t*)take(4 * nt); m.seg_ofs = (uint32_t*)take(4 * nt); m.clu_ofs = (uint32_t*)take(4 * nt);
  m.seg_dst = (uint32_t*)take(4 * nt);
  m.merged = (tpc_merged_track*)take(sizeof(tpc_merged_track) * nt);
  m.seg_index = (uint32_t*)take(4 * nt);
  m.ids = (uint32_t*)take(4 * ((size_t)n_ids + 1));
  m.shared = (uint8_t*)take((size_t)n_ids + 1);
  m.yz = (float2*)take(8 * ((size_t)n_ids + 1));
  m.sr = (uint16_t*)take(2 * ((size_t)n_ids + 1));
  m.counters = (uint32_t*)take(16);
  m.path_ofs = (uint32_t*)take(4 * (nt + 1));
  if (M) *M = m;
  return off;
}
}  // namespace

void tpc_merge_default_params(tpc_merge_params* m) {
  std::memset(m, 0, sizeof(*m));
  m->gap_in_sector = 30; m->gap_adjacent_back = 3; m->gap_adjacent = 10; m->gap_ce = 6;
  m->chi2_max = 20.0f;
  m->sys[0] = 0.3f; m->sys[1] = 0.3f; m->sys[2] = 0.02f; m->sys[3] = 0.02f; m->sys[4] = 0.2f;
  m->ce_sys_z = 3.0f;
  m->pre_dy = 8.0f; m->pre_dz = 8.0f; m->pre_coarse_dz = 40.0f;
  m->stages = 7;
}

size_t tpc_merge_workspace_bytes(const tpc_ctx* ctx, uint64_t n_tracks, uint64_t n_cluster_ids) {
  if (!ctx || n_tracks >= (1ull << 31) || n_cluster_ids >= (1ull << 32)) return 0;
  return carve_merge(ctx, n_tracks, n_cluster_ids, nullptr, nullptr);
}

int tpc_merge_tracks(tpc_ctx* ctx, const tpc_merge_params* params, void* d_ws, size_t ws_bytes, void* cuda_stream) {
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->refit_done) return TPC_E_STATE;
  rc = device_status(ctx);
  if (rc == TPC_E_OVERFLOW) return rc;
  if (!d_ws || ((uintptr_t)d_ws & 255u)) return TPC_E_ARG;
  tpc_merge_params P;
  if (params) P = *params; else tpc_merge_default_params(&P);
  if (!(P.pre_dz > 0.f) || !(P.pre_dy > 0.f) || !(P.chi2_max >= 0.f) || P.gap_in_sector < 0 || P.gap_adjacent < 0 ||
      P.gap_adjacent_back < 0 || P.gap_ce < 0 || P.gap_adjacent_back > ctx->params.min_hits_track - 2)
    return TPC_E_ARG;   // (the last: links must raise the first row, so chains cannot close)
  const uint32_t n_tracks = ctx->h_cnt->n_tracks, n_ids = ctx->h_cnt->n_ids;
  TpcMergeBuffers M;
  const size_t need = carve_merge(ctx, n_tracks, n_ids, (char*)d_ws, &M);
  if (ws_bytes < need) return TPC_E_WORKSPACE;
  M.P = P;
  if (!ctx->buf.trk_yz) { M.yz = nullptr; M.sr = nullptr; }   // (no compact copy of the tracks' clusters: the fit gathers)
  M.inv_w = 1.0f / P.pre_dz;
  const double a = 2.0 * (double)ctx->geom.sector_half_angle_deg * (3.14159265358979323846 / 180.0);
  M.ca = (float)std::cos(a);
  M.sa = (float)std::sin(a);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  (void)cudaGetLastError();
  const int l = (ctx->flags & TPC_DETERMINISTIC) ? tpc_det::run_merge(ctx->buf, &ctx->hconst, M, st, ctx->n_sm)
                                                 : tpc_fast::run_merge(ctx->buf, &ctx->hconst, M, st, ctx->n_sm);
  if (l < 0) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch (merge)");
  cudaError_t e = cudaMemcpyAsync(ctx->h_mcnt, M.counters, 16, cudaMemcpyDeviceToHost, st);
  if (e != cudaSuccess) return set_cuda_err(ctx, e, "cudaMemcpyAsync(merge counters)");
  ctx->mbuf = M;
  ctx->stream = st;
  ctx->synced = false;
  ctx->merged = true;
  ctx->fitted = false;
  ctx->rb_prepared = false; ctx->rebuilt = false;
  ctx->launches = l;
  return TPC_OK;
}

int tpc_get_merged(tpc_ctx* ctx, tpc_merged_view* out) {
  if (!out) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->merged) return TPC_E_STATE;
  const TpcMergeBuffers& M = ctx->mbuf;
  std::memset(out, 0, sizeof(*out));
  out->n_tracks = M.n_tracks;
  out->n_merged = M.n_tracks ? ctx->h_mcnt[0] : 0;
  out->n_links = ctx->h_mcnt[1];
  out->n_cluster_ids = M.n_tracks ? ctx->h_mcnt[2] : 0;
  out->d_merged = M.merged; out->d_seg_index = M.seg_index;
  out->d_cluster_ids = M.ids; out->d_cluster_shared = M.shared;
  out->d_next = M.next; out->d_prev = M.prev; out->d_link_chi2 = M.link_chi2;
  return TPC_OK;
}

// ---------------------------------------------------------------- three-iteration track fit (R10)
namespace {
size_t carve_fit(uint64_t n_merged, uint64_t n_ids, char* base, TpcFitBuffers* T) {
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* p = base ? base + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  };
  TpcFitBuffers t;
  std::memset(&t, 0, sizeof(t));
  t.stored = (uint4*)take(16 * (n_ids + 1));
  t.chi2_cluster = (float*)take(4 * (n_ids + 1));
  t.rejected = (uint8_t*)take(n_ids + 1);
  t.fit = (tpc_track_fit3*)take(sizeof(tpc_track_fit3) * (n_merged + 1));
  t.work = (uint32_t*)take(16);
  if (T) *T = t;
  return off;
}
}  // namespace

void tpc_fit_default_params(tpc_fit_params* f) {
  f->fit_chi2_max = 16.0f;
  f->fit_min_clusters = 10;
  f->ce_var = 10000.0f;
}

size_t tpc_fit_workspace_bytes(const tpc_ctx* ctx, uint64_t n_merged, uint64_t n_cluster_ids) {
  if (!ctx || n_merged >= (1ull << 31) || n_cluster_ids >= (1ull << 32)) return 0;
  return carve_fit(n_merged, n_cluster_ids, nullptr, nullptr);
}

int tpc_fit_tracks(tpc_ctx* ctx, const tpc_fit_params* params, void* d_ws, size_t ws_bytes, void* cuda_stream) {
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->merged) return TPC_E_STATE;
  if (!d_ws || ((uintptr_t)d_ws & 255u)) return TPC_E_ARG;
  tpc_fit_params P;
  if (params) P = *params; else tpc_fit_default_params(&P);
  if (!(P.fit_chi2_max >= 0.f) || P.fit_min_clusters < 2 || !(P.ce_var > 0.f)) return TPC_E_ARG;
  const uint32_t n_merged = ctx->mbuf.n_tracks ? ctx->h_mcnt[0] : 0u, n_ids = ctx->mbuf.n_tracks ? ctx->h_mcnt[2] : 0u;
  TpcFitBuffers T;
  const size_t need = carve_fit(n_merged, n_ids, (char*)d_ws, &T);
  if (ws_bytes < need) return TPC_E_WORKSPACE;
  T.P = P;
  T.ca = ctx->mbuf.ca; T.sa = ctx->mbuf.sa;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  (void)cudaGetLastError();
  const int l = (ctx->flags & TPC_DETERMINISTIC)
                    ? tpc_det::run_fit3(ctx->buf, &ctx->hconst, ctx->mbuf, T, n_merged, st, ctx->n_sm)
                    : tpc_fast::run_fit3(ctx->buf, &ctx->hconst, ctx->mbuf, T, n_merged, st, ctx->n_sm);
  if (l < 0) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch (fit)");
  ctx->fbuf = T;
  ctx->fit_n_merged = n_merged; ctx->fit_n_ids = n_ids;
  ctx->stream = st;
  ctx->synced = false;
  ctx->fitted = true;
  ctx->launches = l;
  return TPC_OK;
}

int tpc_get_fit(tpc_ctx* ctx, tpc_fit_view* out) {
  if (!out) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->fitted) return TPC_E_STATE;
  std::memset(out, 0, sizeof(*out));
  out->n_merged = ctx->fit_n_merged;
  out->n_cluster_ids = ctx->fit_n_ids;
  out->d_fit = ctx->fbuf.fit;
  out->d_chi2_cluster = ctx->fbuf.chi2_cluster;
  out->d_rejected = ctx->fbuf.rejected;
  return TPC_OK;
}

int tpc_fit_tracks_noalloc(tpc_ctx* ctx, const tpc_fit_params* params, const tpc_cluster* d_clusters, uint64_t n_clusters,
                           const tpc_track_fit* d_refit, uint64_t n_tracks, const tpc_merged_track* d_merged,
                           uint64_t n_merged, const uint32_t* d_seg_index, const uint32_t* d_cluster_ids,
                           uint64_t n_cluster_ids, tpc_track_fit3* d_fit_out, float* d_chi2_out, uint8_t* d_rejected_out,
                           uint32_t flags, void* cuda_stream) {
  if (!ctx) return TPC_E_ARG;
  if (n_cluster_ids > TPC_FIT_NOALLOC_MAX_IDS) {
    std::snprintf(ctx->cuda_err, sizeof(ctx->cuda_err),
                  "tpc_fit_tracks_noalloc: %llu cluster ids exceed TPC_FIT_NOALLOC_MAX_IDS = %u (the library's static scratch); "
                  "use tpc_fit_tracks with a workspace", (unsigned long long)n_cluster_ids, (unsigned)TPC_FIT_NOALLOC_MAX_IDS);
    return TPC_E_LIMIT;
  }
  if (n_merged > n_cluster_ids || n_merged > n_tracks || n_clusters >= (1ull << 30) || n_tracks >= (1ull << 30)) return TPC_E_ARG;
  if (n_merged && (!d_clusters || !d_refit || !d_merged || !d_seg_index || !d_cluster_ids || !d_fit_out || !d_chi2_out ||
                   !d_rejected_out))
    return TPC_E_ARG;
  if (((uintptr_t)d_clusters & 15u) || ((uintptr_t)d_refit & 3u) || ((uintptr_t)d_merged & 3u) || ((uintptr_t)d_seg_index & 3u) ||
      ((uintptr_t)d_cluster_ids & 3u) || ((uintptr_t)d_fit_out & 3u) || ((uintptr_t)d_chi2_out & 3u))
    return TPC_E_ARG;
  if (flags & ~TPC_DETERMINISTIC) return TPC_E_ARG;
  tpc_fit_params P;
  if (params) P = *params; else tpc_fit_default_params(&P);
  if (!(P.fit_chi2_max >= 0.f) || P.fit_min_clusters < 2 || !(P.ce_var > 0.f)) return TPC_E_ARG;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) return TPC_E_STATE;   // (the address belongs to ctx's device)
  if (!ctx->noalloc_scratch) {
    std::snprintf(ctx->cuda_err, sizeof(ctx->cuda_err), "tpc_fit_tracks_noalloc: static scratch not resolved at set-up: %s",
                  ctx->noalloc_err);
    return TPC_E_CUDA;
  }
  if (n_merged == 0) return TPC_OK;
  char* scratch = (char*)ctx->noalloc_scratch;
  TpcBuffers B;
  std::memset(&B, 0, sizeof(B));
  B.K = ctx->d_const;
  B.clusters = d_clusters;
  B.n = (uint32_t)n_clusters;
  B.id_base = 0u;
  B.track_fit = const_cast<tpc_track_fit*>(d_refit);          // (read only by the fit)
  TpcMergeBuffers M;
  std::memset(&M, 0, sizeof(M));
  M.n_tracks = (uint32_t)n_tracks;
  M.counters = reinterpret_cast<uint32_t*>(scratch);
  M.merged = const_cast<tpc_merged_track*>(d_merged);
  M.seg_index = const_cast<uint32_t*>(d_seg_index);
  M.ids = const_cast<uint32_t*>(d_cluster_ids);
  TpcFitBuffers T;
  std::memset(&T, 0, sizeof(T));
  T.P = P;
  const double a = 2.0 * (double)ctx->geom.sector_half_angle_deg * (3.14159265358979323846 / 180.0);
  T.ca = (float)std::cos(a);
  T.sa = (float)std::sin(a);
  T.work = reinterpret_cast<uint32_t*>(scratch + 16);
  T.stored = reinterpret_cast<uint4*>(scratch + TPC_FIT_NOALLOC_HDR);
  T.chi2_cluster = d_chi2_out;
  T.rejected = d_rejected_out;
  T.fit = d_fit_out;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  (void)cudaGetLastError();
  k_fit_noalloc_header<<<1, 32, 0, st>>>((uint32_t)n_merged);   // what must start at zero, and the count the kernel reads
  const int l = (flags & TPC_DETERMINISTIC) ? tpc_det::run_fit3(B, &ctx->hconst, M, T, (uint32_t)n_merged, st, ctx->n_sm)
                                            : tpc_fast::run_fit3(B, &ctx->hconst, M, T, (uint32_t)n_merged, st, ctx->n_sm);
  if (l < 0 || cudaPeekAtLastError() != cudaSuccess) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch (fit, no allocation)");
  return TPC_OK;
}

// ---------------------------------------------------------------- Phase-II rebuild (R11)
namespace {
size_t carve_rebuild(uint64_t n_steps, uint64_t n_merged, uint64_t n_clusters, char* base, TpcRebuildBuffers* R) {
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* p = base ? base + off : nullptr;
    off = align_up(off + bytes, 256);
    return p;
  };
  TpcRebuildBuffers r;
  std::memset(&r, 0, sizeof(r));
  const size_t ns = n_steps + 1, nm = n_merged + 1, nc = n_clusters + 1;
  r.stored = (uint4*)take(16 * ns);
  r.cand_id = (int32_t*)take(4 * 3 * ns);
  r.cand_chi2 = (float*)take(4 * 3 * ns);
  r.attached = (int32_t*)take(4 * ns);
  r.shared = (uint8_t*)take(ns); r.used = (uint8_t*)take(ns);
  r.step_track = (uint32_t*)take(4 * ns);
  r.Qkey = (uint32_t*)take(4 * nm);
  r.tkey = (unsigned long long*)take(8 * nm);
  r.list_n = (uint32_t*)take(32);
  r.alive = (uint8_t*)take(nm);
  r.stq2 = (float*)take(12 * nm);
  r.best = (unsigned long long*)take(8 * nc);
  r.bestId = (unsigned long long*)take(8 * nc);
  r.fit = (tpc_track_fit3*)take(sizeof(tpc_track_fit3) * nm);
  if (R) *R = r;
  return off;
}
}  // namespace

void tpc_rebuild_default_params(tpc_rebuild_params* r) {
  r->cand_chi2_max = 16.0f;
  r->final_chi2_max = 16.0f;
  r->min_clusters = 10;
  r->ce_var = 10000.0f;
}

int tpc_rebuild_prepare(tpc_ctx* ctx, void* cuda_stream, uint64_t* n_steps) {
  if (!n_steps) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->merged) return TPC_E_STATE;
  if (ctx->buf.id_base != 0u) return TPC_E_STATE;   // (whole-frame runs only: cluster ids index the frame)
  cudaStream_t st = (cudaStream_t)cuda_stream;
  *n_steps = 0;
  if (ctx->mbuf.n_tracks) {
    (void)cudaGetLastError();
    const int l = (ctx->flags & TPC_DETERMINISTIC) ? tpc_det::run_rebuild_paths(ctx->buf, ctx->mbuf, st, ctx->n_sm)
                                                   : tpc_fast::run_rebuild_paths(ctx->buf, ctx->mbuf, st, ctx->n_sm);
    if (l < 0) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch (rebuild paths)");
    cudaError_t e = cudaMemcpyAsync(ctx->h_mcnt, ctx->mbuf.counters, 16, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return set_cuda_err(ctx, e, "rebuild paths");
    *n_steps = ctx->h_mcnt[3];
  }
  ctx->rb_n_steps = *n_steps;
  ctx->rb_prepared = true;
  ctx->rebuilt = false;
  return TPC_OK;
}

size_t tpc_rebuild_workspace_bytes(const tpc_ctx* ctx, uint64_t n_steps, uint64_t n_merged, uint64_t n_clusters) {
  if (!ctx || n_steps >= (1ull << 32) || n_merged >= (1ull << 31) || n_clusters >= (1ull << 31)) return 0;
  return carve_rebuild(n_steps, n_merged, n_clusters, nullptr, nullptr);
}

int tpc_rebuild_tracks(tpc_ctx* ctx, const tpc_rebuild_params* params, void* d_ws, size_t ws_bytes, void* cuda_stream) {
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->merged || !ctx->rb_prepared) return TPC_E_STATE;
  if (!d_ws || ((uintptr_t)d_ws & 255u)) return TPC_E_ARG;
  tpc_rebuild_params P;
  if (params) P = *params; else tpc_rebuild_default_params(&P);
  if (!(P.cand_chi2_max >= 0.f) || !(P.final_chi2_max >= 0.f) || P.min_clusters < 2 || !(P.ce_var > 0.f)) return TPC_E_ARG;
  const uint32_t n_merged = ctx->mbuf.n_tracks ? ctx->h_mcnt[0] : 0u;
  if (n_merged >= 0x3FFFFFFFu) return TPC_E_OVERFLOW;   // (the track index shares a word with the round tag)
  TpcRebuildBuffers R;
  const size_t need = carve_rebuild(ctx->rb_n_steps, n_merged, ctx->buf.n, (char*)d_ws, &R);
  if (ws_bytes < need) return TPC_E_WORKSPACE;
  R.P = P;
  R.ca = ctx->mbuf.ca; R.sa = ctx->mbuf.sa;
  R.n_merged = n_merged; R.n_steps = (uint32_t)ctx->rb_n_steps; R.n_clusters = ctx->buf.n;
  R.step_ofs = ctx->mbuf.path_ofs;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  (void)cudaGetLastError();
  const int l = (ctx->flags & TPC_DETERMINISTIC) ? tpc_det::run_rebuild(ctx->buf, &ctx->hconst, ctx->mbuf, R, st, ctx->n_sm)
                                                 : tpc_fast::run_rebuild(ctx->buf, &ctx->hconst, ctx->mbuf, R, st, ctx->n_sm);
  if (l < 0) return set_cuda_err(ctx, cudaGetLastError(), "kernel launch (rebuild)");
  ctx->rbuf = R;
  ctx->stream = st;
  ctx->synced = false;
  ctx->rebuilt = true;
  ctx->launches = l;
  return TPC_OK;
}

int tpc_get_rebuild(tpc_ctx* ctx, tpc_rebuild_view* out) {
  if (!out) return TPC_E_ARG;
  int rc = sync_run(ctx);
  if (rc != TPC_OK) return rc;
  if (!ctx->rebuilt) return TPC_E_STATE;
  const TpcRebuildBuffers& R = ctx->rbuf;
  std::memset(out, 0, sizeof(*out));
  out->n_merged = R.n_merged; out->n_steps = R.n_steps;
  out->d_step_ofs = R.step_ofs; out->d_cand_id = R.cand_id; out->d_cand_chi2 = R.cand_chi2;
  out->d_attached = R.attached; out->d_shared = R.shared; out->d_used = R.used; out->d_fit = R.fit;
  return TPC_OK;
}

int tpc_last_launch_count(const tpc_ctx* ctx) { return ctx ? ctx->launches : 0; }

void tpc_destroy(tpc_ctx* c) {
  if (!c) return;
  for (int i = 0; i < TPC_N_STAGES; ++i)
    if (c->events.ev[i]) cudaEventDestroy(c->events.ev[i]);
  for (int i = 0; i <= TPC_MAX_KERNELS; ++i)
    if (c->events.kev[i]) cudaEventDestroy(c->events.kev[i]);
  if (c->d_const) cudaFree(c->d_const);
  if (c->d_cnt) cudaFree(c->d_cnt);
  if (c->d_row_stat) cudaFree(c->d_row_stat);
  if (c->h_cnt) cudaFreeHost(c->h_cnt);
  if (c->h_mcnt) cudaFreeHost(c->h_mcnt);
  if (c->d_sector_seen) cudaFree(c->d_sector_seen);
  if (c->s_in) cudaStreamDestroy(c->s_in);
  if (c->s_out) cudaStreamDestroy(c->s_out);
  for (int i = 0; i < 2; ++i) {
    if (c->ev_in[i]) cudaEventDestroy(c->ev_in[i]);
    if (c->ev_done[i]) cudaEventDestroy(c->ev_done[i]);
    if (c->ev_out[i]) cudaEventDestroy(c->ev_out[i]);
  }
  delete c;
}

const char* tpc_strerror(int err) {
  switch (err) {
    case TPC_OK: return "ok";
    case TPC_E_ARG: return "bad argument (null/misaligned pointer, bad descriptor, or a cluster outside the geometry)";
    case TPC_E_WORKSPACE: return "workspace too small";
    case TPC_E_OVERFLOW: return "device capacity exceeded (bins, seeds or tracks); results invalid";
    case TPC_E_CUDA: return "CUDA runtime error";
    case TPC_E_STATE: return "call order violated";
    case TPC_E_LIMIT: return "size beyond the fixed maximum of the no-allocation entry point";
    default: return "unknown error";
  }
}

const char* tpc_last_cuda_error(const tpc_ctx* ctx) { return ctx ? ctx->cuda_err : ""; }

}  // extern "C"
