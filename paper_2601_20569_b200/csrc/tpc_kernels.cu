// tpc_kernels.cu — sm_100a CUDA kernels of the TPC sector tracking (section 2,
// PAPER.md:57,59 section 3; readings R0..R6 of DESIGN.md).
//
// This translation unit is compiled TWICE:
//   -DTPC_DET=1 --fmad=false  -> namespace tpc_det  : deterministic mode: no FMA
//                                contraction, stable grid order; bit-comparable to the CPU oracle
//   -DTPC_DET=0 --fmad=true --use_fast_math -> namespace tpc_fast : FMA contraction, approximate
//                                division / sqrt, no in-bin sort
// Both use only + - * / sqrt on the decision path; every argmin carries an integer tie-break on
// the ORIGINAL cluster index (rule D2), so atomics / thread order never change a result.
//
// Kernel groups:  K1 grid (row stats -> row descriptors -> per-row build in shared memory, or,
//                 for unordered input, histogram -> per-row scan -> scatter [-> in-bin sort]),
//                 K2 neighbour finder,  K3 link cleanup + seeds,  K4 Kalman track follower
//                 (outward / refit / inward kernels),  K5 ambiguity solving.
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "tpc_internal.h"

#ifndef TPC_DET
#error "compile with -DTPC_DET=0 or 1"
#endif
#if TPC_DET
#define TPC_NS tpc_det
#else
#define TPC_NS tpc_fast
#endif

namespace TPC_NS {

// ------------------------------------------------------------------ small device helpers
__device__ __forceinline__ uint32_t f2key(float f) {  // order-preserving float -> uint
  uint32_t b = __float_as_uint(f);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float key2f(uint32_t k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7FFFFFFFu) : ~k);
}
__device__ __forceinline__ int bin_coord(float v, float v0, float inv_d, int n) {
  int b = (int)floorf((v - v0) * inv_d);
  b = b < 0 ? 0 : b;
  return b > n - 1 ? n - 1 : b;
}
__device__ __forceinline__ bool finite2(float a, float b) {
  return (fabsf(a) <= 3.402823466e38f) && (fabsf(b) <= 3.402823466e38f);  // false for NaN/Inf
}
__device__ __forceinline__ uint4 ld_stream16(const void* p) {  // streaming 16-byte load
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// L2 residency control (createpolicy + .L2::cache_hint): streams that are read once are marked
// evict_first so that they do not push out the randomly accessed tables marked evict_last.
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ int32_t ld_i32_hint(const int32_t* p, uint64_t pol) {  // streaming, not kept in L1
  int32_t v;
  asm volatile("ld.global.L1::no_allocate.L2::cache_hint.b32 %0, [%1], %2;" : "=r"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ unsigned long long ld_u64_hint(const unsigned long long* p, uint64_t pol) {
  unsigned long long v;
  asm volatile("ld.global.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(v) : "l"(p), "l"(pol));
  return v;
}
__device__ __forceinline__ void red_max_u64_hint(unsigned long long* p, unsigned long long v, uint64_t pol) {
  asm volatile("red.global.max.L2::cache_hint.u64 [%0], %1, %2;" ::"l"(p), "l"(v), "l"(pol) : "memory");
}

// Classify one input cluster. Returns: 0 in grid, 1 ignored (NaN/Inf), 2 dropped (|y| beyond
// the row + 2 cm), 3 bad (sector/row outside the geometry).  R1 of DESIGN.md.
__device__ __forceinline__ int classify(const uint4& raw, const TpcConst* __restrict__ K, int& sr, float& y,
                                        float& z, int& row) {
  y = __uint_as_float(raw.x);
  z = __uint_as_float(raw.y);
  const int sector = raw.w & 0xFF;
  row = (raw.w >> 8) & 0xFF;
  sr = sector * K->n_rows + row;
  if (sector >= K->n_sectors || row >= K->n_rows) return 3;
  if (!finite2(y, z)) return 1;
  if (!(fabsf(y) <= K->ylim[row])) return 2;
  return 0;
}

// ================================================================== K1 grid
// K1a: per (sector,row) min/max z and cluster count.  One coalesced 16-byte load per cluster.
// Inputs usually arrive grouped by (sector,row) (clusteriser order), so a warp whose lanes
// all hit the same row does 3 atomics instead of 96.
__global__ void __launch_bounds__(256) k_row_stats(TpcBuffers B) {
  const TpcConst* __restrict__ K = B.K;
  uint32_t n_ign = 0, n_drop = 0, n_bad = 0;
  const uint32_t stride = gridDim.x * blockDim.x, n_up = (B.n + 31u) & ~31u;
  float2* __restrict__ yz_all = reinterpret_cast<float2*>(B.owner);   // (the owner words are not in use yet)
  for (uint32_t i0 = blockIdx.x * blockDim.x + threadIdx.x; i0 < n_up; i0 += 4 * stride) {
   uint4 raw4[4];   // four records requested together (bytes in flight)
#pragma unroll
   for (int u = 0; u < 4; ++u) {
     const uint32_t iu = i0 + u * stride;
     raw4[u] = iu < B.n ? ld_stream16(B.clusters + iu) : make_uint4(0u, 0u, 0u, 0u);
   }
#pragma unroll
   for (int u = 0; u < 4; ++u) {
    const uint32_t i = i0 + u * stride;
    if (i >= n_up) break;   // warp-uniform
    int cls = 4, sr = -1, row;
    float y, z = 0.f;
    if (i < B.n) {
      cls = classify(raw4[u], K, sr, y, z, row);
      // compact copy of the frame for the per-row grid build: 8 bytes per record, NaN = not in the grid
      yz_all[i] = cls == 0 ? make_float2(y, z) : make_float2(__uint_as_float(0x7fc00000u), 0.f);
    }
    n_ign += cls == 1;
    n_drop += cls == 2;
    n_bad += cls == 3;
    const bool ok = cls == 0;
    const bool in_row = cls <= 2;   // carries a valid (sector,row), kept in the grid or not
    const unsigned rowmask = __ballot_sync(0xffffffffu, in_row);
    if (rowmask == 0) continue;
    const unsigned okmask = __ballot_sync(0xffffffffu, ok);
    const int leader = __ffs(rowmask) - 1;
    const int sr0 = __shfl_sync(0xffffffffu, sr, leader);
    const bool uniform = __all_sync(0xffffffffu, !in_row || sr == sr0);
    const uint32_t zk = f2key(z);
    if (uniform) {
      const uint32_t mn = __reduce_min_sync(0xffffffffu, ok ? zk : 0xFFFFFFFFu);
      const uint32_t mx = __reduce_max_sync(0xffffffffu, ok ? zk : 0u);
      if ((int)(threadIdx.x & 31) == leader) {
        TpcRowStat* rs = &B.row_stat[sr0];
        if (okmask) {
          atomicMin(&rs->zmin_key, mn);
          atomicMax(&rs->zmax_key, mx);
          atomicAdd(&rs->count, (uint32_t)__popc(okmask));
        }
        atomicAdd(&rs->n_all, (uint32_t)__popc(rowmask));
        atomicMin(&rs->first, i);                                  // the leader is the lowest lane
        atomicMax(&rs->last, (i - (uint32_t)leader) + (31u - (uint32_t)__clz(rowmask)));
      }
    } else if (in_row) {
      TpcRowStat* rs = &B.row_stat[sr];
      if (ok) {
        atomicMin(&rs->zmin_key, zk);
        atomicMax(&rs->zmax_key, zk);
        atomicAdd(&rs->count, 1u);
      }
      atomicAdd(&rs->n_all, 1u);
      atomicMin(&rs->first, i);
      atomicMax(&rs->last, i);
    }
   }
  }
  n_ign = __reduce_add_sync(0xffffffffu, n_ign);
  n_drop = __reduce_add_sync(0xffffffffu, n_drop);
  n_bad = __reduce_add_sync(0xffffffffu, n_bad);
  if ((threadIdx.x & 31) == 0) {
    if (n_ign) atomicAdd(&B.cnt->n_ignored, n_ign);
    if (n_drop) atomicAdd(&B.cnt->n_dropped, n_drop);
    if (n_bad) {
      atomicAdd(&B.cnt->n_bad, n_bad);
      atomicOr(&B.cnt->error, TPC_DEVERR_BAD_CLUSTER);
    }
  }
}

// Block-wide exclusive scan of one value per thread (blockDim.x <= 1024); returns the
// exclusive prefix, *total = block sum.  Warp-level scans with shuffles + one smem hop.
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* total, uint32_t* smem33) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  uint32_t inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane >= d) inc += t;
  }
  __syncthreads();  // smem33 may still be in use from a previous call
  if (lane == 31) smem33[w] = inc;
  __syncthreads();
  if (w == 0) {
    const int nw = (blockDim.x + 31) >> 5;
    uint32_t s = lane < nw ? smem33[lane] : 0u;
    uint32_t si = s;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, si, d);
      if (lane >= d) si += t;
    }
    smem33[lane] = si - s;
    if (lane == 31) smem33[32] = si;
  }
  __syncthreads();
  *total = smem33[32];
  return smem33[w] + inc - v;
}

// K1b: row descriptors (one CTA).  nz from the z range, exclusive scans over the (sector,row)
// list for the first bin, first sorted cluster and first neighbour-finder tile of each row.
__global__ void __launch_bounds__(1024) k_row_desc(TpcBuffers B) {
  __shared__ uint32_t sm[33];
  const TpcConst* __restrict__ K = B.K;
  uint32_t base_bin = 0, base_clu = 0, base_tile = 0;
  unsigned long long bins64 = 0;
  bool overflow = false;
  uint32_t n_generic = 0;   // rows that do not qualify for the per-row grid build (k_row_sort)
  for (uint32_t s0 = 0; s0 < B.n_sr; s0 += blockDim.x) {
    const uint32_t sr = s0 + threadIdx.x;
    uint32_t cnt = 0, nb = 0, nt = 0, by_row = 1u;
    int nz = 0, ny = 0;
    float z0 = 0.f, y0 = 0.f;
    if (sr < B.n_sr) {
      const int row = sr % K->n_rows;
      cnt = B.row_stat[sr].count;
      ny = K->ny[row];
      y0 = -K->ylim[row];
      if (cnt) {
        z0 = key2f(B.row_stat[sr].zmin_key);
        const float zhi = key2f(B.row_stat[sr].zmax_key);
        const float fz = floorf((zhi - z0) * K->inv_dz);
        // bound nz so that ny*nz cannot wrap; a frame this sparse overflows max_bins anyway
        nz = fz >= 16777216.f ? 16777216 : (int)fz + 1;
        nz = nz < 1 ? 1 : nz;
        const unsigned long long nb64 = (unsigned long long)ny * (unsigned long long)nz;
        if (nb64 > B.max_bins) { overflow = true; nb = 0; nz = 0; }
        else nb = (uint32_t)nb64;
        nt = (cnt + TPC_NF_TILE - 1) / TPC_NF_TILE;
        // k_row_sort needs the row's input records in one contiguous range, and its bin
        // counters + permutation in the cluster's shared memory
        const TpcRowStat rs = B.row_stat[sr];
        const uint32_t bytes = 4u * ((nb + 1) / 2) + 2u * cnt;
        if (rs.last - rs.first + 1u != rs.n_all || rs.n_all > 65535u || bytes > TPC_RS_SMEM_BYTES) { by_row = 0u; ++n_generic; }
      }
    }
    if (B.chunk_tag && sr < B.n_sr && B.row_stat[sr].n_all) {   // chunked frame: sectors must not straddle chunks
      const uint32_t seen = atomicCAS(&B.sector_seen[sr / (uint32_t)K->n_rows], 0u, B.chunk_tag);
      if (seen != 0u && seen != B.chunk_tag) atomicOr(&B.cnt->error, TPC_DEVERR_CHUNKS);
    }
    uint32_t tot_b, tot_c, tot_t;
    const uint32_t pb = block_excl_scan(nb, &tot_b, sm);
    const uint32_t pc = block_excl_scan(cnt, &tot_c, sm);
    const uint32_t pt = block_excl_scan(nt, &tot_t, sm);
    if (sr < B.n_sr) {
      tpc_row_desc d;
      d.y0 = y0; d.z0 = z0; d.ny = ny; d.nz = nz;
      d.bin_ofs = base_bin + pb;
      d.clu_ofs = base_clu + pc;
      d.count = cnt;
      d.pad_ = by_row;   // 1: this row's grid is built by k_row_sort, 0: by the generic kernels
      B.row_desc[sr] = d;
      B.tile_ofs[sr] = base_tile + pt;
    }
    bins64 += tot_b;
    base_bin += tot_b; base_clu += tot_c; base_tile += tot_t;
  }
  overflow = __syncthreads_or(overflow || bins64 > B.max_bins);
  __shared__ uint32_t s_generic;
  if (threadIdx.x == 0) s_generic = 0u;
  __syncthreads();
  if (n_generic) atomicAdd(&s_generic, n_generic);
  __syncthreads();
  if (threadIdx.x == 0) {
    B.cnt->n_rows_generic = s_generic;
    B.cnt->grid_rows = (s_generic == 0u && !overflow) ? 1u : 0u;
    B.tile_ofs[B.n_sr] = base_tile;
    B.cnt->n_sorted = base_clu;
    B.cnt->n_tiles = base_tile;
    if (overflow) {
      atomicOr(&B.cnt->error, TPC_DEVERR_BINS);
      B.cnt->n_bins = 0;
    } else {
      B.cnt->n_bins = base_bin;
    }
  }
}

// (sector,row) of every neighbour-finder tile, so that K2 needs no search.
__global__ void __launch_bounds__(128) k_tile_rows(TpcBuffers B) {
  for (uint32_t sr = blockIdx.x; sr < B.n_sr; sr += gridDim.x) {
    const uint32_t t0 = B.tile_ofs[sr], t1 = B.tile_ofs[sr + 1];
    for (uint32_t t = t0 + threadIdx.x; t < t1; t += blockDim.x) B.tile_sr[t] = (uint16_t)sr;
  }
}

__global__ void __launch_bounds__(256) k_zero_bins(TpcBuffers B) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < B.n_sr * TPC_SEED_SLABS; i += gridDim.x * blockDim.x)
    B.item_cnt[i] = 0u;
  if ((B.cnt->error & TPC_DEVERR_BINS) || B.cnt->n_rows_generic == 0u) return;
  // the bin counters of the rows the generic kernels build (the others belong to k_row_sort)
  for (uint32_t sr = blockIdx.x; sr < B.n_sr; sr += gridDim.x) {
    const tpc_row_desc d = B.row_desc[sr];
    if (d.pad_ || d.count == 0) continue;
    const uint32_t nb = (uint32_t)d.ny * (uint32_t)d.nz;
    for (uint32_t b = threadIdx.x; b < nb; b += blockDim.x) B.bin_start[d.bin_ofs + b] = 0u;
  }
}

__device__ __forceinline__ uint32_t bin_of(const tpc_row_desc& d, const TpcConst* __restrict__ K, float y, float z) {
  const int by = bin_coord(y, d.y0, K->inv_dy, d.ny);
  const int bz = bin_coord(z, d.z0, K->inv_dz, d.nz);
  return d.bin_ofs + (uint32_t)bz * (uint32_t)d.ny + (uint32_t)by;
}

// K1c: histogram.  slot[i] = rank of cluster i inside its bin (the value the atomic returns),
// so the scatter needs no second atomic.
__global__ void __launch_bounds__(256) k_bin_hist(TpcBuffers B) {
  const TpcConst* __restrict__ K = B.K;
  if ((B.cnt->error & TPC_DEVERR_BINS) || B.cnt->n_rows_generic == 0u) return;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < B.n; i += gridDim.x * blockDim.x) {
    const uint4 raw = ld_stream16(B.clusters + i);
    int sr, row;
    float y, z;
    uint32_t s = 0xFFFFFFFFu;
    if (classify(raw, K, sr, y, z, row) == 0) {
      const tpc_row_desc d = B.row_desc[sr];
      if (!d.pad_) s = atomicAdd(&B.bin_start[bin_of(d, K, y, z)], 1u);   // (rows of k_row_sort are not ours)
    }
    B.slot[i] = s;
  }
}

// K1d: per-row exclusive scan of the bin counts -> bin_start (global sorted positions).
// One CTA per (sector,row); warp-level shuffles scan 8 bins per thread per step
// (north star: "a per-row bin index built by a warp-level scan").
__global__ void __launch_bounds__(512) k_bin_scan(TpcBuffers B) {
  __shared__ uint32_t sm[33];
  if ((B.cnt->error & TPC_DEVERR_BINS) || B.cnt->n_rows_generic == 0u) return;
  for (uint32_t sr = blockIdx.x; sr < B.n_sr; sr += gridDim.x) {
    const tpc_row_desc d = B.row_desc[sr];
    if (d.pad_) continue;
    const uint32_t nb = (uint32_t)d.ny * (uint32_t)d.nz;
    uint32_t* p = B.bin_start + d.bin_ofs;
    uint32_t carry = d.clu_ofs;
    for (uint32_t b0 = 0; b0 < nb; b0 += blockDim.x * 8) {
      const uint32_t b = b0 + threadIdx.x * 8;
      uint32_t v[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = (b + k < nb) ? p[b + k] : 0u;
      uint32_t s = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) s += v[k];
      uint32_t tot;
      uint32_t pre = carry + block_excl_scan(s, &tot, sm);
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        if (b + k < nb) p[b + k] = pre;
        pre += v[k];
      }
      carry += tot;
    }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) B.bin_start[B.cnt->n_bins] = B.cnt->n_sorted;
}

// K1e: scatter into bin order: sorted (y,z) pairs + original index.
__global__ void __launch_bounds__(256) k_scatter(TpcBuffers B) {
  const TpcConst* __restrict__ K = B.K;
  if ((B.cnt->error & TPC_DEVERR_BINS) || B.cnt->n_rows_generic == 0u) return;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < B.n; i += gridDim.x * blockDim.x) {
    const uint32_t s = B.slot[i];
    if (s == 0xFFFFFFFFu) continue;
    const uint4 raw = ld_stream16(B.clusters + i);
    int sr, row;
    float y, z;
    classify(raw, K, sr, y, z, row);
    const tpc_row_desc d = B.row_desc[sr];
    const uint32_t pos = B.bin_start[bin_of(d, K, y, z)] + s;
    // The destination sectors are written 8 / 4 bytes at a time by different threads; a store
    // that misses in L2 goes to DRAM as a partial sector (read-modify-write there), so the
    // sectors are pulled into L2 first (measured on the C4 frame: 10.7 -> 8.6 ms).
    asm volatile("prefetch.global.L2 [%0];" ::"l"(B.yz + pos));
    asm volatile("prefetch.global.L2 [%0];" ::"l"(B.orig_id + pos));
    B.yz[pos] = make_float2(y, z);
    B.orig_id[pos] = B.id_base + i;
  }
}

#if TPC_DET
// K1f (deterministic mode only): order the clusters of every bin by ascending original index,
// so that the sorted order is a function of the input alone (stable sort).
__global__ void __launch_bounds__(256) k_bin_sort(TpcBuffers B) {
  if ((B.cnt->error & TPC_DEVERR_BINS) || B.cnt->n_rows_generic == 0u) return;
  for (uint32_t sr = blockIdx.x; sr < B.n_sr; sr += gridDim.x) {
    const tpc_row_desc d = B.row_desc[sr];
    if (d.pad_ || d.count == 0) continue;
    const uint32_t nb = (uint32_t)d.ny * (uint32_t)d.nz;
    for (uint32_t bb = threadIdx.x; bb < nb; bb += blockDim.x) {
      const uint32_t b = d.bin_ofs + bb;
      const uint32_t lo = B.bin_start[b], hi = B.bin_start[b + 1];
      for (uint32_t i = lo + 1; i < hi; ++i) {  // insertion sort, bins hold a few clusters
        const uint32_t id = B.orig_id[i];
        const float2 v = B.yz[i];
        uint32_t j = i;
        while (j > lo && B.orig_id[j - 1] > id) {
          B.orig_id[j] = B.orig_id[j - 1];
          B.yz[j] = B.yz[j - 1];
          --j;
        }
        B.orig_id[j] = id;
        B.yz[j] = v;
      }
    }
  }
}
#endif

// ------------------------------------------------------------------ K1 per-row build
// The grid of one (sector,row) built by ONE CTA whose shared memory holds the row's bin
// counters and its permutation (both 16-bit: a qualifying row has < 65536 records).  It works
// on the compact 8-byte (y,z) copy of the frame that k_row_stats leaves in the (not yet used)
// owner words: the copies of the ~148 rows in flight fit in L2, so HBM sees the records twice
// in all (k_row_stats, pass A) and bin_start, yz, orig_id once, coalesced.  Used when every
// row's input records are contiguous (clusteriser order) and fit; otherwise the generic kernels
// above run (k_row_desc decides).
//   A  count: bin of every record -> shared-memory atomics (two 16-bit counters per word)
//   S  scan : exclusive scan of the counters -> bin_start to HBM, counters become cursors
//   B  place: cursor atomics hand out positions; inv[position] = record
//   (deterministic build: records of a bin ordered by input index, rule R1.4)
//   C  write: position-major, coalesced: record = inv[p] -> yz[p], orig_id[p]
__global__ void __launch_bounds__(TPC_RS_THREADS, 1) k_row_sort(TpcBuffers B) {
  extern __shared__ uint32_t rs_mem[];   // [nbw] packed bin counters / cursors | inv (16-bit)
  __shared__ uint32_t sm[33];
  if (B.cnt->error & TPC_DEVERR_BINS) return;
  if (blockIdx.x == 0 && threadIdx.x == 0) B.bin_start[B.cnt->n_bins] = B.cnt->n_sorted;
  const TpcConst* __restrict__ K = B.K;
  const uint32_t tid = threadIdx.x;
  for (uint32_t sr = blockIdx.x; sr < B.n_sr; sr += gridDim.x) {
    const tpc_row_desc d = B.row_desc[sr];
    if (d.count == 0 || !d.pad_) continue;                   // (rows that do not qualify go to the generic kernels)
    const uint32_t nb = (uint32_t)d.ny * (uint32_t)d.nz;
    const uint32_t nbw = (nb + 1) / 2;                       // counter words
    uint16_t* inv = reinterpret_cast<uint16_t*>(rs_mem + nbw);
    const TpcRowStat rs = B.row_stat[sr];
    const uint32_t n_all = rs.n_all;
    const float2* __restrict__ yz_in = reinterpret_cast<const float2*>(B.owner) + rs.first;   // written by k_row_stats
    __syncthreads();                                         // the previous row is done with rs_mem
    for (uint32_t w = tid; w < nbw; w += TPC_RS_THREADS) rs_mem[w] = 0u;
    __syncthreads();
    // ---- A: count, from the compact (y,z) copy k_row_stats left (NaN = record not in the grid).
    // TPC_RS_BATCH records per thread are requested together
    const float2 kNone = make_float2(__uint_as_float(0x7fc00000u), 0.f);
    for (uint32_t e0 = tid; e0 < n_all; e0 += TPC_RS_BATCH * TPC_RS_THREADS) {
      float2 v[TPC_RS_BATCH];
#pragma unroll
      for (int u = 0; u < TPC_RS_BATCH; ++u) {
        const uint32_t e = e0 + u * TPC_RS_THREADS;
        v[u] = e < n_all ? yz_in[e] : kNone;
      }
#pragma unroll
      for (int u = 0; u < TPC_RS_BATCH; ++u) {
        if (!(v[u].x == v[u].x)) continue;
        const uint32_t bb = bin_of(d, K, v[u].x, v[u].y) - d.bin_ofs;
        atomicAdd(&rs_mem[bb >> 1], 1u << ((bb & 1u) * 16u));
      }
    }
    __syncthreads();
    // ---- S: scan.  Each warp owns a contiguous chunk of the counter words and walks it 32 words
    // at a time (lane = word: conflict-free shared-memory access, warp scan by shuffles, coalesced
    // bin_start stores); the chunk totals are scanned by the block in between.
    {
      const uint32_t lane = tid & 31u, wid = tid >> 5;
      const uint32_t chunk = ((nbw + 1023u) / 1024u) * 32u;            // words per warp, a multiple of 32
      const uint32_t c_lo = min(wid * chunk, nbw), c_hi = min(c_lo + chunk, nbw);
      uint32_t part = 0;
      for (uint32_t w = c_lo + lane; w < c_hi; w += 32) { const uint32_t c = rs_mem[w]; part += (c & 0xFFFFu) + (c >> 16); }
      part = __reduce_add_sync(0xffffffffu, part);
      uint32_t tot;
      const uint32_t warp_pre = block_excl_scan(lane == 0 ? part : 0u, &tot, sm);   // exclusive prefix lands on lane 0
      uint32_t carry = __shfl_sync(0xffffffffu, warp_pre, 0);
      for (uint32_t w0 = c_lo; w0 < c_hi; w0 += 32) {
        const uint32_t w = w0 + lane;
        const uint32_t c = w < c_hi ? rs_mem[w] : 0u;
        const uint32_t lo = c & 0xFFFFu, both = lo + (c >> 16);
        uint32_t inc = both;
#pragma unroll
        for (int dlt = 1; dlt < 32; dlt <<= 1) {
          const uint32_t t = __shfl_up_sync(0xffffffffu, inc, dlt);
          if ((int)lane >= dlt) inc += t;
        }
        const uint32_t p0 = carry + inc - both, p1 = p0 + lo;
        if (w < c_hi) {
          rs_mem[w] = p0 | (p1 << 16);                       // cursors, row-relative (< 65536)
          B.bin_start[d.bin_ofs + 2 * w] = d.clu_ofs + p0;
          if (2 * w + 1 < nb) B.bin_start[d.bin_ofs + 2 * w + 1] = d.clu_ofs + p1;
        }
        carry += __shfl_sync(0xffffffffu, inc, 31);
      }
    }
    __syncthreads();
    // ---- B: place (the row's records now come from L2)
    for (uint32_t e0 = tid; e0 < n_all; e0 += TPC_RS_BATCH * TPC_RS_THREADS) {
      float2 v[TPC_RS_BATCH];
#pragma unroll
      for (int u = 0; u < TPC_RS_BATCH; ++u) {
        const uint32_t e = e0 + u * TPC_RS_THREADS;
        v[u] = e < n_all ? yz_in[e] : kNone;
      }
#pragma unroll
      for (int u = 0; u < TPC_RS_BATCH; ++u) {
        if (!(v[u].x == v[u].x)) continue;   // not in the grid
        const uint32_t bb = bin_of(d, K, v[u].x, v[u].y) - d.bin_ofs;
        const uint32_t sh = (bb & 1u) * 16u;
        const uint32_t p = (atomicAdd(&rs_mem[bb >> 1], 1u << sh) >> sh) & 0xFFFFu;
        inv[p] = (uint16_t)(e0 + u * TPC_RS_THREADS);
      }
    }
    __syncthreads();
#if TPC_DET
    // ---- records of a bin in ascending input index (the cursors now point at the bin ends;
    // a cursor that reached 65536 wrapped to 0 and its carry went into the upper half, which
    // only happens for the last bin of a 65536-record row: excluded by k_row_desc)
    for (uint32_t b = tid; b < nb; b += TPC_RS_THREADS) {
      const uint32_t hi = (rs_mem[b >> 1] >> ((b & 1u) * 16u)) & 0xFFFFu;
      const uint32_t lo = b ? ((rs_mem[(b - 1) >> 1] >> (((b - 1) & 1u) * 16u)) & 0xFFFFu) : 0u;
      for (uint32_t i = lo + 1; i < hi; ++i) {   // insertion sort, bins hold a few clusters
        const uint16_t v = inv[i];
        uint32_t j = i;
        while (j > lo && inv[j - 1] > v) { inv[j] = inv[j - 1]; --j; }
        inv[j] = v;
      }
    }
    __syncthreads();
#endif
    // ---- C: write the sorted arrays
    for (uint32_t q0 = tid; q0 < d.count; q0 += TPC_RS_BATCH * TPC_RS_THREADS) {
      uint32_t e[TPC_RS_BATCH];
      uint2 v[TPC_RS_BATCH];
#pragma unroll
      for (int u = 0; u < TPC_RS_BATCH; ++u) {
        const uint32_t q = q0 + u * TPC_RS_THREADS;
        e[u] = q < d.count ? (uint32_t)inv[q] : 0u;
        v[u] = *reinterpret_cast<const uint2*>(yz_in + e[u]);
      }
#pragma unroll
      for (int u = 0; u < TPC_RS_BATCH; ++u) {
        const uint32_t q = q0 + u * TPC_RS_THREADS;
        if (q >= d.count) continue;
        B.yz[d.clu_ofs + q] = make_float2(__uint_as_float(v[u].x), __uint_as_float(v[u].y));
        B.orig_id[d.clu_ofs + q] = B.id_base + rs.first + e[u];
      }
    }
  }
}

// ================================================================== window queries
// Visit the sorted clusters of one row whose bin intersects [ylo,yhi]x[zlo,zhi].  The margins
// make sure rounding can never hide a cluster that satisfies a window inequality; membership
// is always decided by the caller on the inequality itself (rule D3: results do not depend
// on the bin size).
struct BinWindow {
  uint32_t base;  // bin_ofs + by0 of z-row 0
  int ny, by_span, bz0, bz1;
};
__device__ __forceinline__ BinWindow make_window(const tpc_row_desc& d, const TpcConst* __restrict__ K, float ylo,
                                                 float yhi, float zlo, float zhi) {
  const float my = 1e-3f;
  const float mz = 1e-3f + 4e-7f * fmaxf(fabsf(zlo), fabsf(zhi));
  const int by0 = bin_coord(ylo - my, d.y0, K->inv_dy, d.ny);
  const int by1 = bin_coord(yhi + my, d.y0, K->inv_dy, d.ny);
  BinWindow w;
  w.ny = d.ny;
  w.base = d.bin_ofs + (uint32_t)by0;
  w.by_span = by1 - by0 + 1;
  w.bz0 = bin_coord(zlo - mz, d.z0, K->inv_dz, d.nz);
  w.bz1 = bin_coord(zhi + mz, d.z0, K->inv_dz, d.nz);
  return w;
}

// ================================================================== K2 neighbour finder
// PAPER.md:27 "combinatorial seeding based on a cellular automaton"; R2.
// One CTA per tile of TPC_NF_TILE consecutive sorted clusters of one row, one thread per
// cluster.  Bins are z-major, so a tile is a compact z-slab of its row and everything its
// threads can see on rows r+1 / r-1 is ONE contiguous range of the sorted arrays (all y-bins
// of the z-rows the windows touch).  That range (the (y,z) pairs and the slice of the bin
// index) is staged in shared memory with coalesced loads; the candidate search then runs on
// shared memory in two flat loops (window members -> per-thread lists) and one flat pair
// loop, so the lanes of a warp stay converged.  The best (up,down) pair is the lexicographic
// minimum of (d2, original id of up, original id of down) (rule D2), which makes the result
// independent of the visiting order.  Tiles whose slab does not fit (very sparse or very
// dense rows) take the same search on global memory (nf_generic).
#ifndef TPC_NF_SLAB
#define TPC_NF_SLAB 1024   // clusters staged per neighbour row
#endif
#define TPC_NF_BINS 1020   // bins staged per neighbour row (+1 end marker, + alignment slack)
#ifndef TPC_NF_MINBLOCKS
#define TPC_NF_MINBLOCKS 5
#endif
#define TPC_NF_LIST 12     // window members kept per thread and side

// ---- 1-D TMA (cp.async.bulk) + mbarrier: the slabs are contiguous ranges of the sorted arrays
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
  } while (!ok);
}
// bytes: a multiple of 16; src and dst 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// The search of one cluster directly on global memory.
__device__ __forceinline__ void nf_generic(const TpcBuffers& B, const BinWindow& wu, const BinWindow& wd, float yi,
                                           float zi, float ty, float wy, float wz, float max_d2, int32_t& bj,
                                           int32_t& bk) {
  const uint32_t* __restrict__ bin_start = B.bin_start;
  const float2* __restrict__ yz = B.yz;
  const uint32_t* __restrict__ orig = B.orig_id;
  float best = 0.f;
  for (int bzu = wu.bz0; bzu <= wu.bz1; ++bzu) {
    const uint32_t bu = wu.base + (uint32_t)bzu * (uint32_t)wu.ny;
    const uint32_t ju1 = bin_start[bu + wu.by_span];
    for (uint32_t j = bin_start[bu]; j < ju1; ++j) {
      const float2 cj = yz[j];
      if (!(fabsf((cj.x - yi) - ty) <= wy && fabsf(cj.y - zi) <= wz)) continue;
      const float dyu = cj.x - yi, dzu = cj.y - zi;
      for (int bzd = wd.bz0; bzd <= wd.bz1; ++bzd) {
        const uint32_t bd = wd.base + (uint32_t)bzd * (uint32_t)wd.ny;
        const uint32_t k1 = bin_start[bd + wd.by_span];
        for (uint32_t k = bin_start[bd]; k < k1; ++k) {
          const float2 ck = yz[k];
          if (!(fabsf((yi - ck.x) - ty) <= wy && fabsf(zi - ck.y) <= wz)) continue;
          const float dy = dyu + (ck.x - yi);
          const float dz = dzu + (ck.y - zi);
          const float d2 = dy * dy + dz * dz;
          if (!(d2 <= max_d2)) continue;
          bool better = bj < 0 || d2 < best;
          if (!better && d2 == best) {  // exact tie: rule D2 (rare, ids fetched only here)
            const uint32_t jid = orig[j], bjid = orig[bj];
            better = jid < bjid || (jid == bjid && orig[k] < orig[bk]);
          }
          if (better) { best = d2; bj = (int32_t)j; bk = (int32_t)k; }
        }
      }
    }
  }
}

// Collect the window members of one side from the staged slab into the thread's list.
// The window touches at most three z-rows of bins (the caller checks), each a contiguous
// range of the slab; their bounds are fetched together and ONE flat loop then tests every
// cluster of the three ranges.  UP: window inequality of the up row, else of the down row.
// Returns the member count (members beyond TPC_NF_LIST are not stored: the caller then takes
// the nested fallback).
template <bool UP>
__device__ __forceinline__ int nf_collect(const BinWindow& w, int bz_lo, uint32_t bin_ofs, uint32_t c0,
                                          const uint32_t* __restrict__ s_bin, const float2* __restrict__ s_yz,
                                          uint16_t* __restrict__ s_list, float yi, float zi, float ty, float wy,
                                          float wz) {
  const int nzr = w.bz1 - w.bz0;  // 0..2 extra z-rows
  const uint32_t b = (w.base - bin_ofs) + (uint32_t)(w.bz0 - bz_lo) * (uint32_t)w.ny;
  const uint32_t a0 = s_bin[b] - c0, l0 = (s_bin[b + w.by_span] - c0) - a0;
  uint32_t a1 = 0, l1 = 0, a2 = 0, l2 = 0;
  if (nzr >= 1) { a1 = s_bin[b + w.ny] - c0; l1 = (s_bin[b + w.ny + w.by_span] - c0) - a1; }
  if (nzr >= 2) { a2 = s_bin[b + 2 * w.ny] - c0; l2 = (s_bin[b + 2 * w.ny + w.by_span] - c0) - a2; }
  const uint32_t l01 = l0 + l1, total = l01 + l2;
  const uint32_t o1 = a1 - l0, o2 = a2 - l01;
  int n = 0;
  for (uint32_t t = 0; t < total; ++t) {
    const uint32_t j = t + (t < l0 ? a0 : (t < l01 ? o1 : o2));
    const float2 c = s_yz[j];
    const bool in = UP ? (fabsf((c.x - yi) - ty) <= wy && fabsf(c.y - zi) <= wz)
                       : (fabsf((yi - c.x) - ty) <= wy && fabsf(zi - c.y) <= wz);
    if (in) {
      if (n < TPC_NF_LIST) s_list[n * TPC_NF_TILE] = (uint16_t)j;
      ++n;
    }
  }
  return n;
}

// The down side of the search: every member of the down window is paired at once with the
// (few) members of the up window collected before, so that no second list and no separate
// pair loop are needed.  The first two up members sit in registers.  Best pair = minimum of
// (d2, original id of up, original id of down): independent of the visiting order (rule D2).
__device__ __forceinline__ void nf_down_pairs(const BinWindow& w, int bz_lo, uint32_t bin_ofs, uint32_t c0,
                                              const uint32_t* __restrict__ s_bin, const float2* __restrict__ s_yz_d,
                                              const float2* __restrict__ s_yz_u, const uint16_t* __restrict__ s_list_u,
                                              int nU, float yi, float zi, float ty, float wy, float wz, float max_d2,
                                              const uint32_t* __restrict__ orig, uint32_t cu0, uint32_t cd0,
                                              int32_t& bj, int32_t& bk) {
  const int nzr = w.bz1 - w.bz0;  // 0..2 extra z-rows
  const uint32_t b = (w.base - bin_ofs) + (uint32_t)(w.bz0 - bz_lo) * (uint32_t)w.ny;
  const uint32_t a0 = s_bin[b] - c0, l0 = (s_bin[b + w.by_span] - c0) - a0;
  uint32_t a1 = 0, l1 = 0, a2 = 0, l2 = 0;
  if (nzr >= 1) { a1 = s_bin[b + w.ny] - c0; l1 = (s_bin[b + w.ny + w.by_span] - c0) - a1; }
  if (nzr >= 2) { a2 = s_bin[b + 2 * w.ny] - c0; l2 = (s_bin[b + 2 * w.ny + w.by_span] - c0) - a2; }
  const uint32_t l01 = l0 + l1, total = l01 + l2;
  const uint32_t o1 = a1 - l0, o2 = a2 - l01;
  const uint32_t ju0 = s_list_u[0];
  const float2 cj0 = s_yz_u[ju0];
  const float ux0 = cj0.x - yi, uz0 = cj0.y - zi;
  uint32_t ju1 = 0;
  float ux1 = 0.f, uz1 = 0.f;
  if (nU > 1) {
    ju1 = s_list_u[TPC_NF_TILE];
    const float2 cj1 = s_yz_u[ju1];
    ux1 = cj1.x - yi; uz1 = cj1.y - zi;
  }
  float best = 0.f;
  for (uint32_t t = 0; t < total; ++t) {
    const uint32_t kd = t + (t < l0 ? a0 : (t < l01 ? o1 : o2));
    const float2 ck = s_yz_d[kd];
    if (!(fabsf((yi - ck.x) - ty) <= wy && fabsf(zi - ck.y) <= wz)) continue;
    const float vx = ck.x - yi, vz = ck.y - zi;
    auto pair = [&](uint32_t ju, float ux, float uz) {
      const float dy = ux + vx;
      const float dz = uz + vz;
      const float d2 = dy * dy + dz * dz;
      if (d2 <= max_d2) {
        bool better = bj < 0 || d2 < best;
        if (!better && d2 == best) {  // exact tie: rule D2 (rare, ids fetched only here)
          const uint32_t jid = orig[cu0 + ju], bjid = orig[cu0 + (uint32_t)bj];
          better = jid < bjid || (jid == bjid && orig[cd0 + kd] < orig[cd0 + (uint32_t)bk]);
        }
        if (better) { best = d2; bj = (int32_t)ju; bk = (int32_t)kd; }
      }
    };
    pair(ju0, ux0, uz0);
    if (nU > 1) pair(ju1, ux1, uz1);
    for (int a = 2; a < nU; ++a) {
      const uint32_t ju = s_list_u[a * TPC_NF_TILE];
      const float2 cj = s_yz_u[ju];
      pair(ju, cj.x - yi, cj.y - zi);
    }
  }
}

__global__ void __launch_bounds__(TPC_NF_TILE, TPC_NF_MINBLOCKS) k_neighbours(TpcBuffers B) {
  __shared__ __align__(16) float2 s_yz[2][TPC_NF_SLAB + 2];
  __shared__ __align__(16) uint32_t s_bin[2][TPC_NF_BINS + 8];
  __shared__ uint16_t s_list[TPC_NF_LIST * TPC_NF_TILE];                 // up-window members per thread
  __shared__ __align__(8) unsigned long long s_mbar;
  const TpcConst* __restrict__ K = B.K;
  if (B.cnt->error & TPC_DEVERR_BINS) return;
  const uint32_t n_tiles = B.cnt->n_tiles;
  const int R = K->n_rows;
  const float wy = K->wy, wz = K->wz, max_d2 = K->P.nf_max_d2;
  const float dzbin = K->P.grid_dz, inv_dz = K->inv_dz;
  const uint32_t* __restrict__ bin_start = B.bin_start;
  const float2* __restrict__ yz = B.yz;
  const uint32_t* __restrict__ orig = B.orig_id;
  const int tx = threadIdx.x;
  if (tx == 0) mbar_init(&s_mbar, 1);
  __syncthreads();
  uint32_t parity = 0;
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t sr = B.tile_sr[tile];
    const int r = (int)(sr % (uint32_t)R);
    const tpc_row_desc d = B.row_desc[sr];
    const uint32_t tile_first = (tile - B.tile_ofs[sr]) * TPC_NF_TILE;
    const uint32_t local = tile_first + (uint32_t)tx;
    const bool have = local < d.count;
    const uint32_t i = d.clu_ofs + local;
    tpc_row_desc du, dd;
    du.count = 0; dd.count = 0;
    if (r >= 1 && r <= R - 2) { du = B.row_desc[sr + 1]; dd = B.row_desc[sr - 1]; }
    if (du.count == 0 || dd.count == 0) {  // uniform over the CTA: no links on this row
      if (have) { B.link_up[i] = -1; B.link_dn[i] = -1; }
      continue;
    }
    float yi = 0.f, zi = 0.f, ty = 0.f;
    BinWindow wu, wd;
    wu.bz0 = wd.bz0 = 0x7fffffff; wu.bz1 = wd.bz1 = -1;
    wu.base = wd.base = 0; wu.ny = wd.ny = 1; wu.by_span = wd.by_span = 1;
    if (have) {
      const float2 ci = yz[i];
      yi = ci.x; zi = ci.y;
      const float ti = yi / K->x[r];
      ty = ti * K->dx_row;
      wu = make_window(du, K, (yi + ty) - wy, (yi + ty) + wy, zi - wz, zi + wz);
      wd = make_window(dd, K, (yi - ty) - wy, (yi - ty) + wy, zi - wz, zi + wz);
    }
    // ---- the z-rows of bins the tile's windows can touch on either side, WITHOUT a reduction:
    // the tile is a run of the z-major sorted row, so all its clusters lie in the z-rows of bins
    // between those of its first and last cluster (a thread whose window is not covered, which
    // rounding could only cause at a bin edge, takes the per-thread search below)
    const uint32_t tile_last = min(tile_first + TPC_NF_TILE, d.count) - 1u;
    const int bzf = bin_coord(yz[d.clu_ofs + tile_first].y, d.z0, inv_dz, d.nz);
    const int bzl = bin_coord(yz[d.clu_ofs + tile_last].y, d.z0, inv_dz, d.nz);
    const float zmin = d.z0 + (float)bzf * dzbin, zmax = d.z0 + (float)(bzl + 1) * dzbin;
    const float mzt = 2e-3f + 1e-6f * fmaxf(fabsf(zmin), fabsf(zmax));
    const int ulo = bin_coord((zmin - wz) - mzt, du.z0, inv_dz, du.nz), uhi = bin_coord((zmax + wz) + mzt, du.z0, inv_dz, du.nz);
    const int dlo = bin_coord((zmin - wz) - mzt, dd.z0, inv_dz, dd.nz), dhi = bin_coord((zmax + wz) + mzt, dd.z0, inv_dz, dd.nz);
    const uint32_t ub0 = du.bin_ofs + (uint32_t)ulo * (uint32_t)du.ny;
    const uint32_t unb = (uint32_t)(uhi - ulo + 1) * (uint32_t)du.ny;
    const uint32_t db0 = dd.bin_ofs + (uint32_t)dlo * (uint32_t)dd.ny;
    const uint32_t dnb = (uint32_t)(dhi - dlo + 1) * (uint32_t)dd.ny;
    const uint32_t cu0 = bin_start[ub0], cu1 = bin_start[ub0 + unb];
    const uint32_t cd0 = bin_start[db0], cd1 = bin_start[db0 + dnb];
    // 16-byte alignment of the bulk copies: start of the bin slice rounded down to 4 entries, start
    // of the cluster slab to 2; sizes rounded up (the arrays are padded)
    const uint32_t ub0a = ub0 & ~3u, db0a = db0 & ~3u, cu0a = cu0 & ~1u, cd0a = cd0 & ~1u;
    const uint32_t unb_c = (ub0 + unb + 1u - ub0a + 3u) & ~3u, dnb_c = (db0 + dnb + 1u - db0a + 3u) & ~3u;
    const uint32_t ucl_c = (cu1 - cu0a + 1u) & ~1u, dcl_c = (cd1 - cd0a + 1u) & ~1u;
    int32_t bj = -1, bk = -1;
    const bool staged = unb_c <= TPC_NF_BINS + 8 && dnb_c <= TPC_NF_BINS + 8 && ucl_c <= TPC_NF_SLAB + 2 &&
                        dcl_c <= TPC_NF_SLAB + 2;
    bool slow = !staged;   // this thread searches on global memory (nf_generic)
    if (staged) {
      __syncthreads();     // every warp is done with the previous tile's slabs
      if (tx == 0) {
        mbar_expect_tx(&s_mbar, 4u * (unb_c + dnb_c) + 8u * (ucl_c + dcl_c));
        bulk_g2s(s_bin[0], bin_start + ub0a, 4u * unb_c, &s_mbar);
        bulk_g2s(s_bin[1], bin_start + db0a, 4u * dnb_c, &s_mbar);
        if (ucl_c) bulk_g2s(s_yz[0], yz + cu0a, 8u * ucl_c, &s_mbar);
        if (dcl_c) bulk_g2s(s_yz[1], yz + cd0a, 8u * dcl_c, &s_mbar);
      }
      // windows this tile's slabs do not cover, or taller than three z-rows of bins
      const bool covered = have && wu.bz0 >= ulo && wu.bz1 <= uhi && wd.bz0 >= dlo && wd.bz1 <= dhi &&
                           wu.bz1 - wu.bz0 <= 2 && wd.bz1 - wd.bz0 <= 2;
      slow = have && !covered;
      mbar_wait(&s_mbar, parity);
      parity ^= 1u;
      if (covered) {
        const int nU = nf_collect<true>(wu, 0, ub0a, cu0a, s_bin[0], s_yz[0], &s_list[tx], yi, zi, ty, wy, wz);
        if (nU > TPC_NF_LIST) {
          slow = true;                                                   // rare: crowded window
        } else if (nU) {
          nf_down_pairs(wd, 0, db0a, cd0a, s_bin[1], s_yz[1], s_yz[0], &s_list[tx], nU, yi, zi, ty, wy, wz,
                        max_d2, orig, cu0a, cd0a, bj, bk);
          if (bj >= 0) { bj += (int32_t)cu0a; bk += (int32_t)cd0a; }
        }
      }
    } else {
      slow = have;
    }
    if (slow) nf_generic(B, wu, wd, yi, zi, ty, wy, wz, max_d2, bj, bk);
    if (have) { B.link_up[i] = bj; B.link_dn[i] = bk; }
  }
}

// ================================================================== K3 cleanup + seeds
// R3: one evolution step of the automaton — keep reciprocal links only.
__global__ void __launch_bounds__(256) k_link_cleanup(TpcBuffers B) {
  if (B.cnt->error & TPC_DEVERR_BINS) return;
  const uint32_t n = B.cnt->n_sorted;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const int32_t u = B.link_up[i], d = B.link_dn[i];
    B.link_up2[i] = (u >= 0 && B.link_dn[u] == (int32_t)i) ? u : -1;
    B.link_dn2[i] = (d >= 0 && B.link_up[d] == (int32_t)i) ? d : -1;
  }
}

// (sector,row) of sorted position i: last sr with clu_ofs <= i (empty rows share clu_ofs with
// the next non-empty one, so the search lands on the non-empty row).
__device__ __forceinline__ uint32_t sr_of_position(const TpcBuffers& B, uint32_t i) {
  uint32_t lo = 0, hi = B.n_sr;
  while (hi - lo > 1) {
    const uint32_t mid = (lo + hi) >> 1;
    if (B.row_desc[mid].clu_ofs <= i) lo = mid; else hi = mid;
  }
  return lo;
}
// Work item of a seed: (sector,row, z-slab of the start hit); slabs are equal shares of the
// row's z-bins.  Only the ORDER of the seed list depends on it (a locality heuristic), never a
// result.
__device__ __forceinline__ uint32_t seed_item(const TpcBuffers& B, uint32_t sr, uint32_t i) {
  const tpc_row_desc d = B.row_desc[sr];
  const int bz = bin_coord(B.yz[i].y, d.z0, B.K->inv_dz, d.nz);
  const uint32_t slab = (uint32_t)(((unsigned long long)bz * TPC_SEED_SLABS) / (unsigned long long)(d.nz > 0 ? d.nz : 1));
  return sr * TPC_SEED_SLABS + (slab < TPC_SEED_SLABS ? slab : TPC_SEED_SLABS - 1);
}

// R4 pass A: start hits (no down link, an up link, chain >= seed_min_len); per-block counts.
// A block covers TPC_SEED_SPAN consecutive sorted positions, four per thread (16-byte loads of
// the links, one packed store of the four flags).
#define TPC_SEED_BLOCK 256
#define TPC_SEED_SPAN (4 * TPC_SEED_BLOCK)

// (sector,row) of position i, searched upward from the row of the block's first position
// (rows are long against a block's span, so this is zero or one step)
__device__ __forceinline__ uint32_t sr_from(const TpcBuffers& B, uint32_t sr, uint32_t i) {
  while (sr + 1 < B.n_sr && B.row_desc[sr + 1].clu_ofs <= i) ++sr;
  return sr;
}

__global__ void __launch_bounds__(TPC_SEED_BLOCK) k_seed_flags(TpcBuffers B) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_sr;
  if (B.cnt->error & TPC_DEVERR_BINS) return;
  const uint32_t n = B.cnt->n_sorted;
  const int min_len = B.K->P.seed_min_len;
  const uint32_t n_blocks = (n + TPC_SEED_SPAN - 1) / TPC_SEED_SPAN;
  const int32_t* __restrict__ up2 = B.link_up2;
  for (uint32_t blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
    const uint32_t i0 = blk * TPC_SEED_SPAN + threadIdx.x * 4;
    __syncthreads();
    if (threadIdx.x == 0) s_sr = sr_of_position(B, blk * TPC_SEED_SPAN);
    int32_t dn[4] = {0, 0, 0, 0}, up[4] = {-1, -1, -1, -1};
    if (i0 + 3 < n) {   // link arrays are 256-byte aligned, i0 is a multiple of 4
      const int4 d4 = *reinterpret_cast<const int4*>(B.link_dn2 + i0);
      const int4 u4 = *reinterpret_cast<const int4*>(up2 + i0);
      dn[0] = d4.x; dn[1] = d4.y; dn[2] = d4.z; dn[3] = d4.w;
      up[0] = u4.x; up[1] = u4.y; up[2] = u4.z; up[3] = u4.w;
    } else {
      for (int u = 0; u < 4; ++u) if (i0 + u < n) { dn[u] = B.link_dn2[i0 + u]; up[u] = up2[i0 + u]; }
    }
    uint32_t flags = 0, cnt = 0;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (dn[u] < 0 && up[u] >= 0) {
        // only "at least seed_min_len" is decided here; the full chain length is counted by the
        // follower's chain fit, which walks the chain anyway (k_follow_up -> seed_len[])
        int len = 1;
        for (int32_t c = up[u]; c >= 0 && len < min_len; c = up2[c]) ++len;
        if (len >= min_len) { flags |= 1u << (8 * u); ++cnt; }
      }
    }
    __syncthreads();   // s_sr
    if (flags) {
      uint32_t sr = s_sr;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if ((flags >> (8 * u)) & 1u) {
          sr = sr_from(B, sr, i0 + u);
          atomicAdd(&B.item_cnt[seed_item(B, sr, i0 + u)], 1u);
        }
      }
    }
    if (i0 + 3 < n) *reinterpret_cast<uint32_t*>(B.seed_len + i0) = flags;
    else for (int u = 0; u < 4; ++u) if (i0 + u < n) B.seed_len[i0 + u] = (uint8_t)((flags >> (8 * u)) & 1u);
    uint32_t tot;
    block_excl_scan(cnt, &tot, sm);
    if (threadIdx.x == 0) B.scan_partials[blk] = tot;
  }
}

// Exclusive scan of up to scan_blocks partial sums by one CTA; writes the grand total to
// *total_out (clamped to cap, raising err_bit when it does not fit).
__global__ void __launch_bounds__(1024) k_scan_partials(uint32_t* p, const uint32_t* n_items_ptr,
                                                        uint32_t items_per_block, uint32_t* total_out, uint32_t cap,
                                                        uint32_t* error, uint32_t err_bit) {
  __shared__ uint32_t sm[33];
  const uint32_t n = (*n_items_ptr + items_per_block - 1) / items_per_block;
  uint32_t carry = 0;
  for (uint32_t b0 = 0; b0 < n; b0 += blockDim.x) {
    const uint32_t b = b0 + threadIdx.x;
    const uint32_t v = b < n ? p[b] : 0u;
    uint32_t tot;
    const uint32_t pre = block_excl_scan(v, &tot, sm);
    if (b < n) p[b] = carry + pre;
    carry += tot;
  }
  if (threadIdx.x == 0) {
    if (carry > cap) {
      atomicOr(error, err_bit);
      carry = 0;  // later stages see an empty list; the error is reported by tpc_get_tracks
    }
    *total_out = carry;
  }
}

// Seed-list order.  One CTA per sector: exclusive scans of the sector's per-item seed counts
// in sorted order (row, slab) and in list order (slab, row); item_delta = their difference, so
// that list position = rank in sorted order + item_delta[item].  Sectors stay contiguous and
// in the same order in both, so no cross-sector term is needed.
__global__ void __launch_bounds__(1024) k_seed_items(TpcBuffers B) {
  extern __shared__ uint32_t s_cnt[];   // [n_rows][TPC_SEED_SLABS]
  __shared__ uint32_t sm[33];
  const uint32_t R = (uint32_t)B.K->n_rows, S = TPC_SEED_SLABS, n = R * S;
  const uint32_t base = blockIdx.x * n;
  for (uint32_t e = threadIdx.x; e < n; e += blockDim.x) s_cnt[e] = B.item_cnt[base + e];
  __syncthreads();
  const uint32_t L = (n + blockDim.x - 1) / blockDim.x;
  const uint32_t e0 = threadIdx.x * L, e1 = min(e0 + L, n);
  uint32_t tot;
  {  // sorted order: element e = row*S + slab
    uint32_t sum = 0;
    for (uint32_t e = e0; e < e1; ++e) sum += s_cnt[e];
    uint32_t pre = block_excl_scan(sum, &tot, sm);
    for (uint32_t e = e0; e < e1; ++e) { B.item_delta[base + e] = -(int32_t)pre; pre += s_cnt[e]; }
  }
  __syncthreads();
  // list order: groups of TPC_SEED_GROUP z-slabs, row-major inside a group (group 1: slab-major)
  auto list_to_item = [&](uint32_t e) -> uint32_t {
    const uint32_t g = e / (R * TPC_SEED_GROUP), rem = e % (R * TPC_SEED_GROUP);
    return (rem / TPC_SEED_GROUP) * S + g * TPC_SEED_GROUP + rem % TPC_SEED_GROUP;
  };
  {
    uint32_t sum = 0;
    for (uint32_t e = e0; e < e1; ++e) sum += s_cnt[list_to_item(e)];
    uint32_t pre = block_excl_scan(sum, &tot, sm);
    for (uint32_t e = e0; e < e1; ++e) {
      const uint32_t k = list_to_item(e);
      B.item_delta[base + k] += (int32_t)pre;
      pre += s_cnt[k];
    }
  }
}

// R4 pass B: write the seed list, ordered by (sector, z-slab, row, sorted index) — a pure
// function of the input in deterministic mode.
__global__ void __launch_bounds__(TPC_SEED_BLOCK) k_seed_write(TpcBuffers B) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_sr;
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const uint32_t n = B.cnt->n_sorted;
  const uint32_t n_blocks = (n + TPC_SEED_SPAN - 1) / TPC_SEED_SPAN;
  for (uint32_t blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
    const uint32_t i0 = blk * TPC_SEED_SPAN + threadIdx.x * 4;
    __syncthreads();
    if (threadIdx.x == 0) s_sr = sr_of_position(B, blk * TPC_SEED_SPAN);
    uint32_t flags = 0;
    if (i0 + 3 < n) flags = *reinterpret_cast<const uint32_t*>(B.seed_len + i0);
    else for (int u = 0; u < 4; ++u) if (i0 + u < n && B.seed_len[i0 + u]) flags |= 1u << (8 * u);
    flags &= 0x01010101u;
    uint32_t tot;
    uint32_t pre = block_excl_scan((uint32_t)__popc(flags), &tot, sm) + B.scan_partials[blk];   // syncs: s_sr is visible
    if (flags) {
      uint32_t sr = s_sr;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if ((flags >> (8 * u)) & 1u) {
          sr = sr_from(B, sr, i0 + u);
          const uint32_t pos = (uint32_t)((int32_t)pre + B.item_delta[seed_item(B, sr, i0 + u)]);
          B.seeds[pos] = i0 + u;
          B.seed_sr[pos] = (uint16_t)sr;
          ++pre;
        }
      }
    }
  }
}

// ================================================================== K4 track follower
// "the track following fits all seeds and propagates them through the TPC volume
// using the Kalman filter picking up more clusters of the track".  DESIGN.md R5.
// One seed per thread; the 5-parameter state and the 15 covariance entries live in
// registers, fp32 (north star item 4).  Expression order follows DESIGN.md "Formulas" so
// that the deterministic build (no FMA) is bit-comparable with the CPU oracle.
struct KF {
  float y, z, s, t, q;
  float c00, c10, c11, c20, c21, c22, c30, c31, c32, c33, c40, c41, c42, c43, c44;
};

struct FollowConst {
  float dx, cfield, max_sinphi, max_qpt, vy, vz;
  float road_nsigma, road_min, road_max, chi2_max;
  float ivs, ivt, ivq;
  int max_gap, min_hits, R;
};

__device__ __forceinline__ void kf_init_cov(KF& k, const FollowConst& F) {
  k.c00 = F.vy; k.c10 = 0.f; k.c11 = F.vz;
  k.c20 = 0.f; k.c21 = 0.f; k.c22 = F.ivs;
  k.c30 = 0.f; k.c31 = 0.f; k.c32 = 0.f; k.c33 = F.ivt;
  k.c40 = 0.f; k.c41 = 0.f; k.c42 = 0.f; k.c43 = 0.f; k.c44 = F.ivq;
}

// Formulas P: exact circle in xy, z advances with tan(lambda) times the arc length.
__device__ __forceinline__ bool kf_propagate(KF& k, float dx, const FollowConst& F) {
  const float s = k.s, t = k.t;
  const float cf = F.cfield;
  const float kap = cf * k.q;
  const float ex = sqrtf(1.f - s * s);
  const float s1 = s + kap * dx;
  if (!(fabsf(s1) <= F.max_sinphi)) return false;
  const float ex1 = sqrtf(1.f - s1 * s1);
  const float h = 1.f / (ex + ex1);
  const float ss = s + s1;
  const float tt = ss * h;
  const float dy = dx * tt;
  const float dl = dx * sqrtf(1.f + tt * tt);
  const float a = (0.5f * kap) * dl;
  const float a2 = a * a;
  const float dS = dl * (1.f + a2 * ((1.f / 6.f) + a2 * (3.f / 40.f)));
  const float hh = h * h;
  const float g = s / ex + s1 / ex1;
  const float f02 = dx * (2.f * h + (ss * hh) * g);
  const float f04 = ((dx * dx) * cf) * (h + (ss * hh) * (s1 / ex1));
  const float f12 = ((t * dx) * tt) / (ex * ex1);
  const float f13 = dS;
  const float sm = 0.5f * ss;
  const float exm = 0.5f * (ex + ex1);
  const float f14 = (((t * cf) * (0.5f * (dx * dx))) * sm) / ((exm * exm) * exm);
  const float f24 = cf * dx;
  k.y = k.y + dy;
  k.z = k.z + t * dS;
  k.s = s1;
  const float c00 = k.c00, c10 = k.c10, c11 = k.c11, c20 = k.c20, c21 = k.c21, c22 = k.c22;
  const float c30 = k.c30, c31 = k.c31, c32 = k.c32, c33 = k.c33;
  const float c40 = k.c40, c41 = k.c41, c42 = k.c42, c43 = k.c43, c44 = k.c44;
  const float m00 = (c00 + f02 * c20) + f04 * c40;
  const float m02 = (c20 + f02 * c22) + f04 * c42;
  const float m04 = (c40 + f02 * c42) + f04 * c44;
  const float m10 = ((c10 + f12 * c20) + f13 * c30) + f14 * c40;
  const float m11 = ((c11 + f12 * c21) + f13 * c31) + f14 * c41;
  const float m12 = ((c21 + f12 * c22) + f13 * c32) + f14 * c42;
  const float m13 = ((c31 + f12 * c32) + f13 * c33) + f14 * c43;
  const float m14 = ((c41 + f12 * c42) + f13 * c43) + f14 * c44;
  const float m20 = c20 + f24 * c40;
  const float m21 = c21 + f24 * c41;
  const float m22 = c22 + f24 * c42;
  const float m23 = c32 + f24 * c43;
  const float m24 = c42 + f24 * c44;
  k.c00 = (m00 + f02 * m02) + f04 * m04;
  k.c10 = (m10 + f02 * m12) + f04 * m14;
  k.c11 = ((m11 + f12 * m12) + f13 * m13) + f14 * m14;
  k.c20 = (m20 + f02 * m22) + f04 * m24;
  k.c21 = ((m21 + f12 * m22) + f13 * m23) + f14 * m24;
  k.c22 = m22 + f24 * m24;
  k.c30 = (c30 + f02 * c32) + f04 * c43;
  k.c31 = ((c31 + f12 * c32) + f13 * c33) + f14 * c43;
  k.c32 = c32 + f24 * c43;
  k.c40 = (c40 + f02 * c42) + f04 * c44;
  k.c41 = ((c41 + f12 * c42) + f13 * c43) + f14 * c44;
  k.c42 = c42 + f24 * c44;
  return true;
}

struct Gain { float si00, si01, si11; };

// Formulas U: innovation covariance inverse by the 2x2 determinant.
__device__ __forceinline__ Gain kf_gain(const KF& k, const FollowConst& F) {
  const float s00 = k.c00 + F.vy, s01 = k.c10, s11 = k.c11 + F.vz;
  const float det = s00 * s11 - s01 * s01;
  const float inv = 1.f / det;
  Gain g;
  g.si00 = s11 * inv;
  g.si01 = -(s01 * inv);
  g.si11 = s00 * inv;
  return g;
}
__device__ __forceinline__ float kf_chi2(const KF& k, const Gain& g, float ym, float zm) {
  const float r0 = ym - k.y, r1 = zm - k.z;
  return ((r0 * r0) * g.si00 + (2.f * (r0 * r1)) * g.si01) + (r1 * r1) * g.si11;
}
// Kalman update; returns true if the leg must stop (|sin phi| left the range).
__device__ __forceinline__ bool kf_update(KF& k, const Gain& g, float ym, float zm, const FollowConst& F) {
  const float r0 = ym - k.y, r1 = zm - k.z;
  const float a00 = k.c00, a01 = k.c10, a02 = k.c20, a03 = k.c30, a04 = k.c40;  // C_i0
  const float a10 = k.c10, a11 = k.c11, a12 = k.c21, a13 = k.c31, a14 = k.c41;  // C_i1
  const float k00 = a00 * g.si00 + a10 * g.si01, k10 = a00 * g.si01 + a10 * g.si11;
  const float k01 = a01 * g.si00 + a11 * g.si01, k11 = a01 * g.si01 + a11 * g.si11;
  const float k02 = a02 * g.si00 + a12 * g.si01, k12 = a02 * g.si01 + a12 * g.si11;
  const float k03 = a03 * g.si00 + a13 * g.si01, k13 = a03 * g.si01 + a13 * g.si11;
  const float k04 = a04 * g.si00 + a14 * g.si01, k14 = a04 * g.si01 + a14 * g.si11;
  k.y = k.y + (k00 * r0 + k10 * r1);
  k.z = k.z + (k01 * r0 + k11 * r1);
  k.s = k.s + (k02 * r0 + k12 * r1);
  k.t = k.t + (k03 * r0 + k13 * r1);
  k.q = k.q + (k04 * r0 + k14 * r1);
  k.c00 = k.c00 - (k00 * a00 + k10 * a10);
  k.c10 = k.c10 - (k01 * a00 + k11 * a10);
  k.c11 = k.c11 - (k01 * a01 + k11 * a11);
  k.c20 = k.c20 - (k02 * a00 + k12 * a10);
  k.c21 = k.c21 - (k02 * a01 + k12 * a11);
  k.c22 = k.c22 - (k02 * a02 + k12 * a12);
  k.c30 = k.c30 - (k03 * a00 + k13 * a10);
  k.c31 = k.c31 - (k03 * a01 + k13 * a11);
  k.c32 = k.c32 - (k03 * a02 + k13 * a12);
  k.c33 = k.c33 - (k03 * a03 + k13 * a13);
  k.c40 = k.c40 - (k04 * a00 + k14 * a10);
  k.c41 = k.c41 - (k04 * a01 + k14 * a11);
  k.c42 = k.c42 - (k04 * a02 + k14 * a12);
  k.c43 = k.c43 - (k04 * a03 + k14 * a13);
  k.c44 = k.c44 - (k04 * a04 + k14 * a14);
  if (k.q > F.max_qpt) k.q = F.max_qpt;
  if (k.q < -F.max_qpt) k.q = -F.max_qpt;
  if (!(fabsf(k.s) <= F.max_sinphi)) {
    k.s = (k.s < 0.f) ? -F.max_sinphi : F.max_sinphi;
    return true;
  }
  return false;
}

__device__ __forceinline__ float clampf(float v, float lo, float hi) { return v < lo ? lo : (v > hi ? hi : v); }

// Row descriptors are read at every row step of every seed: keep their lines in L1/L2.
__device__ __forceinline__ tpc_row_desc ld_row_desc(const tpc_row_desc* p) {
  uint4 a, b;
  asm volatile("ld.global.nc.L1::evict_last.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(a.x), "=r"(a.y), "=r"(a.z), "=r"(a.w) : "l"(p));
  asm volatile("ld.global.nc.L1::evict_last.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(b.x), "=r"(b.y), "=r"(b.z), "=r"(b.w) : "l"(reinterpret_cast<const char*>(p) + 16));
  tpc_row_desc d;
  d.y0 = __uint_as_float(a.x); d.z0 = __uint_as_float(a.y); d.ny = (int)a.z; d.nz = (int)a.w;
  d.bin_ofs = b.x; d.clu_ofs = b.y; d.count = b.z; d.pad_ = b.w;
  return d;
}

__device__ __forceinline__ void prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// R5.3: best cluster of row sr inside the road around the predicted state: minimum of
// (chi2, original id).  Returns the sorted index or -1; *m_out = its (y,z).
// The road is small against the bins, so the window covers one or two z-rows of bins, each a
// contiguous range of the sorted clusters.  The two ranges are walked as ONE flat sequence in
// batches of four: the four loads of a batch are issued together, so a search costs one
// memory round trip for the index and one per batch instead of one per candidate.
__device__ __forceinline__ int32_t pick_cluster(const TpcBuffers& B, const TpcConst* __restrict__ K, uint32_t sr,
                                                const KF& k, const Gain& g, const FollowConst& F, float* chi2_out,
                                                float2* m_out, uint32_t& n_cand) {
  const tpc_row_desc d = ld_row_desc(B.row_desc + sr);
  if (d.count == 0) return -1;
  const float ry = clampf(F.road_nsigma * sqrtf(k.c00 + F.vy), F.road_min, F.road_max);
  const float rz = clampf(F.road_nsigma * sqrtf(k.c11 + F.vz), F.road_min, F.road_max);
  const BinWindow w = make_window(d, K, k.y - ry, k.y + ry, k.z - rz, k.z + rz);
  int32_t best = -1;
  float best_chi2 = 0.f;
  float2 best_m = make_float2(0.f, 0.f);
  const float2* __restrict__ yz = B.yz;
  const uint32_t* __restrict__ bin_start = B.bin_start;
  auto eval = [&](uint32_t c, const float2 m) {
    if (!(fabsf(m.x - k.y) <= ry && fabsf(m.y - k.z) <= rz)) return;
    const float chi2 = kf_chi2(k, g, m.x, m.y);
    ++n_cand;
    bool better = best < 0 || chi2 < best_chi2;
    if (!better && chi2 == best_chi2) better = B.orig_id[c] < B.orig_id[best];  // rule D2, rare
    if (better) { best = (int32_t)c; best_chi2 = chi2; best_m = m; }
  };
  const bool two_rows = w.bz1 > w.bz0;
  const uint32_t bA = w.base + (uint32_t)w.bz0 * (uint32_t)w.ny;
  const uint32_t bB = bA + (uint32_t)w.ny;
  const uint32_t a0 = bin_start[bA], a1 = bin_start[bA + w.by_span];
  uint32_t b0 = 0, b1 = 0;
  if (two_rows) { b0 = bin_start[bB]; b1 = bin_start[bB + w.by_span]; }
  const uint32_t la = a1 - a0, total = la + (b1 - b0), ob = b0 - la;
  for (uint32_t t = 0; t < total; t += 4) {
    const uint32_t c0 = t + (t < la ? a0 : ob);
    const uint32_t c1 = (t + 1) + (t + 1 < la ? a0 : ob);
    const uint32_t c2 = (t + 2) + (t + 2 < la ? a0 : ob);
    const uint32_t c3 = (t + 3) + (t + 3 < la ? a0 : ob);
    const bool h1 = t + 1 < total, h2 = t + 2 < total, h3 = t + 3 < total;
    float2 m0, m1 = best_m, m2 = best_m, m3 = best_m;
    m0 = yz[c0];
    if (h1) m1 = yz[c1];
    if (h2) m2 = yz[c2];
    if (h3) m3 = yz[c3];
    eval(c0, m0);
    if (h1) eval(c1, m1);
    if (h2) eval(c2, m2);
    if (h3) eval(c3, m3);
  }
  for (int bz = w.bz0 + 2; bz <= w.bz1; ++bz) {  // roads taller than two bins (small grid_dz)
    const uint32_t b = w.base + (uint32_t)bz * (uint32_t)w.ny;
    const uint32_t c1 = bin_start[b + w.by_span];
    for (uint32_t c = bin_start[b]; c < c1; ++c) eval(c, yz[c]);
  }
  *chi2_out = best_chi2;
  *m_out = best_m;
  return best;
}

// ------------------------------------------------------------------ follower kernels
// R5 runs as THREE kernels, one per part of the procedure, so that the lanes of a warp are in
// the same part (a lane searching a road next to lanes that only refit recorded hits would
// leave those idle during the search and vice versa):
//   k_follow_up    R5.1 init, R5.2 chain fit, R5.3 outward extrapolation -> row_hit, turn state
//   k_follow_refit R5.4 turn, R5.5 inward refit through the recorded hits -> tracklet, or
//                  hand-over (state in the tracklet record) when the start row is reached
//   k_follow_down  R5.6 inward extrapolation below the start row, R5.7 output
// Each is ONE uniform loop per thread ("one row step per iteration"); a lane whose seed is
// finished claims the next one at once (chunks from a global counter).  Loads are software-
// pipelined one row ahead.  The arithmetic per seed, and its order, are exactly those of
// R5.1-R5.7, so neither the assignment of seeds to lanes nor the split changes a result.
#ifndef TPC_FOLLOW_BLOCK
#define TPC_FOLLOW_BLOCK 128
#endif
// idle lanes of a warp that trigger a refill from the queue: refilling in groups amortises the
// claim and keeps groups of lanes on neighbouring seeds (measured: 1 -> 4 lanes, -3 ms per frame)
#ifndef TPC_REFILL_UP
#define TPC_REFILL_UP 4
#endif
#ifndef TPC_REFILL_REFIT
#define TPC_REFILL_REFIT 4
#endif
#ifndef TPC_REFILL_DOWN
#define TPC_REFILL_DOWN 4
#endif
#ifndef TPC_FOLLOW_CHUNK
#define TPC_FOLLOW_CHUNK 8    // seeds a warp claims at a time: small keeps the seeds in flight close in the list (64 -> 8: -5 ms)
#endif
#define TPC_NO_BIN 0xFFFFFFFFu
#define TPC_TL_PENDING 1u   // tracklet.pad_: handed from the refit to the inward extrapolation

// Claim work items for the idle lanes of a warp (need = this lane is idle).  Returns true
// and the item index if this lane got one.  chunk_next / chunk_end / exhausted are
// warp-uniform.
__device__ __forceinline__ bool queue_claim(uint32_t* counter, uint32_t n_items, int lane, bool need,
                                            uint32_t& chunk_next, uint32_t& chunk_end, bool& exhausted,
                                            uint32_t& item) {
  bool got = false;
  while (!exhausted) {
    const unsigned want = __ballot_sync(0xffffffffu, need && !got);
    if (!want) break;
    if (chunk_next >= chunk_end) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(counter, (uint32_t)TPC_FOLLOW_CHUNK);
      base = __shfl_sync(0xffffffffu, base, 0);
      if (base >= n_items) { exhausted = true; break; }
      chunk_next = base;
      chunk_end = min(base + (uint32_t)TPC_FOLLOW_CHUNK, n_items);
    }
    const uint32_t rank = (uint32_t)__popc(want & ((1u << lane) - 1u));
    const uint32_t avail = chunk_end - chunk_next;
    if (need && !got && rank < avail) { item = chunk_next + rank; got = true; }
    chunk_next += min((uint32_t)__popc(want), avail);
  }
  return got;
}

// Filled on the host and passed BY VALUE as a kernel parameter: the constants then sit in the
// constant bank and cost no registers in the follower loops.
static inline FollowConst follow_const(const TpcConst* K) {
  FollowConst F;
  F.dx = K->dx_row; F.cfield = K->cfield; F.max_sinphi = K->P.max_sinphi; F.max_qpt = K->P.max_qpt;
  F.vy = K->vy; F.vz = K->vz;
  F.road_nsigma = K->P.road_nsigma; F.road_min = K->P.road_min; F.road_max = K->P.road_max;
  F.chi2_max = K->P.chi2_max_hit;
  F.ivs = K->P.init_var_sinphi; F.ivt = K->P.init_var_tanl; F.ivq = K->P.init_var_qpt;
  F.max_gap = K->P.max_gap_follow; F.min_hits = K->P.min_hits_tracklet; F.R = K->n_rows;
  return F;
}

__device__ __forceinline__ void follow_count_work(const TpcBuffers& B, int which, int lane, uint32_t w_step,
                                                  uint32_t w_upd, uint32_t w_cand) {
  w_step = __reduce_add_sync(0xffffffffu, w_step);
  w_cand = __reduce_add_sync(0xffffffffu, w_cand);
  w_upd = __reduce_add_sync(0xffffffffu, w_upd);
  if (lane == 0 && w_step) {
    atomicAdd(&B.cnt->follow_work[which][0], (unsigned long long)w_step);
    atomicAdd(&B.cnt->follow_work[which][1], (unsigned long long)w_upd);
    atomicAdd(&B.cnt->follow_work[which][2], (unsigned long long)w_cand);
  }
}

#define TPC_SAVE_KIN()                                                                                         \
  do {                                                                                                         \
    s_kin[0][tx] = k.y; s_kin[1][tx] = k.z; s_kin[2][tx] = k.s; s_kin[3][tx] = k.t; s_kin[4][tx] = k.q;        \
    s_kin[5][tx] = k.c00; s_kin[6][tx] = k.c10; s_kin[7][tx] = k.c11; s_kin[8][tx] = k.c20;                    \
    s_kin[9][tx] = k.c21; s_kin[10][tx] = k.c22; s_kin[11][tx] = k.c30; s_kin[12][tx] = k.c31;                 \
    s_kin[13][tx] = k.c32; s_kin[14][tx] = k.c33; s_kin[15][tx] = k.c40; s_kin[16][tx] = k.c41;                \
    s_kin[17][tx] = k.c42; s_kin[18][tx] = k.c43; s_kin[19][tx] = k.c44;                                       \
  } while (0)

// R5.7: write the tracklet of seed sd from the state saved at its innermost accepted hit.
// pending: the record is a hand-over to k_follow_down (n_hits is then the raw count).
__device__ __forceinline__ void write_tracklet(const TpcBuffers& B, uint32_t sd, const float (*s_kin)[TPC_FOLLOW_BLOCK],
                                               int tx, float x, float chi2, int nh, int r_in, int r_out, uint32_t start,
                                               uint32_t sector, int min_hits, bool pending, uint32_t& n_tl) {
  tpc_tracklet t;
  t.x = x;
#pragma unroll
  for (int i = 0; i < 5; ++i) t.p[i] = s_kin[i][tx];
#pragma unroll
  for (int i = 0; i < 15; ++i) t.c[i] = s_kin[5 + i][tx];
  t.chi2 = chi2;
  t.seed_sorted = start;
  t.seed_id = B.orig_id[start];
  const bool keep = nh >= min_hits;
  t.n_hits = (pending || keep) ? (int16_t)nh : (int16_t)0;
  t.row_first = (uint8_t)r_in;
  t.row_last = (uint8_t)r_out;
  t.sector = (uint8_t)sector;
  t.seed_len = B.seed_len[start];
  t.pad_ = pending ? (uint16_t)TPC_TL_PENDING : (uint16_t)0;
  t.pad2_[0] = 0; t.pad2_[1] = 0;
  B.tracklets[sd] = t;
  if (!pending && keep) ++n_tl;   // summed per warp at the end of the kernel (no contended atomic here)
}

// resident CTAs per SM the register budgets are sized for (measured on the C4 frame: fewer,
// fatter CTAs are better for the outward pass, the other two take 6)
#ifndef TPC_FOLLOW_UP_MINBLOCKS
#define TPC_FOLLOW_UP_MINBLOCKS 5
#endif
#ifndef TPC_FOLLOW_DOWN_MINBLOCKS
#define TPC_FOLLOW_DOWN_MINBLOCKS 6
#endif
#ifndef TPC_FOLLOW_REFIT_MINBLOCKS
#define TPC_FOLLOW_REFIT_MINBLOCKS 6
#endif

// ---- R5.1-R5.3: init, chain fit, outward extrapolation
__global__ void __launch_bounds__(TPC_FOLLOW_BLOCK, TPC_FOLLOW_UP_MINBLOCKS) k_follow_up(TpcBuffers B, const __grid_constant__ FollowConst F) {
  __shared__ float s_ylim[TPC_MAX_ROWS];
  const TpcConst* __restrict__ K = B.K;
  for (int r = threadIdx.x; r < K->n_rows; r += blockDim.x) s_ylim[r] = K->ylim[r];
  __syncthreads();
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const float inv_dy = K->inv_dy, inv_dz = K->inv_dz;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const int32_t* __restrict__ up2 = B.link_up2;
  const float2* __restrict__ yz = B.yz;
  const uint32_t* __restrict__ bin_start = B.bin_start;
  const int lane = threadIdx.x & 31;
  uint32_t w_step = 0, w_cand = 0, w_upd = 0;  // work counters (diagnostics only)
  uint32_t chunk_next = 0, chunk_end = 0;      // warp-uniform: the chunk of seeds this warp draws from
  bool exhausted = false;

  enum { PH_CHAIN = 0, PH_UP = 1, PH_IDLE = 2 };
  int phase = PH_IDLE;
  KF k;
  k.y = k.z = k.s = k.t = k.q = 0.f;
  kf_init_cov(k, F);
  uint32_t sd = 0, sr_base = 0;
  int32_t* __restrict__ hit_row = B.row_hit;  // this seed's row -> sorted index table
  int r = 0, r_out = 0, gap = 0, chain_n = 0;
  float snap_s = 0.f, snap_t = 0.f, snap_q = 0.f, snap_y = 0.f, snap_z = 0.f;
  int32_t c_cur = -1, c_nxt = -1;   // chain hit of the coming row and the one after it
  float2 m_cur = make_float2(0.f, 0.f);
  uint32_t pb = TPC_NO_BIN;         // first cluster of the predicted bin on the coming row

  for (;;) {
    if (__popc(__ballot_sync(0xffffffffu, phase == PH_IDLE)) >= TPC_REFILL_UP) {
      uint32_t item = 0;
      if (queue_claim(&B.cnt->follow_next[0], n_seeds, lane, phase == PH_IDLE, chunk_next, chunk_end, exhausted,
                      item)) {
        // ---- R5.1 init from the first two chain clusters
        sd = item;
        const uint32_t start = B.seeds[sd];
        const uint32_t sr0 = B.seed_sr[sd];
        const int r0 = (int)(sr0 % (uint32_t)F.R);
        sr_base = sr0 - (uint32_t)r0;
        hit_row = B.row_hit + (size_t)sd * (size_t)F.R;
        const int32_t c1 = up2[start];
        const float2 m0 = yz[start];
        const float2 m1 = yz[c1];
        c_nxt = up2[c1];
        const float dy = m1.x - m0.x;
        const float dl = sqrtf(F.dx * F.dx + dy * dy);
        k.y = m0.x; k.z = m0.y;
        k.s = dy / dl;
        k.t = (m1.y - m0.y) / dl;
        k.q = 0.f;
        kf_init_cov(k, F);
        hit_row[r0] = (int32_t)start;
        r = r0; r_out = r0;
        snap_s = k.s; snap_t = k.t; snap_q = k.q; snap_y = m0.x; snap_z = m0.y;
        gap = 0;
        c_cur = c1; m_cur = m1;
        chain_n = 1;
        pb = TPC_NO_BIN;
        phase = PH_CHAIN;
      }
      if (__all_sync(0xffffffffu, phase == PH_IDLE)) break;  // nothing left for this warp
    }
    if (phase != PH_IDLE) {
      const bool extrap = phase == PH_UP;
      const int rn = r + 1;
      bool fin = false;
      if (rn >= F.R) {
        fin = true;  // ran off the pad plane
      } else {
        ++w_step;
        const float y_prev = k.y, z_prev = k.z;
        if (!kf_propagate(k, F.dx, F)) {
          fin = true;  // the leg left the |sin phi| range
        } else {
          r = rn;
          // ---- request the next row's data while this row is computed
          int32_t c_nxt2 = -1;
          float2 m_nxt = make_float2(0.f, 0.f);
          if (extrap) {
            // two rows ahead: the bin index entry of row r+2 is requested now, the clusters of
            // row r+1 (entry requested one step ago) are pulled into L1 now
            if (pb != TPC_NO_BIN) prefetch_l1(yz + pb);
            pb = TPC_NO_BIN;
            if (r + 2 < F.R) {
              const tpc_row_desc dn = ld_row_desc(B.row_desc + sr_base + (uint32_t)(r + 2));
              if (dn.count) {  // linear continuation of this step
                const int by = bin_coord(k.y + 2.f * (k.y - y_prev), dn.y0, inv_dy, dn.ny);
                const int bz = bin_coord(k.z + 2.f * (k.z - z_prev), dn.z0, inv_dz, dn.nz);
                pb = bin_start[dn.bin_ofs + (uint32_t)bz * (uint32_t)dn.ny + (uint32_t)by];
              }
            }
          } else if (c_nxt >= 0) {
            m_nxt = yz[c_nxt];
            c_nxt2 = up2[c_nxt];
          }
          const Gain g = kf_gain(k, F);
          int32_t c = -1;
          float chi2h = 0.f;
          float2 m = m_cur;
          if (!extrap) {
            c = c_cur;                                    // R5.2: chain hit, no chi2 cut
          } else if (fabsf(k.y) <= s_ylim[r]) {           // R5.3: road search
            c = pick_cluster(B, K, sr_base + (uint32_t)r, k, g, F, &chi2h, &m, w_cand);
            if (!(c >= 0 && chi2h <= F.chi2_max)) c = -1;
          }
          if (c >= 0) {
            const bool stop = kf_update(k, g, m.x, m.y, F);
            ++w_upd;
            hit_row[r] = c;
            r_out = r;
            snap_s = k.s; snap_t = k.t; snap_q = k.q; snap_y = m.x; snap_z = m.y;
            gap = 0;
            if (stop) fin = true;
          } else if (extrap) {
            hit_row[r] = -1;
            ++gap;
            if (gap > F.max_gap) fin = true;
          }
          if (!extrap) { c_cur = c_nxt; m_cur = m_nxt; c_nxt = c_nxt2; ++chain_n; }
        }
      }
      if (phase == PH_CHAIN && (fin || c_cur < 0)) {
        // chain length of the seed (R4): hits fitted so far + links not reached when the leg
        // ended inside the chain
        int n_chain = chain_n;
        for (int32_t c = c_cur; c >= 0; c = up2[c]) ++n_chain;
        B.seed_len[B.seeds[sd]] = (uint8_t)n_chain;
      }
      if (fin) {
        // state for R5.4 (turn at the outermost accepted hit)
        B.turn[2 * (size_t)sd] = make_uint4(__float_as_uint(snap_y), __float_as_uint(snap_z), __float_as_uint(snap_s),
                                            __float_as_uint(snap_t));
        B.turn[2 * (size_t)sd + 1] = make_uint4(__float_as_uint(snap_q), (uint32_t)r_out, 0u, 0u);
        phase = PH_IDLE;
      } else if (phase == PH_CHAIN && c_cur < 0) {
        phase = PH_UP; gap = 0; pb = TPC_NO_BIN;  // chain fitted
      }
    }
  }
  follow_count_work(B, 0, lane, w_step, w_upd, w_cand);
}

// ---- R5.4-R5.5: turn at the outermost accepted hit, refit inward through the recorded hits
__global__ void __launch_bounds__(TPC_FOLLOW_BLOCK, TPC_FOLLOW_REFIT_MINBLOCKS) k_follow_refit(TpcBuffers B, const __grid_constant__ FollowConst F) {
  __shared__ float s_x[TPC_MAX_ROWS];
  __shared__ float s_kin[20][TPC_FOLLOW_BLOCK];  // state at the innermost accepted hit (R5.7)
  const TpcConst* __restrict__ K = B.K;
  for (int r = threadIdx.x; r < K->n_rows; r += blockDim.x) s_x[r] = K->x[r];
  __syncthreads();
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const float2* __restrict__ yz = B.yz;
  const int lane = threadIdx.x & 31;
  const int tx = threadIdx.x;
  uint32_t w_step = 0, w_upd = 0, n_tl = 0;
  uint32_t chunk_next = 0, chunk_end = 0;
  bool exhausted = false;

  bool active = false;
  KF k;
  k.y = k.z = k.s = k.t = k.q = 0.f;
  kf_init_cov(k, F);
  uint32_t sd = 0, start = 0, sector = 0;
  const int32_t* __restrict__ hit_row = B.row_hit;
  int r = 0, r0 = 0, r_out = 0, r_in = 0, nh = 0;
  float chi2 = 0.f;
  int32_t c_cur = -1, c_nxt = -1;   // recorded hit of the coming row and of the one after it
  float2 m_cur = make_float2(0.f, 0.f);

  for (;;) {
    if (__popc(__ballot_sync(0xffffffffu, !active)) >= TPC_REFILL_REFIT) {
      uint32_t item = 0;
      if (queue_claim(&B.cnt->follow_next[1], n_seeds, lane, !active, chunk_next, chunk_end, exhausted, item)) {
        // ---- R5.4 turn: (y,z) of the outermost hit, (s,t,q) as they were after its update,
        // covariance back to the initial diagonal
        sd = item;
        start = B.seeds[sd];
        const uint32_t sr0 = B.seed_sr[sd];
        r0 = (int)(sr0 % (uint32_t)F.R);
        sector = sr0 / (uint32_t)F.R;
        hit_row = B.row_hit + (size_t)sd * (size_t)F.R;
        const uint4 t0 = B.turn[2 * (size_t)sd], t1 = B.turn[2 * (size_t)sd + 1];
        k.y = __uint_as_float(t0.x); k.z = __uint_as_float(t0.y);
        k.s = __uint_as_float(t0.z); k.t = __uint_as_float(t0.w); k.q = __uint_as_float(t1.x);
        r_out = (int)t1.y;
        kf_init_cov(k, F);
        chi2 = 0.f; nh = 1; r_in = r_out; r = r_out;
        TPC_SAVE_KIN();
        c_cur = -1; c_nxt = -1;
        if (r_out > r0) {
          c_cur = hit_row[r_out - 1];
          c_nxt = (r_out - 2 >= r0) ? hit_row[r_out - 2] : -1;
          if (c_cur >= 0) m_cur = yz[c_cur];
        }
        active = true;
      }
      if (__all_sync(0xffffffffu, !active)) break;
    }
    if (active) {
      bool fin = false;      // the leg ended inside the refit: the tracklet is complete
      if (r > r0) {
        ++w_step;
        if (!kf_propagate(k, -F.dx, F)) {
          fin = true;
        } else {
          --r;
          int32_t c_nxt2 = -1;
          float2 m_nxt = make_float2(0.f, 0.f);
          if (c_nxt >= 0) m_nxt = yz[c_nxt];
          if (r - 2 >= r0) c_nxt2 = hit_row[r - 2];
          if (c_cur >= 0) {     // R5.5: recorded hit (rows without one are pure propagation)
            const Gain g = kf_gain(k, F);
            const float chi2h = kf_chi2(k, g, m_cur.x, m_cur.y);
            const bool stop = kf_update(k, g, m_cur.x, m_cur.y, F);
            ++w_upd;
            chi2 = chi2 + chi2h;
            ++nh;
            r_in = r;
            TPC_SAVE_KIN();
            if (stop) fin = true;
          }
          c_cur = c_nxt; m_cur = m_nxt; c_nxt = c_nxt2;
        }
      }
      if (fin) {
        // (hits below r_in are outside [row_first,row_last] and thereby not part of the tracklet)
        write_tracklet(B, sd, s_kin, tx, s_x[r_in], chi2, nh, r_in, r_out, start, sector, F.min_hits, false, n_tl);
        active = false;
      } else if (r == r0) {
        // the start row is reached (its hit is always present, so the saved state is the live one)
        const bool pending = r0 > 0;   // rows below to extrapolate into
        write_tracklet(B, sd, s_kin, tx, s_x[r_in], chi2, nh, r_in, r_out, start, sector, F.min_hits, pending, n_tl);
        active = false;
      }
    }
  }
  follow_count_work(B, 1, lane, w_step, w_upd, 0u);
  n_tl = __reduce_add_sync(0xffffffffu, n_tl);
  if (lane == 0 && n_tl) atomicAdd(&B.cnt->n_tracklets, n_tl);
}

// ---- R5.6-R5.7: inward extrapolation below the start row, output
__global__ void __launch_bounds__(TPC_FOLLOW_BLOCK, TPC_FOLLOW_DOWN_MINBLOCKS) k_follow_down(TpcBuffers B, const __grid_constant__ FollowConst F) {
  __shared__ float s_ylim[TPC_MAX_ROWS];
  __shared__ float s_x[TPC_MAX_ROWS];
  __shared__ float s_kin[20][TPC_FOLLOW_BLOCK];
  const TpcConst* __restrict__ K = B.K;
  for (int r = threadIdx.x; r < K->n_rows; r += blockDim.x) { s_ylim[r] = K->ylim[r]; s_x[r] = K->x[r]; }
  __syncthreads();
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const float inv_dy = K->inv_dy, inv_dz = K->inv_dz;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const float2* __restrict__ yz = B.yz;
  const uint32_t* __restrict__ bin_start = B.bin_start;
  const int lane = threadIdx.x & 31;
  const int tx = threadIdx.x;
  uint32_t w_step = 0, w_cand = 0, w_upd = 0, n_tl = 0;
  uint32_t chunk_next = 0, chunk_end = 0;
  bool exhausted = false;

  bool active = false;
  KF k;
  k.y = k.z = k.s = k.t = k.q = 0.f;
  kf_init_cov(k, F);
  uint32_t sd = 0, start = 0, sr_base = 0;
  int32_t* __restrict__ hit_row = B.row_hit;
  int r = 0, r_out = 0, r_in = 0, gap = 0, nh = 0;
  float chi2 = 0.f;
  uint32_t pb = TPC_NO_BIN;

  for (;;) {
    if (__popc(__ballot_sync(0xffffffffu, !active)) >= TPC_REFILL_DOWN) {
      uint32_t item = 0;
      // seeds are taken in LIST order (not in the order the refit finished them): the lanes of a
      // warp then hold seeds of the same (sector, z-slab, row), walk the same rows and read
      // neighbouring bins
      if (queue_claim(&B.cnt->follow_next[2], n_seeds, lane, !active, chunk_next, chunk_end, exhausted, item) &&
          B.tracklets[item].pad_ == (uint16_t)TPC_TL_PENDING) {
        sd = item;
        const tpc_tracklet* __restrict__ t = B.tracklets + sd;
        k.y = t->p[0]; k.z = t->p[1]; k.s = t->p[2]; k.t = t->p[3]; k.q = t->p[4];
        k.c00 = t->c[0]; k.c10 = t->c[1]; k.c11 = t->c[2]; k.c20 = t->c[3]; k.c21 = t->c[4]; k.c22 = t->c[5];
        k.c30 = t->c[6]; k.c31 = t->c[7]; k.c32 = t->c[8]; k.c33 = t->c[9];
        k.c40 = t->c[10]; k.c41 = t->c[11]; k.c42 = t->c[12]; k.c43 = t->c[13]; k.c44 = t->c[14];
        chi2 = t->chi2; nh = t->n_hits; start = t->seed_sorted;
        r = r_in = t->row_first; r_out = t->row_last;
        sr_base = (uint32_t)t->sector * (uint32_t)F.R;
        hit_row = B.row_hit + (size_t)sd * (size_t)F.R;
        TPC_SAVE_KIN();
        gap = 0;
        pb = TPC_NO_BIN;
        active = true;
      }
      if (__all_sync(0xffffffffu, !active)) break;
    }
    if (active) {
      const int rn = r - 1;
      bool fin = false;
      if (pb != TPC_NO_BIN) prefetch_l1(yz + pb);
      if (rn < 0) {
        fin = true;
      } else {
        ++w_step;
        const float y_prev = k.y, z_prev = k.z;
        if (!kf_propagate(k, -F.dx, F)) {
          fin = true;
        } else {
          r = rn;
          pb = TPC_NO_BIN;   // (inward legs are short: one row ahead measured better than two)
          if (r - 1 >= 0) {
            const tpc_row_desc dn = ld_row_desc(B.row_desc + sr_base + (uint32_t)(r - 1));
            if (dn.count) {
              const int by = bin_coord(k.y + (k.y - y_prev), dn.y0, inv_dy, dn.ny);
              const int bz = bin_coord(k.z + (k.z - z_prev), dn.z0, inv_dz, dn.nz);
              pb = bin_start[dn.bin_ofs + (uint32_t)bz * (uint32_t)dn.ny + (uint32_t)by];
            }
          }
          int32_t c = -1;
          float chi2h = 0.f;
          float2 m = make_float2(0.f, 0.f);
          const Gain g = kf_gain(k, F);
          if (fabsf(k.y) <= s_ylim[r]) {                  // R5.6: road search
            c = pick_cluster(B, K, sr_base + (uint32_t)r, k, g, F, &chi2h, &m, w_cand);
            if (!(c >= 0 && chi2h <= F.chi2_max)) c = -1;
          }
          if (c >= 0) {
            const bool stop = kf_update(k, g, m.x, m.y, F);
            ++w_upd;
            hit_row[r] = c;
            chi2 = chi2 + chi2h;
            ++nh;
            r_in = r;
            TPC_SAVE_KIN();
            gap = 0;
            if (stop) fin = true;
          } else {
            hit_row[r] = -1;
            ++gap;
            if (gap > F.max_gap) fin = true;
          }
        }
      }
      if (fin) {
        write_tracklet(B, sd, s_kin, tx, s_x[r_in], chi2, nh, r_in, r_out, start, sr_base / (uint32_t)F.R, F.min_hits,
                       false, n_tl);
        active = false;
      }
    }
  }
  follow_count_work(B, 2, lane, w_step, w_upd, w_cand);
  n_tl = __reduce_add_sync(0xffffffffu, n_tl);
  if (lane == 0 && n_tl) atomicAdd(&B.cnt->n_tracklets, n_tl);
}

// ================================================================== K5 ambiguity solving
// PAPER.md:27 ("identifies the best instance of each track, assigns all clusters to this
// instance and removes the clones"; 10 % shared by default) with the Phase-I criterion of
// PAPER.md:57 (chi2 priority; shared clusters counted from the outermost pad row).  R6.
// Layout of the work: everything that touches memory per (tracklet,row) runs with one WARP
// per tracklet and the lanes across its rows (coalesced row_hit reads, 32 independent
// gathers / atomics in flight per warp); the sequential walk of R6.3 runs with one THREAD per
// tracklet on two bit masks in registers (row has a hit / the hit is owned) and touches no
// memory inside its loop.
#define TPC_MASK_WORDS (TPC_MAX_ROWS / 32)   // mask stride per tracklet / track, in words

__global__ void __launch_bounds__(256) k_zero_owner(TpcBuffers B) {
  const uint32_t n = B.cnt->n_sorted;  // owner[] is indexed by sorted position
  uint4* p4 = reinterpret_cast<uint4*>(B.owner);
  const uint32_t n2 = (n + 1) / 2;      // the buffer is padded to 256 bytes
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n2; i += gridDim.x * blockDim.x)
    p4[i] = make_uint4(0, 0, 0, 0);
}

// K5a / K5b work on TILES of 32 consecutive tracklets of the seed list (one CTA per tile at a
// time, lane = tracklet, the 8 warps share the rows in groups of four: one 16-byte load per
// lane, the other half of each sector is read by the next warp).  The tracklets of a tile (and
// of the tiles that run at the same time) come from the same z-slab of one sector and are
// processed row by row, so their owner words sit in a few KB per row and stay in L2.  The per-row ballots are transposed through shared
// memory into per-tracklet row masks, stored [word][tracklet].
#ifndef TPC_SEL_BLOCK
#define TPC_SEL_BLOCK 256
#endif
#define TPC_SEL_UNROLL 4   // rows per load: row_hit rows are 16-byte aligned when n_rows % 4 == 0

// hits of rows rb..rb+3 of one tracklet (p = its row_hit row), -1 where `want` is false
__device__ __forceinline__ void load_hits4(const int32_t* __restrict__ p, int rb, int R, bool vec, const bool (&want)[4],
                                           int32_t (&c)[4]) {
  c[0] = c[1] = c[2] = c[3] = -1;
  if (!(want[0] || want[1] || want[2] || want[3])) return;
  if (vec) {
    const int4 v = __ldcs(reinterpret_cast<const int4*>(p + rb));
    if (want[0]) c[0] = v.x;
    if (want[1]) c[1] = v.y;
    if (want[2]) c[2] = v.z;
    if (want[3]) c[3] = v.w;
  } else {
#pragma unroll
    for (int u = 0; u < 4; ++u) if (want[u] && rb + u < R) c[u] = __ldcs(p + rb + u);
  }
}

__device__ __forceinline__ unsigned long long tracklet_key(const tpc_tracklet* __restrict__ t, float w) {
  const int nh = t->n_hits;
  if (nh <= 0) return 0ull;
  const int ndf = 2 * nh - 5;
  const float Q = (float)nh - w * (t->chi2 / (float)ndf);
  return ((unsigned long long)f2key(Q) << 32) | (unsigned long long)(0xFFFFFFFFu - t->seed_id);
}

// bits[r] holds, for row r, one bit per tracklet of the tile -> word w of tracklet `lane`
__device__ __forceinline__ uint32_t transpose_rows(const uint32_t* __restrict__ bits, int w, int lane, int R) {
  uint32_t m = 0u;
#pragma unroll 8
  for (int b = 0; b < 32; ++b) {
    const int r = w * 32 + b;
    if (r < R) m |= ((bits[r] >> lane) & 1u) << b;
  }
  return m;
}

// K5a (R6.1, R6.2): weight -> 64-bit key; per-cluster owner = max key (64-bit atomicMax).
// Also writes, per tracklet, the mask of rows with a hit and the mask of rows where this
// tracklet's key was the maximum when it looked ("tentative": only those can still be owned
// at the end, a hit that lost once has lost for good because owner words only grow).
__global__ void __launch_bounds__(TPC_SEL_BLOCK) k_sel_owner(TpcBuffers B) {
  __shared__ unsigned long long s_key[32];
  __shared__ int s_r0[32], s_r1[32];
  __shared__ uint32_t s_has[TPC_MAX_ROWS], s_tent[TPC_MAX_ROWS];
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const int R = B.K->n_rows;
  const int W = (R + 31) >> 5;
  const float w = B.K->P.sel_chi2_weight;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t hstride = B.max_seeds;
  const uint32_t n_tiles = (n_seeds + 31u) >> 5;
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t sd = tile * 32u + (uint32_t)lane;
    __syncthreads();   // the previous tile is done with the shared arrays
    if (warp == 0) {
      unsigned long long key = 0ull;
      int r0 = 0x7fffffff, r1 = -1;
      if (sd < n_seeds) {
        const tpc_tracklet* __restrict__ t = B.tracklets + sd;
        key = tracklet_key(t, w);
        if (key) { r0 = t->row_first; r1 = t->row_last; }
        B.tl_key[sd] = key;
      }
      s_key[lane] = key; s_r0[lane] = r0; s_r1[lane] = r1;
    }
    for (int r = threadIdx.x; r < R; r += TPC_SEL_BLOCK) { s_has[r] = 0u; s_tent[r] = 0u; }
    __syncthreads();
    const unsigned long long key = s_key[lane];
    const int r0 = s_r0[lane], r1 = s_r1[lane];
    const int t0 = __reduce_min_sync(0xffffffffu, r0), t1 = __reduce_max_sync(0xffffffffu, r1);
    // a tile without a single accepted tracklet (t0 = INT_MAX, t1 = -1: e.g. 32 consecutive short
    // stubs) has no rows to visit and no masks to write; CTA-uniform, the next iteration's first
    // barrier is the only one skipped ahead of
    if (t1 < 0) continue;
    const int32_t* __restrict__ hits = B.row_hit + (size_t)sd * (size_t)R;
    const bool vec = (R & 3) == 0;
    // two row groups per iteration: eight independent hit -> owner chains in flight per lane
    constexpr int kStride = (TPC_SEL_BLOCK / 32) * TPC_SEL_UNROLL;
    for (int rb0 = (t0 & ~3) + warp * TPC_SEL_UNROLL; rb0 <= t1; rb0 += 2 * kStride) {
      int32_t c[2][TPC_SEL_UNROLL];
      unsigned long long o[2][TPC_SEL_UNROLL];
#pragma unroll
      for (int g = 0; g < 2; ++g) {
        const int rb = rb0 + g * kStride;
        bool want[TPC_SEL_UNROLL];
#pragma unroll
        for (int u = 0; u < TPC_SEL_UNROLL; ++u) want[u] = rb + u >= r0 && rb + u <= r1;
        load_hits4(hits, rb, R, vec && rb + 3 < R, want, c[g]);
      }
#pragma unroll
      for (int g = 0; g < 2; ++g)
#pragma unroll
        for (int u = 0; u < TPC_SEL_UNROLL; ++u) o[g][u] = c[g][u] >= 0 ? __ldcg(&B.owner[c[g][u]]) : ~0ull;
#pragma unroll
      for (int g = 0; g < 2; ++g) {
        const int rb = rb0 + g * kStride;
#pragma unroll
        for (int u = 0; u < TPC_SEL_UNROLL; ++u) {
          // read first: most hits lose against the current owner and then need no atomic
          const bool tent = o[g][u] < key;
          if (tent) atomicMax(&B.owner[c[g][u]], key);
          const uint32_t hm = __ballot_sync(0xffffffffu, c[g][u] >= 0);
          const uint32_t tm = __ballot_sync(0xffffffffu, tent);
          if (lane == 0 && rb + u < R) { s_has[rb + u] = hm; s_tent[rb + u] = tm; }
        }
      }
    }
    __syncthreads();
    if (warp < W && sd < n_seeds && key) {
      B.tl_mask[(size_t)warp * hstride + sd] = transpose_rows(s_has, warp, lane, R);
      B.tl_mask[(size_t)(TPC_MASK_WORDS + warp) * hstride + sd] = transpose_rows(s_tent, warp, lane, R);
    }
  }
}

// K5b: "the hit is owned" mask of R6.3: the tentative rows whose owner word still is this
// tracklet's key once all tracklets have been through K5a.
__global__ void __launch_bounds__(TPC_SEL_BLOCK) k_sel_masks(TpcBuffers B) {
  __shared__ uint32_t s_tw[TPC_MASK_WORDS][32];   // tentative words of the tile's tracklets
  __shared__ uint32_t s_own[TPC_MAX_ROWS];
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const int R = B.K->n_rows;
  const int W = (R + 31) >> 5;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t hstride = B.max_seeds;
  const uint32_t n_tiles = (n_seeds + 31u) >> 5;
  for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const uint32_t sd = tile * 32u + (uint32_t)lane;
    const unsigned long long key = sd < n_seeds ? B.tl_key[sd] : 0ull;
    __syncthreads();
    if (warp < W) s_tw[warp][lane] = key ? B.tl_mask[(size_t)(TPC_MASK_WORDS + warp) * hstride + sd] : 0u;
    for (int r = threadIdx.x; r < R; r += TPC_SEL_BLOCK) s_own[r] = 0u;
    __syncthreads();
    // a tracklet whose tentative hits are too few for any segment (the bound of walk_tracklet;
    // owned hits are a subset of the tentative ones) is not looked at: its owned mask is left
    // empty, which the count pass rejects by the same bound
    if (warp == 0) {
      int n_tent = 0;
      for (int w = 0; w < W; ++w) n_tent += __popc(s_tw[w][lane]);
      const tpc_params& P = B.K->P;
      const bool hopeless = P.shared_fixed_cap
                                ? n_tent * 1000 + P.shared_permille * (int)(sd < n_seeds ? B.tracklets[sd].n_hits : 0) < P.min_hits_track * 1000
                                : n_tent * 1000 < P.min_hits_track * (1000 - P.shared_permille);
      if (hopeless)
        for (int w = 0; w < W; ++w) s_tw[w][lane] = 0u;
    }
    __syncthreads();
    const int32_t* __restrict__ hits = B.row_hit + (size_t)sd * (size_t)R;
    const bool vec = (R & 3) == 0;
    for (int rb = warp * TPC_SEL_UNROLL; rb < R; rb += (TPC_SEL_BLOCK / 32) * TPC_SEL_UNROLL) {
      int32_t c[TPC_SEL_UNROLL];
      bool own[TPC_SEL_UNROLL];
      bool want[TPC_SEL_UNROLL];
      bool any = false;
#pragma unroll
      for (int u = 0; u < TPC_SEL_UNROLL; ++u) {
        const int r = rb + u;
        want[u] = r < R && ((s_tw[r >> 5][lane] >> (r & 31)) & 1u);
        any |= want[u];
      }
      if (!__any_sync(0xffffffffu, any)) continue;
      load_hits4(hits, rb, R, vec, want, c);
#pragma unroll
      for (int u = 0; u < TPC_SEL_UNROLL; ++u) own[u] = c[u] >= 0 && __ldcg(&B.owner[c[u]]) == key;
#pragma unroll
      for (int u = 0; u < TPC_SEL_UNROLL; ++u) {
        const uint32_t om = __ballot_sync(0xffffffffu, own[u]);
        if (lane == 0 && rb + u < R) s_own[rb + u] = om;
      }
    }
    __syncthreads();
    if (warp < W && key) B.tl_mask[(size_t)(TPC_MASK_WORDS + warp) * hstride + sd] = transpose_rows(s_own, warp, lane, R);
  }
}

// The walk of R6.3 on the two masks: from the outermost row inward with the running shared
// budget; segments split at holes > max_gap_select; EMIT=false counts, EMIT=true writes the
// track records and, per track, the masks of its accepted / shared rows (k_sel_ids turns
// them into cluster lists).
template <bool EMIT>
__device__ __forceinline__ void walk_tracklet(const TpcBuffers& B, uint32_t sd, uint32_t& n_seg_out, uint32_t& n_id_out,
                                              uint32_t trk_ofs, uint32_t id_ofs) {
  const tpc_params& P = B.K->P;
  const tpc_tracklet& tl = B.tracklets[sd];
  const int r0 = tl.row_first, r1 = tl.row_last;
  const int min_hits = P.min_hits_track, max_gap = P.max_gap_select;
  const int permille = P.shared_permille;
  const bool fixed_cap = P.shared_fixed_cap != 0;   // variant: the rule before Phase I
  const int R = B.K->n_rows;
  uint32_t has[TPC_MASK_WORDS], own[TPC_MASK_WORDS], acc[TPC_MASK_WORDS], shm[TPC_MASK_WORDS];
#pragma unroll
  for (int w = 0; w < TPC_MASK_WORDS; ++w) {
    has[w] = 0u; own[w] = 0u; acc[w] = 0u; shm[w] = 0u;
    if (w * 32 < R) {
      has[w] = B.tl_mask[(size_t)w * B.max_seeds + sd];                      // [word][tracklet]
      own[w] = B.tl_mask[(size_t)(TPC_MASK_WORDS + w) * B.max_seeds + sd];
    }
  }
  int n_acc = 0, n_sh = 0, gap = 0, seg_last = -1, seg_first = -1;
  uint32_t n_seg = 0, n_id = 0;
  if (!EMIT) {
    // A segment holds at least (1 - shared fraction) owned hits at every moment of the walk
    // (running rule of R6.3), so a tracklet that owns too few hits cannot reach min_hits_track
    // in any segment: most clone instances leave here.
    int n_own = 0;
#pragma unroll
    for (int w = 0; w < TPC_MASK_WORDS; ++w) n_own += __popc(own[w]);
    if (fixed_cap ? n_own * 1000 + permille * (int)tl.n_hits < min_hits * 1000
                  : n_own * 1000 < min_hits * (1000 - permille)) { n_seg_out = 0; n_id_out = 0; return; }
  }
  auto close = [&]() {
    if (n_acc >= min_hits) {
      if (EMIT) {
        const uint32_t ti = trk_ofs + n_seg;
#pragma unroll
        for (int w = 0; w < TPC_MASK_WORDS; ++w) {
          if (w * 32 < R) {
            B.trk_mask[(size_t)ti * (2 * TPC_MASK_WORDS) + w] = acc[w];
            B.trk_mask[(size_t)ti * (2 * TPC_MASK_WORDS) + TPC_MASK_WORDS + w] = shm[w];
          }
        }
        B.trk_sd[ti] = sd;
        tpc_track t;
        t.x = tl.x;
#pragma unroll
        for (int i = 0; i < 5; ++i) t.p[i] = tl.p[i];
#pragma unroll
        for (int i = 0; i < 15; ++i) t.c[i] = tl.c[i];
        t.chi2 = tl.chi2;
        t.cluster_ofs = id_ofs + n_id;
        t.seed_id = tl.seed_id;
        t.n_clusters = (uint16_t)n_acc;
        t.n_shared = (uint16_t)n_sh;
        t.sector = tl.sector;
        t.row_first = (uint8_t)seg_first;
        t.row_last = (uint8_t)seg_last;
        t.flags = (seg_first == r0) ? 0 : TPC_TRACK_PARAMS_STALE;
        t.n_hits_tracklet = (uint16_t)tl.n_hits;
        t.segment = (uint8_t)n_seg;
        t.pad_ = 0;
        B.tracks[ti] = t;
      }
      ++n_seg;
      n_id += (uint32_t)n_acc;
    }
    if (EMIT) {
#pragma unroll
      for (int w = 0; w < TPC_MASK_WORDS; ++w) { acc[w] = 0u; shm[w] = 0u; }
    }
    n_acc = 0; n_sh = 0; seg_last = -1; seg_first = -1;
  };
#pragma unroll
  for (int w = TPC_MASK_WORDS - 1; w >= 0; --w) {
    if (w * 32 > r1 || w * 32 + 31 < r0) continue;
    const int b_hi = min(31, r1 - w * 32), b_lo = max(0, r0 - w * 32);
    const uint32_t hw = has[w], ow = own[w];
    for (int b = b_hi; b >= b_lo; --b) {
      const int r = w * 32 + b;
      bool c = (hw >> b) & 1u;
      bool sh = false;
      if (c && !((ow >> b) & 1u)) {
        if ((n_sh + 1) * 1000 <= (fixed_cap ? permille * (int)tl.n_hits : permille * (n_acc + 1))) sh = true;
        else c = false;
      }
      if (c) {
        if (n_acc == 0) seg_last = r;
        seg_first = r;
        if (EMIT) {
          acc[w] |= 1u << b;
          if (sh) shm[w] |= 1u << b;
        }
        ++n_acc;
        if (sh) ++n_sh;
        gap = 0;
      } else {
        ++gap;
        if (gap > max_gap && n_acc > 0) close();
      }
    }
  }
  close();
  n_seg_out = n_seg;
  n_id_out = n_id;
}

// K5c: count tracks / cluster ids per tracklet + per-block partial sums (for the scans).
__global__ void __launch_bounds__(256) k_sel_count(TpcBuffers B) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_ns[256], s_ni[256];
  __shared__ uint16_t s_list[256];
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS)) return;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const uint32_t n_blocks = (n_seeds + blockDim.x - 1) / blockDim.x;
  uint32_t* part_seg = B.scan_partials;
  uint32_t* part_id = B.scan_partials + (B.scan_blocks + 1) / 2;
  for (uint32_t blk = blockIdx.x; blk < n_blocks; blk += gridDim.x) {
    const uint32_t sd = blk * blockDim.x + threadIdx.x;
    // tracklets that can hold a segment at all (the bound of walk_tracklet) are compacted and
    // walked with full warps; the others count zero
    bool cand = false;
    if (sd < n_seeds && B.tl_key[sd] != 0ull) {
      int n_own = 0;
#pragma unroll
      for (int w = 0; w < TPC_MASK_WORDS; ++w)
        if (w * 32 < B.K->n_rows) n_own += __popc(B.tl_mask[(size_t)(TPC_MASK_WORDS + w) * B.max_seeds + sd]);
      const tpc_params& P = B.K->P;
      cand = P.shared_fixed_cap ? n_own * 1000 + P.shared_permille * (int)B.tracklets[sd].n_hits >= P.min_hits_track * 1000
                                : n_own * 1000 >= P.min_hits_track * (1000 - P.shared_permille);
    }
    s_ns[threadIdx.x] = 0u; s_ni[threadIdx.x] = 0u;
    uint32_t n_cand;
    const uint32_t slot = block_excl_scan(cand ? 1u : 0u, &n_cand, sm);
    if (cand) s_list[slot] = (uint16_t)threadIdx.x;
    __syncthreads();
    if (threadIdx.x < n_cand) {
      const uint32_t t = s_list[threadIdx.x];
      uint32_t a = 0, b = 0;
      walk_tracklet<false>(B, blk * blockDim.x + t, a, b, 0, 0);
      s_ns[t] = a; s_ni[t] = b;
    }
    __syncthreads();
    const uint32_t ns = s_ns[threadIdx.x], ni = s_ni[threadIdx.x];
    uint32_t tot_s, tot_i;
    const uint32_t ps = block_excl_scan(ns, &tot_s, sm);
    const uint32_t pi = block_excl_scan(ni, &tot_i, sm);
    if (sd < n_seeds) { B.seg_cnt[sd] = ns ? ps : 0xFFFFFFFFu; B.id_cnt[sd] = pi; }  // block-local exclusive prefix
    if (threadIdx.x == 0) { part_seg[blk] = tot_s; part_id[blk] = tot_i; }
  }
}

// K5d: emit the track records at their scanned offsets (order = seed order).  Only about one
// tracklet in five emits anything, so a CTA first compacts the emitting tracklets of a span of
// TPC_EMIT_SPAN seeds into shared memory and then walks them with full warps.
#define TPC_EMIT_SPAN 1024
__global__ void __launch_bounds__(256) k_sel_emit(TpcBuffers B) {
  __shared__ uint32_t sm[33];
  __shared__ uint32_t s_list[TPC_EMIT_SPAN];
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS | TPC_DEVERR_TRACKS)) return;
  const uint32_t n_seeds = B.cnt->n_seeds;
  const uint32_t* part_seg = B.scan_partials;
  const uint32_t* part_id = B.scan_partials + (B.scan_blocks + 1) / 2;
  const uint32_t n_spans = (n_seeds + TPC_EMIT_SPAN - 1) / TPC_EMIT_SPAN;
  for (uint32_t span = blockIdx.x; span < n_spans; span += gridDim.x) {
    const uint32_t sd0 = span * TPC_EMIT_SPAN + threadIdx.x * 4;
    uint32_t ps[4];
    uint32_t cnt = 0;
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      ps[u] = sd0 + u < n_seeds ? B.seg_cnt[sd0 + u] : 0xFFFFFFFFu;
      cnt += ps[u] != 0xFFFFFFFFu;   // has a surviving segment
    }
    uint32_t tot;
    uint32_t pre = block_excl_scan(cnt, &tot, sm);   // (its first barrier also frees s_list of the previous span)
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (ps[u] != 0xFFFFFFFFu) s_list[pre++] = sd0 + u;
    __syncthreads();
    for (uint32_t e = threadIdx.x; e < tot; e += blockDim.x) {
      const uint32_t sd = s_list[e];
      const uint32_t blk = sd / 256u;   // block of k_sel_count that scanned this tracklet
      uint32_t ns, ni;
      walk_tracklet<true>(B, sd, ns, ni, part_seg[blk] + B.seg_cnt[sd], part_id[blk] + B.id_cnt[sd]);
    }
  }
}

// K5e: cluster lists (original ids ascending in row) and shared flags, one warp per track.
__global__ void __launch_bounds__(256) k_sel_ids(TpcBuffers B) {
  if (B.cnt->error & (TPC_DEVERR_BINS | TPC_DEVERR_SEEDS | TPC_DEVERR_TRACKS)) return;
  const uint32_t n_tracks = B.cnt->n_tracks;
  const uint32_t R = (uint32_t)B.K->n_rows;
  const int lane = threadIdx.x & 31;
  const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t ti = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; ti < n_tracks; ti += n_warps) {
    const tpc_track* __restrict__ t = B.tracks + ti;
    const int r0 = t->row_first, r1 = t->row_last;
    uint32_t o = t->cluster_ofs;
    const uint32_t sd = B.trk_sd[ti];
    const int32_t* __restrict__ hits = B.row_hit + (size_t)sd * R;
    const uint32_t* __restrict__ mk = B.trk_mask + (size_t)ti * (2 * TPC_MASK_WORDS);
    for (int wd = r0 >> 5; wd <= (r1 >> 5); ++wd) {
      const uint32_t am = mk[wd], sm = mk[TPC_MASK_WORDS + wd];
      if ((am >> lane) & 1u) {
        const uint32_t pos = o + (uint32_t)__popc(am & ((1u << lane) - 1u));
        B.cluster_ids[pos] = B.orig_id[hits[wd * 32 + lane]];
        B.cluster_shared[pos] = (uint8_t)((sm >> lane) & 1u);
      }
      o += (uint32_t)__popc(am);
    }
  }
}

__global__ void k_init(TpcBuffers B) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < B.n_sr) {
    TpcRowStat s;
    s.zmin_key = 0xFFFFFFFFu; s.zmax_key = 0u; s.count = 0u; s.n_all = 0u;
    s.first = 0xFFFFFFFFu; s.last = 0u; s.pad_[0] = s.pad_[1] = 0u;
    B.row_stat[i] = s;
  }
  if (i == 0) {
    TpcCounters c;
    c.n_sorted = c.n_ignored = c.n_dropped = c.n_bad = 0;
    c.n_bins = c.n_tiles = c.n_seeds = c.n_tracklets = 0;
    c.n_tracks = c.n_ids = c.error = 0;
    c.grid_rows = 0; c.n_rows_generic = 0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) c.follow_work[a][b] = 0ull;
    c.follow_next[0] = c.follow_next[1] = c.follow_next[2] = 0u; c.pad_ = 0u;
    *B.cnt = c;
  }
}

// ================================================================== R8 sector-track refit
// "a sector track refit at the beginning of the track merging was added,
// guaranteeing reasonable initial parameters".  One thread per output track: a pure Kalman fit
// through the track's own cluster list (outward pass, turn, inward pass; no search, no chi2
// cut) with the propagation / update statements of the follower.  The clusters are read from
// the input frame through their original indices.
// A cluster record gathered by original index is used once: the load bypasses L1 allocation
// (TPC_GATHER_NA = 1) so that the lines of the per-thread streams (id lists, stored predictions) survive there.
#ifndef TPC_GATHER_NA
#define TPC_GATHER_NA 1
#endif
__device__ __forceinline__ uint4 ld_cluster_once(const tpc_cluster* p) {
#if TPC_GATHER_NA
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
#else
  return *reinterpret_cast<const uint4*>(p);
#endif
}

// ---- work distribution of the per-track kernels (fit, rebuild).  Tracks next to each other in merge order start in the
// same region of the chamber (their grid lines and pages are shared: a global sort by length was
// measured 35 % slower), but their path lengths differ by up to 10x, and a warp runs as long as its
// longest track.  So: CTAs fetch chunks of TPC_RB_CHUNK consecutive tracks from a counter, sort the
// chunk by path length in shared memory, and the warps fetch groups of 32 tracks of similar length.
#define TPC_RB_CHUNK 512
#ifndef TPC_RB_MINB
#define TPC_RB_MINB 5
#endif
struct RbChunkShared { uint32_t key[TPC_RB_CHUNK]; uint32_t chunk, group; };
// len(i): work of item i (any monotone measure)
template <class LenFn>
__device__ __forceinline__ bool rb_chunk_begin(uint32_t n_items, LenFn len_of, uint32_t* counter, RbChunkShared& S, uint32_t& base) {
  __syncthreads();   // (everybody is done with the previous chunk's keys)
  if (threadIdx.x == 0) { S.chunk = atomicAdd(counter, 1u); S.group = 0u; }
  __syncthreads();
  base = S.chunk * (uint32_t)TPC_RB_CHUNK;
  if (base >= n_items) return false;
  for (uint32_t i = threadIdx.x; i < TPC_RB_CHUNK; i += blockDim.x) {
    const uint32_t mi = base + i;
    uint32_t len = mi < n_items ? len_of(mi) : 0u;
    if (len > 0x3FFFFFu) len = 0x3FFFFFu;
    S.key[i] = (len << 9) | i;
  }
  __syncthreads();
  for (uint32_t size = 2; size <= TPC_RB_CHUNK; size <<= 1)         // bitonic sort, descending
    for (uint32_t stride = size >> 1; stride > 0; stride >>= 1) {
      for (uint32_t i = threadIdx.x; i < TPC_RB_CHUNK / 2; i += blockDim.x) {
        const uint32_t lo = 2u * i - (i & (stride - 1u)), hi = lo + stride;
        const uint32_t a = S.key[lo], b = S.key[hi];
        const bool desc = (lo & size) == 0u;
        if ((a < b) == desc) { S.key[lo] = b; S.key[hi] = a; }
      }
      __syncthreads();
    }
  return true;
}
// the warp's next group of 32 tracks of the chunk; false: none left
__device__ __forceinline__ bool rb_group_next(uint32_t n_items, RbChunkShared& S, uint32_t base, uint32_t& mi, bool& valid) {
  uint32_t g = 0u;
  if ((threadIdx.x & 31u) == 0u) g = atomicAdd(&S.group, 1u);
  g = __shfl_sync(0xFFFFFFFFu, g, 0);
  if (g >= TPC_RB_CHUNK / 32) return false;
  mi = base + (S.key[g * 32u + (threadIdx.x & 31u)] & (uint32_t)(TPC_RB_CHUNK - 1));
  valid = mi < n_items;
  return true;
}

template <bool COMPACT>   // leave / use the compact copy of the tracks' clusters (B.trk_yz, B.trk_sr)
__global__ void __launch_bounds__(128) k_track_refit(TpcBuffers B, const __grid_constant__ FollowConst F, uint32_t n_tracks) {
  __shared__ RbChunkShared S;
  uint32_t base, ti;
  bool valid;
  auto len_of = [&](uint32_t i) { return (uint32_t)B.tracks[i].n_clusters; };
  while (rb_chunk_begin(n_tracks, len_of, &B.cnt->refit_next, S, base))
  while (rb_group_next(n_tracks, S, base, ti, valid)) {
    if (!valid) continue;
    const tpc_track* __restrict__ t = B.tracks + ti;
    const uint32_t* __restrict__ ids = B.cluster_ids + t->cluster_ofs;
    const int n = t->n_clusters;
    tpc_track_fit out;
    out.x = 0.f; out.chi2 = 0.f; out.n_clusters = (uint32_t)n; out.flags = 1u;
    out.x_out = 0.f; out.pad_[0] = out.pad_[1] = out.pad_[2] = 0u;
#pragma unroll
    for (int i = 0; i < 5; ++i) { out.p[i] = 0.f; out.p_out[i] = 0.f; }
#pragma unroll
    for (int i = 0; i < 15; ++i) { out.c[i] = 0.f; out.c_out[i] = 0.f; }
    int r_last = 0;
    // The outward pass gathers the 16-byte records of the frame by original index (a 64-byte DRAM access
    // each) and leaves a compact copy in list order (10 bytes per cluster); the inward pass, the merging's
    // copy, the fit and the rebuild read that instead of gathering again.
    // (COMPACT is a template parameter on purpose: a run-time choice of the source inside these loaders made
    // the compiler lose the lock-step of the lanes in the fit -- 4x the instructions at 5 lanes each)
    float2* __restrict__ cyz = COMPACT ? B.trk_yz + t->cluster_ofs : nullptr;
    uint16_t* __restrict__ csr = COMPACT ? B.trk_sr + t->cluster_ofs : nullptr;
    int n_copied = 0;
    auto rec = [&](int i, float& y, float& z, int& row) {          // gather (+ copy)
      const uint4 raw = ld_cluster_once(B.clusters + (ids[i] - B.id_base));
      y = __uint_as_float(raw.x); z = __uint_as_float(raw.y); row = (int)((raw.w >> 8) & 0xFF);
      if (COMPACT) {
        if (i >= n_copied) { cyz[i] = make_float2(y, z); csr[i] = (uint16_t)(((raw.w & 0xFFu) << 8) | ((raw.w >> 8) & 0xFFu)); n_copied = i + 1; }
      }
    };
    auto rec_back = [&](int i, float& y, float& z, int& row) {     // from the compact copy if there is one
      if (COMPACT) { const float2 v = cyz[i]; y = v.x; z = v.y; row = (int)(csr[i] & 0xFFu); }
      else rec(i, y, z, row);
    };
    bool ok = n >= 2;
    if (ok) {
      KF k;
      float y0, z0, y1, z1;
      int r0, r1;
      rec(0, y0, z0, r0);
      rec(1, y1, z1, r1);
      {  // R8.1
        const float dx = (float)(r1 - r0) * F.dx;
        const float dy = y1 - y0;
        const float dl = sqrtf(dx * dx + dy * dy);
        k.y = y0; k.z = z0;
        k.s = dy / dl;
        k.t = (z1 - z0) / dl;
        k.q = 0.f;
        kf_init_cov(k, F);
      }
      float snap_s = k.s, snap_t = k.t, snap_q = k.q;
      float ym = y0, zm = z0;
      int r = r0;
      for (int i = 1; i < n && ok; ++i) {  // R8.2 outward
        int ri;
        rec(i, ym, zm, ri);
        for (; r < ri && ok; ++r) ok = kf_propagate(k, F.dx, F);
        if (!ok) break;
        const Gain g = kf_gain(k, F);
        if (kf_update(k, g, ym, zm, F)) ok = false;
        snap_s = k.s; snap_t = k.t; snap_q = k.q;
      }
      if (ok) {  // the outer end (R9 extends it): the state after the outward pass at the last cluster
        r_last = r;
        out.p_out[0] = k.y; out.p_out[1] = k.z; out.p_out[2] = k.s; out.p_out[3] = k.t; out.p_out[4] = k.q;
        out.c_out[0] = k.c00; out.c_out[1] = k.c10; out.c_out[2] = k.c11; out.c_out[3] = k.c20; out.c_out[4] = k.c21;
        out.c_out[5] = k.c22; out.c_out[6] = k.c30; out.c_out[7] = k.c31; out.c_out[8] = k.c32; out.c_out[9] = k.c33;
        out.c_out[10] = k.c40; out.c_out[11] = k.c41; out.c_out[12] = k.c42; out.c_out[13] = k.c43; out.c_out[14] = k.c44;
      }
      if (ok) {  // R8.3 turn
        k.y = ym; k.z = zm; k.s = snap_s; k.t = snap_t; k.q = snap_q;
        kf_init_cov(k, F);
      }
      float chi2 = 0.f;
      for (int i = n - 2; i >= 0 && ok; --i) {  // R8.4 inward
        int ri;
        rec_back(i, ym, zm, ri);
        for (; r > ri && ok; --r) ok = kf_propagate(k, -F.dx, F);
        if (!ok) break;
        const Gain g = kf_gain(k, F);
        const float c2 = kf_chi2(k, g, ym, zm);
        if (kf_update(k, g, ym, zm, F)) ok = false;
        chi2 = chi2 + c2;
      }
      if (ok) {
        out.x = B.K->x[r0];
        out.p[0] = k.y; out.p[1] = k.z; out.p[2] = k.s; out.p[3] = k.t; out.p[4] = k.q;
        out.c[0] = k.c00; out.c[1] = k.c10; out.c[2] = k.c11; out.c[3] = k.c20; out.c[4] = k.c21; out.c[5] = k.c22;
        out.c[6] = k.c30; out.c[7] = k.c31; out.c[8] = k.c32; out.c[9] = k.c33;
        out.c[10] = k.c40; out.c[11] = k.c41; out.c[12] = k.c42; out.c[13] = k.c43; out.c[14] = k.c44;
        out.chi2 = chi2;
        out.x_out = B.K->x[r_last];
        out.flags = 0u;
      }
    }
    if (COMPACT)   // (a pass that stopped early: the copy is completed all the same, other kernels rely on it)
      for (int i = n_copied; i < n; ++i) { float y, z; int row; rec(i, y, z, row); }
    B.track_fit[ti] = out;
  }
}

// ================================================================== R9 track merging
// PAPER.md:29 (section 2): "merges tracks first inside the TPC sectors, then between adjacent
// sectors of the TPC halves, and then across the central electrode"; on top of the
// sector-track refit.  DESIGN.md reading R9.  Layout of the work:
//   k_merge_bin_*   the INNER ends of the tracks with a valid refit are binned by (sector, first row,
//                   z slab of pre_dz) -- a counting sort that also lays down compact 64-byte records
//                   (state, diagonal variances, tie-break key, track index) in cell order;
//   k_merge_sweep   one thread per track a with a free outer end carries its outer state along the
//                   stage's path (row steps / rotation + one step) and looks the candidates of every
//                   row it reaches up in the cells around its own z.  Pass 1: own best partner and
//                   atomicMin of chi2 on the partner's word; pass 2 (same sweep again): the tracks that
//                   hold a partner's minimum chi2 settle exact ties by their 64-bit key;
//   k_merge_link    mutual choice -> next / prev;
//   k_merge_chain_* chains -> merged records, segment lists, concatenated cluster lists.
#define TPC_MG_ZB 1024   // z slabs per (sector,row), periodic (a slab is pre_dz wide)

__device__ __forceinline__ unsigned long long merge_key(const tpc_track& t) {
  return ((unsigned long long)t.sector << 41) | ((unsigned long long)((t.flags >> 1) & 1u) << 40) |
         ((unsigned long long)t.seed_id << 8) | (unsigned long long)t.segment;
}
__device__ __forceinline__ uint32_t merge_cell(const TpcMergeBuffers& M, uint32_t sector, uint32_t row, float z) {
  const int zb = ((int)floorf(z * M.inv_w)) & (TPC_MG_ZB - 1);
  return (sector * M.n_rows + row) * TPC_MG_ZB + (uint32_t)zb;
}

__global__ void __launch_bounds__(256) k_merge_init(TpcBuffers B, TpcMergeBuffers M) {
  const uint32_t stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  for (uint32_t c = i0; c < M.n_cells + 1; c += stride) M.cell_start[c] = 0u;
  for (uint32_t t = i0; t < M.n_tracks; t += stride) { M.next[t] = -1; M.prev[t] = -1; M.link_chi2[t] = 0.f; }
  if (i0 < 4) M.counters[i0] = 0u;
}
__global__ void __launch_bounds__(256) k_merge_bin_count(TpcBuffers B, TpcMergeBuffers M) {
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < M.n_tracks; t += gridDim.x * blockDim.x) {
    const tpc_track_fit* f = B.track_fit + t;
    if (f->flags) continue;
    atomicAdd(&M.cell_start[merge_cell(M, B.tracks[t].sector, B.tracks[t].row_first, f->p[1])], 1u);
  }
}
// exclusive scan of a[0..n) in blocks of 1024: local prefixes in place, block totals to partials
__global__ void __launch_bounds__(1024) k_scan_blocks(uint32_t* a, uint32_t n, uint32_t* partials) {
  __shared__ uint32_t sm[33];
  const uint32_t i = blockIdx.x * 1024u + threadIdx.x;
  const uint32_t v = i < n ? a[i] : 0u;
  uint32_t tot;
  const uint32_t pre = block_excl_scan(v, &tot, sm);
  if (i < n) a[i] = pre;
  if (threadIdx.x == 0) partials[blockIdx.x] = tot;
}
__global__ void __launch_bounds__(1024) k_scan_top(uint32_t* partials, uint32_t n_blocks, uint32_t* total_out) {
  __shared__ uint32_t sm[33];
  uint32_t carry = 0;
  for (uint32_t b0 = 0; b0 < n_blocks; b0 += 1024) {
    const uint32_t b = b0 + threadIdx.x;
    const uint32_t v = b < n_blocks ? partials[b] : 0u;
    uint32_t tot;
    const uint32_t pre = block_excl_scan(v, &tot, sm);
    if (b < n_blocks) partials[b] = carry + pre;
    carry += tot;
  }
  if (threadIdx.x == 0 && total_out) *total_out = carry;
}
__global__ void __launch_bounds__(1024) k_scan_add(uint32_t* a, uint32_t n, const uint32_t* partials, uint32_t* end_out) {
  const uint32_t i = blockIdx.x * 1024u + threadIdx.x;
  if (i < n) a[i] += partials[blockIdx.x];
  (void)end_out;
}
__global__ void __launch_bounds__(256) k_merge_bin_fill(TpcBuffers B, TpcMergeBuffers M) {
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < M.n_tracks; t += gridDim.x * blockDim.x) {
    const tpc_track_fit* f = B.track_fit + t;
    if (f->flags) continue;
    const tpc_track tr = B.tracks[t];
    const uint32_t cell = merge_cell(M, tr.sector, tr.row_first, f->p[1]);
    const uint32_t pos = M.cell_start[cell] + atomicAdd(&M.cell_cursor[cell], 1u);
    const unsigned long long key = merge_key(tr);
    uint4* rec = reinterpret_cast<uint4*>(M.ends + (size_t)pos * 16);
    rec[0] = make_uint4(__float_as_uint(f->p[0]), __float_as_uint(f->p[1]), __float_as_uint(f->p[2]), __float_as_uint(f->p[3]));
    rec[1] = make_uint4(__float_as_uint(f->p[4]), __float_as_uint(f->c[0]), __float_as_uint(f->c[2]), __float_as_uint(f->c[5]));
    rec[2] = make_uint4(__float_as_uint(f->c[9]), __float_as_uint(f->c[14]), (uint32_t)key, (uint32_t)(key >> 32));
    rec[3] = make_uint4(t, 0u, 0u, 0u);
  }
}
__global__ void __launch_bounds__(256) k_merge_stage_reset(TpcMergeBuffers M) {
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < M.n_tracks; t += gridDim.x * blockDim.x) {
    M.best_out[t] = -1; M.best_out_chi[t] = 0xFFFFFFFFu; M.best_in_chi[t] = 0xFFFFFFFFu; M.best_in_key[t] = ~0ull;
    M.cand_cnt[t] = 0u;
  }
}

// rotation of a state at local x into the neighbouring sector's frame (sa carries the sign): same
// point, direction phi' = phi - alpha, parameters on the plane x' = const through the point;
// first-order Jacobian dy'/dy = ca - sa*tan(phi'), dz'/dy = -sa*t/cos(phi'), ds'/ds = ca + sa*s/cos(phi)
__device__ __forceinline__ bool merge_rotate(KF& k, float& x, float ca, float sa, float max_sinphi) {
  const float s = k.s;
  const float cphi = sqrtf(1.f - s * s);
  const float s1 = s * ca - cphi * sa;
  if (!(fabsf(s1) <= max_sinphi)) return false;
  const float cphi1 = sqrtf(1.f - s1 * s1);
  const float xn = x * ca + k.y * sa;
  const float yn = k.y * ca - x * sa;
  const float a = ca - sa * (s1 / cphi1);
  const float b = -(sa * (k.t / cphi1));
  const float r = ca + sa * (s / cphi);
  const float c00 = k.c00, c10 = k.c10, c11 = k.c11, c20 = k.c20, c21 = k.c21, c22 = k.c22;
  const float c30 = k.c30, c31 = k.c31, c32 = k.c32, c40 = k.c40, c41 = k.c41, c42 = k.c42;
  k.c00 = (a * a) * c00;
  k.c10 = a * (b * c00 + c10);
  k.c11 = ((b * b) * c00 + (2.f * b) * c10) + c11;
  k.c20 = (a * r) * c20;
  k.c21 = r * (b * c20 + c21);
  k.c22 = (r * r) * c22;
  k.c30 = a * c30;
  k.c31 = b * c30 + c31;
  k.c32 = r * c32;
  k.c40 = a * c40;
  k.c41 = b * c40 + c41;
  k.c42 = r * c42;
  x = xn; k.y = yn; k.s = s1;
  return true;
}

template <int STAGE, int PASS>
__global__ void __launch_bounds__(128) k_merge_sweep(TpcBuffers B, TpcMergeBuffers M, const __grid_constant__ FollowConst F) {
  const tpc_merge_params& P = M.P;
  const int R = (int)M.n_rows;
  for (uint32_t a = blockIdx.x * blockDim.x + threadIdx.x; a < M.n_tracks; a += gridDim.x * blockDim.x) {
    if (M.next[a] >= 0) continue;                      // outer end already linked by an earlier stage
    if (PASS == 2 && M.cand_cnt[a] <= TPC_MG_CAND) continue;   // settled from the cached candidates (k_merge_resolve)
    uint32_t n_cand = 0u;
    const tpc_track_fit* fa = B.track_fit + a;
    if (fa->flags) continue;
    const tpc_track ta = B.tracks[a];
    const unsigned long long key_a = merge_key(ta);
    const int la = ta.row_last;
    const float za_out = fa->p_out[1];
    KF k0;
    k0.y = fa->p_out[0]; k0.z = fa->p_out[1]; k0.s = fa->p_out[2]; k0.t = fa->p_out[3]; k0.q = fa->p_out[4];
    k0.c00 = fa->c_out[0]; k0.c10 = fa->c_out[1]; k0.c11 = fa->c_out[2]; k0.c20 = fa->c_out[3]; k0.c21 = fa->c_out[4];
    k0.c22 = fa->c_out[5]; k0.c30 = fa->c_out[6]; k0.c31 = fa->c_out[7]; k0.c32 = fa->c_out[8]; k0.c33 = fa->c_out[9];
    k0.c40 = fa->c_out[10]; k0.c41 = fa->c_out[11]; k0.c42 = fa->c_out[12]; k0.c43 = fa->c_out[13]; k0.c44 = fa->c_out[14];
    int32_t best = -1;
    float best_chi2 = 0.f;
    unsigned long long best_key = 0ull;
    // candidates on row `row` of sector `sb` for the transported state k
    auto visit = [&](uint32_t sb, int row, const KF& k) {
      const float zc = STAGE == 3 ? -k.z : k.z;
      const int zb0 = (int)floorf(((zc - P.pre_dz) - 0.01f) * M.inv_w), zb1 = (int)floorf(((zc + P.pre_dz) + 0.01f) * M.inv_w);   // (margin: rounding never hides a candidate; the cuts below decide)
      for (int zb = zb0; zb <= zb1; ++zb) {
        const uint32_t cell = (sb * M.n_rows + (uint32_t)row) * TPC_MG_ZB + (uint32_t)(zb & (TPC_MG_ZB - 1));
        const uint32_t e1 = M.cell_start[cell + 1];
        for (uint32_t e = M.cell_start[cell]; e < e1; ++e) {
          const uint4* rec = reinterpret_cast<const uint4*>(M.ends + (size_t)e * 16);
          const uint4 r0 = rec[0];
          const float yb = __uint_as_float(r0.x), zbv = __uint_as_float(r0.y);
          // pre-cuts: coarse on the end states as they are, fine on the transported state
          const float dzc = STAGE == 3 ? zbv + za_out : zbv - za_out;
          if (!(fabsf(dzc) <= P.pre_coarse_dz)) continue;
          const float dzf = STAGE == 3 ? zbv + k.z : zbv - k.z;
          if (!(fabsf(dzf) <= P.pre_dz)) continue;
          if (!(fabsf(yb - k.y) <= P.pre_dy)) continue;
          const uint4 r1 = rec[1], r2 = rec[2];
          const uint32_t b = rec[3].x;
          if (b == a || M.prev[b] >= 0) continue;        // inner end already linked by an earlier stage
          const float pb[5] = {yb, zbv, __uint_as_float(r0.z), __uint_as_float(r0.w), __uint_as_float(r1.x)};
          const float vb[5] = {__uint_as_float(r1.y), __uint_as_float(r1.z), __uint_as_float(r1.w), __uint_as_float(r2.x),
                               __uint_as_float(r2.y)};
          const float pa[5] = {k.y, k.z, k.s, k.t, k.q};
          const float va[5] = {k.c00, k.c11, k.c22, k.c33, k.c44};
          float chi2 = 0.f;
#pragma unroll
          for (int i = 0; i < 5; ++i) {
            float d = pb[i] - pa[i];
            float sys = P.sys[i];
            if (i == 1 && STAGE == 3) { d = pb[1] + pa[1]; sys = P.ce_sys_z; }
            const float var = (va[i] + vb[i]) + sys * sys;
            chi2 = chi2 + (d * d) / var;
          }
          if (!(chi2 <= P.chi2_max)) continue;
          const unsigned long long key_b = ((unsigned long long)r2.w << 32) | r2.z;
          if (PASS == 1) {
            if (best < 0 || chi2 < best_chi2 || (chi2 == best_chi2 && key_b < best_key)) {
              best = (int32_t)b; best_chi2 = chi2; best_key = key_b;
            }
            atomicMin(&M.best_in_chi[b], __float_as_uint(chi2));      // chi2 >= 0: bit order = value order
            if (n_cand < TPC_MG_CAND) M.cand[(size_t)a * TPC_MG_CAND + n_cand] = make_uint2(b, __float_as_uint(chi2));
            ++n_cand;
          } else if (__float_as_uint(chi2) == M.best_in_chi[b]) {
            atomicMin(&M.best_in_key[b], key_a);
          }
        }
      }
    };
    if (STAGE == 2) {
      const uint32_t side = ta.sector / 18u, s18 = ta.sector % 18u;
      for (int dir = 0; dir < 2; ++dir) {
        const uint32_t sb = side * 18u + (dir == 0 ? (s18 + 1u) % 18u : (s18 + 17u) % 18u);
        if (sb >= B.n_sectors) continue;
        KF kr = k0;
        float xr = B.K->x[la];
        if (!merge_rotate(kr, xr, M.ca, dir == 0 ? M.sa : -M.sa, F.max_sinphi)) continue;
        const int r_lo = max(0, la - P.gap_adjacent_back), r_hi = min(R - 1, la + P.gap_adjacent);
        for (int row = r_lo; row <= r_hi; ++row) {
          KF k = kr;
          if (!kf_propagate(k, B.K->x[row] - xr, F)) continue;
          visit(sb, row, k);
        }
      }
    } else {
      const uint32_t sb = STAGE == 1 ? ta.sector : (ta.sector < 18u ? ta.sector + 18u : ta.sector - 18u);
      if (sb < B.n_sectors) {
        KF k = k0;
        const int G = STAGE == 1 ? P.gap_in_sector : P.gap_ce;
        for (int g = 1; g <= G && la + g < R; ++g) {
          if (!kf_propagate(k, F.dx, F)) break;
          visit(sb, la + g, k);
        }
      }
    }
    if (PASS == 1) { M.best_out[a] = best; M.best_out_chi[a] = __float_as_uint(best_chi2); M.cand_cnt[a] = n_cand; }
  }
}

// Pass 2 for the tracks whose accepted candidates fit the cache (nearly all): among the holders of a
// partner's minimum chi2 the least 64-bit id wins.  The others repeat the sweep (k_merge_sweep<., 2>).
// (The cached chi2 bits are pass 1's own, so the comparison with the minimum cannot miss by a rounding
// difference between two compilations of the sweep, which the fast build's repeated sweep could.)
__global__ void __launch_bounds__(256) k_merge_resolve(TpcBuffers B, TpcMergeBuffers M) {
  for (uint32_t a = blockIdx.x * blockDim.x + threadIdx.x; a < M.n_tracks; a += gridDim.x * blockDim.x) {
    const uint32_t n = M.cand_cnt[a];
    if (n == 0u || n > TPC_MG_CAND) continue;
    const unsigned long long key_a = merge_key(B.tracks[a]);
    for (uint32_t i = 0; i < n; ++i) {
      const uint2 c = M.cand[(size_t)a * TPC_MG_CAND + i];
      if (c.y == M.best_in_chi[c.x]) atomicMin(&M.best_in_key[c.x], key_a);
    }
  }
}

__global__ void __launch_bounds__(256) k_merge_link(TpcBuffers B, TpcMergeBuffers M) {
  for (uint32_t a = blockIdx.x * blockDim.x + threadIdx.x; a < M.n_tracks; a += gridDim.x * blockDim.x) {
    const int32_t b = M.best_out[a];
    if (b < 0) continue;
    if (M.best_out_chi[a] == M.best_in_chi[b] && M.best_in_key[b] == merge_key(B.tracks[a])) {
      M.next[a] = b; M.prev[b] = (int32_t)a;
      M.link_chi2[a] = __uint_as_float(M.best_out_chi[a]);
      atomicAdd(&M.counters[1], 1u);
    }
  }
}

// chains: per head the number of segments / clusters -> three scans -> records, lists
__global__ void __launch_bounds__(256) k_merge_chain_count(TpcBuffers B, TpcMergeBuffers M) {
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < M.n_tracks; t += gridDim.x * blockDim.x) {
    uint32_t ns = 0, nc = 0;
    if (M.prev[t] < 0) {
      for (int32_t k = (int32_t)t; k >= 0; k = M.next[k]) { ++ns; nc += B.tracks[k].n_clusters; }
    }
    M.head_ofs[t] = ns ? 1u : 0u; M.seg_ofs[t] = ns; M.clu_ofs[t] = nc;
  }
}
__global__ void __launch_bounds__(256) k_merge_chain_emit(TpcBuffers B, TpcMergeBuffers M) {
  for (uint32_t t = blockIdx.x * blockDim.x + threadIdx.x; t < M.n_tracks; t += gridDim.x * blockDim.x) {
    if (M.prev[t] >= 0) continue;
    tpc_merged_track m;
    m.head = t; m.n_segments = 0; m.n_clusters = 0; m.n_shared = 0;
    m.cluster_ofs = M.clu_ofs[t]; m.seg_ofs = M.seg_ofs[t];
    m.row_first = B.tracks[t].row_first; m.sector_first = B.tracks[t].sector;
    m.row_last = 0; m.sector_last = 0;
    for (int32_t k = (int32_t)t; k >= 0; k = M.next[k]) {
      const tpc_track tk = B.tracks[k];
      M.seg_index[m.seg_ofs + m.n_segments] = (uint32_t)k;
      M.seg_dst[k] = m.cluster_ofs + m.n_clusters;
      ++m.n_segments; m.n_clusters += tk.n_clusters; m.n_shared += tk.n_shared;
      m.row_last = tk.row_last; m.sector_last = tk.sector;
    }
    M.merged[M.head_ofs[t]] = m;
  }
}
__global__ void __launch_bounds__(256) k_merge_copy_ids(TpcBuffers B, TpcMergeBuffers M) {
  const int lane = threadIdx.x & 31;
  const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
  for (uint32_t t = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; t < M.n_tracks; t += n_warps) {
    const uint32_t src = B.tracks[t].cluster_ofs, n = B.tracks[t].n_clusters, dst = M.seg_dst[t];
    for (uint32_t i = lane; i < n; i += 32) {
      M.ids[dst + i] = B.cluster_ids[src + i];
      M.shared[dst + i] = B.cluster_shared[src + i];
      if (M.yz) { M.yz[dst + i] = B.trk_yz[src + i]; M.sr[dst + i] = B.trk_sr[src + i]; }
    }
  }
}

// ================================================================== R10 three-iteration track fit
// PAPER.md:31,37 (section 2) and PAPER.md:57 (section 3, Phase I): three passes over the cluster list
// of every merged track -- inward (the predicted position and its covariance are STORED at every
// cluster, in half precision), outward (the prediction is interpolated with the stored one, the
// cluster's chi2 against the interpolation is cut: marking only), inward again through the unmarked
// clusters.  One thread per merged track; the stored predictions live in a 16-byte record per
// cluster of the merged list.  DESIGN.md reading R10.
__device__ __forceinline__ float fit_round_half(float v) { return __half2float(__float2half_rn(v)); }

__device__ __forceinline__ bool link_transport(KF& k, int sec0, int row0, int sec1, int row1, float zc,
                                               const TpcConst* __restrict__ K, const FollowConst& F, float ca, float sa,
                                               float ce_var) {
  if (sec0 == sec1 || sec0 - sec1 == 18 || sec1 - sec0 == 18) {
    const int n = row1 > row0 ? row1 - row0 : row0 - row1;
    const float dx = row1 > row0 ? F.dx : -F.dx;
    for (int i = 0; i < n; ++i)
      if (!kf_propagate(k, dx, F)) return false;
    if (sec0 != sec1) {   // central electrode: z re-based on the measurement, its correlations dropped
      k.z = zc;
      k.c10 = 0.f; k.c21 = 0.f; k.c31 = 0.f; k.c41 = 0.f;
      k.c11 = ce_var;
    }
    return true;
  }
  const float sgn = (sec1 % 18 == (sec0 % 18 + 1) % 18) ? 1.f : -1.f;
  float x = K->x[row0];
  if (!merge_rotate(k, x, ca, sgn * sa, F.max_sinphi)) return false;
  return kf_propagate(k, K->x[row1] - x, F);
}
__device__ __forceinline__ bool fit_transport(KF& k, int sec0, int row0, int sec1, int row1, float zc,
                                              const TpcConst* __restrict__ K, const FollowConst& F,
                                              const TpcFitBuffers& T) {
  return link_transport(k, sec0, row0, sec1, row1, zc, K, F, T.ca, T.sa, T.P.ce_var);
}
__device__ __forceinline__ void fit_turn(KF& k, float y, float z, const FollowConst& F) {
  k.y = y; k.z = z;
  kf_init_cov(k, F);
}
__device__ __forceinline__ float fit_chi2_2x2(float r0, float r1, float a, float b, float d, float vy, float vz) {
  const float s00 = a + vy, s01 = b, s11 = d + vz;
  const float det = s00 * s11 - s01 * s01;
  const float inv = 1.f / det;
  const float i00 = s11 * inv, i01 = -(s01 * inv), i11 = s00 * inv;
  return ((r0 * r0) * i00 + (2.f * (r0 * r1)) * i01) + (r1 * r1) * i11;
}

template <bool COMPACT>   // clusters from the compact copy of the merged lists (M.yz, M.sr) / gathered from the frame
__global__ void __launch_bounds__(128) k_track_fit3(TpcBuffers B, TpcMergeBuffers M, TpcFitBuffers T,
                                                    const __grid_constant__ FollowConst F) {
  const TpcConst* __restrict__ K = B.K;
  const uint32_t n_merged = M.counters[0];
  __shared__ RbChunkShared S;
  uint32_t base, mi;
  bool valid;
  auto len_of = [&](uint32_t i) { return M.merged[i].n_clusters; };
  while (rb_chunk_begin(n_merged, len_of, T.work, S, base))
  while (rb_group_next(n_merged, S, base, mi, valid)) {
    const unsigned vm = __ballot_sync(0xffffffffu, valid);   // the lanes of this group: their loops below run in lock-step
    if (!valid) continue;
    const tpc_merged_track m = M.merged[mi];
    const uint32_t* __restrict__ ids = M.ids + m.cluster_ofs;
    const int n = (int)m.n_clusters;
    tpc_track_fit3 out;
    out.x = 0.f; out.chi2 = 0.f; out.n_clusters = (uint32_t)n; out.n_used = 0u; out.flags = 1u;
#pragma unroll
    for (int i = 0; i < 5; ++i) out.p[i] = 0.f;
#pragma unroll
    for (int i = 0; i < 15; ++i) out.c[i] = 0.f;
    float* __restrict__ chi_c = T.chi2_cluster + m.cluster_ofs;
    uint8_t* __restrict__ rej = T.rejected + m.cluster_ofs;
    uint4* __restrict__ store = T.stored + m.cluster_ofs;
    for (int i = 0; i < n; ++i) { chi_c[i] = 0.f; rej[i] = 0; }
    const float2* __restrict__ cyz = M.yz + m.cluster_ofs;
    const uint16_t* __restrict__ csr = M.sr + m.cluster_ofs;
    auto rec = [&](int i, float& y, float& z, int& sec, int& row) {
      if (COMPACT) {
        const float2 v = cyz[i]; const uint32_t w = csr[i];
        y = v.x; z = v.y; sec = (int)(w >> 8); row = (int)(w & 0xFFu);
      } else {
        const uint4 raw = ld_cluster_once(B.clusters + (ids[i] - B.id_base));
        y = __uint_as_float(raw.x); z = __uint_as_float(raw.y); sec = (int)(raw.w & 0xFF); row = (int)((raw.w >> 8) & 0xFF);
      }
    };
    const uint32_t tail = M.seg_index[m.seg_ofs + m.n_segments - 1];
    const tpc_track_fit* ft = B.track_fit + tail;
    bool ok = n >= 2 && ft->flags == 0u;
    KF k;
    k.y = k.z = 0.f;
    k.s = ft->p_out[2]; k.t = ft->p_out[3]; k.q = ft->p_out[4];
    kf_init_cov(k, F);
    float yc, zc, yp, zp;
    int sc, rc, sp, rp;
    // Transport between consecutive clusters, ONE ROW STEP PER LOOP ITERATION (as the follower): the plan for
    // the next cluster gives the number of row steps; an iteration propagates one step and, when none is left,
    // processes the cluster.  A lane crossing a hole of three rows then costs its warp three cheap
    // iterations, not three propagations inside every other lane's cluster step.  Arithmetic and its order
    // per track are those of link_transport: the row steps, then (electrode) the z re-base; (adjacent sector)
    // rotation and one step over the x distance, done when the plan is made.
    int steps = 0;
    float dxs = 0.f;
    bool ce = false;
    auto plan = [&](int s0, int r0, int s1, int r1) -> bool {
      if (s0 == s1 || s0 - s1 == 18 || s1 - s0 == 18) {
        steps = r1 > r0 ? r1 - r0 : r0 - r1;
        dxs = r1 > r0 ? F.dx : -F.dx;
        ce = s0 != s1;
        return true;
      }
      steps = 0; ce = false;
      const float sgn = (s1 % 18 == (s0 % 18 + 1) % 18) ? 1.f : -1.f;
      float x = K->x[r0];
      if (!merge_rotate(k, x, T.ca, sgn * T.sa, F.max_sinphi)) return false;
      return kf_propagate(k, K->x[r1] - x, F);
    };
    auto arrive = [&](float z_cluster) {     // after the last row step: the electrode re-base
      if (ce) {
        k.z = z_cluster;
        k.c10 = 0.f; k.c21 = 0.f; k.c31 = 0.f; k.c41 = 0.f;
        k.c11 = T.P.ce_var;
      }
    };
    // ---- iteration 1: inward from c_{n-1}; predictions stored in half precision
    {
      int i = -1;
      if (ok) {
        rec(n - 1, yp, zp, sp, rp);
        fit_turn(k, yp, zp, F);
        i = n - 2;
        if (i >= 0) { rec(i, yc, zc, sc, rc); if (!plan(sp, rp, sc, rc)) ok = false; }
      }
      // (the loop condition is a vote of the group's lanes: they meet at the top of every iteration)
      for (bool act = ok && i >= 0; __any_sync(vm, act); act = ok && i >= 0) {
        if (!act) continue;
        if (steps > 0) { if (!kf_propagate(k, dxs, F)) ok = false; else --steps; }
        if (ok && steps == 0) {
          arrive(zc);
          const uint32_t h0 = (uint32_t)__half_as_ushort(__float2half_rn(k.y - yc)) | ((uint32_t)__half_as_ushort(__float2half_rn(k.z - zc)) << 16);
          const uint32_t h1 = (uint32_t)__half_as_ushort(__float2half_rn(k.c00)) | ((uint32_t)__half_as_ushort(__float2half_rn(k.c10)) << 16);
          const uint32_t h2 = (uint32_t)__half_as_ushort(__float2half_rn(k.c11));
          store[i] = make_uint4(h0, h1, h2, 0u);
          const Gain g = kf_gain(k, F);
          if (kf_update(k, g, yc, zc, F)) ok = false;
          else {
            sp = sc; rp = rc;
            --i;
            if (i >= 0) { rec(i, yc, zc, sc, rc); if (!plan(sp, rp, sc, rc)) ok = false; }
          }
        }
      }
    }
    // ---- iteration 2: outward from c_0; interpolation, chi2 cut (marking only)
    int used = 0;
    {
      int i = n;
      if (ok) {
      rec(0, yp, zp, sp, rp);
      fit_turn(k, yp, zp, F);
      {
        const uint4 st = store[0];
        const float s_ry = __half2float(__ushort_as_half((unsigned short)(st.x & 0xFFFFu))), s_rz = __half2float(__ushort_as_half((unsigned short)(st.x >> 16)));
        const float a1 = __half2float(__ushort_as_half((unsigned short)(st.y & 0xFFFFu))), b1 = __half2float(__ushort_as_half((unsigned short)(st.y >> 16)));
        const float d1 = __half2float(__ushort_as_half((unsigned short)(st.z & 0xFFFFu)));
        const float chi2 = fit_chi2_2x2(s_ry, s_rz, a1, b1, d1, F.vy, F.vz);
        chi_c[0] = chi2;
        if (!(chi2 <= T.P.fit_chi2_max)) rej[0] = 1; else ++used;
      }
      i = 1;
      if (i < n) { rec(i, yc, zc, sc, rc); if (!plan(sp, rp, sc, rc)) ok = false; }
      }
      for (bool act = ok && i < n; __any_sync(vm, act); act = ok && i < n) {
        if (!act) continue;
        if (steps > 0) { if (!kf_propagate(k, dxs, F)) ok = false; else --steps; }
        if (ok && steps == 0) {
          arrive(zc);
          const float r2y = k.y - yc, r2z = k.z - zc;
          const float a2 = k.c00, b2 = k.c10, d2 = k.c11;
          float chi2;
          if (i == n - 1) {
            chi2 = fit_chi2_2x2(r2y, r2z, a2, b2, d2, F.vy, F.vz);
          } else {
            const uint4 st = store[i];
            const float s_ry = __half2float(__ushort_as_half((unsigned short)(st.x & 0xFFFFu))), s_rz = __half2float(__ushort_as_half((unsigned short)(st.x >> 16)));
            const float a1 = __half2float(__ushort_as_half((unsigned short)(st.y & 0xFFFFu))), b1 = __half2float(__ushort_as_half((unsigned short)(st.y >> 16)));
            const float d1 = __half2float(__ushort_as_half((unsigned short)(st.z & 0xFFFFu)));
            const float det1 = a1 * d1 - b1 * b1, det2 = a2 * d2 - b2 * b2;
            const float n1 = 1.f / det1, n2 = 1.f / det2;
            const float i1a = d1 * n1, i1b = -(b1 * n1), i1d = a1 * n1;
            const float i2a = d2 * n2, i2b = -(b2 * n2), i2d = a2 * n2;
            const float ia = i1a + i2a, ib = i1b + i2b, id = i1d + i2d;
            const float detw = ia * id - ib * ib;
            const float nw = 1.f / detw;
            const float wa = id * nw, wb = -(ib * nw), wd = ia * nw;
            const float hy = (i1a * s_ry + i1b * s_rz) + (i2a * r2y + i2b * r2z);
            const float hz = (i1b * s_ry + i1d * s_rz) + (i2b * r2y + i2d * r2z);
            const float ry = wa * hy + wb * hz, rz = wb * hy + wd * hz;
            chi2 = fit_chi2_2x2(ry, rz, wa, wb, wd, F.vy, F.vz);
          }
          chi_c[i] = chi2;
          if (!(chi2 <= T.P.fit_chi2_max)) rej[i] = 1; else ++used;
          const Gain g = kf_gain(k, F);
          if (kf_update(k, g, yc, zc, F)) ok = false;
          else {
            sp = sc; rp = rc;
            ++i;
            if (i < n) { rec(i, yc, zc, sc, rc); if (!plan(sp, rp, sc, rc)) ok = false; }
          }
        }
      }
    }
    // ---- iteration 3: inward through the unmarked clusters
    if (ok) {
      out.n_used = (uint32_t)used;
      if (used < T.P.fit_min_clusters || used < 2) ok = false;
    }
    {
      float chi2 = 0.f;
      int i = -1;
      if (ok) {
        int last = n - 1;
        while (rej[last]) --last;
        rec(last, yp, zp, sp, rp);
        fit_turn(k, yp, zp, F);
        i = last - 1;
        while (i >= 0 && rej[i]) --i;
        if (i >= 0) { rec(i, yc, zc, sc, rc); if (!plan(sp, rp, sc, rc)) ok = false; }
      }
      for (bool act = ok && i >= 0; __any_sync(vm, act); act = ok && i >= 0) {
        if (!act) continue;
        if (steps > 0) { if (!kf_propagate(k, dxs, F)) ok = false; else --steps; }
        if (ok && steps == 0) {
          arrive(zc);
          const Gain g = kf_gain(k, F);
          const float c2 = kf_chi2(k, g, yc, zc);
          if (kf_update(k, g, yc, zc, F)) ok = false;
          else {
            chi2 = chi2 + c2;
            sp = sc; rp = rc;
            --i;
            while (i >= 0 && rej[i]) --i;
            if (i >= 0) { rec(i, yc, zc, sc, rc); if (!plan(sp, rp, sc, rc)) ok = false; }
          }
        }
      }
      if (ok) {
        out.x = K->x[rp];
        out.p[0] = k.y; out.p[1] = k.z; out.p[2] = k.s; out.p[3] = k.t; out.p[4] = k.q;
        out.c[0] = k.c00; out.c[1] = k.c10; out.c[2] = k.c11; out.c[3] = k.c20; out.c[4] = k.c21; out.c[5] = k.c22;
        out.c[6] = k.c30; out.c[7] = k.c31; out.c[8] = k.c32; out.c[9] = k.c33;
        out.c[10] = k.c40; out.c[11] = k.c41; out.c[12] = k.c42; out.c[13] = k.c43; out.c[14] = k.c44;
        out.chi2 = chi2;
        out.flags = 0u;
      }
    }
    T.fit[mi] = out;
  }
}

// ================================================================== R11 Phase-II track rebuild
// PAPER.md:59,65 (section 3, Phase II); reading R11.  Kernels:
//   k_rb_path_len   length of every merged track's path of (sector,row) steps (-> scan -> step offsets)
//   k_rb_step_track warp per merged track: the track index of every step
//   k_rb_pass12     thread per merged track: pass 1 inward through the original clusters (prediction
//                   stored at every step), pass 2 outward (interpolation, candidates of the step's row
//                   from the search grid of the sector tracking, best three kept, update with the best)
//   k_rb_round      thread per step (round 1) / per loser-list entry (rounds 2, 3): propose (64-bit
//                   atomicMax of weight | round | track) and resolve; k_rb_ties settles equal weights
//   k_rb_pass3      thread per merged track: one inward walk = shared attachment + pass 3 with the
//                   plain chi2 cut
// Iterator over the steps of a merged track, forward (outward) or backward; it also tells which
// original cluster of the merged list, if any, sits on the step.
template <bool COMPACT>   // original clusters from the compact copy of the merged lists / gathered from the frame
struct RbPath {
  const uint32_t* segs; const tpc_track* tracks; const uint32_t* ids; const tpc_cluster* cl;
  const float2* cyz; const uint16_t* csr;
  int n_seg, n_ids;
  uint32_t id_base;
  int g, row, ci, hole_end;
  bool hole;
  int sec, f, l;                       // current segment
  int c_sec, c_row; float c_y, c_z; uint32_t c_id; bool c_ok;   // the next original cluster in walking order
  __device__ __forceinline__ void load_seg() { const tpc_track t = tracks[segs[g]]; sec = t.sector; f = t.row_first; l = t.row_last; }
  __device__ __forceinline__ void load_cluster() {
    c_ok = ci >= 0 && ci < n_ids;
    if (c_ok) {
      c_id = ids[ci];
      if (COMPACT) {
        const float2 v = cyz[ci]; const uint32_t w = csr[ci];
        c_y = v.x; c_z = v.y; c_sec = (int)(w >> 8); c_row = (int)(w & 0xFFu);
      } else {
        const uint4 raw = ld_cluster_once(cl + (c_id - id_base));
        c_y = __uint_as_float(raw.x); c_z = __uint_as_float(raw.y); c_sec = (int)(raw.w & 0xFF); c_row = (int)((raw.w >> 8) & 0xFF);
      }
    }
  }
  __device__ __forceinline__ void begin_fwd() { g = 0; load_seg(); row = f; hole = false; ci = 0; load_cluster(); }
  __device__ __forceinline__ void begin_bwd_rows() { g = n_seg - 1; load_seg(); row = l; hole = false; ci = -1; c_ok = false; }
  __device__ __forceinline__ void begin_bwd() { g = n_seg - 1; load_seg(); row = l; hole = false; ci = n_ids - 1; load_cluster(); }
  // the original cluster on the current step: true + (id, y, z); the cursor moves on by dir
  __device__ __forceinline__ bool take_orig(int dir, int32_t& id, float& y, float& z) {
    if (hole || !c_ok || c_sec != sec || c_row != row) return false;
    id = (int32_t)c_id; y = c_y; z = c_z;
    ci += dir;
    load_cluster();
    return true;
  }
  __device__ __forceinline__ bool next_fwd() {
    if (!hole) {
      if (row < l) { ++row; return true; }
      if (g + 1 >= n_seg) return false;
      const tpc_track tn = tracks[segs[g + 1]];
      if ((int)tn.sector == sec && (int)tn.row_first > l + 1) { hole = true; row = l + 1; hole_end = tn.row_first; return true; }
      ++g; load_seg(); row = f;
      return true;
    }
    if (row + 1 < hole_end) { ++row; return true; }
    hole = false; ++g; load_seg(); row = f;
    return true;
  }
  __device__ __forceinline__ bool next_bwd() {
    if (!hole) {
      if (row > f) { --row; return true; }
      if (g == 0) return false;
      const tpc_track tp = tracks[segs[g - 1]];
      if ((int)tp.sector == sec && f > (int)tp.row_last + 1) { hole = true; row = f - 1; hole_end = tp.row_last; return true; }
      --g; load_seg(); row = l;
      return true;
    }
    if (row - 1 > hole_end) { --row; return true; }
    hole = false; --g; load_seg(); row = l;
    return true;
  }
};
template <bool COMPACT>
__device__ __forceinline__ RbPath<COMPACT> rb_path(const TpcBuffers& B, const TpcMergeBuffers& M, const tpc_merged_track& m) {
  RbPath<COMPACT> P;
  P.cyz = COMPACT ? M.yz + m.cluster_ofs : nullptr; P.csr = COMPACT ? M.sr + m.cluster_ofs : nullptr;
  P.segs = M.seg_index + m.seg_ofs; P.tracks = B.tracks; P.ids = M.ids + m.cluster_ofs; P.cl = B.clusters;
  P.n_seg = (int)m.n_segments; P.n_ids = (int)m.n_clusters; P.id_base = B.id_base;
  P.hole = false; P.hole_end = 0; P.c_ok = false;
  return P;
}

__global__ void __launch_bounds__(256) k_rb_path_len(TpcBuffers B, TpcMergeBuffers M) {
  const uint32_t n_merged = M.counters[0];
  for (uint32_t mi = blockIdx.x * blockDim.x + threadIdx.x; mi < M.n_tracks + 1; mi += gridDim.x * blockDim.x) {
    uint32_t n = 0;
    if (mi < n_merged) {
      const tpc_merged_track m = M.merged[mi];
      const uint32_t* segs = M.seg_index + m.seg_ofs;
      for (uint32_t g = 0; g < m.n_segments; ++g) {
        const tpc_track t = B.tracks[segs[g]];
        n += (uint32_t)(t.row_last - t.row_first + 1);
        if (g + 1 < m.n_segments) {
          const tpc_track tn = B.tracks[segs[g + 1]];
          if (tn.sector == t.sector && tn.row_first > t.row_last + 1) n += (uint32_t)(tn.row_first - t.row_last - 1);
        }
      }
    }
    M.path_ofs[mi] = n;
  }
}

// warp per merged track: the track of every step
__global__ void __launch_bounds__(256) k_rb_step_track(TpcRebuildBuffers Rb) {
  const uint32_t lane = threadIdx.x & 31u, wpb = blockDim.x >> 5;
  for (uint32_t mi = blockIdx.x * wpb + (threadIdx.x >> 5); mi < Rb.n_merged; mi += gridDim.x * wpb) {
    const uint32_t s0 = Rb.step_ofs[mi], s1 = Rb.step_ofs[mi + 1];
    for (uint32_t e = s0 + lane; e < s1; e += 32u) Rb.step_track[e] = mi;
  }
}

__device__ __forceinline__ uint32_t rb_half2(float a, float b) {
  return (uint32_t)__half_as_ushort(__float2half_rn(a)) | ((uint32_t)__half_as_ushort(__float2half_rn(b)) << 16);
}
__device__ __forceinline__ float rb_unhalf(uint32_t w, int hi) {
  return __half2float(__ushort_as_half((unsigned short)(hi ? (w >> 16) : (w & 0xFFFFu))));
}

template <bool COMPACT>
__global__ void __launch_bounds__(128, TPC_RB_MINB) k_rb_pass12(TpcBuffers B, TpcMergeBuffers M, TpcRebuildBuffers Rb,
                                                   const __grid_constant__ FollowConst F) {
  const TpcConst* __restrict__ K = B.K;
  const float w_sel = K->P.sel_chi2_weight;
  __shared__ RbChunkShared S;
  uint32_t base, mi;
  bool valid;
  auto len_of = [&](uint32_t i) { return Rb.step_ofs[i + 1] - Rb.step_ofs[i]; };
  while (rb_chunk_begin(Rb.n_merged, len_of, Rb.list_n + 4, S, base))
  while (rb_group_next(Rb.n_merged, S, base, mi, valid)) {
    if (!valid) continue;
    const tpc_merged_track m = M.merged[mi];
    const uint32_t s0 = Rb.step_ofs[mi];
    const int n = (int)(Rb.step_ofs[mi + 1] - s0);
    // a track that fails holds no candidates (pass 2 writes all three entries of every step it reaches)
    auto no_candidates = [&]() {
      for (int kk = 0; kk < n; ++kk)
#pragma unroll
        for (int j = 0; j < TPC_RB_NCAND; ++j) { Rb.cand_id[(size_t)(s0 + kk) * TPC_RB_NCAND + j] = -1; Rb.cand_chi2[(size_t)(s0 + kk) * TPC_RB_NCAND + j] = 0.f; }
    };
    Rb.alive[mi] = 0; Rb.Qkey[mi] = 0u;
    Rb.tkey[mi] = merge_key(B.tracks[m.head]);
    const uint32_t tail = M.seg_index[m.seg_ofs + m.n_segments - 1];
    const tpc_track_fit* ft = B.track_fit + tail;
    if (ft->flags != 0u || n < 2) { no_candidates(); continue; }
    RbPath<COMPACT> P = rb_path<COMPACT>(B, M, m);
    KF k;
    k.y = k.z = 0.f;
    k.s = ft->p_out[2]; k.t = ft->p_out[3]; k.q = ft->p_out[4];
    kf_init_cov(k, F);
    int32_t oid; float oy, oz;
    bool ok = true;
    // ---- pass 1: inward through the original clusters; the prediction is stored at every step
    P.begin_bwd();
    if (!P.take_orig(-1, oid, oy, oz)) { no_candidates(); continue; }   // (cannot happen: a segment's last row holds its last cluster)
    fit_turn(k, oy, oz, F);
    float chi1 = 0.f;
    int n1 = 1, ps = P.sec, pr = P.row;
    for (int kk = n - 2; kk >= 0 && ok; --kk) {
      P.next_bwd();
      const bool has = P.take_orig(-1, oid, oy, oz);
      if (!link_transport(k, ps, pr, P.sec, P.row, has ? oz : 0.f, K, F, Rb.ca, Rb.sa, Rb.P.ce_var)) { ok = false; break; }
      Rb.stored[s0 + (uint32_t)kk] = make_uint4(__float_as_uint(k.y), __float_as_uint(k.z), rb_half2(k.c00, k.c10),
                                                rb_half2(k.c11, 0.f) | (has ? 0x10000u : 0u));
      if (has) {
        const Gain g = kf_gain(k, F);
        const float c2 = kf_chi2(k, g, oy, oz);
        if (kf_update(k, g, oy, oz, F)) { ok = false; break; }
        chi1 = chi1 + c2;
        ++n1;
      }
      ps = P.sec; pr = P.row;
    }
    if (!ok) { no_candidates(); continue; }
    {
      const int ndf = 2 * n1 - 5;
      const float Q = (float)n1 - w_sel * (chi1 / (float)(ndf > 0 ? ndf : 1));
      Rb.Qkey[mi] = f2key(Q);
    }
    // ---- pass 2: outward; interpolation, candidates from the search grid, update with the best.  The
    // stored record says whether the step holds an original cluster; the cluster itself is only read
    // where the electrode is crossed (z re-based on it).
    P.begin_fwd();
    fit_turn(k, P.c_y, P.c_z, F);
    int ci = 1;
    ps = P.sec; pr = P.row;
    for (int kk = 0; kk < n && ok; ++kk) {
      const uint4 st = Rb.stored[s0 + (uint32_t)kk];
      if (kk > 0) {
        P.next_fwd();
        const bool has = (st.w >> 16) & 1u;
        float zc = 0.f;
        if (has) {
          if (P.sec != ps) zc = COMPACT ? P.cyz[ci].y : B.clusters[P.ids[ci] - B.id_base].z;
          ++ci;
        }
        if (!link_transport(k, ps, pr, P.sec, P.row, zc, K, F, Rb.ca, Rb.sa, Rb.P.ce_var)) { ok = false; break; }
      }
      const uint32_t sr = (uint32_t)P.sec * (uint32_t)F.R + (uint32_t)P.row;
      float py, pz, wa, wb, wd;
      if (kk == 0) {
        py = __uint_as_float(st.x); pz = __uint_as_float(st.y); wa = rb_unhalf(st.z, 0); wb = rb_unhalf(st.z, 1); wd = rb_unhalf(st.w, 0);
      } else if (kk == n - 1) {
        py = k.y; pz = k.z; wa = k.c00; wb = k.c10; wd = k.c11;
      } else {
        const float r1y = __uint_as_float(st.x) - k.y, r1z = __uint_as_float(st.y) - k.z;
        const float a1 = rb_unhalf(st.z, 0), b1 = rb_unhalf(st.z, 1), d1 = rb_unhalf(st.w, 0), a2 = k.c00, b2 = k.c10, d2 = k.c11;
        const float det1 = a1 * d1 - b1 * b1, det2 = a2 * d2 - b2 * b2;
        const float n1i = 1.f / det1, n2i = 1.f / det2;
        const float i1a = d1 * n1i, i1b = -(b1 * n1i), i1d = a1 * n1i;
        const float i2a = d2 * n2i, i2b = -(b2 * n2i), i2d = a2 * n2i;
        const float ia = i1a + i2a, ib = i1b + i2b, id = i1d + i2d;
        const float detw = ia * id - ib * ib;
        const float nw = 1.f / detw;
        wa = id * nw; wb = -(ib * nw); wd = ia * nw;
        const float hy = i1a * r1y + i1b * r1z, hz = i1b * r1y + i1d * r1z;
        py = k.y + (wa * hy + wb * hz);
        pz = k.z + (wb * hy + wd * hz);
      }
      const float ry = clampf(F.road_nsigma * sqrtf(wa + F.vy), F.road_min, F.road_max);
      const float rz = clampf(F.road_nsigma * sqrtf(wd + F.vz), F.road_min, F.road_max);
      // ---- all clusters of the step's (sector,row) inside the road and the chi2 cut: best three by
      // (chi2, original id); kept by sorted position, the ids are read at the end (and on a chi2 tie)
      static_assert(TPC_RB_NCAND == 3, "the insertion below is written out for three candidates");
      uint32_t bpos[TPC_RB_NCAND] = {0u, 0u, 0u};
      float bchi[TPC_RB_NCAND] = {INFINITY, INFINITY, INFINITY};   // (an empty entry sorts behind every candidate)
      float by0 = 0.f, bz0 = 0.f;
      int nb = 0;
      const tpc_row_desc d = ld_row_desc(B.row_desc + sr);
      if (d.count) {
        const BinWindow w = make_window(d, K, py - ry, py + ry, pz - rz, pz + rz);
        uint32_t b = w.base + (uint32_t)w.bz0 * (uint32_t)w.ny;
        uint32_t c = B.bin_start[b], c1 = B.bin_start[b + w.by_span];
        for (int bz = w.bz0; bz <= w.bz1; ++bz) {
          uint32_t cn = 0u, cn1 = 0u;
          if (bz < w.bz1) { cn = B.bin_start[b + (uint32_t)w.ny]; cn1 = B.bin_start[b + (uint32_t)w.ny + w.by_span]; }   // next z-row: requested before this one is scanned
          // (four clusters of the range requested together: one memory round trip per batch, not per cluster)
          auto consider = [&](uint32_t cc, const float2 mm) {
            if (!(fabsf(mm.x - py) <= ry && fabsf(mm.y - pz) <= rz)) return;
            const float c2 = fit_chi2_2x2(mm.x - py, mm.y - pz, wa, wb, wd, F.vy, F.vz);
            if (!(c2 <= Rb.P.cand_chi2_max)) return;
            auto before = [&](int j) { return c2 < bchi[j] || (c2 == bchi[j] && B.orig_id[cc] < B.orig_id[bpos[j]]); };
            if (before(0)) {
              bpos[2] = bpos[1]; bchi[2] = bchi[1]; bpos[1] = bpos[0]; bchi[1] = bchi[0]; bpos[0] = cc; bchi[0] = c2;
              by0 = mm.x; bz0 = mm.y;
            } else if (before(1)) {
              bpos[2] = bpos[1]; bchi[2] = bchi[1]; bpos[1] = cc; bchi[1] = c2;
            } else if (before(2)) {
              bpos[2] = cc; bchi[2] = c2;
            } else {
              return;
            }
            if (nb < TPC_RB_NCAND) ++nb;
          };
          for (; c < c1; c += 4) {
            const bool h1 = c + 1 < c1, h2 = c + 2 < c1, h3 = c + 3 < c1;
            const float2 m0 = B.yz[c];
            float2 m1 = m0, m2 = m0, m3 = m0;
            if (h1) m1 = B.yz[c + 1];
            if (h2) m2 = B.yz[c + 2];
            if (h3) m3 = B.yz[c + 3];
            consider(c, m0);
            if (h1) consider(c + 1, m1);
            if (h2) consider(c + 2, m2);
            if (h3) consider(c + 3, m3);
          }
          b += (uint32_t)w.ny; c = cn; c1 = cn1;
        }
      }
      const size_t so = (size_t)(s0 + (uint32_t)kk) * TPC_RB_NCAND;
#pragma unroll
      for (int j = 0; j < TPC_RB_NCAND; ++j) {
        const bool in = j < nb;
        Rb.cand_id[so + j] = in ? (int32_t)B.orig_id[bpos[j]] : -1;
        Rb.cand_chi2[so + j] = in ? bchi[j] : 0.f;
      }
      if (kk > 0 && nb > 0) {
        const Gain g = kf_gain(k, F);
        if (kf_update(k, g, by0, bz0, F)) { ok = false; break; }
      }
      ps = P.sec; pr = P.row;
    }
    if (!ok) { no_candidates(); continue; }
    Rb.alive[mi] = 1;
    Rb.stq2[3 * (size_t)mi] = k.s; Rb.stq2[3 * (size_t)mi + 1] = k.t; Rb.stq2[3 * (size_t)mi + 2] = k.q;
  }
}

// ---- second ambiguity solving: three proposal rounds.  A cluster goes to the proposing
// track of largest (Q, then least 64-bit id).  One 64-bit word per cluster, best[c] = Q key << 32 |
// round tag << 30 | (0x3FFFFFFF - merged track): an atomicMax gives the largest Q (and, provisionally, the
// least track INDEX among equal Q); the winner is whoever finds its own word there.  Exactly equal
// weights of two tracks are rare: such proposers are flagged in the loser list and a pair of small
// kernels settles them by the 64-bit id (atomicMin into bestId, take-over from the provisional winner).
// A cluster is owned iff its word carries the tag of an EARLIER round (ownership is final, so no word is
// ever reset).  Round 1: every step of every live track proposes its first candidate; rounds 2 and 3
// run over the loser lists (their order is irrelevant: the atomics commute).
#define TPC_RB_M_MASK 0x3FFFFFFFu
__device__ __forceinline__ unsigned long long rb_word(uint32_t qkey, int round, uint32_t m) {
  return ((unsigned long long)qkey << 32) | (unsigned long long)(((uint32_t)(3 - round) << 30) | (TPC_RB_M_MASK - m));
}
__device__ __forceinline__ uint32_t rb_word_track(unsigned long long w) { return TPC_RB_M_MASK - ((uint32_t)w & TPC_RB_M_MASK); }
__device__ __forceinline__ bool rb_owned_before(unsigned long long w, int round) {
  return w != 0ull && (int)(((uint32_t)w >> 30) & 3u) > 3 - round;
}
__device__ __forceinline__ void rb_append(uint2* list, uint32_t* n, bool lose, uint32_t e, uint32_t flag) {
  const uint32_t mask = __ballot_sync(0xFFFFFFFFu, lose);
  if (!mask) return;
  const uint32_t lane = threadIdx.x & 31u;
  uint32_t base = 0u;
  if (lane == (uint32_t)(__ffs(mask) - 1)) base = atomicAdd(n, (uint32_t)__popc(mask));
  base = __shfl_sync(0xFFFFFFFFu, base, __ffs(mask) - 1);
  if (lose) list[base + __popc(mask & ((1u << lane) - 1u))] = make_uint2(e, flag);
}
// PHASE 0: propose; PHASE 1: resolve.  ROUND 1 runs over all steps (list == nullptr), the others over `list`.
template <int ROUND, int PHASE>
__global__ void __launch_bounds__(256) k_rb_round(TpcRebuildBuffers Rb, uint2* list, const uint32_t* n_list, uint2* losers,
                                                  uint32_t* n_losers) {
  const uint32_t n = ROUND == 1 ? Rb.n_steps : *n_list, n_pad = (n + 31u) & ~31u;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_pad; i += gridDim.x * blockDim.x) {
    int32_t c = -1;
    uint32_t e = 0u, m = 0u;
    if (i < n) {
      if (ROUND == 1) {
        e = i;
        m = Rb.step_track[e];
        if (Rb.alive[m]) c = Rb.cand_id[(size_t)e * TPC_RB_NCAND];
      } else {
        const uint2 it = list[i];
        e = it.x;
        m = Rb.step_track[e];
        if (PHASE == 0) {
          // the best candidate without an owner (owners are final, so the search restarts at the first);
          // a step that took a cluster over in the tie kernels is done
          if (Rb.attached[e] < 0)
            for (int p = 0; p < TPC_RB_NCAND; ++p) {
              const int32_t cc = Rb.cand_id[(size_t)e * TPC_RB_NCAND + p];
              if (cc < 0) break;
              if (!rb_owned_before(Rb.best[cc], ROUND)) { c = cc; break; }
            }
          list[i].y = (uint32_t)c;
        } else {
          c = (int32_t)it.y;
        }
      }
    }
    if (PHASE == 0) {
      if (c >= 0) atomicMax(&Rb.best[c], rb_word(Rb.Qkey[m], ROUND, m));
    } else {
      bool win = false, tie = false;
      if (c >= 0) {
        const unsigned long long w = Rb.best[c], mine = rb_word(Rb.Qkey[m], ROUND, m);
        win = w == mine;
        tie = !win && (uint32_t)(w >> 32) == (uint32_t)(mine >> 32);
        if (win) Rb.attached[e] = c;
      }
      rb_append(losers, n_losers, c >= 0 && !win, e, tie ? 1u : 0u);
    }
  }
}
// the flagged entries of a loser list: equal weight as the provisional winner of cluster c
template <int PHASE>
__global__ void __launch_bounds__(256) k_rb_ties(TpcRebuildBuffers Rb, uint2* list, uint32_t* n_list, int round) {
  const uint32_t n = *n_list;
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const uint2 it = list[i];
    if (it.y != 1u) continue;
    const uint32_t e = it.x, m = Rb.step_track[e];
    // (the step's proposal of this round: its first candidate that was not owned before)
    int32_t c = -1;
    for (int p = 0; p < TPC_RB_NCAND; ++p) {
      const int32_t cc = Rb.cand_id[(size_t)e * TPC_RB_NCAND + p];
      if (cc < 0) break;
      if (!rb_owned_before(Rb.best[cc], round)) { c = cc; break; }
    }
    if (c < 0) continue;
    if (PHASE == 0) {
      atomicMin(&Rb.bestId[c], Rb.tkey[m]);
      atomicMin(&Rb.bestId[c], Rb.tkey[rb_word_track(Rb.best[c])]);
    } else if (Rb.bestId[c] == Rb.tkey[m]) {
      const unsigned long long old = atomicExch(&Rb.best[c], rb_word(Rb.Qkey[m], round, m));
      const uint32_t mw = rb_word_track(old);
      Rb.attached[e] = c;
      if (mw != m)
        for (uint32_t e2 = Rb.step_ofs[mw]; e2 < Rb.step_ofs[mw + 1]; ++e2)
          if (Rb.attached[e2] == c) {
            Rb.attached[e2] = -1;
            list[atomicAdd(n_list, 1u)] = make_uint2(e2, 0u);
          }
    }
  }
}

__global__ void __launch_bounds__(128) k_rb_pass3(TpcBuffers B, TpcMergeBuffers M, TpcRebuildBuffers Rb,
                                                  const __grid_constant__ FollowConst F) {
  const TpcConst* __restrict__ K = B.K;
  const int permille = K->P.shared_permille;
  // (plain order: the chunked distribution of pass 1+2 was measured 5 % slower here)
  for (uint32_t mi = blockIdx.x * blockDim.x + threadIdx.x; mi < Rb.n_merged; mi += gridDim.x * blockDim.x) {
    tpc_track_fit3 out;
    out.x = 0.f; out.chi2 = 0.f; out.n_clusters = 0u; out.n_used = 0u; out.flags = 1u;
#pragma unroll
    for (int i = 0; i < 5; ++i) out.p[i] = 0.f;
#pragma unroll
    for (int i = 0; i < 15; ++i) out.c[i] = 0.f;
    if (!Rb.alive[mi]) { Rb.fit[mi] = out; continue; }
    const tpc_merged_track m = M.merged[mi];
    const uint32_t s0 = Rb.step_ofs[mi];
    const int n = (int)(Rb.step_ofs[mi + 1] - s0);
    // The record of the cluster a step owns is requested one step ahead (attached[] of the next step and its
    // record travel while this step is computed); a cluster attached as shared during this walk is loaded
    // on demand.
    int32_t pre_id = n > 0 ? Rb.attached[s0 + (uint32_t)(n - 1)] : -1;
    uint4 pre_raw = make_uint4(0u, 0u, 0u, 0u);
    if (pre_id >= 0) pre_raw = ld_cluster_once(B.clusters + ((uint32_t)pre_id - B.id_base));
    int32_t cur_id = -1;
    uint4 cur_raw = pre_raw;
    auto cluster_yz = [&](int32_t id, float& y, float& z) {
      const uint4 raw = id == cur_id ? cur_raw : ld_cluster_once(B.clusters + ((uint32_t)id - B.id_base));
      y = __uint_as_float(raw.x); z = __uint_as_float(raw.y);
    };
    // One walk from the outermost step inward does both: the shared attachment (the rule of R6.3: its
    // decision at a step depends on the steps outside of it only) and, from the outermost attached step
    // on, pass 3 with the plain chi2 cut.  After a failed transport / update the walk goes on for the
    // attachment marks alone.
    RbPath<false> P = rb_path<false>(B, M, m);
    P.begin_bwd_rows();
    KF k, kin;
    k.s = Rb.stq2[3 * (size_t)mi]; k.t = Rb.stq2[3 * (size_t)mi + 1]; k.q = Rb.stq2[3 * (size_t)mi + 2];
    k.y = k.z = 0.f;
    kf_init_cov(k, F);
    kin = k;
    int n_acc = 0, n_sh = 0, nu = 0, row_in = 0, ps = 0, pr = 0;
    float chi3 = 0.f;
    bool ok = true, started = false;
    for (int kk = n - 1; kk >= 0; --kk) {
      if (kk < n - 1) P.next_bwd();
      const uint32_t e = s0 + (uint32_t)kk;
      int32_t ca = pre_id;
      cur_id = pre_id; cur_raw = pre_raw;
      if (kk > 0) {
        pre_id = Rb.attached[e - 1u];
        if (pre_id >= 0) pre_raw = ld_cluster_once(B.clusters + ((uint32_t)pre_id - B.id_base));
      }
      if (ca >= 0) {
        ++n_acc;
      } else {
        const int32_t c = Rb.cand_id[(size_t)e * TPC_RB_NCAND];
        if (c >= 0 && (long long)(n_sh + 1) * 1000 <= (long long)permille * (n_acc + 1)) {
          Rb.attached[e] = c; Rb.shared[e] = 1; ++n_acc; ++n_sh;
          ca = c;
        }
      }
      if (!ok) continue;
      float ay = 0.f, az = 0.f;
      if (!started) {
        if (ca < 0) continue;
        cluster_yz(ca, ay, az);
        fit_turn(k, ay, az, F);
        Rb.used[e] = 1;
        kin = k; nu = 1; row_in = P.row; ps = P.sec; pr = P.row;
        started = true;
        continue;
      }
      float zc = k.z;
      if (ca >= 0) { cluster_yz(ca, ay, az); zc = az; }
      else if (P.sec != ps && (P.sec - ps == 18 || ps - P.sec == 18)) {
        // the electrode is crossed onto a step without an attached cluster: z is re-based on the
        // step's original cluster if it has one (rare: the merged list is searched)
        for (int i = 0; i < P.n_ids; ++i) {
          const uint4 raw = *reinterpret_cast<const uint4*>(P.cl + (P.ids[i] - P.id_base));
          if ((int)(raw.w & 0xFF) == P.sec && (int)((raw.w >> 8) & 0xFF) == P.row) { zc = __uint_as_float(raw.y); break; }
        }
      }
      if (!link_transport(k, ps, pr, P.sec, P.row, zc, K, F, Rb.ca, Rb.sa, Rb.P.ce_var)) { ok = false; continue; }
      ps = P.sec; pr = P.row;
      if (ca < 0) continue;
      const Gain g = kf_gain(k, F);
      const float c2 = kf_chi2(k, g, ay, az);
      if (!(c2 <= Rb.P.final_chi2_max)) continue;   // plain cut: the cluster is dropped, no update
      if (kf_update(k, g, ay, az, F)) { ok = false; continue; }
      chi3 = chi3 + c2;
      Rb.used[e] = 1;
      ++nu;
      kin = k;
      row_in = P.row;
    }
    out.n_clusters = (uint32_t)n_acc;
    out.n_used = (uint32_t)nu;
    if (started && ok && nu >= Rb.P.min_clusters) {
      out.flags = 0u;
      out.chi2 = chi3;
      out.x = K->x[row_in];
      out.p[0] = kin.y; out.p[1] = kin.z; out.p[2] = kin.s; out.p[3] = kin.t; out.p[4] = kin.q;
      out.c[0] = kin.c00; out.c[1] = kin.c10; out.c[2] = kin.c11; out.c[3] = kin.c20; out.c[4] = kin.c21; out.c[5] = kin.c22;
      out.c[6] = kin.c30; out.c[7] = kin.c31; out.c[8] = kin.c32; out.c[9] = kin.c33;
      out.c[10] = kin.c40; out.c[11] = kin.c41; out.c[12] = kin.c42; out.c[13] = kin.c43; out.c[14] = kin.c44;
    }
    Rb.fit[mi] = out;
  }
}

// ================================================================== host: enqueue the path
#define TPC_LAUNCH_CHECK(name)                                      \
  do {                                                              \
    if (cudaPeekAtLastError() != cudaSuccess) return -1;            \
    if (timers && launches < TPC_MAX_KERNELS) {                     \
      E.kname[launches] = name;                                     \
      cudaEventRecord(E.kev[launches + 1], st);                     \
    }                                                               \
    ++launches;                                                     \
  } while (0)

// CTAs of `kernel` that are resident on one SM at this block size / dynamic shared memory.
// Every kernel here is a grid-stride (persistent) loop: a grid larger than what is resident
// runs in waves and leaves a tail, a smaller one leaves SMs short of warps.
template <class K>
static inline int resident_ctas(K kernel, int block, size_t smem = 0) {
  int n = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kernel, block, smem) != cudaSuccess || n < 1) n = 1;
  return n;
}

static inline int grid_for(uint64_t n, int block, int n_sm, int ctas_per_sm) {
  uint64_t g = (n + block - 1) / block;
  const uint64_t cap = (uint64_t)n_sm * ctas_per_sm;
  if (g > cap) g = cap;
  return g < 1 ? 1 : (int)g;
}

int run_refit(const TpcBuffers& B, const TpcConst* hK, uint32_t n_tracks, cudaStream_t st, int n_sm) {
  if (n_tracks == 0) return 0;
  const FollowConst F = follow_const(hK);
  cudaMemsetAsync(&B.cnt->refit_next, 0, 4, st);
  if (B.trk_yz) k_track_refit<true><<<grid_for(n_tracks, 128, n_sm, resident_ctas(k_track_refit<true>, 128)), 128, 0, st>>>(B, F, n_tracks);
  else k_track_refit<false><<<grid_for(n_tracks, 128, n_sm, resident_ctas(k_track_refit<false>, 128)), 128, 0, st>>>(B, F, n_tracks);
  return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

static inline void scan_u32(uint32_t* a, uint32_t n, uint32_t* partials, uint32_t* total_out, cudaStream_t st) {
  const uint32_t nb = (n + 1023u) / 1024u;
  if (!nb) return;
  k_scan_blocks<<<nb, 1024, 0, st>>>(a, n, partials);
  k_scan_top<<<1, 1024, 0, st>>>(partials, nb, total_out);
  k_scan_add<<<nb, 1024, 0, st>>>(a, n, partials, nullptr);
}

// Returns the number of kernels launched, or -1 on a launch error.
int run_merge(const TpcBuffers& B, const TpcConst* hK, const TpcMergeBuffers& M, cudaStream_t st, int n_sm) {
  const FollowConst F = follow_const(hK);
  int launches = 0;
  const int g256 = grid_for((uint64_t)M.n_tracks + 1, 256, n_sm, 8);
  k_merge_init<<<grid_for((uint64_t)M.n_cells + 1, 256, n_sm, 8), 256, 0, st>>>(B, M);
  cudaMemsetAsync(M.cell_cursor, 0, 4 * (size_t)M.n_cells, st);
  ++launches;
  if (M.n_tracks) {
    k_merge_bin_count<<<g256, 256, 0, st>>>(B, M);
    scan_u32(M.cell_start, M.n_cells + 1, M.partials, nullptr, st);
    k_merge_bin_fill<<<g256, 256, 0, st>>>(B, M);
    launches += 5;
    const int gs = grid_for(M.n_tracks, 128, n_sm, 8);
    for (int stage = 1; stage <= 3; ++stage) {
      if (!((M.P.stages >> (stage - 1)) & 1)) continue;
      k_merge_stage_reset<<<g256, 256, 0, st>>>(M);
      if (stage == 1) { k_merge_sweep<1, 1><<<gs, 128, 0, st>>>(B, M, F); k_merge_resolve<<<g256, 256, 0, st>>>(B, M); k_merge_sweep<1, 2><<<gs, 128, 0, st>>>(B, M, F); }
      if (stage == 2) { k_merge_sweep<2, 1><<<gs, 128, 0, st>>>(B, M, F); k_merge_resolve<<<g256, 256, 0, st>>>(B, M); k_merge_sweep<2, 2><<<gs, 128, 0, st>>>(B, M, F); }
      if (stage == 3) { k_merge_sweep<3, 1><<<gs, 128, 0, st>>>(B, M, F); k_merge_resolve<<<g256, 256, 0, st>>>(B, M); k_merge_sweep<3, 2><<<gs, 128, 0, st>>>(B, M, F); }
      k_merge_link<<<g256, 256, 0, st>>>(B, M);
      launches += 5;
    }
    k_merge_chain_count<<<g256, 256, 0, st>>>(B, M);
    scan_u32(M.head_ofs, M.n_tracks, M.partials, &M.counters[0], st);
    scan_u32(M.seg_ofs, M.n_tracks, M.partials, nullptr, st);
    scan_u32(M.clu_ofs, M.n_tracks, M.partials, &M.counters[2], st);
    k_merge_chain_emit<<<g256, 256, 0, st>>>(B, M);
    k_merge_copy_ids<<<grid_for((uint64_t)M.n_tracks * 32, 256, n_sm, 8), 256, 0, st>>>(B, M);
    launches += 12;
  }
  return cudaPeekAtLastError() == cudaSuccess ? launches : -1;
}

int run_fit3(const TpcBuffers& B, const TpcConst* hK, const TpcMergeBuffers& M, const TpcFitBuffers& T, uint32_t n_merged,
             cudaStream_t st, int n_sm) {
  if (n_merged == 0) return 0;
  const FollowConst F = follow_const(hK);
  cudaMemsetAsync(T.work, 0, 16, st);
  if (M.yz) k_track_fit3<true><<<grid_for(n_merged, 128, n_sm, resident_ctas(k_track_fit3<true>, 128)), 128, 0, st>>>(B, M, T, F);
  else k_track_fit3<false><<<grid_for(n_merged, 128, n_sm, resident_ctas(k_track_fit3<false>, 128)), 128, 0, st>>>(B, M, T, F);
  return cudaPeekAtLastError() == cudaSuccess ? 1 : -1;
}

int run_rebuild_paths(const TpcBuffers& B, const TpcMergeBuffers& M, cudaStream_t st, int n_sm) {
  k_rb_path_len<<<grid_for((uint64_t)M.n_tracks + 1, 256, n_sm, 8), 256, 0, st>>>(B, M);
  scan_u32(M.path_ofs, M.n_tracks + 1, M.partials, &M.counters[3], st);
  return cudaPeekAtLastError() == cudaSuccess ? 4 : -1;
}

int run_rebuild(const TpcBuffers& B, const TpcConst* hK, const TpcMergeBuffers& M, const TpcRebuildBuffers& Rb, cudaStream_t st,
                int n_sm) {
  if (Rb.n_merged == 0) return 0;
  const FollowConst F = follow_const(hK);
  const int gw = grid_for((uint64_t)Rb.n_merged * 32, 256, n_sm, 8);
  const int gs = grid_for((uint64_t)Rb.n_steps + 32, 256, n_sm, 8);
  const size_t ns = Rb.n_steps, nc = Rb.n_clusters;
  cudaMemsetAsync(Rb.list_n, 0, 32, st);
  cudaMemsetAsync(Rb.attached, 0xFF, 4 * ns, st);
  cudaMemsetAsync(Rb.shared, 0, ns, st);
  cudaMemsetAsync(Rb.used, 0, ns, st);
  cudaMemsetAsync(Rb.best, 0, 8 * nc, st);
  cudaMemsetAsync(Rb.bestId, 0xFF, 8 * nc, st);
  k_rb_step_track<<<gw, 256, 0, st>>>(Rb);
  if (M.yz) k_rb_pass12<true><<<grid_for(Rb.n_merged, 128, n_sm, resident_ctas(k_rb_pass12<true>, 128)), 128, 0, st>>>(B, M, Rb, F);
  else k_rb_pass12<false><<<grid_for(Rb.n_merged, 128, n_sm, resident_ctas(k_rb_pass12<false>, 128)), 128, 0, st>>>(B, M, Rb, F);
  // the stored predictions are dead now: their region holds the loser lists (round 3's goes where round 2's was)
  uint2* list2 = reinterpret_cast<uint2*>(Rb.stored);
  uint2* list3 = list2 + ns;
  uint32_t* cnt = Rb.list_n;
  const int gl = grid_for((uint64_t)Rb.n_steps / 8 + 32, 256, n_sm, 8);
  k_rb_round<1, 0><<<gs, 256, 0, st>>>(Rb, nullptr, nullptr, nullptr, nullptr);
  k_rb_round<1, 1><<<gs, 256, 0, st>>>(Rb, nullptr, nullptr, list2, cnt);
  k_rb_ties<0><<<gl, 256, 0, st>>>(Rb, list2, cnt, 1);
  k_rb_ties<1><<<gl, 256, 0, st>>>(Rb, list2, cnt, 1);
  k_rb_round<2, 0><<<gl, 256, 0, st>>>(Rb, list2, cnt, nullptr, nullptr);
  k_rb_round<2, 1><<<gl, 256, 0, st>>>(Rb, list2, cnt, list3, cnt + 1);
  k_rb_ties<0><<<gl, 256, 0, st>>>(Rb, list3, cnt + 1, 2);
  k_rb_ties<1><<<gl, 256, 0, st>>>(Rb, list3, cnt + 1, 2);
  k_rb_round<3, 0><<<gl, 256, 0, st>>>(Rb, list3, cnt + 1, nullptr, nullptr);
  k_rb_round<3, 1><<<gl, 256, 0, st>>>(Rb, list3, cnt + 1, list2, cnt + 2);
  k_rb_ties<0><<<gl, 256, 0, st>>>(Rb, list2, cnt + 2, 3);
  k_rb_ties<1><<<gl, 256, 0, st>>>(Rb, list2, cnt + 2, 3);
  k_rb_pass3<<<grid_for(Rb.n_merged, 128, n_sm, resident_ctas(k_rb_pass3, 128)), 128, 0, st>>>(B, M, Rb, F);
  return cudaPeekAtLastError() == cudaSuccess ? 15 : -1;
}

// Returns the number of kernels launched, or -1 on a launch error.
int run_pipeline(const TpcBuffers& B, const TpcConst* hK, cudaStream_t st, uint32_t flags, TpcStageEvents& E, int n_sm) {
  int launches = 0;
  const FollowConst F = follow_const(hK);
  const bool timers = E.enabled;
  if (timers) cudaEventRecord(E.kev[0], st);
  k_init<<<(B.n_sr + 255) / 256, 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_init");
  if (timers) cudaEventRecord(E.ev[0], st);
  // ---- K1 grid
  k_row_stats<<<grid_for(B.n, 256, n_sm, resident_ctas(k_row_stats, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_row_stats");
  k_row_desc<<<1, 1024, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_row_desc");
  k_tile_rows<<<grid_for((uint64_t)B.n_sr * 128, 128, n_sm, 8), 128, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_tile_rows");
  cudaFuncSetAttribute(k_row_sort, cudaFuncAttributeMaxDynamicSharedMemorySize, TPC_RS_SMEM_BYTES);
  k_row_sort<<<min((uint32_t)n_sm, B.n_sr), TPC_RS_THREADS, TPC_RS_SMEM_BYTES, st>>>(B);
  TPC_LAUNCH_CHECK("k_row_sort");
  k_zero_bins<<<grid_for((uint64_t)B.n_sr * 256, 256, n_sm, 8), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_zero_bins");
  k_bin_hist<<<grid_for(B.n, 256, n_sm, resident_ctas(k_bin_hist, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_bin_hist");
  k_bin_scan<<<grid_for((uint64_t)B.n_sr * 512, 512, n_sm, resident_ctas(k_bin_scan, 512)), 512, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_bin_scan");
  k_scatter<<<grid_for(B.n, 256, n_sm, resident_ctas(k_scatter, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_scatter");
#if TPC_DET
  k_bin_sort<<<grid_for((uint64_t)B.n_sr * 256, 256, n_sm, resident_ctas(k_bin_sort, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_bin_sort");
#endif
  if (timers) cudaEventRecord(E.ev[1], st);
  if (flags & TPC_GRID_ONLY) {   // the tracks come from tpc_set_tracks
    if (timers) for (int i = 2; i <= 5; ++i) cudaEventRecord(E.ev[i], st);
    E.n_kernels = launches < TPC_MAX_KERNELS ? launches : TPC_MAX_KERNELS;
    return launches;
  }
  // ---- K2 neighbour finder
  k_neighbours<<<grid_for((uint64_t)(B.n / TPC_NF_TILE + B.n_sr) * TPC_NF_TILE, TPC_NF_TILE, n_sm, resident_ctas(k_neighbours, TPC_NF_TILE)), TPC_NF_TILE, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_neighbours");
  if (timers) cudaEventRecord(E.ev[2], st);
  // ---- K3 cleanup + seeds
  k_link_cleanup<<<grid_for(B.n, 256, n_sm, resident_ctas(k_link_cleanup, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_link_cleanup");
  k_seed_flags<<<grid_for((B.n + 3) / 4, TPC_SEED_BLOCK, n_sm, resident_ctas(k_seed_flags, TPC_SEED_BLOCK)), TPC_SEED_BLOCK, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_seed_flags");
  k_scan_partials<<<1, 1024, 0, st>>>(B.scan_partials, &B.cnt->n_sorted, 1024u, &B.cnt->n_seeds, B.max_seeds,
                                      &B.cnt->error, TPC_DEVERR_SEEDS);
  TPC_LAUNCH_CHECK("k_scan_partials");
  {
    const size_t smem = (size_t)B.n_rows * TPC_SEED_SLABS * sizeof(uint32_t);
    cudaFuncSetAttribute(k_seed_items, cudaFuncAttributeMaxDynamicSharedMemorySize,
                         (int)(TPC_MAX_ROWS * TPC_SEED_SLABS * sizeof(uint32_t)));
    k_seed_items<<<B.n_sectors, 1024, smem, st>>>(B);
  }
  TPC_LAUNCH_CHECK("k_seed_items");
  k_seed_write<<<grid_for((B.n + 3) / 4, TPC_SEED_BLOCK, n_sm, resident_ctas(k_seed_write, TPC_SEED_BLOCK)), TPC_SEED_BLOCK, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_seed_write");
  if (timers) cudaEventRecord(E.ev[3], st);
  // ---- K4 follower
  k_follow_up<<<grid_for(B.max_seeds, TPC_FOLLOW_BLOCK, n_sm, resident_ctas(k_follow_up, TPC_FOLLOW_BLOCK)), TPC_FOLLOW_BLOCK, 0, st>>>(B, F);
  TPC_LAUNCH_CHECK("k_follow_up");
  k_follow_refit<<<grid_for(B.max_seeds, TPC_FOLLOW_BLOCK, n_sm, resident_ctas(k_follow_refit, TPC_FOLLOW_BLOCK)), TPC_FOLLOW_BLOCK, 0, st>>>(B, F);
  TPC_LAUNCH_CHECK("k_follow_refit");
  k_follow_down<<<grid_for(B.max_seeds, TPC_FOLLOW_BLOCK, n_sm, resident_ctas(k_follow_down, TPC_FOLLOW_BLOCK)), TPC_FOLLOW_BLOCK, 0, st>>>(B, F);
  TPC_LAUNCH_CHECK("k_follow_down");
  if (timers) cudaEventRecord(E.ev[4], st);
  // ---- K5 ambiguity solving
  k_zero_owner<<<grid_for(B.n / 2 + 1, 256, n_sm, 8), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_zero_owner");
  k_sel_owner<<<grid_for((uint64_t)(B.max_seeds / 32 + 1) * TPC_SEL_BLOCK, TPC_SEL_BLOCK, n_sm, resident_ctas(k_sel_owner, TPC_SEL_BLOCK)), TPC_SEL_BLOCK, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_sel_owner");
  k_sel_masks<<<grid_for((uint64_t)(B.max_seeds / 32 + 1) * TPC_SEL_BLOCK, TPC_SEL_BLOCK, n_sm, resident_ctas(k_sel_masks, TPC_SEL_BLOCK)), TPC_SEL_BLOCK, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_sel_masks");
  k_sel_count<<<grid_for(B.max_seeds, 256, n_sm, resident_ctas(k_sel_count, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_sel_count");
  const uint32_t half = (B.scan_blocks + 1) / 2;
  k_scan_partials<<<1, 1024, 0, st>>>(B.scan_partials, &B.cnt->n_seeds, 256u, &B.cnt->n_tracks, B.max_tracks,
                                      &B.cnt->error, TPC_DEVERR_TRACKS);
  TPC_LAUNCH_CHECK("k_scan_partials");
  k_scan_partials<<<1, 1024, 0, st>>>(B.scan_partials + half, &B.cnt->n_seeds, 256u, &B.cnt->n_ids, B.max_ids,
                                      &B.cnt->error, TPC_DEVERR_TRACKS);
  TPC_LAUNCH_CHECK("k_scan_partials");
  k_sel_emit<<<grid_for((uint64_t)(B.max_seeds / TPC_EMIT_SPAN + 1) * 256, 256, n_sm, resident_ctas(k_sel_emit, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_sel_emit");
  k_sel_ids<<<grid_for((uint64_t)B.max_tracks * 32, 256, n_sm, resident_ctas(k_sel_ids, 256)), 256, 0, st>>>(B);
  TPC_LAUNCH_CHECK("k_sel_ids");
  if (timers) cudaEventRecord(E.ev[5], st);
  (void)flags;
  E.n_kernels = launches < TPC_MAX_KERNELS ? launches : TPC_MAX_KERNELS;
  return launches;
}

}  // namespace TPC_NS
