// tpc_oracle.cpp — the CPU ORACLE of the TPC sector tracking (test infrastructure; see
// tpc_oracle.h for what may load it and for the list of pins).
//
// Follows DESIGN.md "Readings" R0..R6 step by step, in the paper's order
// (CA seeding -> Kalman track following -> ambiguity solving; the
// cluster search grid; Phase-I selection criterion).  Plain loops, std::vector,
// one sector at a time.  No blocking, fusion or reordering beyond what the readings state.
// Build: g++ -O2 -std=c++17 -ffp-contract=off (rule D1: no FMA contraction, no fast-math).
#include "tpc_oracle.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <thread>
#include <vector>

#include "tpc_oracle_math.hpp"

namespace {

using tpc_oracle::KFGain;
using tpc_oracle::KFJac;
using tpc_oracle::KFState;

// ------------------------------------------------------------------ R0 geometry tables
// DESIGN.md R0 / rule D5: computed in double, rounded once to float.
// x_r = r_min + r*(r_max-r_min)/(n_rows-1)            (BASELINE.json config 1: radii linear)
// ymax_r = x_r * tan(half_angle)                       (trapezoidal sectors)
// ylim_r = ymax_r + 2 cm                               (acceptance of the grid / follower)
// cfield = -0.00299792458 * Bz                         (curvature per unit q/pT)
struct Tables {
  int n_rows = 0;
  std::vector<float> x, ymax, ylim;
  std::vector<int> ny;
  float dx_row = 0, cfield = 0;
};

Tables make_tables(const orc_geom& g, float grid_dy) {
  Tables t;
  t.n_rows = g.n_rows;
  t.x.resize(g.n_rows);
  t.ymax.resize(g.n_rows);
  t.ylim.resize(g.n_rows);
  t.ny.resize(g.n_rows);
  const double pitch = ((double)g.r_max - (double)g.r_min) / (double)(g.n_rows - 1);
  const double th = std::tan((double)g.sector_half_angle_deg * (3.14159265358979323846 / 180.0));
  for (int r = 0; r < g.n_rows; ++r) {
    const double xr = (double)g.r_min + r * pitch;
    const double ym = xr * th;
    t.x[r] = (float)xr;
    t.ymax[r] = (float)ym;
    t.ylim[r] = (float)(ym + 2.0);
    const int ny = (int)std::ceil(2.0 * (ym + 2.0) / (double)grid_dy);
    t.ny[r] = ny < 1 ? 1 : ny;
  }
  t.dx_row = (float)pitch;
  t.cfield = (float)(-0.00299792458 * (double)g.bz_tesla);
  return t;
}

// ------------------------------------------------------------------ per-sector working set
struct Sector {
  int sector = 0;
  // R1 grid
  std::vector<orc_row_desc> rows;      // [n_rows] (bin_ofs / clu_ofs local to the sector)
  std::vector<uint32_t> bin_start;     // local sorted positions, size n_bins+1
  std::vector<uint32_t> ids;           // sorted position -> original id
  std::vector<float> ys, zs;           // sorted position -> coordinates
  std::vector<int> row_of;             // sorted position -> row
  // R2/R3 links in sorted-position space
  std::vector<int32_t> up, dn, up2, dn2;
  // R4 seeds, R5 tracklets
  std::vector<orc_seed> seeds;
  std::vector<int32_t> seed_pos;       // sorted position of each start hit
  std::vector<orc_tracklet> tracklets;
  std::vector<int32_t> row_hit;        // [n_seeds][n_rows] sorted positions, -1 none
  // R6 output
  std::vector<orc_track> tracks;
  std::vector<uint32_t> cluster_ids;
  std::vector<uint8_t> shared;
  uint64_t n_ignored = 0, n_dropped = 0;
  double t_stage[5] = {0, 0, 0, 0, 0};
  std::vector<orc_trace_rec> trace;    // road-search decisions (only when orc_set_trace(1))
};

int g_trace = 0;  // set by orc_set_trace before orc_run; read-only while sectors run

inline int bin_coord(float v, float v0, float inv_d, int n) {
  int b = (int)std::floor((v - v0) * inv_d);
  if (b < 0) b = 0;
  if (b > n - 1) b = n - 1;
  return b;
}

// ------------------------------------------------------------------ R1 grid
void build_grid(Sector& S, const orc_cluster* cl, const std::vector<uint32_t>& members,
                const Tables& T, const orc_params& P) {
  const int R = T.n_rows;
  const float inv_dy = 1.0f / P.grid_dy, inv_dz = 1.0f / P.grid_dz;
  S.rows.assign(R, orc_row_desc{});
  // kept clusters per row, in ascending original index
  std::vector<std::vector<uint32_t>> per_row(R);
  for (uint32_t id : members) {
    const orc_cluster& c = cl[id];
    if (!(std::isfinite(c.y) && std::isfinite(c.z))) { S.n_ignored++; continue; }
    if (!(std::fabs(c.y) <= T.ylim[c.row])) { S.n_dropped++; continue; }
    per_row[c.row].push_back(id);
  }
  uint32_t bin_ofs = 0, clu_ofs = 0;
  S.bin_start.clear();
  for (int r = 0; r < R; ++r) {
    orc_row_desc& d = S.rows[r];
    d.ny = T.ny[r];
    d.y0 = -T.ylim[r];
    d.bin_ofs = bin_ofs;
    d.clu_ofs = clu_ofs;
    d.count = (uint32_t)per_row[r].size();
    if (per_row[r].empty()) { d.nz = 0; d.z0 = 0.0f; continue; }
    float zlo = cl[per_row[r][0]].z, zhi = zlo;
    for (uint32_t id : per_row[r]) { zlo = std::min(zlo, cl[id].z); zhi = std::max(zhi, cl[id].z); }
    d.z0 = zlo;
    int nz = (int)std::floor((zhi - zlo) * inv_dz) + 1;
    d.nz = nz < 1 ? 1 : nz;
    const uint32_t nb = (uint32_t)d.ny * (uint32_t)d.nz;
    // key = bin (z-major); stable sort keeps ascending original id inside a bin
    std::vector<std::pair<uint32_t, uint32_t>> keyed;
    keyed.reserve(per_row[r].size());
    for (uint32_t id : per_row[r]) {
      const int by = bin_coord(cl[id].y, d.y0, inv_dy, d.ny);
      const int bz = bin_coord(cl[id].z, d.z0, inv_dz, d.nz);
      keyed.emplace_back((uint32_t)bz * (uint32_t)d.ny + (uint32_t)by, id);
    }
    std::stable_sort(keyed.begin(), keyed.end(),
                     [](const auto& a, const auto& b) { return a.first < b.first; });
    std::vector<uint32_t> cnt(nb, 0);
    for (auto& k : keyed) cnt[k.first]++;
    uint32_t run = clu_ofs;
    for (uint32_t b = 0; b < nb; ++b) { S.bin_start.push_back(run); run += cnt[b]; }
    for (auto& k : keyed) {
      S.ids.push_back(k.second);
      S.ys.push_back(cl[k.second].y);
      S.zs.push_back(cl[k.second].z);
      S.row_of.push_back(r);
    }
    bin_ofs += nb;
    clu_ofs += d.count;
  }
  S.bin_start.push_back(clu_ofs);
}

// Visit every cluster of row r whose bin intersects [ylo,yhi] x [zlo,zhi] (a margin is added
// so that rounding can never hide a cluster that satisfies a window inequality; membership
// itself is always decided by the caller on the inequality, rule D3).
template <class F>
inline void for_window(const Sector& S, int r, float ylo, float yhi, float zlo, float zhi,
                       const orc_params& P, F&& f) {
  const orc_row_desc& d = S.rows[r];
  if (d.count == 0) return;
  const float inv_dy = 1.0f / P.grid_dy, inv_dz = 1.0f / P.grid_dz;
  const float my = 0.05f, mz = 0.05f + 1e-6f * std::max(std::fabs(zlo), std::fabs(zhi));
  const int by0 = bin_coord(ylo - my, d.y0, inv_dy, d.ny), by1 = bin_coord(yhi + my, d.y0, inv_dy, d.ny);
  const int bz0 = bin_coord(zlo - mz, d.z0, inv_dz, d.nz), bz1 = bin_coord(zhi + mz, d.z0, inv_dz, d.nz);
  for (int bz = bz0; bz <= bz1; ++bz) {
    const uint32_t b0 = d.bin_ofs + (uint32_t)bz * (uint32_t)d.ny + (uint32_t)by0;
    const uint32_t b1 = d.bin_ofs + (uint32_t)bz * (uint32_t)d.ny + (uint32_t)by1;
    for (uint32_t i = S.bin_start[b0]; i < S.bin_start[b1 + 1]; ++i) f((int32_t)i);
  }
}

// ------------------------------------------------------------------ R2 neighbour finder
// PAPER.md:27 "combinatorial seeding based on a cellular automaton".  DESIGN.md R2: for each
// cluster i on rows 1..R-2 the best (up j on row r+1, down k on row r-1) pair minimising the
// 3-point straightness d2 = dy^2 + dz^2, dy = (y_j-y_i)+(y_k-y_i), dz likewise, inside the
// windows; ties by (original id of j, original id of k) (rule D2).
void find_neighbours(Sector& S, const Tables& T, const orc_params& P) {
  const size_t n = S.ids.size();
  S.up.assign(n, -1);
  S.dn.assign(n, -1);
  const int R = T.n_rows;
  const float wy = P.nf_slope_y * T.dx_row, wz = P.nf_slope_z * T.dx_row;
  std::vector<int32_t> U, D;
  for (size_t i = 0; i < n; ++i) {
    const int r = S.row_of[i];
    if (r < 1 || r > R - 2) continue;
    const float yi = S.ys[i], zi = S.zs[i];
    const float ti = yi / T.x[r];
    const float ty = ti * T.dx_row;
    U.clear();
    D.clear();
    for_window(S, r + 1, (yi + ty) - wy, (yi + ty) + wy, zi - wz, zi + wz, P, [&](int32_t j) {
      if (std::fabs((S.ys[j] - yi) - ty) <= wy && std::fabs(S.zs[j] - zi) <= wz) U.push_back(j);
    });
    if (U.empty()) continue;
    for_window(S, r - 1, (yi - ty) - wy, (yi - ty) + wy, zi - wz, zi + wz, P, [&](int32_t k) {
      if (std::fabs((yi - S.ys[k]) - ty) <= wy && std::fabs(zi - S.zs[k]) <= wz) D.push_back(k);
    });
    bool have = false;
    float best = 0;
    int32_t bj = -1, bk = -1;
    for (int32_t j : U)
      for (int32_t k : D) {
        const float dy = (S.ys[j] - yi) + (S.ys[k] - yi);
        const float dz = (S.zs[j] - zi) + (S.zs[k] - zi);
        const float d2 = dy * dy + dz * dz;
        if (!(d2 <= P.nf_max_d2)) continue;
        bool better = !have || d2 < best;
        if (have && d2 == best) {
          if (S.ids[j] < S.ids[bj]) better = true;
          else if (S.ids[j] == S.ids[bj] && S.ids[k] < S.ids[bk]) better = true;
        }
        if (better) { have = true; best = d2; bj = j; bk = k; }
      }
    if (have) { S.up[i] = bj; S.dn[i] = bk; }
  }
}

// ------------------------------------------------------------------ R3 link cleanup
// One evolution step of the cellular automaton: keep reciprocal links only.
void cleanup_links(Sector& S) {
  const size_t n = S.ids.size();
  S.up2.assign(n, -1);
  S.dn2.assign(n, -1);
  for (size_t i = 0; i < n; ++i) {
    const int32_t u = S.up[i], d = S.dn[i];
    if (u >= 0 && S.dn[u] == (int32_t)i) S.up2[i] = u;
    if (d >= 0 && S.up[d] == (int32_t)i) S.dn2[i] = d;
  }
}

// ------------------------------------------------------------------ R4 start hits / seeds
// Start hit: no down link, an up link, chain length >= seed_min_len.  Seeds in ascending
// original id of the start hit (rule D4).
void find_seeds(Sector& S, const orc_params& P) {
  const size_t n = S.ids.size();
  std::vector<std::pair<uint32_t, int32_t>> starts;  // (orig id, sorted pos)
  for (size_t i = 0; i < n; ++i)
    if (S.dn2[i] < 0 && S.up2[i] >= 0) starts.emplace_back(S.ids[i], (int32_t)i);
  std::sort(starts.begin(), starts.end());
  for (auto& st : starts) {
    int len = 1;
    for (int32_t c = S.up2[st.second]; c >= 0; c = S.up2[c]) ++len;
    if (len < P.seed_min_len) continue;
    orc_seed sd;
    sd.start_id = st.first;
    sd.len = len;
    sd.sector = S.sector;
    sd.row = S.row_of[st.second];
    S.seeds.push_back(sd);
    S.seed_pos.push_back(st.second);
  }
}

// ------------------------------------------------------------------ R5 track following
// "the track following fits all seeds and propagates them through the TPC
// volume using the Kalman filter picking up more clusters of the track".  DESIGN.md R5.
struct FollowCtx {
  const Sector& S;
  const Tables& T;
  const orc_params& P;
  float vy, vz;
  std::vector<orc_trace_rec>* trace = nullptr;  // observation only: never read by the algorithm
  int32_t trace_seed = 0;
};

inline void init_cov(KFState<float>& st, const FollowCtx& X) {
  for (int i = 0; i < 15; ++i) st.c[i] = 0.0f;
  st.c[0] = X.vy;
  st.c[2] = X.vz;
  st.c[5] = X.P.init_var_sinphi;
  st.c[9] = X.P.init_var_tanl;
  st.c[14] = X.P.init_var_qpt;
}

inline float clampf(float v, float lo, float hi) { return v < lo ? lo : (v > hi ? hi : v); }

// Best candidate on row r for the predicted state: minimum (chi2, original id) among the
// clusters inside the road (R5.3).  Returns the sorted position or -1; chi2 in *chi2_out.
inline int32_t pick_cluster(const FollowCtx& X, int r, const KFState<float>& st, const KFGain<float>& g,
                            float* chi2_out) {
  const orc_params& P = X.P;
  const float ry = clampf(P.road_nsigma * std::sqrt(st.c[0] + X.vy), P.road_min, P.road_max);
  const float rz = clampf(P.road_nsigma * std::sqrt(st.c[2] + X.vz), P.road_min, P.road_max);
  int32_t best = -1;
  float best_chi2 = 0;
  for_window(X.S, r, st.y - ry, st.y + ry, st.z - rz, st.z + rz, P, [&](int32_t c) {
    if (!(std::fabs(X.S.ys[c] - st.y) <= ry && std::fabs(X.S.zs[c] - st.z) <= rz)) return;
    const float chi2 = tpc_oracle::kf_chi2(st, g, X.S.ys[c], X.S.zs[c]);
    if (best < 0 || chi2 < best_chi2 || (chi2 == best_chi2 && X.S.ids[c] < X.S.ids[best])) {
      best = c;
      best_chi2 = chi2;
    }
  });
  *chi2_out = best_chi2;
  return best;
}

// Extrapolate from row r_from (exclusive) in direction dir (+1 up, -1 down) picking up
// clusters (R5.3 / R5.6).  `on_hit` is called after every accepted update.
template <class F>
inline void extrapolate(const FollowCtx& X, KFState<float>& st, int r_from, int dir, int32_t* hits,
                        float* chi2_acc, int* n_acc, F&& on_hit) {
  const orc_params& P = X.P;
  const float dx = dir > 0 ? X.T.dx_row : -X.T.dx_row;
  int gap = 0;
  for (int r = r_from + dir; r >= 0 && r < X.T.n_rows; r += dir) {
    if (!tpc_oracle::kf_propagate(st, dx, X.T.cfield, P.max_sinphi)) break;
    bool got = false;
    orc_trace_rec tr;
    if (X.trace) {
      tr.seed = X.trace_seed; tr.row = r; tr.dir = dir; tr.searched = 0;
      tr.y = st.y; tr.z = st.z; tr.c00 = st.c[0]; tr.c10 = st.c[1]; tr.c11 = st.c[2];
      tr.chi2 = 0; tr.picked_id = -1; tr.accepted = 0;
    }
    if (std::fabs(st.y) <= X.T.ylim[r]) {
      const KFGain<float> g = tpc_oracle::kf_gain(st, X.vy, X.vz);
      float chi2 = 0;
      const int32_t c = pick_cluster(X, r, st, g, &chi2);
      if (X.trace) {
        tr.searched = 1; tr.chi2 = chi2; tr.picked_id = c < 0 ? -1 : (int32_t)X.S.ids[c];
        tr.accepted = (c >= 0 && chi2 <= P.chi2_max_hit) ? 1 : 0;
      }
      if (c >= 0 && chi2 <= P.chi2_max_hit) {
        const bool stop = tpc_oracle::kf_update(st, g, X.S.ys[c], X.S.zs[c], P.max_sinphi, P.max_qpt);
        hits[r] = c;
        *chi2_acc = *chi2_acc + chi2;
        *n_acc = *n_acc + 1;
        on_hit(r);
        got = true;
        gap = 0;
        if (X.trace) X.trace->push_back(tr);
        if (stop) break;
      }
    }
    if (X.trace && !got) X.trace->push_back(tr);
    if (!got) {
      ++gap;
      if (gap > P.max_gap_follow) break;
    }
  }
}

void follow_seed(const FollowCtx& X, int32_t start, int seed_len, uint32_t seed_id, orc_tracklet& out,
                 int32_t* hits /*[n_rows]*/) {
  const Sector& S = X.S;
  const orc_params& P = X.P;
  const int R = X.T.n_rows;
  const float dxr = X.T.dx_row;
  for (int r = 0; r < R; ++r) hits[r] = -1;
  std::memset(&out, 0, sizeof(out));
  out.seed_id = seed_id;
  out.sector = S.sector;
  out.seed_len = seed_len;

  // R5.1 init from the first two chain clusters
  const int r0 = S.row_of[start];
  const int32_t c1 = S.up2[start];
  KFState<float> st;
  {
    const float dy = S.ys[c1] - S.ys[start];
    const float dl = std::sqrt(dxr * dxr + dy * dy);
    st.y = S.ys[start];
    st.z = S.zs[start];
    st.s = dy / dl;
    st.t = (S.zs[c1] - S.zs[start]) / dl;
    st.q = 0.0f;
    init_cov(st, X);
  }
  hits[r0] = start;
  int r_out = r0;
  float snap_s = st.s, snap_t = st.t, snap_q = st.q;
  float chi2_up = 0;
  int n_up = 1;
  bool stopped = false;

  // R5.2 chain fit (up), no chi2 cut
  {
    int r = r0;
    for (int32_t c = c1; c >= 0; c = S.up2[c]) {
      ++r;
      if (!tpc_oracle::kf_propagate(st, dxr, X.T.cfield, P.max_sinphi)) { stopped = true; break; }
      const KFGain<float> g = tpc_oracle::kf_gain(st, X.vy, X.vz);
      const bool stop = tpc_oracle::kf_update(st, g, S.ys[c], S.zs[c], P.max_sinphi, P.max_qpt);
      hits[r] = c;
      r_out = r;
      ++n_up;
      snap_s = st.s; snap_t = st.t; snap_q = st.q;
      if (stop) { stopped = true; break; }
    }
  }
  // R5.3 extrapolate up
  if (!stopped)
    extrapolate(X, st, r_out, +1, hits, &chi2_up, &n_up, [&](int r) {
      r_out = r;
      snap_s = st.s; snap_t = st.t; snap_q = st.q;
    });

  // R5.4 turn at the outermost accepted hit
  {
    const int32_t co = hits[r_out];
    st.y = S.ys[co];
    st.z = S.zs[co];
    st.s = snap_s;
    st.t = snap_t;
    st.q = snap_q;
    init_cov(st, X);
  }
  float chi2 = 0;
  int nh = 1;
  int r_in = r_out;
  KFState<float> st_in = st;  // state right after the innermost accepted hit
  stopped = false;

  // R5.5 refit down through the recorded hits
  for (int r = r_out - 1; r >= r0; --r) {
    if (!tpc_oracle::kf_propagate(st, -dxr, X.T.cfield, P.max_sinphi)) { stopped = true; break; }
    const int32_t c = hits[r];
    if (c < 0) continue;
    const KFGain<float> g = tpc_oracle::kf_gain(st, X.vy, X.vz);
    const float c2 = tpc_oracle::kf_chi2(st, g, S.ys[c], S.zs[c]);
    const bool stop = tpc_oracle::kf_update(st, g, S.ys[c], S.zs[c], P.max_sinphi, P.max_qpt);
    chi2 = chi2 + c2;
    ++nh;
    r_in = r;
    st_in = st;
    if (stop) { stopped = true; break; }
  }
  // hits below the point where the refit ended are not part of the tracklet
  for (int r = r0; r < r_in; ++r) hits[r] = -1;

  // R5.6 extrapolate down
  if (!stopped)
    extrapolate(X, st, r_in, -1, hits, &chi2, &nh, [&](int r) {
      r_in = r;
      st_in = st;
    });

  // R5.7 output
  if (nh >= P.min_hits_tracklet) {
    out.n_hits = nh;
    out.row_first = r_in;
    out.row_last = r_out;
    out.x = X.T.x[r_in];
    out.p[0] = st_in.y; out.p[1] = st_in.z; out.p[2] = st_in.s; out.p[3] = st_in.t; out.p[4] = st_in.q;
    for (int i = 0; i < 15; ++i) out.c[i] = st_in.c[i];
    out.chi2 = chi2;
  } else {
    out.n_hits = 0;
    for (int r = 0; r < R; ++r) hits[r] = -1;
  }
}

void follow_all(Sector& S, const Tables& T, const orc_params& P) {
  FollowCtx X{S, T, P, P.err_y * P.err_y, P.err_z * P.err_z};
  if (g_trace) X.trace = &S.trace;
  const size_t ns = S.seeds.size();
  S.tracklets.resize(ns);
  S.row_hit.assign(ns * (size_t)T.n_rows, -1);
  for (size_t k = 0; k < ns; ++k) {
    X.trace_seed = (int32_t)k;
    follow_seed(X, S.seed_pos[k], S.seeds[k].len, S.seeds[k].start_id, S.tracklets[k],
                &S.row_hit[k * (size_t)T.n_rows]);
  }
}

// ------------------------------------------------------------------ R6 ambiguity solving
// "identifies the best instance of each track, assigns all clusters to this
// instance and removes the clones"; "a configurable fraction of a track's clusters, by
// default 10%, are allowed to be shared".  PAPER.md:57 (Phase I): "more priority is given to
// the track with smaller global chi2, reducing the weight of the track length.  Shared
// clusters are counted starting at the outermost pad row".  DESIGN.md R6.
inline uint32_t orderable_u32(float f) {
  uint32_t b;
  std::memcpy(&b, &f, 4);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

inline uint64_t tracklet_key(int n_hits, float chi2, uint32_t seed_id, const orc_params& P) {
  const int ndf = 2 * n_hits - 5;
  const float Q = (float)n_hits - P.sel_chi2_weight * (chi2 / (float)ndf);
  return ((uint64_t)orderable_u32(Q) << 32) | (uint64_t)(0xFFFFFFFFu - seed_id);
}

// tracklets: n_t entries; row_hit[k*R + r] = cluster index (in [0,n_idx)) or -1; to_orig maps a
// cluster index to the original id (nullptr = identity).
void select_tracks(int R, const orc_params& P, size_t n_idx, size_t n_t, const orc_tracklet* tl,
                   const int32_t* row_hit, const uint32_t* to_orig, std::vector<orc_track>& tracks,
                   std::vector<uint32_t>& ids, std::vector<uint8_t>& shared) {
  // R6.1 weight, R6.2 owner = max key over the tracklets containing the cluster
  std::vector<uint64_t> key(n_t, 0), owner(n_idx, 0);
  for (size_t k = 0; k < n_t; ++k) {
    if (tl[k].n_hits <= 0) continue;
    key[k] = tracklet_key(tl[k].n_hits, tl[k].chi2, tl[k].seed_id, P);
    for (int r = tl[k].row_first; r <= tl[k].row_last; ++r) {
      const int32_t c = row_hit[k * (size_t)R + r];
      if (c >= 0 && key[k] > owner[c]) owner[c] = key[k];
    }
  }
  // R6.3 walk from the outermost row inward, R6.4 emit
  std::vector<int32_t> seg_c;
  std::vector<uint8_t> seg_s;
  for (size_t k = 0; k < n_t; ++k) {
    if (tl[k].n_hits <= 0) continue;
    int n_acc = 0, n_sh = 0, gap = 0, segment = 0, seg_last = -1, seg_first = -1;
    seg_c.clear();
    seg_s.clear();
    auto close = [&]() {
      if (n_acc >= P.min_hits_track) {
        orc_track t;
        std::memset(&t, 0, sizeof(t));
        t.x = tl[k].x;
        for (int i = 0; i < 5; ++i) t.p[i] = tl[k].p[i];
        for (int i = 0; i < 15; ++i) t.c[i] = tl[k].c[i];
        t.chi2 = tl[k].chi2;
        t.cluster_ofs = (uint32_t)ids.size();
        t.seed_id = tl[k].seed_id;
        t.n_clusters = n_acc;
        t.n_shared = n_sh;
        t.sector = tl[k].sector;
        t.row_first = seg_first;
        t.row_last = seg_last;
        t.flags = (seg_first == tl[k].row_first) ? 0 : 1;
        t.n_hits_tracklet = tl[k].n_hits;
        t.segment = segment;
        tracks.push_back(t);
        for (int i = (int)seg_c.size() - 1; i >= 0; --i) {  // ascending in row
          ids.push_back(to_orig ? to_orig[seg_c[i]] : (uint32_t)seg_c[i]);
          shared.push_back(seg_s[i]);
        }
        ++segment;
      }
      n_acc = 0; n_sh = 0; seg_last = -1; seg_first = -1;
      seg_c.clear();
      seg_s.clear();
    };
    for (int r = tl[k].row_last; r >= tl[k].row_first; --r) {
      int32_t c = row_hit[k * (size_t)R + r];
      bool sh = false;
      if (c >= 0 && owner[c] != key[k]) {
        // R6.3: Phase-I running fraction counted from the outermost row, or, as the
        // variant of SURVEY.md 8(f), the fixed cap of the rule before Phase I (shared_fixed_cap)
        const int64_t budget = P.shared_fixed_cap ? (int64_t)P.shared_permille * tl[k].n_hits
                                                  : (int64_t)P.shared_permille * (n_acc + 1);
        if ((int64_t)(n_sh + 1) * 1000 <= budget) sh = true;
        else c = -1;
      }
      if (c >= 0) {
        if (n_acc == 0) seg_last = r;
        seg_first = r;
        ++n_acc;
        if (sh) ++n_sh;
        seg_c.push_back(c);
        seg_s.push_back(sh ? 1 : 0);
        gap = 0;
      } else {
        ++gap;
        if (gap > P.max_gap_select && n_acc > 0) close();
      }
    }
    close();
  }
}

double now_s() {
  return std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

void run_sector(Sector& S, const orc_cluster* cl, const std::vector<uint32_t>& members, const Tables& T,
                const orc_params& P) {
  double t0 = now_s();
  build_grid(S, cl, members, T, P);
  double t1 = now_s();
  find_neighbours(S, T, P);
  double t2 = now_s();
  cleanup_links(S);
  find_seeds(S, P);
  double t3 = now_s();
  follow_all(S, T, P);
  double t4 = now_s();
  select_tracks(T.n_rows, P, S.ids.size(), S.tracklets.size(), S.tracklets.data(), S.row_hit.data(),
                S.ids.data(), S.tracks, S.cluster_ids, S.shared);
  double t5 = now_s();
  S.t_stage[0] = t1 - t0; S.t_stage[1] = t2 - t1; S.t_stage[2] = t3 - t2;
  S.t_stage[3] = t4 - t3; S.t_stage[4] = t5 - t4;
}

}  // namespace

struct orc_result {
  uint64_t n = 0;
  int n_rows = 0, sector_lo = 0, sector_hi = 0;
  uint64_t n_bad = 0;
  std::vector<Sector> sectors;
};

extern "C" {

void orc_default_params(orc_params* p) {
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
  p->shared_fixed_cap = 0;
  p->grid_dy = 2.0f; p->grid_dz = 2.0f;
}

orc_result* orc_run(const orc_cluster* clusters, uint64_t n, const orc_geom* g, const orc_params* pp,
                    int sector_lo, int sector_hi, int n_threads) {
  if (!g || (!clusters && n) || g->n_rows < 3 || g->n_rows > 255 || g->n_sectors < 1 || n >= (1ull << 31))
    return nullptr;
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  if (sector_lo < 0) sector_lo = 0;
  if (sector_hi > g->n_sectors) sector_hi = g->n_sectors;
  const Tables T = make_tables(*g, P.grid_dy);
  auto* res = new orc_result();
  res->n = n;
  res->n_rows = g->n_rows;
  res->sector_lo = sector_lo;
  res->sector_hi = sector_hi;
  const int ns = sector_hi > sector_lo ? sector_hi - sector_lo : 0;
  res->sectors.resize(ns);
  std::vector<std::vector<uint32_t>> members(ns);
  for (uint64_t i = 0; i < n; ++i) {
    const orc_cluster& c = clusters[i];
    if (c.sector >= g->n_sectors || c.row >= g->n_rows) { res->n_bad++; continue; }
    if (c.sector >= sector_lo && c.sector < sector_hi) members[c.sector - sector_lo].push_back((uint32_t)i);
  }
  for (int s = 0; s < ns; ++s) res->sectors[s].sector = sector_lo + s;
  if (n_threads <= 1) {
    for (int s = 0; s < ns; ++s) run_sector(res->sectors[s], clusters, members[s], T, P);
  } else {
    std::vector<std::thread> thr;
    for (int t = 0; t < n_threads; ++t)
      thr.emplace_back([&, t]() {
        for (int s = t; s < ns; s += n_threads) run_sector(res->sectors[s], clusters, members[s], T, P);
      });
    for (auto& th : thr) th.join();
  }
  return res;
}

void orc_free(orc_result* r) { delete r; }

void orc_sizes(const orc_result* r, uint64_t out[10]) {
  for (int i = 0; i < 10; ++i) out[i] = 0;
  out[0] = (uint64_t)r->sectors.size() * r->n_rows;
  out[8] = r->n_bad;
  for (const Sector& S : r->sectors) {
    out[1] += S.bin_start.empty() ? 0 : S.bin_start.size() - 1;
    out[2] += S.ids.size();
    out[3] += S.seeds.size();
    out[4] += S.tracks.size();
    out[5] += S.cluster_ids.size();
    out[6] += S.n_ignored;
    out[7] += S.n_dropped;
    for (const orc_tracklet& t : S.tracklets) out[9] += t.n_hits > 0;
  }
}

void orc_set_trace(int on) { g_trace = on; }

uint64_t orc_trace_size(const orc_result* r) {
  uint64_t n = 0;
  for (const Sector& S : r->sectors) n += S.trace.size();
  return n;
}

void orc_fetch_trace(const orc_result* r, orc_trace_rec* out) {
  size_t k = 0;
  int32_t seed_base = 0;
  for (const Sector& S : r->sectors) {
    for (const orc_trace_rec& t : S.trace) {
      out[k] = t;
      out[k++].seed += seed_base;   // index into the concatenated seed / tracklet arrays
    }
    seed_base += (int32_t)S.seeds.size();
  }
}

void orc_stage_seconds(const orc_result* r, double out[5]) {
  for (int i = 0; i < 5; ++i) out[i] = 0;
  for (const Sector& S : r->sectors)
    for (int i = 0; i < 5; ++i) out[i] += S.t_stage[i];
}

// Grid of the processed sectors, concatenated sector-major with global offsets.
void orc_fetch_grid(const orc_result* r, orc_row_desc* rows, uint32_t* bin_start, uint32_t* sorted_ids) {
  uint32_t bin_base = 0, clu_base = 0;
  size_t row_i = 0;
  for (const Sector& S : r->sectors) {
    for (int rr = 0; rr < r->n_rows; ++rr, ++row_i) {
      if (!rows) continue;
      rows[row_i] = S.rows[rr];
      rows[row_i].bin_ofs += bin_base;
      rows[row_i].clu_ofs += clu_base;
    }
    const size_t nb = S.bin_start.empty() ? 0 : S.bin_start.size() - 1;
    if (bin_start)
      for (size_t b = 0; b < nb; ++b) bin_start[bin_base + b] = S.bin_start[b] + clu_base;
    if (sorted_ids)
      for (size_t i = 0; i < S.ids.size(); ++i) sorted_ids[clu_base + i] = S.ids[i];
    bin_base += (uint32_t)nb;
    clu_base += (uint32_t)S.ids.size();
  }
  if (bin_start) bin_start[bin_base] = clu_base;
}

void orc_fetch_links(const orc_result* r, int32_t* up, int32_t* dn, int32_t* up2, int32_t* dn2) {
  int32_t* outs[4] = {up, dn, up2, dn2};
  for (int a = 0; a < 4; ++a)
    if (outs[a])
      for (uint64_t i = 0; i < r->n; ++i) outs[a][i] = -1;
  for (const Sector& S : r->sectors) {
    const std::vector<int32_t>* src[4] = {&S.up, &S.dn, &S.up2, &S.dn2};
    for (int a = 0; a < 4; ++a) {
      if (!outs[a]) continue;
      for (size_t i = 0; i < S.ids.size(); ++i) {
        const int32_t v = (*src[a])[i];
        outs[a][S.ids[i]] = v < 0 ? -1 : (int32_t)S.ids[v];
      }
    }
  }
}

void orc_fetch_seeds(const orc_result* r, orc_seed* seeds) {
  size_t k = 0;
  for (const Sector& S : r->sectors)
    for (const orc_seed& s : S.seeds) seeds[k++] = s;
}

void orc_fetch_tracklets(const orc_result* r, orc_tracklet* t, int32_t* row_hit) {
  size_t k = 0;
  for (const Sector& S : r->sectors) {
    for (size_t i = 0; i < S.tracklets.size(); ++i, ++k) {
      if (t) t[k] = S.tracklets[i];
      if (row_hit)
        for (int rr = 0; rr < r->n_rows; ++rr) {
          const int32_t v = S.row_hit[i * (size_t)r->n_rows + rr];
          row_hit[k * (size_t)r->n_rows + rr] = v < 0 ? -1 : (int32_t)S.ids[v];
        }
    }
  }
}

void orc_fetch_tracks(const orc_result* r, orc_track* t, uint32_t* cluster_ids, uint8_t* shared) {
  size_t k = 0, ofs = 0;
  for (const Sector& S : r->sectors) {
    for (size_t i = 0; i < S.tracks.size(); ++i, ++k) {
      if (!t) continue;
      t[k] = S.tracks[i];
      t[k].cluster_ofs += (uint32_t)ofs;
    }
    if (cluster_ids) std::memcpy(cluster_ids + ofs, S.cluster_ids.data(), S.cluster_ids.size() * 4);
    if (shared) std::memcpy(shared + ofs, S.shared.data(), S.shared.size());
    ofs += S.cluster_ids.size();
  }
}

// ------------------------------------------------------------------ single-step entry points
void orc_geom_tables(const orc_geom* g, float* x, float* ymax, float* consts) {
  const Tables T = make_tables(*g, 2.0f);
  for (int r = 0; r < g->n_rows; ++r) {
    if (x) x[r] = T.x[r];
    if (ymax) ymax[r] = T.ymax[r];
  }
  if (consts) { consts[0] = T.dx_row; consts[1] = T.cfield; }
}

}  // extern "C"
template <class T>
static int propagate_any(T* state, T dx, T cfield, T max_sinphi, T* jac6) {
  KFState<T> st;
  st.y = state[0]; st.z = state[1]; st.s = state[2]; st.t = state[3]; st.q = state[4];
  for (int i = 0; i < 15; ++i) st.c[i] = state[5 + i];
  KFJac<T> J;
  const bool ok = tpc_oracle::kf_propagate(st, dx, cfield, max_sinphi, &J);
  if (!ok) return 0;
  state[0] = st.y; state[1] = st.z; state[2] = st.s; state[3] = st.t; state[4] = st.q;
  for (int i = 0; i < 15; ++i) state[5 + i] = st.c[i];
  if (jac6) { jac6[0] = J.f02; jac6[1] = J.f04; jac6[2] = J.f12; jac6[3] = J.f13; jac6[4] = J.f14; jac6[5] = J.f24; }
  return 1;
}
extern "C" {
int orc_propagate_f(float* s, float dx, float c, float m, float* j) { return propagate_any<float>(s, dx, c, m, j); }
int orc_propagate_d(double* s, double dx, double c, double m, double* j) { return propagate_any<double>(s, dx, c, m, j); }

}  // extern "C"
template <class T>
static T update_any(T* state, T ym, T zm, T vy, T vz, T max_sinphi, T max_qpt, int* stop) {
  KFState<T> st;
  st.y = state[0]; st.z = state[1]; st.s = state[2]; st.t = state[3]; st.q = state[4];
  for (int i = 0; i < 15; ++i) st.c[i] = state[5 + i];
  const KFGain<T> g = tpc_oracle::kf_gain(st, vy, vz);
  const T chi2 = tpc_oracle::kf_chi2(st, g, ym, zm);
  const bool s = tpc_oracle::kf_update(st, g, ym, zm, max_sinphi, max_qpt);
  if (stop) *stop = s ? 1 : 0;
  state[0] = st.y; state[1] = st.z; state[2] = st.s; state[3] = st.t; state[4] = st.q;
  for (int i = 0; i < 15; ++i) state[5 + i] = st.c[i];
  return chi2;
}
extern "C" {
float orc_update_f(float* s, float ym, float zm, float vy, float vz, float ms, float mq, int* stop) {
  return update_any<float>(s, ym, zm, vy, vz, ms, mq, stop);
}
double orc_update_d(double* s, double ym, double zm, double vy, double vz, double ms, double mq, int* stop) {
  return update_any<double>(s, ym, zm, vy, vz, ms, mq, stop);
}

// Fit a given list of hits exactly as follow_seed does for hits it has accepted: the hits are
// put into a one-sector working set whose link chain is the list itself, roads are disabled
// by making every other row empty, so R5.1, R5.2, R5.4, R5.5 run and R5.3/R5.6 find nothing.
float orc_fit_hits(const orc_geom* g, const orc_params* pp, const int32_t* rows, const float* y,
                   const float* z, int n, float* out_state) {
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  P.min_hits_tracklet = 2;
  const Tables T = make_tables(*g, P.grid_dy);
  if (n < 2 || rows[1] != rows[0] + 1) return -1.0f;
  std::vector<orc_cluster> cl(n);
  std::vector<uint32_t> members(n);
  for (int i = 0; i < n; ++i) {
    cl[i].y = y[i]; cl[i].z = z[i]; cl[i].q = 0; cl[i].sector = 0; cl[i].row = (uint8_t)rows[i]; cl[i].flags = 0;
    members[i] = (uint32_t)i;
  }
  Sector S;
  build_grid(S, cl.data(), members, T, P);
  // chain = the first run of consecutive rows; later hits are found by the road search
  const size_t ns = S.ids.size();
  S.up.assign(ns, -1); S.dn.assign(ns, -1); S.up2.assign(ns, -1); S.dn2.assign(ns, -1);
  std::vector<int32_t> pos_of(n, -1);
  for (size_t i = 0; i < ns; ++i) pos_of[S.ids[i]] = (int32_t)i;
  int chain = 1;
  while (chain < n && rows[chain] == rows[chain - 1] + 1) ++chain;
  for (int i = 0; i + 1 < chain; ++i) {
    S.up2[pos_of[i]] = pos_of[i + 1];
    S.dn2[pos_of[i + 1]] = pos_of[i];
  }
  FollowCtx X{S, T, P, P.err_y * P.err_y, P.err_z * P.err_z};
  orc_tracklet tl;
  std::vector<int32_t> hits(T.n_rows);
  follow_seed(X, pos_of[0], chain, 0, tl, hits.data());
  if (tl.n_hits <= 0) return -1.0f;
  out_state[0] = tl.x;
  for (int i = 0; i < 5; ++i) out_state[1 + i] = tl.p[i];
  for (int i = 0; i < 15; ++i) out_state[6 + i] = tl.c[i];
  out_state[21] = (float)tl.n_hits;
  out_state[22] = (float)tl.row_first;
  return tl.chi2;
}

// R8 sector-track refit ("a sector track refit at the beginning of the track merging
// was added, guaranteeing reasonable initial parameters"; reading R8).  A pure Kalman fit
// of a GIVEN cluster list (rows strictly ascending, holes allowed), no search and no chi2 cut:
//   R8.1 init at the first cluster from the first two (dx = row distance * pitch), C = initial diagonal
//   R8.2 outward: row by row to every further cluster (pure propagation on rows in between), update
//   R8.3 turn at the last cluster as R5.4 (s,t,q after its update; y,z measured; C reset)
//   R8.4 inward: back through the clusters to the first one, chi2 accumulated in this pass
// out_state = x, p[5], c[15], n at the first cluster's row, then x_out, p_out[5], c_out[15]: the state
// after the outward pass R8.2 at the last cluster (43 floats).  Returns chi2, or -1 if a propagation
// or an update left the |sin phi| range (the fit failed; out_state untouched).
float orc_refit_hits(const orc_geom* g, const orc_params* pp, const int32_t* rows, const float* y,
                     const float* z, int n, float* out_state) {
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  const Tables T = make_tables(*g, P.grid_dy);
  if (n < 2) return -1.0f;
  const float vy = P.err_y * P.err_y, vz = P.err_z * P.err_z;
  KFState<float> st;
  auto reset_cov = [&]() {
    for (int i = 0; i < 15; ++i) st.c[i] = 0.0f;
    st.c[0] = vy; st.c[2] = vz; st.c[5] = P.init_var_sinphi; st.c[9] = P.init_var_tanl; st.c[14] = P.init_var_qpt;
  };
  {  // R8.1
    const float dx = (float)(rows[1] - rows[0]) * T.dx_row;   // the pitch the propagation steps use
    const float dy = y[1] - y[0];
    const float dl = std::sqrt(dx * dx + dy * dy);
    st.y = y[0]; st.z = z[0];
    st.s = dy / dl;
    st.t = (z[1] - z[0]) / dl;
    st.q = 0.0f;
    reset_cov();
  }
  float snap_s = st.s, snap_t = st.t, snap_q = st.q;
  for (int i = 1; i < n; ++i) {  // R8.2
    for (int r = rows[i - 1]; r < rows[i]; ++r)
      if (!tpc_oracle::kf_propagate(st, T.dx_row, T.cfield, P.max_sinphi)) return -1.0f;
    const KFGain<float> gn = tpc_oracle::kf_gain(st, vy, vz);
    if (tpc_oracle::kf_update(st, gn, y[i], z[i], P.max_sinphi, P.max_qpt)) return -1.0f;
    snap_s = st.s; snap_t = st.t; snap_q = st.q;
  }
  // the OUTER end (used by the merging, R9): the state after the outward pass at the last cluster
  const KFState<float> st_out = st;
  st.y = y[n - 1]; st.z = z[n - 1]; st.s = snap_s; st.t = snap_t; st.q = snap_q;  // R8.3
  reset_cov();
  float chi2 = 0.0f;
  for (int i = n - 2; i >= 0; --i) {  // R8.4
    for (int r = rows[i + 1]; r > rows[i]; --r)
      if (!tpc_oracle::kf_propagate(st, -T.dx_row, T.cfield, P.max_sinphi)) return -1.0f;
    const KFGain<float> gn = tpc_oracle::kf_gain(st, vy, vz);
    const float c2 = tpc_oracle::kf_chi2(st, gn, y[i], z[i]);
    if (tpc_oracle::kf_update(st, gn, y[i], z[i], P.max_sinphi, P.max_qpt)) return -1.0f;
    chi2 = chi2 + c2;
  }
  out_state[0] = T.x[rows[0]];
  out_state[1] = st.y; out_state[2] = st.z; out_state[3] = st.s; out_state[4] = st.t; out_state[5] = st.q;
  for (int i = 0; i < 15; ++i) out_state[6 + i] = st.c[i];
  out_state[21] = (float)n;
  out_state[22] = T.x[rows[n - 1]];
  out_state[23] = st_out.y; out_state[24] = st_out.z; out_state[25] = st_out.s; out_state[26] = st_out.t; out_state[27] = st_out.q;
  for (int i = 0; i < 15; ++i) out_state[28 + i] = st_out.c[i];
  return chi2;
}

orc_result* orc_select_only(const orc_geom* g, const orc_params* pp, uint64_t n_clusters, int n_tracklets,
                            const int32_t* row_hit, const int32_t* n_hits, const float* chi2,
                            const uint32_t* seed_id) {
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  const int R = g->n_rows;
  auto* res = new orc_result();
  res->n = n_clusters;
  res->n_rows = R;
  res->sector_hi = 1;
  res->sectors.resize(1);
  Sector& S = res->sectors[0];
  S.tracklets.resize(n_tracklets);
  for (int k = 0; k < n_tracklets; ++k) {
    orc_tracklet& t = S.tracklets[k];
    std::memset(&t, 0, sizeof(t));
    t.n_hits = n_hits[k];
    t.chi2 = chi2[k];
    t.seed_id = seed_id[k];
    t.row_first = R; t.row_last = -1;
    for (int r = 0; r < R; ++r)
      if (row_hit[k * (size_t)R + r] >= 0) { t.row_first = std::min(t.row_first, r); t.row_last = std::max(t.row_last, r); }
  }
  select_tracks(R, P, n_clusters, n_tracklets, S.tracklets.data(), row_hit, nullptr, S.tracks, S.cluster_ids, S.shared);
  return res;
}

}  // extern "C"
