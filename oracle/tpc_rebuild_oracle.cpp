// tpc_rebuild_oracle.cpp — CPU ORACLE of the Phase-II track rebuild, reading R11 of DESIGN.md (TEST
// INFRASTRUCTURE, see tpc_oracle.h for what may load it; shares no code with the CUDA path).
//
// PAPER.md:59 (section 3, Phase II): "the track is practically rebuilt during iterations 2 and 3 of
// the fit, i. e. the cluster-to-track attachment is performed again from scratch.  Instead of
// performing a chi2 cut for cluster rejection in the second iteration, the fast cluster search grid
// from the sector tracking is queried for all clusters compatible with the chi2 cut and all candidates
// together with their residuals are written to temporary storage.  When iteration 2 has finished for
// all tracks, a second ambiguity solving step is executed. [...] candidates are assigned to the track
// with the best combination of global chi2 and track length [...] allowing a configurable amount of
// cluster sharing.  However, tracks failing to get their best candidate attached are still eligible
// for the second candidate, and so on.  Only after this final cluster-to-track attachment, the third
// fit iteration is executed"; "it performs a simple chi2 cut for final cluster rejection
// without interpolation."  The reading R11, step by step:
//
//   PATH of a merged track: the (sector, row) steps it passes: every row of every segment from its
//   first to its last row, plus the rows of the hole between two consecutive segments of one sector.
//   Transport between consecutive steps: one row step inside a sector, the link transport of R10
//   (rotation + one step / row steps + z re-based) where the sector changes.
//   pass 1, inward, through the ORIGINAL clusters (those of the merged list): at every step the
//     predicted position (fp32) and its covariance C00, C10, C11 (half precision) are stored; update
//     where the step holds an original cluster; its chi2 sum and cluster count give the track's weight
//     Q = n - w*chi2/(2n-5) (the formula of R6);
//   pass 2, outward: at every step the prediction from inside is interpolated with the stored one
//     (as R10: information form on the 2x2 position blocks); all clusters of the step's (sector, row)
//     inside the road |dy| <= ry, |dz| <= rz (ry = clamp(nsigma*sqrt(W00+Vy), road_min, road_max)) with
//     chi2 = r^T (W+V)^-1 r <= cand_chi2_max are CANDIDATES; the best ORC_RB_NCAND by (chi2, original id)
//     are kept with their chi2; the filter is updated with the best one;
//   second ambiguity solving, ORC_RB_NCAND rounds: every step without a cluster proposes its best
//     candidate not yet owned; a cluster goes to the proposing track of largest (Q, then least id);
//     the others move on to their next candidate in the next round; afterwards, walking each track
//     from its outermost step inward, a step still without a cluster takes its best candidate as
//     SHARED iff (n_shared+1)*1000 <= shared_permille*(n_attached+1) (the rule of R6.3);
//   pass 3, inward, through the attached clusters: plain cut chi2_hit <= final_chi2_max, else the
//     cluster is dropped (no update); result = state at the innermost used cluster.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#include "tpc_oracle.h"
#include "tpc_oracle_math.hpp"

namespace {

using tpc_oracle::KFGain;
using tpc_oracle::KFState;

// ---- IEEE binary16 round-to-nearest-even (the oracle's own; pinned against numpy through orc_float_to_half)
float round_half(float f) { return orc_half_to_float(orc_float_to_half(f)); }

struct Geo {
  std::vector<float> x, ylim;
  float dx_row, cfield, ca, sa;
};
Geo make_geo(const orc_geom& g) {   // rule D5
  Geo G;
  const double pitch = ((double)g.r_max - (double)g.r_min) / (double)(g.n_rows - 1);
  const double th = std::tan((double)g.sector_half_angle_deg * (3.14159265358979323846 / 180.0));
  G.x.resize(g.n_rows); G.ylim.resize(g.n_rows);
  for (int r = 0; r < g.n_rows; ++r) {
    const double xr = (double)g.r_min + r * pitch;
    G.x[r] = (float)xr;
    G.ylim[r] = (float)(xr * th + 2.0);
  }
  G.dx_row = (float)pitch;
  G.cfield = (float)(-0.00299792458 * (double)g.bz_tesla);
  const double a = 2.0 * (double)g.sector_half_angle_deg * (3.14159265358979323846 / 180.0);
  G.ca = (float)std::cos(a);
  G.sa = (float)std::sin(a);
  return G;
}

bool rotate_state(KFState<float>& st, float& x, float ca, float sa, float max_sinphi) {   // R9 stage 2, restated
  const float s = st.s;
  const float cphi = std::sqrt(1.0f - s * s);
  const float s1 = s * ca - cphi * sa;
  if (!(tpc_oracle::o_abs(s1) <= max_sinphi)) return false;
  const float cphi1 = std::sqrt(1.0f - s1 * s1);
  const float xn = x * ca + st.y * sa;
  const float yn = st.y * ca - x * sa;
  const float a = ca - sa * (s1 / cphi1);
  const float b = -(sa * (st.t / cphi1));
  const float r = ca + sa * (s / cphi);
  float* c = st.c;
  const float c00 = c[0], c10 = c[1], c11 = c[2], c20 = c[3], c21 = c[4], c22 = c[5];
  const float c30 = c[6], c31 = c[7], c32 = c[8], c40 = c[10], c41 = c[11], c42 = c[12];
  c[0] = (a * a) * c00;
  c[1] = a * (b * c00 + c10);
  c[2] = ((b * b) * c00 + (2.0f * b) * c10) + c11;
  c[3] = (a * r) * c20;
  c[4] = r * (b * c20 + c21);
  c[5] = (r * r) * c22;
  c[6] = a * c30;
  c[7] = b * c30 + c31;
  c[8] = r * c32;
  c[10] = a * c40;
  c[11] = b * c40 + c41;
  c[12] = r * c42;
  x = xn; st.y = yn; st.s = s1;
  return true;
}

struct Step {
  int32_t sector, row;
  int32_t orig;   // original cluster of the merged track on this step (index into clusters), -1 none
};

struct Ctx {
  const Geo& G;
  const orc_params& P;
  const orc_rebuild_params& R;
  float vy, vz;
};

// one path step from a to b (b is the next step outward if dir > 0, inward if dir < 0)
bool transport(const Ctx& X, KFState<float>& st, const Step& a, const Step& b, float zc) {
  if (a.sector == b.sector) {
    const int n = b.row > a.row ? b.row - a.row : a.row - b.row;   // 1 inside a segment or a hole
    const float dx = b.row > a.row ? X.G.dx_row : -X.G.dx_row;
    for (int i = 0; i < n; ++i)
      if (!tpc_oracle::kf_propagate(st, dx, X.G.cfield, X.P.max_sinphi)) return false;
    return true;
  }
  if (a.sector - b.sector == 18 || b.sector - a.sector == 18) {
    const int n = b.row > a.row ? b.row - a.row : a.row - b.row;
    const float dx = b.row > a.row ? X.G.dx_row : -X.G.dx_row;
    for (int i = 0; i < n; ++i)
      if (!tpc_oracle::kf_propagate(st, dx, X.G.cfield, X.P.max_sinphi)) return false;
    st.z = zc;
    st.c[1] = 0.0f; st.c[4] = 0.0f; st.c[7] = 0.0f; st.c[11] = 0.0f;
    st.c[2] = X.R.ce_var;
    return true;
  }
  const float sgn = (b.sector % 18 == (a.sector % 18 + 1) % 18) ? 1.0f : -1.0f;
  float x = X.G.x[a.row];
  if (!rotate_state(st, x, X.G.ca, sgn * X.G.sa, X.P.max_sinphi)) return false;
  return tpc_oracle::kf_propagate(st, X.G.x[b.row] - x, X.G.cfield, X.P.max_sinphi);
}

inline void turn(const Ctx& X, KFState<float>& st, float y, float z) {
  st.y = y; st.z = z;
  for (int i = 0; i < 15; ++i) st.c[i] = 0.0f;
  st.c[0] = X.vy; st.c[2] = X.vz;
  st.c[5] = X.P.init_var_sinphi; st.c[9] = X.P.init_var_tanl; st.c[14] = X.P.init_var_qpt;
}

inline float chi2_2x2(float r0, float r1, float a, float b, float d, float vy, float vz) {
  const float s00 = a + vy, s01 = b, s11 = d + vz;
  const float det = s00 * s11 - s01 * s01;
  const float inv = 1.0f / det;
  const float i00 = s11 * inv, i01 = -(s01 * inv), i11 = s00 * inv;
  return ((r0 * r0) * i00 + (2.0f * (r0 * r1)) * i01) + (r1 * r1) * i11;
}
inline float clampf(float v, float lo, float hi) { return v < lo ? lo : (v > hi ? hi : v); }

inline uint32_t orderable_u32(float f) {
  uint32_t b;
  std::memcpy(&b, &f, 4);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

}  // namespace

extern "C" {

void orc_rebuild_default_params(orc_rebuild_params* r) {
  r->cand_chi2_max = 16.0f;
  r->final_chi2_max = 16.0f;
  r->min_clusters = 10;
  r->ce_var = 10000.0f;
}

int64_t orc_rebuild_path_len(const orc_rb_segment* seg, int32_t n_seg) {
  int64_t n = 0;
  for (int g = 0; g < n_seg; ++g) {
    n += seg[g].row_last - seg[g].row_first + 1;
    if (g + 1 < n_seg && seg[g + 1].sector == seg[g].sector && seg[g + 1].row_first > seg[g].row_last + 1)
      n += seg[g + 1].row_first - seg[g].row_last - 1;
  }
  return n;
}

int orc_rebuild(const orc_geom* g, const orc_params* pp, const orc_rebuild_params* rp, const orc_cluster* cl, uint64_t n_cl,
                int32_t n_merged, const int32_t* seg_ofs, const orc_rb_segment* segs, const int64_t* clu_ofs,
                const uint32_t* cluster_ids, const float* start_stq, const uint8_t* valid, const uint64_t* key_id,
                const int64_t* step_ofs, int32_t* cand_id, float* cand_chi2, int32_t* attached, uint8_t* shared,
                uint8_t* used, float* fit, float* chi2_out, int32_t* n_attached, int32_t* n_used, uint8_t* flags) {
  if (!g || !cl || n_merged < 0) return -1;
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  orc_rebuild_params R;
  if (rp) R = *rp; else orc_rebuild_default_params(&R);
  const Geo G = make_geo(*g);
  const Ctx X{G, P, R, P.err_y * P.err_y, P.err_z * P.err_z};
  const int NR = g->n_rows;
  // clusters of every (sector,row) that the search grid holds (R1: finite, inside the acceptance)
  std::vector<std::vector<uint32_t>> row_ids((size_t)g->n_sectors * NR);
  for (uint64_t i = 0; i < n_cl; ++i) {
    const orc_cluster& c = cl[i];
    if (c.sector >= g->n_sectors || c.row >= NR) continue;
    if (!(std::isfinite(c.y) && std::isfinite(c.z))) continue;
    if (!(std::fabs(c.y) <= G.ylim[c.row])) continue;
    row_ids[(size_t)c.sector * NR + c.row].push_back((uint32_t)i);
  }
  const int64_t n_steps_all = step_ofs[n_merged];
  for (int64_t k = 0; k < n_steps_all; ++k) {
    attached[k] = -1; shared[k] = 0; used[k] = 0;
    for (int j = 0; j < ORC_RB_NCAND; ++j) { cand_id[k * ORC_RB_NCAND + j] = -1; cand_chi2[k * ORC_RB_NCAND + j] = 0.0f; }
  }
  std::vector<std::vector<Step>> paths(n_merged);
  std::vector<uint32_t> Qkey(n_merged, 0);
  std::vector<uint8_t> alive(n_merged, 0);
  std::vector<KFState<float>> state2(n_merged);   // (s,t,q) after pass 2, the start values of pass 3
  for (int32_t m = 0; m < n_merged; ++m) {
    fit[m * 21] = 0; chi2_out[m] = 0; n_attached[m] = 0; n_used[m] = 0; flags[m] = 1;
    // ---- the path
    std::vector<Step>& path = paths[m];
    int64_t ci = clu_ofs[m];
    for (int s = seg_ofs[m]; s < seg_ofs[m + 1]; ++s) {
      const orc_rb_segment& sg = segs[s];
      for (int r = sg.row_first; r <= sg.row_last; ++r) {
        Step st{sg.sector, r, -1};
        if (ci < clu_ofs[m + 1] && cl[cluster_ids[ci]].sector == sg.sector &&
            cl[cluster_ids[ci]].row == r) {
          st.orig = (int32_t)cluster_ids[ci];
          ++ci;
        }
        path.push_back(st);
      }
      if (s + 1 < seg_ofs[m + 1] && segs[s + 1].sector == sg.sector)
        for (int r = sg.row_last + 1; r < segs[s + 1].row_first; ++r) path.push_back(Step{sg.sector, r, -1});
    }
    const int n = (int)path.size();
    if ((int64_t)n != step_ofs[m + 1] - step_ofs[m] || ci != clu_ofs[m + 1]) return -2;   // inconsistent input
    if (!valid[m] || n < 2) continue;
    // ---- pass 1: inward through the original clusters; predictions stored at every step
    KFState<float> st;
    st.s = start_stq[3 * m]; st.t = start_stq[3 * m + 1]; st.q = start_stq[3 * m + 2];
    std::vector<float> sy(n, 0.0f), sz(n, 0.0f), s00(n, 0.0f), s10(n, 0.0f), s11(n, 0.0f);
    turn(X, st, cl[path[n - 1].orig].y, cl[path[n - 1].orig].z);
    float chi1 = 0.0f;
    int n1 = 1;
    bool ok = true;
    for (int k = n - 2; k >= 0 && ok; --k) {
      const float zc = path[k].orig >= 0 ? cl[path[k].orig].z : 0.0f;
      if (!transport(X, st, path[k + 1], path[k], zc)) { ok = false; break; }
      sy[k] = st.y; sz[k] = st.z;
      s00[k] = round_half(st.c[0]); s10[k] = round_half(st.c[1]); s11[k] = round_half(st.c[2]);
      if (path[k].orig >= 0) {
        const orc_cluster& c = cl[path[k].orig];
        const KFGain<float> gn = tpc_oracle::kf_gain(st, X.vy, X.vz);
        const float c2 = tpc_oracle::kf_chi2(st, gn, c.y, c.z);
        if (tpc_oracle::kf_update(st, gn, c.y, c.z, P.max_sinphi, P.max_qpt)) { ok = false; break; }
        chi1 = chi1 + c2;
        ++n1;
      }
    }
    if (!ok) continue;
    {
      const int ndf = 2 * n1 - 5;
      const float Q = (float)n1 - P.sel_chi2_weight * (chi1 / (float)(ndf > 0 ? ndf : 1));
      Qkey[m] = orderable_u32(Q);
    }
    // ---- pass 2: outward; interpolation, candidates from the row's clusters, update with the best
    turn(X, st, cl[path[0].orig].y, cl[path[0].orig].z);
    for (int k = 0; k < n && ok; ++k) {
      if (k > 0) {
        const float zc = path[k].orig >= 0 ? cl[path[k].orig].z : 0.0f;
        if (!transport(X, st, path[k - 1], path[k], zc)) { ok = false; break; }
      }
      float py, pz, wa, wb, wd;
      if (k == 0) {
        py = sy[0]; pz = sz[0]; wa = s00[0]; wb = s10[0]; wd = s11[0];
      } else if (k == n - 1) {
        py = st.y; pz = st.z; wa = st.c[0]; wb = st.c[1]; wd = st.c[2];
      } else {
        // residual of the stored prediction against the inner one; r2 = 0
        const float r1y = sy[k] - st.y, r1z = sz[k] - st.z;
        const float a1 = s00[k], b1 = s10[k], d1 = s11[k], a2 = st.c[0], b2 = st.c[1], d2 = st.c[2];
        const float det1 = a1 * d1 - b1 * b1, det2 = a2 * d2 - b2 * b2;
        const float n1i = 1.0f / det1, n2i = 1.0f / det2;
        const float i1a = d1 * n1i, i1b = -(b1 * n1i), i1d = a1 * n1i;
        const float i2a = d2 * n2i, i2b = -(b2 * n2i), i2d = a2 * n2i;
        const float ia = i1a + i2a, ib = i1b + i2b, id = i1d + i2d;
        const float detw = ia * id - ib * ib;
        const float nw = 1.0f / detw;
        wa = id * nw; wb = -(ib * nw); wd = ia * nw;
        const float hy = i1a * r1y + i1b * r1z, hz = i1b * r1y + i1d * r1z;
        py = st.y + (wa * hy + wb * hz);
        pz = st.z + (wb * hy + wd * hz);
      }
      const float ry = clampf(P.road_nsigma * std::sqrt(wa + X.vy), P.road_min, P.road_max);
      const float rz = clampf(P.road_nsigma * std::sqrt(wd + X.vz), P.road_min, P.road_max);
      // all clusters of the step's (sector,row): plain linear scan
      int32_t bid[ORC_RB_NCAND];
      float bchi[ORC_RB_NCAND];
      int nb = 0;
      for (uint32_t id : row_ids[(size_t)path[k].sector * NR + path[k].row]) {
        const orc_cluster& c = cl[id];
        if (!(std::fabs(c.y - py) <= ry && std::fabs(c.z - pz) <= rz)) continue;
        const float c2 = chi2_2x2(c.y - py, c.z - pz, wa, wb, wd, X.vy, X.vz);
        if (!(c2 <= R.cand_chi2_max)) continue;
        // insert into the best list by (chi2, id)
        int pos = nb;
        while (pos > 0 && (c2 < bchi[pos - 1] || (c2 == bchi[pos - 1] && (int32_t)id < bid[pos - 1]))) --pos;
        if (pos >= ORC_RB_NCAND) continue;
        const int last = nb < ORC_RB_NCAND ? nb : ORC_RB_NCAND - 1;
        for (int j = last; j > pos; --j) { bid[j] = bid[j - 1]; bchi[j] = bchi[j - 1]; }
        bid[pos] = (int32_t)id; bchi[pos] = c2;
        if (nb < ORC_RB_NCAND) ++nb;
      }
      const int64_t so = (step_ofs[m] + k) * ORC_RB_NCAND;
      for (int j = 0; j < nb; ++j) { cand_id[so + j] = bid[j]; cand_chi2[so + j] = bchi[j]; }
      if (k > 0 && nb > 0) {
        const orc_cluster& c = cl[bid[0]];
        const KFGain<float> gn = tpc_oracle::kf_gain(st, X.vy, X.vz);
        if (tpc_oracle::kf_update(st, gn, c.y, c.z, P.max_sinphi, P.max_qpt)) { ok = false; break; }
      }
    }
    if (!ok) {   // a track that failed holds no candidates
      for (int k = 0; k < n; ++k)
        for (int j = 0; j < ORC_RB_NCAND; ++j) { cand_id[(step_ofs[m] + k) * ORC_RB_NCAND + j] = -1; cand_chi2[(step_ofs[m] + k) * ORC_RB_NCAND + j] = 0.0f; }
      continue;
    }
    alive[m] = 1;
    state2[m] = st;
  }
  // ---- second ambiguity solving: ORC_RB_NCAND rounds of proposals
  std::vector<int32_t> owner(n_cl, -1);        // cluster -> merged track that owns it
  std::vector<uint8_t> ptr(n_steps_all, 0);
  std::vector<uint32_t> bestQ(n_cl);
  std::vector<uint64_t> bestId(n_cl);
  for (int round = 0; round < ORC_RB_NCAND; ++round) {
    std::fill(bestQ.begin(), bestQ.end(), 0u);
    std::fill(bestId.begin(), bestId.end(), ~0ull);
    auto proposal = [&](int32_t m, int64_t k) -> int32_t {   // the step's best candidate not yet owned, -1 none
      if (attached[k] >= 0) return -1;
      while (ptr[k] < ORC_RB_NCAND) {
        const int32_t c = cand_id[k * ORC_RB_NCAND + ptr[k]];
        if (c < 0) return -1;
        if (owner[c] < 0) return c;
        ++ptr[k];
      }
      (void)m;
      return -1;
    };
    for (int32_t m = 0; m < n_merged; ++m) {
      if (!alive[m]) continue;
      for (int64_t k = step_ofs[m]; k < step_ofs[m + 1]; ++k) {
        const int32_t c = proposal(m, k);
        if (c >= 0 && Qkey[m] > bestQ[c]) bestQ[c] = Qkey[m];
      }
    }
    for (int32_t m = 0; m < n_merged; ++m) {
      if (!alive[m]) continue;
      for (int64_t k = step_ofs[m]; k < step_ofs[m + 1]; ++k) {
        const int32_t c = proposal(m, k);
        if (c >= 0 && Qkey[m] == bestQ[c] && key_id[m] < bestId[c]) bestId[c] = key_id[m];
      }
    }
    // resolve: winners attach (ownership is final: later rounds cannot take the cluster away)
    std::vector<std::pair<int64_t, int32_t>> wins;      // (step, cluster), applied after the scan of all proposals
    std::vector<int32_t> win_track;
    for (int32_t m = 0; m < n_merged; ++m) {
      if (!alive[m]) continue;
      for (int64_t k = step_ofs[m]; k < step_ofs[m + 1]; ++k) {
        const int32_t c = proposal(m, k);
        if (c < 0) continue;
        // (a step that lost keeps its pointer: in the next round the cluster is owned and skipped)
        if (Qkey[m] == bestQ[c] && key_id[m] == bestId[c]) { wins.emplace_back(k, c); win_track.push_back(m); }
      }
    }
    for (size_t w = 0; w < wins.size(); ++w) {
      attached[wins[w].first] = wins[w].second;
      owner[wins[w].second] = win_track[w];
    }
  }
  // ---- shared attachment from the outermost step inward, then pass 3
  for (int32_t m = 0; m < n_merged; ++m) {
    if (!alive[m]) continue;
    const std::vector<Step>& path = paths[m];
    const int n = (int)path.size();
    const int64_t s0 = step_ofs[m];
    int n_acc = 0, n_sh = 0;
    for (int k = n - 1; k >= 0; --k) {
      if (attached[s0 + k] >= 0) { ++n_acc; continue; }
      const int32_t c = cand_id[(s0 + k) * ORC_RB_NCAND];
      if (c < 0) continue;
      if ((int64_t)(n_sh + 1) * 1000 <= (int64_t)P.shared_permille * (n_acc + 1)) {
        attached[s0 + k] = c; shared[s0 + k] = 1; ++n_acc; ++n_sh;
      }
    }
    n_attached[m] = n_acc;
    int last = n - 1;
    while (last >= 0 && attached[s0 + last] < 0) --last;
    if (last < 0) continue;
    KFState<float> st = state2[m];
    turn(X, st, cl[attached[s0 + last]].y, cl[attached[s0 + last]].z);
    used[s0 + last] = 1;
    KFState<float> st_in = st;          // state right after the innermost used cluster
    int nu = 1, row_in = path[last].row;
    float chi3 = 0.0f;
    bool ok = true;
    for (int k = last - 1; k >= 0 && ok; --k) {
      const int32_t ca = attached[s0 + k];
      // (the electrode re-base needs a measured z on the step behind it: the attached cluster's, else
      // the original cluster's -- the end rows of a segment always hold one)
      const float zc = ca >= 0 ? cl[ca].z : (path[k].orig >= 0 ? cl[path[k].orig].z : st.z);
      if (!transport(X, st, path[k + 1], path[k], zc)) { ok = false; break; }
      if (ca < 0) continue;
      const orc_cluster& c = cl[ca];
      const KFGain<float> gn = tpc_oracle::kf_gain(st, X.vy, X.vz);
      const float c2 = tpc_oracle::kf_chi2(st, gn, c.y, c.z);
      if (!(c2 <= R.final_chi2_max)) continue;   // plain cut: the cluster is dropped, no update
      if (tpc_oracle::kf_update(st, gn, c.y, c.z, P.max_sinphi, P.max_qpt)) { ok = false; break; }
      chi3 = chi3 + c2;
      used[s0 + k] = 1;
      ++nu;
      st_in = st;
      row_in = path[k].row;
    }
    n_used[m] = nu;
    if (!ok || nu < R.min_clusters) continue;
    flags[m] = 0;
    chi2_out[m] = chi3;
    float* o = fit + (size_t)m * 21;
    o[0] = G.x[row_in];
    o[1] = st_in.y; o[2] = st_in.z; o[3] = st_in.s; o[4] = st_in.t; o[5] = st_in.q;
    for (int i = 0; i < 15; ++i) o[6 + i] = st_in.c[i];
  }
  return 0;
}

}  // extern "C"
