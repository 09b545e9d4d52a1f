// tpc_merge_oracle.cpp — CPU ORACLE of the track merging, reading R9 of DESIGN.md (TEST
// INFRASTRUCTURE, see tpc_oracle.h for what may load it; shares no code with the CUDA path).
//
// PAPER.md:29 (section 2): "The track merging merges tracks first inside the TPC sectors, then
// between adjacent sectors of the TPC halves, and then across the central electrode."
// PAPER.md:57 (section 3): "a sector track refit at the beginning of the track merging was added,
// guaranteeing reasonable initial parameters" (R8, orc_refit_hits: it gives every sector track
// its state at the innermost cluster, I_k, and at the outermost cluster, O_k).
// The paper says no more; everything below is the reading R9, written out plainly:
//
//   three stages in the paper's order; in each stage, for every ordered pair (a, b) of sector
//   tracks with a FREE outer end (next[a] < 0) and a FREE inner end (prev[b] < 0) that the stage
//   pairs up, the outer state O_a is transported to the x of b's innermost row and compared with
//   I_b:   chi2 = sum_i (p_b,i - p_a',i)^2 / (C_a'[ii] + C_b[ii] + sys_i^2),  i = y, z, sin phi,
//   tan lambda, q/pT.  A pair matches if chi2 <= chi2_max.  best_out[a] = the matching b of least
//   (chi2, id_b), best_in[b] = the matching a of least (chi2, id_a); a and b are linked iff they
//   chose each other (as the cellular automaton's links, R3).  id = (sector, iteration, seed id,
//   segment), unique per track.
//     stage 1, inside a sector:  same sector, 1 <= f_b - l_a <= gap_in_sector; transport = that many
//              row steps of the follower's propagation (formulas P);
//     stage 2, adjacent sectors of one half:  sector_b = sector_a +- 1 (mod 18, same side),
//              -gap_adjacent_back <= f_b - l_a <= gap_adjacent; transport = rotation of O_a by
//              +-20 degrees into b's frame, then ONE propagation step to x[f_b];
//     stage 3, across the central electrode:  sector_b = sector_a +- 18, 1 <= f_b - l_a <= gap_ce,
//              row steps; z compared as z_b + z_a' (the two drift sides see z_true -+ v t, so the
//              sum vanishes where the track crosses the electrode) with sys_z replaced by ce_sys_z.
//   Pre-cuts (part of the definition; they also bound the search): coarse, on the two end states as
//   they are, |z_b - z_a| <= pre_coarse_dz (stage 3: |z_b + z_a|); fine, on the TRANSPORTED state,
//   |y_b - y_a'| <= pre_dy and |z_b - z_a'| <= pre_dz (stage 3: |z_b + z_a'|).
//   Tracks whose refit failed take no part.  Every link raises row_first by >= min_hits_track - 1 -
//   gap_adjacent_back > 0 rows, so the links form simple chains.
#include <cmath>
#include <cstdint>
#include <vector>

#include "tpc_oracle.h"
#include "tpc_oracle_math.hpp"

namespace {

using tpc_oracle::KFState;

struct Geo {
  std::vector<float> x;
  float dx_row, cfield, ca, sa;   // cos / sin of one sector step (2 * half angle)
};

Geo make_geo(const orc_geom& g) {   // rule D5: tables in double, rounded once
  Geo G;
  const double pitch = ((double)g.r_max - (double)g.r_min) / (double)(g.n_rows - 1);
  G.x.resize(g.n_rows);
  for (int r = 0; r < g.n_rows; ++r) G.x[r] = (float)((double)g.r_min + r * pitch);
  G.dx_row = (float)pitch;
  G.cfield = (float)(-0.00299792458 * (double)g.bz_tesla);
  const double a = 2.0 * (double)g.sector_half_angle_deg * (3.14159265358979323846 / 180.0);
  G.ca = (float)std::cos(a);
  G.sa = (float)std::sin(a);
  return G;
}

inline void load_state(KFState<float>& st, const float* p, const float* c) {
  st.y = p[0]; st.z = p[1]; st.s = p[2]; st.t = p[3]; st.q = p[4];
  for (int i = 0; i < 15; ++i) st.c[i] = c[i];
}

// Rotation of a state at local x into the frame of the neighbouring sector (alpha = +-one sector
// step; sa carries the sign).  Same point, direction phi' = phi - alpha; the parameters are then
// those on the plane x' = const through the point.  First-order Jacobian (new w.r.t. old):
//   dy'/dy = ca - sa*tan(phi'),  dz'/dy = -sa*t/cos(phi'),  ds'/ds = ca + sa*s/cos(phi); others 1 / 0.
inline bool rotate_state(KFState<float>& st, float& x, float ca, float sa, float max_sinphi) {
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

struct Key {
  int32_t sector, iter;
  uint32_t seed_id;
  int32_t segment;
};
inline bool key_less(const Key& a, const Key& b) {
  if (a.sector != b.sector) return a.sector < b.sector;
  if (a.iter != b.iter) return a.iter < b.iter;
  if (a.seed_id != b.seed_id) return a.seed_id < b.seed_id;
  return a.segment < b.segment;
}
inline Key key_of(const orc_merge_track& t) { return Key{t.sector, t.iter, t.seed_id, t.segment}; }

// chi2 of the match of a's transported outer state with b's inner state; false = no match
bool match(const Geo& G, const orc_params& P, const orc_merge_params& M, const orc_merge_track& a,
           const orc_merge_track& b, int stage, float* chi2_out) {
  const int gap = b.row_first - a.row_last;
  // coarse pre-cut on the untransported end states
  const float dz_coarse = stage == 3 ? b.p_in[1] + a.p_out[1] : b.p_in[1] - a.p_out[1];
  if (!(tpc_oracle::o_abs(dz_coarse) <= M.pre_coarse_dz)) return false;
  KFState<float> st;
  load_state(st, a.p_out, a.c_out);
  if (stage == 2) {
    // b = a + 1 (mod 18): b's frame is turned by +one sector step
    const int sa18 = a.sector % 18, sb18 = b.sector % 18;
    const float sgn = (sb18 == (sa18 + 1) % 18) ? 1.0f : -1.0f;
    float x = G.x[a.row_last];
    if (!rotate_state(st, x, G.ca, sgn * G.sa, P.max_sinphi)) return false;
    if (!tpc_oracle::kf_propagate(st, G.x[b.row_first] - x, G.cfield, P.max_sinphi)) return false;
  } else {
    for (int i = 0; i < gap; ++i)
      if (!tpc_oracle::kf_propagate(st, G.dx_row, G.cfield, P.max_sinphi)) return false;
  }
  // fine pre-cuts on the transported state
  const float dz_pre = stage == 3 ? b.p_in[1] + st.z : b.p_in[1] - st.z;
  if (!(tpc_oracle::o_abs(dz_pre) <= M.pre_dz)) return false;
  if (!(tpc_oracle::o_abs(b.p_in[0] - st.y) <= M.pre_dy)) return false;
  const float pa[5] = {st.y, st.z, st.s, st.t, st.q};
  const int diag[5] = {0, 2, 5, 9, 14};
  float chi2 = 0.0f;
  for (int i = 0; i < 5; ++i) {
    float d = b.p_in[i] - pa[i];
    float sys = M.sys[i];
    if (i == 1 && stage == 3) { d = b.p_in[1] + pa[1]; sys = M.ce_sys_z; }
    const float var = (st.c[diag[i]] + b.c_in[diag[i]]) + sys * sys;
    chi2 = chi2 + (d * d) / var;
  }
  *chi2_out = chi2;
  return chi2 <= M.chi2_max;
}

bool stage_pairs(const orc_merge_params& M, const orc_merge_track& a, const orc_merge_track& b, int stage) {
  const int gap = b.row_first - a.row_last;
  if (stage == 1) return a.sector == b.sector && gap >= 1 && gap <= M.gap_in_sector;
  if (stage == 2) {
    if (a.sector / 18 != b.sector / 18) return false;
    const int sa = a.sector % 18, sb = b.sector % 18;
    if (sb != (sa + 1) % 18 && sb != (sa + 17) % 18) return false;
    return gap >= -M.gap_adjacent_back && gap <= M.gap_adjacent;
  }
  const int d = a.sector - b.sector;
  return (d == 18 || d == -18) && gap >= 1 && gap <= M.gap_ce;
}

}  // namespace

extern "C" {

void orc_merge_default_params(orc_merge_params* m) {
  m->gap_in_sector = 30; m->gap_adjacent_back = 3; m->gap_adjacent = 10; m->gap_ce = 6;
  m->chi2_max = 20.0f;
  m->sys[0] = 0.3f; m->sys[1] = 0.3f; m->sys[2] = 0.02f; m->sys[3] = 0.02f; m->sys[4] = 0.2f;
  m->ce_sys_z = 3.0f;
  m->pre_dy = 8.0f; m->pre_dz = 8.0f; m->pre_coarse_dz = 40.0f;
  m->stages = 7;
}

// next[k] / prev[k]: index of the track linked behind / before track k, -1 none; link_chi2[k] = the
// match chi2 of the link k -> next[k].  Returns the number of links, or -1 on a bad argument.
int orc_merge_links(const orc_geom* g, const orc_params* pp, const orc_merge_params* mp,
                    const orc_merge_track* t, int32_t n, int32_t* next, int32_t* prev, float* link_chi2) {
  if (!g || !t || !next || !prev || n < 0) return -1;
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  orc_merge_params M;
  if (mp) M = *mp; else orc_merge_default_params(&M);
  const Geo G = make_geo(*g);
  for (int32_t k = 0; k < n; ++k) { next[k] = -1; prev[k] = -1; if (link_chi2) link_chi2[k] = 0.0f; }
  // tracks of each sector (only a speed-up of the plain double loop: the stage rules pair sectors)
  std::vector<std::vector<int32_t>> by_sector(g->n_sectors);
  for (int32_t k = 0; k < n; ++k)
    if (t[k].valid && t[k].sector >= 0 && t[k].sector < g->n_sectors) by_sector[t[k].sector].push_back(k);
  int n_links = 0;
  std::vector<int32_t> best_out(n), best_in(n);
  std::vector<float> chi_out(n), chi_in(n);
  for (int stage = 1; stage <= 3; ++stage) {
    if (!((M.stages >> (stage - 1)) & 1)) continue;
    for (int32_t k = 0; k < n; ++k) { best_out[k] = -1; best_in[k] = -1; }
    for (int sa = 0; sa < g->n_sectors; ++sa) {
      int partners[2], np = 0;
      if (stage == 1) partners[np++] = sa;
      else if (stage == 2) {
        const int base = (sa / 18) * 18, s18 = sa % 18;
        partners[np++] = base + (s18 + 1) % 18;
        if ((s18 + 17) % 18 != (s18 + 1) % 18) partners[np++] = base + (s18 + 17) % 18;
      } else partners[np++] = sa < 18 ? sa + 18 : sa - 18;
      for (int ip = 0; ip < np; ++ip) {
        const int sb = partners[ip];
        if (sb < 0 || sb >= g->n_sectors) continue;
        for (int32_t a : by_sector[sa]) {
          if (next[a] >= 0) continue;
          for (int32_t b : by_sector[sb]) {
            if (prev[b] >= 0 || a == b) continue;
            if (!stage_pairs(M, t[a], t[b], stage)) continue;
            float chi2;
            if (!match(G, P, M, t[a], t[b], stage, &chi2)) continue;
            if (best_out[a] < 0 || chi2 < chi_out[a] ||
                (chi2 == chi_out[a] && key_less(key_of(t[b]), key_of(t[best_out[a]])))) {
              best_out[a] = b; chi_out[a] = chi2;
            }
            if (best_in[b] < 0 || chi2 < chi_in[b] ||
                (chi2 == chi_in[b] && key_less(key_of(t[a]), key_of(t[best_in[b]])))) {
              best_in[b] = a; chi_in[b] = chi2;
            }
          }
        }
      }
    }
    for (int32_t a = 0; a < n; ++a) {
      const int32_t b = best_out[a];
      if (b >= 0 && best_in[b] == a) {
        next[a] = b; prev[b] = a;
        if (link_chi2) link_chi2[a] = chi_out[a];
        ++n_links;
      }
    }
  }
  return n_links;
}

// single-step entry points for the pins
int orc_merge_rotate(const orc_geom* g, float* state20, float* x, int sign, float max_sinphi) {
  const Geo G = make_geo(*g);
  KFState<float> st;
  load_state(st, state20, state20 + 5);
  if (!rotate_state(st, *x, G.ca, (sign >= 0 ? 1.0f : -1.0f) * G.sa, max_sinphi)) return 0;
  state20[0] = st.y; state20[1] = st.z; state20[2] = st.s; state20[3] = st.t; state20[4] = st.q;
  for (int i = 0; i < 15; ++i) state20[5 + i] = st.c[i];
  return 1;
}

}  // extern "C"
