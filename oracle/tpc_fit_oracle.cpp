// tpc_fit_oracle.cpp — CPU ORACLE of the three-iteration track fit with the Phase-I interpolation
// rejection, reading R10 of DESIGN.md (TEST INFRASTRUCTURE, see tpc_oracle.h for what may load it;
// shares no code with the CUDA path).
//
// PAPER.md:31 (section 2): the track fit "performs three iterations, first inward, then outward,
// then inward"; cluster rejection by "an interpolation approach": one iteration
// "stores the current track position and covariance at every TPC pad row in reduced precision",
// a later one performs the chi2 cut "against the interpolation between the current position and
// covariance with the values stored ... for this pad row".  PAPER.md:57 (section 3, Phase I):
// "position and covariance are stored in the first, inward iteration.  The interpolation and the
// chi2 cut are performed in the second, outward iteration.  Cluster rejection happens later in the
// third iteration."  The paper gives no formula; the reading R10, step by step:
//
//   input: the cluster list of one (merged) track in chain order c_0 .. c_{n-1}: (sector, row, y, z),
//          and start parameters (s, t, q) at the outermost cluster (the refit's outer state, R8).
//   transport between consecutive clusters: same sector: |row difference| row steps of formulas P;
//          adjacent sector (a stage-2 link of R9): rotation by one sector step, then ONE propagation
//          step to the cluster's row; across the central electrode (stage 3): row steps, then the z of
//          the state is re-based on the measured z (the two sides see z_true -+ v t with t unknown):
//          z <- z_cluster, C_1j <- 0 (j != 1), C_11 <- ce_var.
//   start of an iteration (a "turn", as R5.4): (y, z) = the start cluster's measured position,
//          (s, t, q) = current estimate, C = the initial diagonal; the start cluster counts as fitted.
//   iteration 1, inward from c_{n-1}: at every further cluster: transport, STORE the predicted
//          residual (y_pred - y_c, z_pred - z_c) and (C00, C10, C11), each rounded to IEEE half
//          precision ("reduced precision"), then update with the cluster.
//   iteration 2, outward from c_0: at every further cluster: transport; INTERPOLATE the prediction
//          (from the inner clusters) with the stored one (from the outer clusters): both exclude the
//          cluster itself: W = (C2^-1 + C1^-1)^-1, r = W (C2^-1 r2 + C1^-1 r1) (2x2, residuals taken
//          against the cluster), chi2_c = r^T (W + V)^-1 r; the cluster is MARKED if chi2_c >
//          fit_chi2_max; then update with the cluster (marked or not: rejection happens later).  At c_0
//          only the stored prediction exists, at c_{n-1} only the inner one: the chi2 is one-sided.
//   iteration 3, inward from the outermost UNMARKED cluster, through the unmarked clusters only;
//          chi2 of this pass and the state at the innermost unmarked cluster are the result.
//   A fit fails (flag) if a transport or an update leaves |sin phi| <= max_sinphi, or if fewer than
//   fit_min_clusters clusters stay unmarked.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#include "tpc_oracle.h"
#include "tpc_oracle_math.hpp"

namespace {

using tpc_oracle::KFGain;
using tpc_oracle::KFState;

// ---- IEEE 754 binary16 rounding of a float (round to nearest even), returned as a float
uint16_t float_to_half_bits(float f) {
  uint32_t x;
  std::memcpy(&x, &f, 4);
  const uint32_t sign = (x >> 16) & 0x8000u;
  const uint32_t absx = x & 0x7FFFFFFFu;
  if (absx >= 0x7F800000u) return (uint16_t)(sign | (absx > 0x7F800000u ? 0x7E00u : 0x7C00u));  // NaN / Inf
  if (absx >= 0x477FF000u) return (uint16_t)(sign | 0x7C00u);                                     // rounds to Inf (>= 65520)
  if (absx < 0x33000001u) return (uint16_t)sign;                                                   // rounds to 0 (<= 2^-25)
  const int e = (int)(absx >> 23) - 127;
  uint32_t man = (absx & 0x7FFFFFu) | 0x800000u;   // 24 bits with the hidden one
  int shift;                                        // bits to drop
  uint32_t hexp;
  if (e < -14) { shift = 13 + (-14 - e); hexp = 0; }   // subnormal half
  else { shift = 13; hexp = (uint32_t)(e + 15); }
  const uint32_t keep = man >> shift;
  const uint32_t rem = man & ((1u << shift) - 1u), halfway = 1u << (shift - 1);
  uint32_t r = keep;
  if (rem > halfway || (rem == halfway && (keep & 1u))) ++r;
  // r holds the hidden bit for normals (bit 10): adding the exponent field handles the carry
  const uint32_t h = hexp ? ((hexp - 1) << 10) + r : r;
  return (uint16_t)(sign | h);
}
float half_bits_to_float(uint16_t h) {
  const uint32_t sign = (uint32_t)(h & 0x8000u) << 16;
  const uint32_t e = (h >> 10) & 0x1Fu, m = h & 0x3FFu;
  uint32_t x;
  if (e == 0) {
    if (m == 0) x = sign;
    else {  // subnormal: m * 2^-24
      const float v = (float)m * 5.9604644775390625e-08f;
      std::memcpy(&x, &v, 4);
      x |= sign;
    }
  } else if (e == 31) x = sign | 0x7F800000u | (m << 13);
  else x = sign | ((e + 112u) << 23) | (m << 13);
  float f;
  std::memcpy(&f, &x, 4);
  return f;
}
inline float round_half(float f) { return half_bits_to_float(float_to_half_bits(f)); }

struct Geo {
  std::vector<float> x;
  float dx_row, cfield, ca, sa;
};
Geo make_geo(const orc_geom& g) {   // rule D5
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

// rotation into the neighbouring sector's frame: the statements of R9 stage 2 (tpc_merge_oracle.cpp),
// restated here so that the two oracles stay independent files
bool rotate_state(KFState<float>& st, float& x, float ca, float sa, float max_sinphi) {
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

struct Ctx {
  const Geo& G;
  const orc_params& P;
  const orc_fit_params& F;
  float vy, vz;
};

// transport the state from cluster (sec0,row0) to cluster (sec1,row1); zc = measured z of the target
bool transport(const Ctx& X, KFState<float>& st, int sec0, int row0, int sec1, int row1, float zc) {
  if (sec0 == sec1 || sec0 - sec1 == 18 || sec1 - sec0 == 18) {
    const int n = row1 > row0 ? row1 - row0 : row0 - row1;
    const float dx = row1 > row0 ? X.G.dx_row : -X.G.dx_row;
    for (int i = 0; i < n; ++i)
      if (!tpc_oracle::kf_propagate(st, dx, X.G.cfield, X.P.max_sinphi)) return false;
    if (sec0 != sec1) {   // central electrode: z re-based on the measurement, its correlations dropped
      st.z = zc;
      st.c[1] = 0.0f; st.c[4] = 0.0f; st.c[7] = 0.0f; st.c[11] = 0.0f;
      st.c[2] = X.F.ce_var;
    }
    return true;
  }
  // adjacent sectors of one half: sec1 = sec0 + 1 (mod 18) turns the frame by +one sector step
  const float sgn = (sec1 % 18 == (sec0 % 18 + 1) % 18) ? 1.0f : -1.0f;
  float x = X.G.x[row0];
  if (!rotate_state(st, x, X.G.ca, sgn * X.G.sa, X.P.max_sinphi)) return false;
  return tpc_oracle::kf_propagate(st, X.G.x[row1] - x, X.G.cfield, X.P.max_sinphi);
}

inline void turn(const Ctx& X, KFState<float>& st, float y, float z) {
  st.y = y; st.z = z;
  for (int i = 0; i < 15; ++i) st.c[i] = 0.0f;
  st.c[0] = X.vy; st.c[2] = X.vz;
  st.c[5] = X.P.init_var_sinphi; st.c[9] = X.P.init_var_tanl; st.c[14] = X.P.init_var_qpt;
}

// chi2 of the residual r against covariance [[a,b],[b,d]] + V
inline float chi2_2x2(float r0, float r1, float a, float b, float d, float vy, float vz) {
  const float s00 = a + vy, s01 = b, s11 = d + vz;
  const float det = s00 * s11 - s01 * s01;
  const float inv = 1.0f / det;
  const float i00 = s11 * inv, i01 = -(s01 * inv), i11 = s00 * inv;
  return ((r0 * r0) * i00 + (2.0f * (r0 * r1)) * i01) + (r1 * r1) * i11;
}

}  // namespace

extern "C" {

void orc_fit_default_params(orc_fit_params* f) {
  f->fit_chi2_max = 16.0f;
  f->fit_min_clusters = 10;
  f->ce_var = 10000.0f;
}

uint16_t orc_float_to_half(float f) { return float_to_half_bits(f); }
float orc_half_to_float(uint16_t h) { return half_bits_to_float(h); }

// One track.  sector/row/y/z: n clusters in chain order; start_stq: (s, t, q) at the outermost cluster.
// out_state: x, p[5], c[15] at the innermost unmarked cluster's row (21 floats); chi2_cluster[n]: the
// interpolation chi2 of iteration 2; rejected[n]: 1 = marked.  Returns the chi2 of iteration 3, *n_used,
// or -1 (fit failed; outputs undefined except chi2_cluster / rejected as far as computed).
float orc_fit_track(const orc_geom* g, const orc_params* pp, const orc_fit_params* fp, const int32_t* sector,
                    const int32_t* row, const float* y, const float* z, int n, const float* start_stq,
                    float* out_state, float* chi2_cluster, uint8_t* rejected, int32_t* n_used) {
  orc_params P;
  if (pp) P = *pp; else orc_default_params(&P);
  orc_fit_params F;
  if (fp) F = *fp; else orc_fit_default_params(&F);
  const Geo G = make_geo(*g);
  const Ctx X{G, P, F, P.err_y * P.err_y, P.err_z * P.err_z};
  for (int i = 0; i < n; ++i) { chi2_cluster[i] = 0.0f; rejected[i] = 0; }
  *n_used = 0;
  if (n < 2) return -1.0f;
  KFState<float> st;
  st.s = start_stq[0]; st.t = start_stq[1]; st.q = start_stq[2];
  // stored predictions of iteration 1 (reduced precision)
  std::vector<float> s_ry(n, 0.0f), s_rz(n, 0.0f), s_c00(n, 0.0f), s_c10(n, 0.0f), s_c11(n, 0.0f);
  // ---- iteration 1: inward from c_{n-1}
  turn(X, st, y[n - 1], z[n - 1]);
  for (int i = n - 2; i >= 0; --i) {
    if (!transport(X, st, sector[i + 1], row[i + 1], sector[i], row[i], z[i])) return -1.0f;
    s_ry[i] = round_half(st.y - y[i]);
    s_rz[i] = round_half(st.z - z[i]);
    s_c00[i] = round_half(st.c[0]);
    s_c10[i] = round_half(st.c[1]);
    s_c11[i] = round_half(st.c[2]);
    const KFGain<float> gn = tpc_oracle::kf_gain(st, X.vy, X.vz);
    if (tpc_oracle::kf_update(st, gn, y[i], z[i], P.max_sinphi, P.max_qpt)) return -1.0f;
  }
  // ---- iteration 2: outward from c_0, interpolation + chi2 cut (marking only)
  turn(X, st, y[0], z[0]);
  {  // c_0: only the stored (outer-side) prediction exists
    chi2_cluster[0] = chi2_2x2(s_ry[0], s_rz[0], s_c00[0], s_c10[0], s_c11[0], X.vy, X.vz);
    if (!(chi2_cluster[0] <= F.fit_chi2_max)) rejected[0] = 1;
  }
  for (int i = 1; i < n; ++i) {
    if (!transport(X, st, sector[i - 1], row[i - 1], sector[i], row[i], z[i])) return -1.0f;
    const float r2y = st.y - y[i], r2z = st.z - z[i];
    const float a2 = st.c[0], b2 = st.c[1], d2 = st.c[2];
    float chi2;
    if (i == n - 1) {  // only the inner-side prediction exists
      chi2 = chi2_2x2(r2y, r2z, a2, b2, d2, X.vy, X.vz);
    } else {
      // information form: I = C^-1 for both predictions, W = (I1 + I2)^-1, r = W (I1 r1 + I2 r2)
      const float a1 = s_c00[i], b1 = s_c10[i], d1 = s_c11[i];
      const float det1 = a1 * d1 - b1 * b1, det2 = a2 * d2 - b2 * b2;
      const float n1 = 1.0f / det1, n2 = 1.0f / det2;
      const float i1a = d1 * n1, i1b = -(b1 * n1), i1d = a1 * n1;
      const float i2a = d2 * n2, i2b = -(b2 * n2), i2d = a2 * n2;
      const float ia = i1a + i2a, ib = i1b + i2b, id = i1d + i2d;
      const float detw = ia * id - ib * ib;
      const float nw = 1.0f / detw;
      const float wa = id * nw, wb = -(ib * nw), wd = ia * nw;
      const float hy = (i1a * s_ry[i] + i1b * s_rz[i]) + (i2a * r2y + i2b * r2z);
      const float hz = (i1b * s_ry[i] + i1d * s_rz[i]) + (i2b * r2y + i2d * r2z);
      const float ry = wa * hy + wb * hz, rz = wb * hy + wd * hz;
      chi2 = chi2_2x2(ry, rz, wa, wb, wd, X.vy, X.vz);
    }
    chi2_cluster[i] = chi2;
    if (!(chi2 <= F.fit_chi2_max)) rejected[i] = 1;
    const KFGain<float> gn = tpc_oracle::kf_gain(st, X.vy, X.vz);
    if (tpc_oracle::kf_update(st, gn, y[i], z[i], P.max_sinphi, P.max_qpt)) return -1.0f;
  }
  // ---- iteration 3: inward through the unmarked clusters only
  int used = 0;
  for (int i = 0; i < n; ++i) used += rejected[i] ? 0 : 1;
  *n_used = used;
  if (used < F.fit_min_clusters || used < 2) return -1.0f;
  int last = n - 1;
  while (rejected[last]) --last;
  // the state of iteration 2 sits on c_{n-1}; bring (s, t, q) as they are to the outermost unmarked cluster
  turn(X, st, y[last], z[last]);
  float chi2 = 0.0f;
  int prev = last;
  for (int i = last - 1; i >= 0; --i) {
    if (rejected[i]) continue;
    if (!transport(X, st, sector[prev], row[prev], sector[i], row[i], z[i])) return -1.0f;
    const KFGain<float> gn = tpc_oracle::kf_gain(st, X.vy, X.vz);
    const float c2 = tpc_oracle::kf_chi2(st, gn, y[i], z[i]);
    if (tpc_oracle::kf_update(st, gn, y[i], z[i], P.max_sinphi, P.max_qpt)) return -1.0f;
    chi2 = chi2 + c2;
    prev = i;
  }
  out_state[0] = G.x[row[prev]];
  out_state[1] = st.y; out_state[2] = st.z; out_state[3] = st.s; out_state[4] = st.t; out_state[5] = st.q;
  for (int i = 0; i < 15; ++i) out_state[6 + i] = st.c[i];
  return chi2;
}

}  // extern "C"
