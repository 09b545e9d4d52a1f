// tpc_oracle_math.hpp — Kalman-filter arithmetic of the CPU ORACLE (test infrastructure).
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Nothing under paper_2601_20569_b200/
// includes, links or calls it; only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs do.  It shares no code with the CUDA path.
//
// What it follows: the track following of the ALICE sector tracking, "the track following
// fits all seeds and propagates them through the TPC volume using the Kalman filter picking
// up more clusters of the track" (section 2).  The paper gives no formula
// (it defers to its ref. [7]); the track model below is DESIGN.md reading R5 (textbook
// helix in a uniform solenoid field + linear Kalman update), written step by step in the
// order of DESIGN.md section 3 "Formulas".  Rule D1: only + - * / sqrt, IEEE
// round-to-nearest, no FMA contraction (compile with -ffp-contract=off), no reassociation.
//
// Templated on the scalar type so the pins (tests/test_oracle_*.py) can run the very same
// statements in double next to the float instantiation the path uses.
//
// State at local x (row plane): p = (y, z, s = sin(phi), t = tan(lambda) = dz/dl_xy,
// q = q/pT); covariance C lower-triangular, 15 entries:
//   c[0]=C00 c[1]=C10 c[2]=C11 c[3]=C20 c[4]=C21 c[5]=C22 c[6]=C30 c[7]=C31 c[8]=C32
//   c[9]=C33 c[10]=C40 c[11]=C41 c[12]=C42 c[13]=C43 c[14]=C44
#ifndef TPC_ORACLE_MATH_HPP
#define TPC_ORACLE_MATH_HPP

#include <cmath>

namespace tpc_oracle {

template <class T>
struct KFState {
  T y, z, s, t, q;
  T c[15];
};

// Jacobian entries of one propagation step that differ from the identity.
template <class T>
struct KFJac {
  T f02, f04, f12, f13, f14, f24;
};

template <class T>
inline T o_abs(T v) { return v < T(0) ? -v : v; }

// Propagate the state from x to x+dx (dx of either sign) on the exact circle in the xy
// plane; z advances by tan(lambda) times the arc length.  `cfield` = signed curvature per
// unit q/pT (R0: c = -0.00299792458*Bz, rounded once to the scalar type).
// Returns false (state untouched) when |sin(phi)| would exceed max_sinphi: the leg ends.
// DESIGN.md section 3, block P.
template <class T>
inline bool kf_propagate(KFState<T>& st, T dx, T cfield, T max_sinphi, KFJac<T>* jac_out = nullptr) {
  const T s = st.s, t = st.t, q = st.q;
  const T k = cfield * q;
  const T ex = std::sqrt(T(1) - s * s);
  const T s1 = s + k * dx;
  if (!(o_abs(s1) <= max_sinphi)) return false;
  const T ex1 = std::sqrt(T(1) - s1 * s1);
  const T h = T(1) / (ex + ex1);
  const T ss = s + s1;
  const T tt = ss * h;
  const T dy = dx * tt;
  const T dl = dx * std::sqrt(T(1) + tt * tt);  // SIGNED chord (negative for dx<0)
  const T a = (T(0.5) * k) * dl;
  const T a2 = a * a;
  // asin(a)/a = 1 + a^2/6 + 3 a^4/40 + O(a^6)
  const T dS = dl * (T(1) + a2 * (T(1) / T(6) + a2 * (T(3) / T(40))));

  const T hh = h * h;
  const T g = s / ex + s1 / ex1;
  const T f02 = dx * (T(2) * h + (ss * hh) * g);
  const T f04 = ((dx * dx) * cfield) * (h + (ss * hh) * (s1 / ex1));
  const T f12 = ((t * dx) * tt) / (ex * ex1);
  const T f13 = dS;
  const T sm = T(0.5) * ss;
  const T exm = T(0.5) * (ex + ex1);
  const T f14 = (((t * cfield) * (T(0.5) * (dx * dx))) * sm) / ((exm * exm) * exm);
  const T f24 = cfield * dx;

  st.y = st.y + dy;
  st.z = st.z + t * dS;
  st.s = s1;

  // C' = F C F^T, F = I + {f02,f04 | f12,f13,f14 | f24}.  M = F C (rows 0..2), then C' = M F^T.
  T* c = st.c;
  const T c00 = c[0], c10 = c[1], c11 = c[2], c20 = c[3], c21 = c[4], c22 = c[5];
  const T c30 = c[6], c31 = c[7], c32 = c[8], c33 = c[9];
  const T c40 = c[10], c41 = c[11], c42 = c[12], c43 = c[13], c44 = c[14];
  // row 0 of M
  const T m00 = (c00 + f02 * c20) + f04 * c40;
  const T m02 = (c20 + f02 * c22) + f04 * c42;
  const T m04 = (c40 + f02 * c42) + f04 * c44;
  // row 1 of M
  const T m10 = ((c10 + f12 * c20) + f13 * c30) + f14 * c40;
  const T m11 = ((c11 + f12 * c21) + f13 * c31) + f14 * c41;
  const T m12 = ((c21 + f12 * c22) + f13 * c32) + f14 * c42;
  const T m13 = ((c31 + f12 * c32) + f13 * c33) + f14 * c43;
  const T m14 = ((c41 + f12 * c42) + f13 * c43) + f14 * c44;
  // row 2 of M
  const T m20 = c20 + f24 * c40;
  const T m21 = c21 + f24 * c41;
  const T m22 = c22 + f24 * c42;
  const T m23 = c32 + f24 * c43;
  const T m24 = c42 + f24 * c44;
  // C' lower triangle
  c[0] = (m00 + f02 * m02) + f04 * m04;
  c[1] = (m10 + f02 * m12) + f04 * m14;
  c[2] = ((m11 + f12 * m12) + f13 * m13) + f14 * m14;
  c[3] = (m20 + f02 * m22) + f04 * m24;
  c[4] = ((m21 + f12 * m22) + f13 * m23) + f14 * m24;
  c[5] = m22 + f24 * m24;
  c[6] = (c30 + f02 * c32) + f04 * c43;
  c[7] = ((c31 + f12 * c32) + f13 * c33) + f14 * c43;
  c[8] = c32 + f24 * c43;
  // c[9] = c33 unchanged
  c[10] = (c40 + f02 * c42) + f04 * c44;
  c[11] = ((c41 + f12 * c42) + f13 * c43) + f14 * c44;
  c[12] = c42 + f24 * c44;
  // c[13], c[14] unchanged

  if (jac_out) {
    jac_out->f02 = f02; jac_out->f04 = f04; jac_out->f12 = f12;
    jac_out->f13 = f13; jac_out->f14 = f14; jac_out->f24 = f24;
  }
  return true;
}

// Innovation covariance inverse for a measurement (y,z) with V = diag(vy, vz).
// DESIGN.md section 3, block U.
template <class T>
struct KFGain {
  T si00, si01, si11;
};

template <class T>
inline KFGain<T> kf_gain(const KFState<T>& st, T vy, T vz) {
  const T s00 = st.c[0] + vy;
  const T s01 = st.c[1];
  const T s11 = st.c[2] + vz;
  const T det = s00 * s11 - s01 * s01;
  const T inv = T(1) / det;
  KFGain<T> g;
  g.si00 = s11 * inv;
  g.si01 = -(s01 * inv);
  g.si11 = s00 * inv;
  return g;
}

// chi2 of a candidate measurement against the predicted state.
template <class T>
inline T kf_chi2(const KFState<T>& st, const KFGain<T>& g, T ym, T zm) {
  const T r0 = ym - st.y;
  const T r1 = zm - st.z;
  return ((r0 * r0) * g.si00 + (T(2) * (r0 * r1)) * g.si01) + (r1 * r1) * g.si11;
}

// Kalman update with measurement (ym, zm).  Returns true if the leg must STOP afterwards
// (|sin(phi)| left the allowed range; it is clamped to +-max_sinphi so the state stays
// finite).  |q/pT| is clamped to max_qpt.
template <class T>
inline bool kf_update(KFState<T>& st, const KFGain<T>& g, T ym, T zm, T max_sinphi, T max_qpt) {
  T* c = st.c;
  const T r0 = ym - st.y;
  const T r1 = zm - st.z;
  // columns 0 and 1 of C (H picks y and z)
  const T a0[5] = {c[0], c[1], c[3], c[6], c[10]};   // C_i0
  const T a1[5] = {c[1], c[2], c[4], c[7], c[11]};   // C_i1
  T k0[5], k1[5];
  for (int i = 0; i < 5; ++i) {
    k0[i] = a0[i] * g.si00 + a1[i] * g.si01;
    k1[i] = a0[i] * g.si01 + a1[i] * g.si11;
  }
  st.y = st.y + (k0[0] * r0 + k1[0] * r1);
  st.z = st.z + (k0[1] * r0 + k1[1] * r1);
  st.s = st.s + (k0[2] * r0 + k1[2] * r1);
  st.t = st.t + (k0[3] * r0 + k1[3] * r1);
  st.q = st.q + (k0[4] * r0 + k1[4] * r1);
  // C_ij -= K_i0*C_j0 + K_i1*C_j1   (lower triangle, i >= j)
  int idx = 0;
  for (int i = 0; i < 5; ++i)
    for (int j = 0; j <= i; ++j, ++idx) c[idx] = c[idx] - (k0[i] * a0[j] + k1[i] * a1[j]);
  if (st.q > max_qpt) st.q = max_qpt;
  if (st.q < -max_qpt) st.q = -max_qpt;
  bool stop = false;
  if (!(o_abs(st.s) <= max_sinphi)) {
    st.s = (st.s < T(0)) ? -max_sinphi : max_sinphi;  // NaN also lands here -> +max
    stop = true;
  }
  return stop;
}

}  // namespace tpc_oracle
#endif
