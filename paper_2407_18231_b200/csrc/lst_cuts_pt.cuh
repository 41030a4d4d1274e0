// lst_cuts_pt.cuh -- CUTS.md section 7: pLS x T3 / T5 linking (readings S6, S7).
#pragma once
#include "lst_cuts.cuh"

namespace lst {

struct Seed {  // per-pLS quantities that do not depend on the candidate (CUTS.md section 7)
  float x1, y1, z1;
  float vx, vy, lv;  // P1 - P0 and its transverse length
  float kp;          // (-q) / (pt * KR)
  float slope;       // (z1 - z0) / lv
  float tolk;        // PT_K_TOL0 + PT_K_TOL1 * |kp|
};

__device__ __forceinline__ Seed make_seed(const Cuts& c, float pt, int q, float x0, float y0, float z0,
                                          float x1, float y1, float z1) {
  Seed s;
  s.x1 = x1;
  s.y1 = y1;
  s.z1 = z1;
  float qf = (float)q;
  s.kp = (-qf) / (pt * c.kr);
  s.vx = x1 - x0;
  s.vy = y1 - y0;
  s.lv = sqrtf(s.vx * s.vx + s.vy * s.vy);
  s.slope = (z1 - z0) / s.lv;
  s.tolk = c.pt_k_tol0 + c.pt_k_tol1 * fabsf(s.kp);
  return s;
}

// Gate on the first MD anchor (ax, ay).  Returns ACC if the gate passes, NEAR if the gcrs cut was
// evaluated and is near-threshold (the strict gdot > 0 cut is never flagged).
__device__ __forceinline__ unsigned pt_gate(const Cuts& c, const Seed& s, float ax, float ay) {
  float wx = ax - s.x1, wy = ay - s.y1;
  float gdot = s.vx * wx + s.vy * wy;
  if (!(gdot > 0.0f)) return 0;
  float lw = sqrtf(wx * wx + wy * wy);
  float gcrs = fabsf(s.vx * wy - s.vy * wx);
  float glim = (s.lv * lw) * (lw * c.inv_2rmin + c.pt_gate_tol);
  unsigned res = near_thr(c, gcrs, glim) ? NEAR : 0u;
  if (gcrs <= glim) res |= ACC;
  return res;
}

// r-z extrapolation cut at anchor Q (CUTS.md section 7, loop over Q in (A, L))
__device__ __forceinline__ unsigned pt_rz(const Cuts& c, const Seed& s, float kx, float4 Q, bool eQ) {
  float qx = Q.x - s.x1, qy = Q.y - s.y1;
  float lq = sqrtf(qx * qx + qy * qy);
  float tq = (lq * kx) * 0.5f;
  float sq = lq * g_poly(tq * tq);
  float zq = fabsf(Q.z - (s.z1 + s.slope * sq));
  float zt = eQ ? c.pt_z_tol * (1.0f + fabsf(Q.z) / Q.w) : c.pt_z_tol;
  unsigned res = near_thr(c, zq, zt) ? NEAR : 0u;
  if (zq <= zt) res |= ACC;
  return res;
}

// Cuts after the gate.  kt[0..n_kt) = stored curvatures (k3 of a T3; ki, ko of a T5);
// base = 0 for a pT3, the T5 score for a pT5.  A = first MD anchor, L = last MD anchor.
template <int N_KT>
__device__ __forceinline__ unsigned pt_after_gate(const Cuts& c, const Seed& s, float4 A, bool eA,
                                                  float4 L, bool eL, const float (&kt)[N_KT],
                                                  float base, float& score_out) {
  float l0, l1;
  float kx = kappa3(s.x1, s.y1, A.x, A.y, L.x, L.y, l0, l1);
  float dp = kx - s.kp;
  unsigned res = near_thr(c, fabsf(dp), s.tolk) ? NEAR : 0u;
  if (!(fabsf(dp) <= s.tolk)) return res;
  float score = dp * dp;
#pragma unroll
  for (int i = 0; i < N_KT; ++i) {
    float dk = kx - kt[i];
    if (near_thr(c, fabsf(dk), s.tolk)) res |= NEAR;
    if (!(fabsf(dk) <= s.tolk)) return res;
    score = score + dk * dk;
  }
  unsigned r = pt_rz(c, s, kx, A, eA);
  res |= (r & NEAR);
  if (!(r & ACC)) return res;
  r = pt_rz(c, s, kx, L, eL);
  res |= (r & NEAR);
  if (!(r & ACC)) return res;
  score_out = score + base;
  return res | ACC;
}

// Necessary condition of the curvature match |kx - kp| <= tolk, kx = kappa3(P1, A, L) (CUTS.md
// section 7), without sqrt or division: compares kx^2 = 4 crs^2 / (|P1A|^2 |AL|^2 |P1L|^2) with
// (|kp| -+ tolk)^2.  false = the exact cut rejects AND is not near-threshold.
// Inequality chain.  Let k2/prod = kx~^2 be what is computed here and kx the spec's binary32 value: crs is
// formed exactly as in kappa3 (same operands, same order), the rest differs by |kx~ - kx| <= d |kx| with
// d < 4e-6 (three sqrt, four products and one division on the spec's side, five products here).  The exact
// cut flags or accepts only if |kp| - tolk (1 + 1e-5) <= |kx| <= |kp| + tolk (1 + 1e-5).  With
// m = 1e-3 (|kp| + tolk):
//   reject high: |kx~| > hi = |kp| + tolk + m   =>  |kx| >= |kx~| (1 - d) > |kp| + tolk (1 + 1e-5)
//   reject low:  |kx~| < lo = |kp| - tolk - m   =>  |kx| <= |kx~| (1 + d) < |kp| - tolk (1 + 1e-5)
// because m - d (|kp| + tolk + m) > 1e-5 tolk (m is taken relative to |kp| + tolk, NOT to |kp| - tolk: the
// latter margin vanishes where |kp| ~ tolk, i.e. for seeds of pT ~ 20.4 GeV).  The sign test needs lo > 0.
// kp = (-q) / (pt * KR), tolk = PT_K_TOL0 + PT_K_TOL1 * |kp| (as in make_seed).
__device__ __forceinline__ bool pt_curv_possible(float kp, float tolk, float x1, float y1, float2 A, float2 L) {
  const float ax = A.x - x1, ay = A.y - y1;
  const float bx = L.x - A.x, by = L.y - A.y;
  const float cx = L.x - x1, cy = L.y - y1;
  const float crs = ax * cy - ay * cx;
  const float prod = ((ax * ax + ay * ay) * (bx * bx + by * by)) * (cx * cx + cy * cy);
  const float k2 = 4.0f * (crs * crs);
  const float m = 1e-3f * (fabsf(kp) + tolk);
  const float hi = (fabsf(kp) + tolk) + m;
  if (k2 > (hi * hi) * prod) return false;
  const float lo = (fabsf(kp) - tolk) - m;
  if (lo > 0.0f) {
    if (k2 < (lo * lo) * prod) return false;
    if ((crs > 0.0f) != (kp > 0.0f)) return false;  // |kx| >= lo (1 - d) > 0 with the wrong sign: |kx - kp| > |kp| > tolk (1 + 1e-5)
  }
  return true;
}

}  // namespace lst
