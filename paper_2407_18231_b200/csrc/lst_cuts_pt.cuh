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

// ---- approximate cascade: which candidates can the exact cuts accept or flag? -------------------------
// The seed linking evaluates ~1e7 (seed, T3 / T5) candidates per batch behind the gate and accepts 0.06 %.
// The exact cut list (precise sqrt and division, ~700 thread instructions) is therefore run only on the
// candidates that an APPROXIMATE evaluation of the same cuts, in the same order, cannot reject for sure:
//   * kx~ ~ kappa3(P1, A, L): crs is formed exactly as in kappa3 (same operands, same order, no FMA), the
//     three lengths by ONE rsqrt.approx of the product of the squared lengths.  Against the spec's binary32
//     kx: |kx~ - kx| <= d |kx|, d < 1.2e-6 (spec side: three sqrt, two products, one division <= 9 ulp;
//     here: three fused squares, two products, rsqrt.approx (2^-22), one product <= 8 ulp; 1 ulp = 6e-8);
//     the bands below take d = 4e-6.
//   * a cut v <= t is classified with a band b >= |v~ - v| + 1e-5 t (the near-threshold window):
//     v~ > t + b: the exact cut fails and is not near; v~ < t - b: it passes and is not near; otherwise
//     (or when an operand is NaN / out of the approximation's range) the candidate goes to the exact cuts.
//   * a candidate is dropped only at a cut that surely fails AFTER cuts that surely pass: it is then
//     rejected by the spec at that cut without a near flag, so objects AND counters are unchanged
//     (CUTS.md section 0: evaluation stops at the first failed cut).
// Bands: curvature cuts b = 1.2e-5 tolk + 4e-6 |kx~| (|dp~ - dp| <= d |kx|);
//        r-z cuts      b = 1.2e-5 zt + 8e-6 |slope sq~| + 1e-6 (|z1| + |zQ|)
//        (sq = lq g((lq kx / 2)^2): rel. error <= 3 ulp (lq) + 0.43 * 2 (d + 5 ulp) (g, u g'/g <= 0.43 on
//        u <= 1) + polynomial rounding < 5e-6; the last term covers the roundings of the sum).
// kx~; ok = false when the product of the squared lengths leaves the range where the bound holds
__device__ __forceinline__ float kx_approx(float x1, float y1, float xa, float ya, float xl, float yl, bool& ok) {
  const float ax = xa - x1, ay = ya - y1;
  const float bx = xl - xa, by = yl - ya;
  const float cx = xl - x1, cy = yl - y1;
  const float crs = ax * cy - ay * cx;  // no FMA contraction in this translation unit: the spec's crs
  const float prod = (fmaf(ax, ax, ay * ay) * fmaf(bx, bx, by * by)) * fmaf(cx, cx, cy * cy);
  ok = prod >= 1e-30f && prod <= 1e30f;
  return (2.0f * crs) * rsqrt_approx(prod);
}

__device__ __forceinline__ int pt_class_curv(float kx, float kref, float tolk, bool ok) {
  return classify(fabsf(kx - kref), tolk, 1.2e-5f * fabsf(tolk) + 4e-6f * fabsf(kx), ok);
}

// r-z cut at Q = (x, y, z, r | endcap << 31)
__device__ __forceinline__ int pt_class_rz(const Cuts& c, float x1, float y1, float z1, float slope, float kx,
                                           float4 Q, bool ok) {
  const float qx = Q.x - x1, qy = Q.y - y1;
  const float lq2 = fmaf(qx, qx, qy * qy);
  ok = ok && lq2 >= 1e-30f && lq2 <= 1e30f;
  const float lq = lq2 * rsqrt_approx(lq2);
  const float tq = (lq * kx) * 0.5f;
  const float sq = lq * g_poly(tq * tq);
  const float pred = slope * sq;
  const float zq = fabsf(Q.z - (z1 + pred));
  const bool eQ = __float_as_int(Q.w) < 0;
  const float zt = eQ ? c.pt_z_tol * (1.0f + __fdividef(fabsf(Q.z), fabsf(Q.w))) : c.pt_z_tol;
  const float band = 1.2e-5f * fabsf(zt) + 8e-6f * fabsf(pred) + 1e-6f * (fabsf(z1) + fabsf(Q.z));
  return classify(zq, zt, band, ok && fabsf(tq) <= 1.0f);
}

}  // namespace lst
