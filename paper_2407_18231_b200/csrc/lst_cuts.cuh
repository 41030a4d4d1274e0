// lst_cuts.cuh -- device transcription of CUTS.md (the selection spec) for sm_100a.
// binary32, evaluated exactly as parenthesised in CUTS.md; the translation unit is compiled with
// -fmad=false (no FMA contraction), precise div/sqrt, no flush-to-zero.  Intrinsics __fmul_rn /
// __fadd_rn are NOT needed under -fmad=false; plain operators keep the code readable.
#pragma once
#include <cuda_runtime.h>

namespace lst {

struct Cuts {  // CUTS.md section 1: primary constants + derived (computed on the host in binary32)
  float z0_max;
  float md_b_phi_tol, md_z_tol, md_e_slope, md_e_tol;
  float ls_kappa_max, ls_z_tol, ls_dir_tol;
  float t3_kappa_max, t3_z_tol0, t3_z_tol1;
  float t5_tol0, t5_tol1;
  float pt_gate_tol, pt_k_tol0, pt_k_tol1, pt_z_tol;
  float near_rel;
  float kr, r_min, inv_2rmin;
  int stage_mask;
  // extensions: CUTS.md section 10 (T4) and section 11 (learned T5 selection)
  float t4_tol0, t4_tol1;
  float t5_mlp_scale, t5_mlp_thr;
  float t5_mlp[65];  // W1[8][6] row-major, b1[8], W2[8], b2
};

// CUTS.md section 0: near-threshold flag of a cut v <= t
__device__ __forceinline__ bool near_thr(const Cuts& c, float v, float t) {
  return fabsf(v - t) <= c.near_rel * fabsf(t);
}

// CUTS.md section 1: g(u) ~ asin(sqrt u)/sqrt u, Horner innermost first
__device__ __forceinline__ float g_poly(float u) {
  float t = u * 0.030381944f;
  t = 0.044642857f + t;
  t = u * t;
  t = 0.075f + t;
  t = u * t;
  t = 0.16666667f + t;
  t = u * t;
  return 1.0f + t;
}

// CUTS.md section 5: signed circumcircle curvature of P, Q, S (transverse plane)
__device__ __forceinline__ float kappa3(float xp, float yp, float xq, float yq, float xs, float ys,
                                        float& lpq, float& lqs) {
  float ax = xq - xp, ay = yq - yp;
  float bx = xs - xq, by = ys - yq;
  float cx = xs - xp, cy = ys - yp;
  lpq = sqrtf(ax * ax + ay * ay);
  lqs = sqrtf(bx * bx + by * by);
  float lps = sqrtf(cx * cx + cy * cy);
  float crs = ax * cy - ay * cx;
  return (2.0f * crs) / ((lpq * lqs) * lps);
}

// result bits of a candidate test
enum : unsigned { ACC = 1u, NEAR = 2u };

// CUTS.md section 3.  a = lower hit, b = upper hit, float4 = (x, y, z, r).
// On accept of a barrel pair, (ux, uy) receives the unit direction.
__device__ __forceinline__ unsigned md_test(const Cuts& c, bool endcap, float4 a, float4 b, float& ux,
                                            float& uy) {
  unsigned res = 0;
  if (!endcap) {
    float dx = b.x - a.x, dy = b.y - a.y;
    float dd = sqrtf(dx * dx + dy * dy);
    float dot = a.x * dx + a.y * dy;
    float crs = a.x * dy - a.y * dx;
    float lim = (a.w * dd) * (a.w * c.inv_2rmin + c.md_b_phi_tol);
    float zv = fabsf(b.z * a.w - a.z * b.w);
    float zl = c.z0_max * (b.w - a.w) + c.md_z_tol * a.w;
    if (dot > 0.0f) {
      if (near_thr(c, fabsf(crs), lim)) res |= NEAR;
      if (fabsf(crs) <= lim) {
        if (near_thr(c, zv, zl)) res |= NEAR;
        if (zv <= zl) {
          res |= ACC;
          ux = dx / dd;
          uy = dy / dd;
        }
      }
    }
  } else {
    float crs = a.x * b.y - a.y * b.x;
    float dz = fabsf(b.z - a.z);
    float den = fabsf(a.z) - c.z0_max;
    float lim = b.w * (((((a.w * a.w) * dz) * c.inv_2rmin) * c.md_e_slope) / den + c.md_e_tol);
    float rv = fabsf(b.w * a.z - a.w * b.z);
    float rl = c.z0_max * fabsf(b.w - a.w) + c.md_z_tol * fabsf(a.z);
    if (near_thr(c, fabsf(crs), lim)) res |= NEAR;
    if (fabsf(crs) <= lim) {
      if (near_thr(c, rv, rl)) res |= NEAR;
      if (rv <= rl) {
        res |= ACC;
        ux = 0.0f;
        uy = 0.0f;
      }
    }
  }
  return res;
}

// CUTS.md section 4.  A, B = MD anchors (x, y, z, r); uA, uB = unit directions.
__device__ __forceinline__ unsigned ls_test(const Cuts& c, float4 A, float2 uA, bool eA, float4 B,
                                            float2 uB, bool eB, float& kappa_out) {
  float ex = B.x - A.x, ey = B.y - A.y;
  float cc = sqrtf(ex * ex + ey * ey);
  float crs = A.x * B.y - A.y * B.x;
  float kappa = (2.0f * crs) / ((A.w * B.w) * cc);
  float kv = fabsf(kappa) * c.r_min;
  unsigned res = 0;
  if (near_thr(c, kv, c.ls_kappa_max)) res |= NEAR;
  if (!(kv <= c.ls_kappa_max)) return res;
  float tA = (A.w * kappa) * 0.5f;
  float gA = g_poly(tA * tA);
  float tB = (B.w * kappa) * 0.5f;
  float gB = g_poly(tB * tB);
  float rho = (B.w * gB) / (A.w * gA);
  bool e = eA || eB;
  float ztol = e ? c.ls_z_tol * (1.0f + fabsf(B.z) / B.w) : c.ls_z_tol;
  float zv = fabsf(B.z - A.z * rho);
  float zl = c.z0_max * (rho - 1.0f) + ztol;
  if (near_thr(c, zv, zl)) res |= NEAR;
  if (!(zv <= zl)) return res;
  float half = (cc * kappa) * 0.5f;
  if (!eA) {
    float sA = (uA.x * ey - uA.y * ex) / cc;
    float dA = fabsf(sA - half);
    if (near_thr(c, dA, c.ls_dir_tol)) res |= NEAR;
    if (!(dA <= c.ls_dir_tol)) return res;
  }
  if (!eB) {
    float sB = (uB.x * ey - uB.y * ex) / cc;
    float dB = fabsf(sB + half);
    if (near_thr(c, dB, c.ls_dir_tol)) res |= NEAR;
    if (!(dB <= c.ls_dir_tol)) return res;
  }
  kappa_out = kappa;
  return res | ACC;
}

// CUTS.md section 5 (reading S2).  e = endcap(A) || endcap(B) || endcap(C).
__device__ __forceinline__ unsigned t3_test(const Cuts& c, float4 A, float4 B, float4 C, bool e,
                                            float& k3_out) {
  float lpq, lqs;
  float k3 = kappa3(A.x, A.y, B.x, B.y, C.x, C.y, lpq, lqs);
  float kv = fabsf(k3) * c.r_min;
  unsigned res = 0;
  if (near_thr(c, kv, c.t3_kappa_max)) res |= NEAR;
  if (!(kv <= c.t3_kappa_max)) return res;
  float ratio = lqs / lpq;
  float zpred = B.z + (B.z - A.z) * ratio;
  float tol = c.t3_z_tol0 + c.t3_z_tol1 * ratio;
  tol = e ? tol * (1.0f + fabsf(C.z) / C.w) : tol;
  float zv = fabsf(C.z - zpred);
  if (near_thr(c, zv, tol)) res |= NEAR;
  if (!(zv <= tol)) return res;
  k3_out = k3;
  return res | ACC;
}

// CUTS.md section 6 (reading S3).  B, C, D = anchors of the bridge MDs.  With stage-mask bit 7
// the three pairwise cuts are replaced by the one cut of CUTS.md section 11.
__device__ __forceinline__ unsigned t5_test(const Cuts& c, float ki, float ko, float4 B, float4 C,
                                            float4 D, float& score_out) {
  float l0, l1;
  float kb = kappa3(B.x, B.y, C.x, C.y, D.x, D.y, l0, l1);
  float d1 = ki - kb, d2 = kb - ko, d3 = ki - ko;
  unsigned res = 0;
  if (c.stage_mask & 128) {
    const float S = c.t5_mlp_scale;
    const float f[6] = {fabsf(ki) * S, fabsf(kb) * S, fabsf(ko) * S, fabsf(d1) * S, fabsf(d2) * S, fabsf(d3) * S};
    float s = c.t5_mlp[64];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      float a = c.t5_mlp[48 + j];
#pragma unroll
      for (int i = 0; i < 6; ++i) a = a + c.t5_mlp[6 * j + i] * f[i];
      s = s + c.t5_mlp[56 + j] * fmaxf(a, 0.0f);
    }
    if (near_thr(c, s, c.t5_mlp_thr)) res |= NEAR;
    if (!(s <= c.t5_mlp_thr)) return res;
  } else {
    float tol = c.t5_tol0 + c.t5_tol1 * fmaxf(fabsf(ki), fabsf(ko));
    if (near_thr(c, fabsf(d1), tol)) res |= NEAR;
    if (!(fabsf(d1) <= tol)) return res;
    if (near_thr(c, fabsf(d2), tol)) res |= NEAR;
    if (!(fabsf(d2) <= tol)) return res;
    if (near_thr(c, fabsf(d3), tol)) res |= NEAR;
    if (!(fabsf(d3) <= tol)) return res;
  }
  score_out = (d1 * d1 + d2 * d2) + d3 * d3;
  return res | ACC;
}

// CUTS.md section 10: T4 = two T3s sharing two MDs; k1, k2 = their stored curvatures
__device__ __forceinline__ unsigned t4_test(const Cuts& c, float k1, float k2, float& score_out) {
  const float tol = c.t4_tol0 + c.t4_tol1 * fmaxf(fabsf(k1), fabsf(k2));
  const float dd = k1 - k2;
  unsigned res = near_thr(c, fabsf(dd), tol) ? NEAR : 0u;
  if (!(fabsf(dd) <= tol)) return res;
  score_out = dd * dd;
  return res | ACC;
}

// ---- approximate classification of a cut v <= t (used by the pre-filters of MD, LS and the seed linking) ----
// A pre-filter evaluates a cut with cheaper arithmetic (rsqrt.approx, approximate division, FMA) and a band
// b >= |v~ - v| + |t~ - t| + 1e-5 |t| (the near-threshold window of CUTS.md section 0):
//   v~ > t~ + b  =>  the exact cut fails and is not near     (PT_FAIL)
//   v~ < t~ - b  =>  the exact cut passes and is not near    (PT_PASS)
//   otherwise, or when an operand is NaN / outside the range where the error bound holds: PT_UNSURE,
//   and the exact arithmetic of the spec decides.
// A candidate is dropped only at a cut that surely fails AFTER cuts that surely pass: the spec rejects it at
// that cut without a near flag (evaluation stops at the first failed cut), so objects AND counters are unchanged.
enum PtClass : int { PT_FAIL = 0, PT_PASS = 1, PT_UNSURE = 2 };

__device__ __forceinline__ float rsqrt_approx(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

__device__ __forceinline__ int classify(float v, float t, float band, bool ok) {
  if (ok && v > t + band) return PT_FAIL;
  if (ok && v < t - band) return PT_PASS;
  return PT_UNSURE;  // includes every NaN
}

// CUTS.md section 3 without sqrt or division.  Barrel: crs, dot, K = ra INV_2RMIN + tol, zv, zl are formed
// exactly as in the spec; only lim = (ra dd) K is replaced by lim^2 ~ ((ra ra)(dx^2 + dy^2))(K K) (relative
// error < 5e-7), compared with crs^2 at +-1e-4 (= +-5e-5 on |crs| / lim, 5x the near window).  The second
// cut is the spec's own arithmetic.  Endcap: bend / den by approximate division (2^-22), band 3e-5.
__device__ __forceinline__ int md_class(const Cuts& c, bool endcap, float4 a, float4 b) {
  if (!endcap) {
    const float dx = b.x - a.x, dy = b.y - a.y;
    const float dot = a.x * dx + a.y * dy;
    const float crs = a.x * dy - a.y * dx;
    if (!(dot > 0.0f)) return PT_FAIL;  // strict cut, never flagged (a NaN fails it, as in the spec)
    const float K = a.w * c.inv_2rmin + c.md_b_phi_tol;
    const float lim2 = ((a.w * a.w) * fmaf(dx, dx, dy * dy)) * (K * K);
    const float c2 = crs * crs;
    const bool ok = K >= 0.0f && lim2 >= 1e-30f && lim2 <= 1e30f;
    if (ok && c2 > lim2 * 1.0001f) return PT_FAIL;
    if (!(ok && c2 < lim2 * 0.9999f)) return PT_UNSURE;
    const float zv = fabsf(b.z * a.w - a.z * b.w);
    const float zl = c.z0_max * (b.w - a.w) + c.md_z_tol * a.w;
    if (near_thr(c, zv, zl) || !(zl == zl)) return PT_UNSURE;
    return zv <= zl ? PT_PASS : PT_FAIL;
  }
  const float crs = a.x * b.y - a.y * b.x;
  const float dz = fabsf(b.z - a.z);
  const float den = fabsf(a.z) - c.z0_max;
  const float q = __fdividef((((a.w * a.w) * dz) * c.inv_2rmin) * c.md_e_slope, den);
  const float lim = b.w * (q + c.md_e_tol);
  const float band = 3e-5f * (fabsf(lim) + fabsf(b.w * q));
  const int c1 = classify(fabsf(crs), lim, band, fabsf(den) >= 1e-30f && fabsf(den) <= 1e30f);
  if (c1 != PT_PASS) return c1;
  const float rv = fabsf(b.w * a.z - a.w * b.z);
  const float rl = c.z0_max * fabsf(b.w - a.w) + c.md_z_tol * fabsf(a.z);
  if (near_thr(c, rv, rl) || !(rl == rl)) return PT_UNSURE;
  return rv <= rl ? PT_PASS : PT_FAIL;
}

// CUTS.md section 4 with one rsqrt.approx per length and approximate divisions.  PT_FAIL = surely rejected and
// not near; anything else needs the exact cut list (an accepted LS needs its exact kappa anyway).
// Errors against the spec's binary32 values: kappa 1e-6 relative (crs exact); g(t^2) 1e-6 (u g'/g <= 0.43 for
// u <= 1, same polynomial); rho 3e-6; c and 1/c 4e-7.
__device__ __forceinline__ int ls_class(const Cuts& c, float4 A, float2 uA, bool eA, float4 B, float2 uB, bool eB) {
  const float ex = B.x - A.x, ey = B.y - A.y;
  const float c2 = fmaf(ex, ex, ey * ey);
  const float crs = A.x * B.y - A.y * B.x;
  const float rr = A.w * B.w;
  const float den2 = (rr * rr) * c2;
  bool ok = den2 >= 1e-30f && den2 <= 1e30f && c2 >= 1e-30f && c2 <= 1e30f && rr >= 0.0f;
  const float kappa = (2.0f * crs) * rsqrt_approx(den2);  // rA, rB >= 0 (square roots) or NaN (-> not ok)
  const float kv = fabsf(kappa) * c.r_min;
  int cl = classify(kv, c.ls_kappa_max, 2e-5f * fabsf(c.ls_kappa_max) + 3e-6f * kv, ok);
  if (cl != PT_PASS) return cl;
  const float tA = (A.w * kappa) * 0.5f, tB = (B.w * kappa) * 0.5f;
  ok = ok && fabsf(tA) <= 1.0f && fabsf(tB) <= 1.0f;
  const float rho = __fdividef(B.w * g_poly(tB * tB), A.w * g_poly(tA * tA));
  const float ztol = (eA || eB) ? c.ls_z_tol * (1.0f + __fdividef(fabsf(B.z), B.w)) : c.ls_z_tol;
  const float zar = A.z * rho;
  const float zv = fabsf(B.z - zar);
  const float zl = c.z0_max * (rho - 1.0f) + ztol;
  cl = classify(zv, zl, 1.2e-5f * fabsf(zl) + 5e-6f * (fabsf(zar) + fabsf(c.z0_max * rho)) + 1e-6f * (fabsf(B.z) + fabsf(ztol)), ok);
  if (cl != PT_PASS) return cl;
  const float icc = rsqrt_approx(c2);
  const float half = ((c2 * icc) * kappa) * 0.5f;
  if (!eA) {
    const float sA = (uA.x * ey - uA.y * ex) * icc;
    cl = classify(fabsf(sA - half), c.ls_dir_tol, 1.2e-5f * fabsf(c.ls_dir_tol) + 3e-6f * (fabsf(sA) + fabsf(half)), ok);
    if (cl != PT_PASS) return cl;
  }
  if (!eB) {
    const float sB = (uB.x * ey - uB.y * ex) * icc;
    cl = classify(fabsf(sB + half), c.ls_dir_tol, 1.2e-5f * fabsf(c.ls_dir_tol) + 3e-6f * (fabsf(sB) + fabsf(half)), ok);
    if (cl != PT_PASS) return cl;
  }
  return PT_PASS;
}

}  // namespace lst
