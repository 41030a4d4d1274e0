/* lst_oracle.c -- CPU oracle of the LST object-building chain.  TEST INFRASTRUCTURE ONLY.
 * See lst_oracle.h.  Every function cites the CUTS.md section (and PAPER.md passage) it follows.
 * Plain loops, no blocking, no reordering; binary32 arithmetic written exactly as parenthesised in
 * CUTS.md.  Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC.
 */
#include "lst_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------------------------- */
/* CUTS.md section 1 */
void orc_default_params(orc_params* p) {
  p->b_field = 3.8f;
  p->pt_min = 0.8f;
  p->z0_max = 15.0f;
  p->md_b_phi_tol = 0.06f;
  p->md_z_tol = 0.9f;
  p->md_e_slope = 1.15f;
  p->md_e_tol = 0.015f;
  p->ls_kappa_max = 1.05f;
  p->ls_z_tol = 1.0f;
  p->ls_dir_tol = 0.05f;
  p->t3_kappa_max = 1.10f;
  p->t3_z_tol0 = 1.0f;
  p->t3_z_tol1 = 0.6f;
  p->t5_tol0 = 4e-4f;
  p->t5_tol1 = 0.05f;
  p->pt_gate_tol = 0.05f;
  p->pt_k_tol0 = 5e-4f;
  p->pt_k_tol1 = 0.10f;
  p->pt_z_tol = 2.0f;
  p->near_rel = 1e-5f;
  p->stage_mask = 0x3f;
  p->t4_tol0 = 4e-4f;
  p->t4_tol1 = 0.05f;
  p->t5_mlp_scale = 100.0f;
  p->t5_mlp_thr = 1.0f;
  for (int i = 0; i < 65; ++i) p->t5_mlp[i] = 0.0f;
}

void orc_derived(const orc_params* p, float out[3]) {
  float kr = 100.0f / (0.3f * p->b_field);
  float r_min = p->pt_min * kr;
  float inv_2rmin = 1.0f / (2.0f * r_min);
  out[0] = kr;
  out[1] = r_min;
  out[2] = inv_2rmin;
}

/* CUTS.md section 0: near-threshold flag of a cut v <= t */
static int near_thr(const orc_params* p, float v, float t) {
  return fabsf(v - t) <= p->near_rel * fabsf(t);
}

/* CUTS.md section 1 */
float orc_g(float u) {
  float t = u * 0.030381944f;
  t = 0.044642857f + t;
  t = u * t;
  t = 0.075f + t;
  t = u * t;
  t = 0.16666667f + t;
  t = u * t;
  return 1.0f + t;
}

/* CUTS.md section 5 */
float orc_kappa3(float xp, float yp, float xq, float yq, float xs, float ys, float* len) {
  float ax = xq - xp, ay = yq - yp;
  float bx = xs - xq, by = ys - yq;
  float cx = xs - xp, cy = ys - yp;
  float lpq = sqrtf(ax * ax + ay * ay);
  float lqs = sqrtf(bx * bx + by * by);
  float lps = sqrtf(cx * cx + cy * cy);
  float crs = ax * cy - ay * cx;
  if (len) {
    len[0] = lpq;
    len[1] = lqs;
    len[2] = lps;
  }
  return (2.0f * crs) / ((lpq * lqs) * lps);
}

/* CUTS.md section 3 (hit pair on the two sensors of a module, window tuned to
 * pT >= 0.8 GeV) */
int orc_md_test(const orc_params* p, int endcap, float xa, float ya, float za, float xb, float yb,
                float zb, float* vals, int* near) {
  float d[3];
  orc_derived(p, d);
  float inv_2rmin = d[2];
  float ra = sqrtf(xa * xa + ya * ya);
  float rb = sqrtf(xb * xb + yb * yb);
  int nr = 0, acc = 0;
  if (!endcap) {
    float dx = xb - xa, dy = yb - ya;
    float dd = sqrtf(dx * dx + dy * dy);
    float dot = xa * dx + ya * dy;
    float crs = xa * dy - ya * dx;
    float lim = (ra * dd) * (ra * inv_2rmin + p->md_b_phi_tol);
    float zv = fabsf(zb * ra - za * rb);
    float zl = p->z0_max * (rb - ra) + p->md_z_tol * ra;
    if (dot > 0.0f) {
      nr |= near_thr(p, fabsf(crs), lim);
      if (fabsf(crs) <= lim) {
        nr |= near_thr(p, zv, zl);
        if (zv <= zl) acc = 1;
      }
    }
    if (vals) {
      vals[0] = dd; vals[1] = dot; vals[2] = crs; vals[3] = lim; vals[4] = zv; vals[5] = zl;
      vals[6] = dx / dd; vals[7] = dy / dd;
    }
  } else {
    float crs = xa * yb - ya * xb;
    float dz = fabsf(zb - za);
    float den = fabsf(za) - p->z0_max;
    float lim = rb * (((((ra * ra) * dz) * inv_2rmin) * p->md_e_slope) / den + p->md_e_tol);
    float rv = fabsf(rb * za - ra * zb);
    float rl = p->z0_max * fabsf(rb - ra) + p->md_z_tol * fabsf(za);
    nr |= near_thr(p, fabsf(crs), lim);
    if (fabsf(crs) <= lim) {
      nr |= near_thr(p, rv, rl);
      if (rv <= rl) acc = 1;
    }
    if (vals) {
      vals[0] = crs; vals[1] = lim; vals[2] = rv; vals[3] = rl;
      vals[4] = vals[5] = vals[6] = vals[7] = 0.0f;
    }
  }
  if (near) *near = nr;
  return acc;
}

/* CUTS.md section 4 (two MDs on connected modules linked into a Line Segment) */
int orc_ls_test(const orc_params* p, const float* A, int eA, const float* B, int eB, float* vals,
                int* near) {
  float d[3];
  orc_derived(p, d);
  float r_min = d[1];
  float xA = A[0], yA = A[1], zA = A[2], rA = A[3], uxA = A[4], uyA = A[5];
  float xB = B[0], yB = B[1], zB = B[2], rB = B[3], uxB = B[4], uyB = B[5];
  float ex = xB - xA, ey = yB - yA;
  float c = sqrtf(ex * ex + ey * ey);
  float crs = xA * yB - yA * xB;
  float kappa = (2.0f * crs) / ((rA * rB) * c);
  float kv = fabsf(kappa) * r_min;
  float tA = (rA * kappa) * 0.5f;
  float gA = orc_g(tA * tA);
  float tB = (rB * kappa) * 0.5f;
  float gB = orc_g(tB * tB);
  float rho = (rB * gB) / (rA * gA);
  int e = eA || eB;
  float ztol = e ? p->ls_z_tol * (1.0f + fabsf(zB) / rB) : p->ls_z_tol;
  float zv = fabsf(zB - zA * rho);
  float zl = p->z0_max * (rho - 1.0f) + ztol;
  float half = (c * kappa) * 0.5f;
  float dA = 0.0f, dB = 0.0f;
  if (!eA) {
    float sA = (uxA * ey - uyA * ex) / c;
    dA = fabsf(sA - half);
  }
  if (!eB) {
    float sB = (uxB * ey - uyB * ex) / c;
    dB = fabsf(sB + half);
  }
  int nr = 0, acc = 0;
  nr |= near_thr(p, kv, p->ls_kappa_max);
  if (kv <= p->ls_kappa_max) {
    nr |= near_thr(p, zv, zl);
    if (zv <= zl) {
      int okA = 1;
      if (!eA) {
        nr |= near_thr(p, dA, p->ls_dir_tol);
        okA = dA <= p->ls_dir_tol;
      }
      if (okA) {
        int okB = 1;
        if (!eB) {
          nr |= near_thr(p, dB, p->ls_dir_tol);
          okB = dB <= p->ls_dir_tol;
        }
        if (okB) acc = 1;
      }
    }
  }
  if (vals) {
    vals[0] = kappa; vals[1] = kv; vals[2] = rho; vals[3] = zv; vals[4] = zl; vals[5] = half;
    vals[6] = dA; vals[7] = dB;
  }
  if (near) *near = nr;
  return acc;
}

/* CUTS.md section 5 (two LSs with a common MD form a T3; reading S2 = chain) */
int orc_t3_test(const orc_params* p, const float* A, int eA, const float* B, int eB, const float* C,
                int eC, float* vals, int* near) {
  float d[3];
  orc_derived(p, d);
  float r_min = d[1];
  float len[3];
  float k3 = orc_kappa3(A[0], A[1], B[0], B[1], C[0], C[1], len);
  float kv = fabsf(k3) * r_min;
  float ratio = len[1] / len[0];
  float zA = A[2], zB = B[2], zC = C[2], rC = C[3];
  float zpred = zB + (zB - zA) * ratio;
  int e = eA || eB || eC;
  float tol = p->t3_z_tol0 + p->t3_z_tol1 * ratio;
  tol = e ? tol * (1.0f + fabsf(zC) / rC) : tol;
  float zv = fabsf(zC - zpred);
  int nr = 0, acc = 0;
  nr |= near_thr(p, kv, p->t3_kappa_max);
  if (kv <= p->t3_kappa_max) {
    nr |= near_thr(p, zv, tol);
    if (zv <= tol) acc = 1;
  }
  if (vals) {
    vals[0] = k3; vals[1] = ratio; vals[2] = zv; vals[3] = tol;
  }
  if (near) *near = nr;
  return acc;
}

/* CUTS.md section 6 (two T3s with a common MD form a T5; reading S3) */
int orc_t5_test(const orc_params* p, float ki, float ko, const float* B, const float* C,
                const float* D, float* vals, int* near) {
  float kb = orc_kappa3(B[0], B[1], C[0], C[1], D[0], D[1], 0);
  float tol = p->t5_tol0 + p->t5_tol1 * fmaxf(fabsf(ki), fabsf(ko));
  float d1 = ki - kb, d2 = kb - ko, d3 = ki - ko;
  int nr = 0, acc = 0;
  float s = 0.0f;
  if (p->stage_mask & 128) {
    /* CUTS.md section 11: one cut on a 6-8-1 rectifier perceptron */
    const float* W1 = p->t5_mlp;
    const float* b1 = p->t5_mlp + 48;
    const float* W2 = p->t5_mlp + 56;
    float S = p->t5_mlp_scale;
    float f[6] = {fabsf(ki) * S, fabsf(kb) * S, fabsf(ko) * S, fabsf(d1) * S, fabsf(d2) * S, fabsf(d3) * S};
    float h[8];
    for (int j = 0; j < 8; ++j) {
      float a = b1[j];
      for (int i = 0; i < 6; ++i) a = a + W1[6 * j + i] * f[i];
      h[j] = fmaxf(a, 0.0f);
    }
    s = p->t5_mlp[64];
    for (int j = 0; j < 8; ++j) s = s + W2[j] * h[j];
    nr |= near_thr(p, s, p->t5_mlp_thr);
    if (s <= p->t5_mlp_thr) acc = 1;
  } else {
    nr |= near_thr(p, fabsf(d1), tol);
    if (fabsf(d1) <= tol) {
      nr |= near_thr(p, fabsf(d2), tol);
      if (fabsf(d2) <= tol) {
        nr |= near_thr(p, fabsf(d3), tol);
        if (fabsf(d3) <= tol) acc = 1;
      }
    }
  }
  if (vals) {
    vals[0] = kb; vals[1] = tol; vals[2] = (d1 * d1 + d2 * d2) + d3 * d3; vals[3] = s;
  }
  if (near) *near = nr;
  return acc;
}

/* CUTS.md section 10 ("more objects": a 4-MD object from two T3s sharing two MDs) */
int orc_t4_test(const orc_params* p, float k1, float k2, float* vals, int* near) {
  float tol = p->t4_tol0 + p->t4_tol1 * fmaxf(fabsf(k1), fabsf(k2));
  float d = k1 - k2;
  int nr = near_thr(p, fabsf(d), tol);
  int acc = fabsf(d) <= tol;
  if (vals) {
    vals[0] = d; vals[1] = tol; vals[2] = d * d; vals[3] = 0.0f;
  }
  if (near) *near = nr;
  return acc;
}

/* CUTS.md section 7 (T3s and T5s combined with IT tracks (pLSs) into pT3s / pT5s) */
int orc_pt_test(const orc_params* p, const float* pls, const float* A, int eA, const float* L,
                int eL, const float* kt, int n_kt, float base_score, float* vals, int* near) {
  float d[3];
  orc_derived(p, d);
  float kr = d[0], inv_2rmin = d[2];
  float pt = pls[0], q = pls[1];
  float x0 = pls[2], y0 = pls[3], z0 = pls[4], x1 = pls[5], y1 = pls[6], z1 = pls[7];
  float kp = (-q) / (pt * kr);
  float vx = x1 - x0, vy = y1 - y0;
  float lv = sqrtf(vx * vx + vy * vy);
  float wx = A[0] - x1, wy = A[1] - y1;
  float lw = sqrtf(wx * wx + wy * wy);
  float gdot = vx * wx + vy * wy;
  float gcrs = fabsf(vx * wy - vy * wx);
  float glim = (lv * lw) * (lw * inv_2rmin + p->pt_gate_tol);
  float kx = orc_kappa3(x1, y1, A[0], A[1], L[0], L[1], 0);
  float tolk = p->pt_k_tol0 + p->pt_k_tol1 * fabsf(kp);
  float dp = kx - kp;
  float slope = (z1 - z0) / lv;
  float zq[2], zt[2];
  const float* Q[2] = {A, L};
  int eQ[2] = {eA, eL};
  for (int i = 0; i < 2; ++i) {
    float qx = Q[i][0] - x1, qy = Q[i][1] - y1;
    float lq = sqrtf(qx * qx + qy * qy);
    float tq = (lq * kx) * 0.5f;
    float sq = lq * orc_g(tq * tq);
    float zQ = Q[i][2], rQ = Q[i][3];
    zq[i] = fabsf(zQ - (z1 + slope * sq));
    zt[i] = eQ[i] ? p->pt_z_tol * (1.0f + fabsf(zQ) / rQ) : p->pt_z_tol;
  }
  float score = dp * dp;
  for (int i = 0; i < n_kt; ++i) {
    float dk = kx - kt[i];
    score = score + dk * dk;
  }
  score = score + base_score;

  int nr = 0, acc = 0;
  if (gdot > 0.0f) {
    nr |= near_thr(p, gcrs, glim);
    if (gcrs <= glim) {
      nr |= near_thr(p, fabsf(dp), tolk);
      if (fabsf(dp) <= tolk) {
        int ok = 1;
        for (int i = 0; i < n_kt && ok; ++i) {
          float dk = kx - kt[i];
          nr |= near_thr(p, fabsf(dk), tolk);
          ok = fabsf(dk) <= tolk;
        }
        for (int i = 0; i < 2 && ok; ++i) {
          nr |= near_thr(p, zq[i], zt[i]);
          ok = zq[i] <= zt[i];
        }
        acc = ok;
      }
    }
  }
  if (vals) {
    vals[0] = kp; vals[1] = gdot; vals[2] = gcrs; vals[3] = glim; vals[4] = kx; vals[5] = zq[0];
    vals[6] = zq[1]; vals[7] = score;
  }
  if (near) *near = nr;
  return acc;
}

/* ------------------------------------------------------------------------------------------- */
/* growable arrays */
typedef struct { int* v; int n, cap; } ivec;
typedef struct { float* v; int n, cap; } fvec;
static void ipush(ivec* a, int x) {
  if (a->n == a->cap) {
    a->cap = a->cap ? 2 * a->cap : 1024;
    a->v = (int*)realloc(a->v, sizeof(int) * (size_t)a->cap);
  }
  a->v[a->n++] = x;
}
static void fpush(fvec* a, float x) {
  if (a->n == a->cap) {
    a->cap = a->cap ? 2 * a->cap : 1024;
    a->v = (float*)realloc(a->v, sizeof(float) * (size_t)a->cap);
  }
  a->v[a->n++] = x;
}

struct orc_event {
  int n[ORC_N_KINDS];
  ivec i32[ORC_N_KINDS];
  fvec f32[ORC_N_KINDS];
  long long near[ORC_N_STAGES];
  long long n_tests[ORC_N_STAGES];
};

static const int KIND_W[ORC_N_KINDS] = {3, 2, 5, 7, 2, 2, 16, 6};
static const int KIND_FW[ORC_N_KINDS] = {6, 1, 1, 1, 1, 1, 0, 1};

int orc_count(const orc_event* ev, int kind) { return ev->n[kind]; }
void orc_copy_i32(const orc_event* ev, int kind, int* dst) {
  memcpy(dst, ev->i32[kind].v, sizeof(int) * (size_t)ev->n[kind] * (size_t)KIND_W[kind]);
}
void orc_copy_f32(const orc_event* ev, int kind, float* dst) {
  memcpy(dst, ev->f32[kind].v, sizeof(float) * (size_t)ev->n[kind] * (size_t)KIND_FW[kind]);
}
void orc_counters(const orc_event* ev, long long* near, long long* n_tests) {
  for (int s = 0; s < ORC_N_STAGES; ++s) {
    near[s] = ev->near[s];
    n_tests[s] = ev->n_tests[s];
  }
}
void orc_free_event(orc_event* ev) {
  if (!ev) return;
  for (int k = 0; k < ORC_N_KINDS; ++k) {
    free(ev->i32[k].v);
    free(ev->f32[k].v);
  }
  free(ev);
}

/* accessors into the flat records */
#define MD_I(ev, i) ((ev)->i32[ORC_K_MD].v + 3 * (i))  /* h_lo, h_hi, module */
#define MD_F(ev, i) ((ev)->f32[ORC_K_MD].v + 6 * (i))  /* x y z r ux uy */
#define LS_I(ev, i) ((ev)->i32[ORC_K_LS].v + 2 * (i))
#define T3_I(ev, i) ((ev)->i32[ORC_K_T3].v + 5 * (i))
#define T5_I(ev, i) ((ev)->i32[ORC_K_T5].v + 7 * (i))
#define PT3_I(ev, i) ((ev)->i32[ORC_K_PT3].v + 2 * (i))
#define PT5_I(ev, i) ((ev)->i32[ORC_K_PT5].v + 2 * (i))
#define T4_I(ev, i) ((ev)->i32[ORC_K_T4].v + 6 * (i))

/* CUTS.md section 8: number of MDs common to two MD lists */
static int share(const int* a, int na, const int* b, int nb) {
  int s = 0;
  for (int i = 0; i < na; ++i)
    for (int j = 0; j < nb; ++j)
      if (a[i] == b[j]) ++s;
  return s;
}

/* CUTS.md section 8: key = (pls,) + (h_lo, h_hi) of each MD in order; lexicographic compare */
static int key_less(const int* md_hits, int plsY, const int* mdY, int plsX, const int* mdX, int nmd) {
  if (plsY != plsX) return plsY < plsX;
  for (int i = 0; i < nmd; ++i) {
    const int* hy = md_hits + 2 * mdY[i];
    const int* hx = md_hits + 2 * mdX[i];
    if (hy[0] != hx[0]) return hy[0] < hx[0];
    if (hy[1] != hx[1]) return hy[1] < hx[1];
  }
  return 0;
}
static int better(const int* md_hits, float sY, int plsY, const int* mdY, float sX, int plsX,
                  const int* mdX, int nmd) {
  if (sY < sX) return 1;
  if (sY == sX) return key_less(md_hits, plsY, mdY, plsX, mdX, nmd);
  return 0;
}

/* CUTS.md section 8, rules 1-4, on plain arrays:
 * md_hits [n_md][2]; t3_md [n_t3][3]; t5_md [n_t5][5] + t5_score; pt3 [n_pt3][2] = (pls, t3) +
 * pt3_score; pt5 [n_pt5][2] = (pls, t5) + pt5_score.  Outputs: keep5[n_pt5], keep3[n_pt3],
 * keepT[n_t5] (1 = survivor), linked[n_pls] (1 = seed of a surviving pT5/pT3). */
void orc_dedup(const int* md_hits, const int* t3_md, int n_t3, const int* t5_md, int n_t5,
               const float* t5_score, const int* pt3, int n_pt3, const float* pt3_score,
               const int* pt5, int n_pt5, const float* pt5_score, int n_pls, char* keep5,
               char* keep3, char* keepT, char* linked) {
  (void)n_t3;
  /* rule 1: pT5 */
  for (int X = 0; X < n_pt5; ++X) {
    int pX = pt5[2 * X];
    const int* mX = t5_md + 5 * pt5[2 * X + 1];
    keep5[X] = 1;
    for (int Y = 0; Y < n_pt5; ++Y) {
      if (Y == X) continue;
      int pY = pt5[2 * Y];
      const int* mY = t5_md + 5 * pt5[2 * Y + 1];
      if ((pY == pX || share(mY, 5, mX, 5) >= 3) &&
          better(md_hits, pt5_score[Y], pY, mY, pt5_score[X], pX, mX, 5))
        keep5[X] = 0;
    }
  }
  /* rule 2: pT3 */
  for (int X = 0; X < n_pt3; ++X) {
    int pX = pt3[2 * X];
    const int* mX = t3_md + 3 * pt3[2 * X + 1];
    keep3[X] = 1;
    for (int Y = 0; Y < n_pt3; ++Y) {
      if (Y == X) continue;
      int pY = pt3[2 * Y];
      const int* mY = t3_md + 3 * pt3[2 * Y + 1];
      if ((pY == pX || share(mY, 3, mX, 3) >= 2) &&
          better(md_hits, pt3_score[Y], pY, mY, pt3_score[X], pX, mX, 3))
        keep3[X] = 0;
    }
    for (int Z = 0; Z < n_pt5; ++Z) {
      if (!keep5[Z]) continue;
      const int* mZ = t5_md + 5 * pt5[2 * Z + 1];
      if (pt5[2 * Z] == pX || share(mX, 3, mZ, 5) >= 2) keep3[X] = 0;
    }
  }
  /* rule 3: T5 */
  for (int X = 0; X < n_t5; ++X) {
    const int* mX = t5_md + 5 * X;
    keepT[X] = 1;
    for (int Y = 0; Y < n_t5; ++Y) {
      if (Y == X) continue;
      const int* mY = t5_md + 5 * Y;
      if (share(mY, 5, mX, 5) >= 3 && better(md_hits, t5_score[Y], -1, mY, t5_score[X], -1, mX, 5))
        keepT[X] = 0;
    }
    for (int Z = 0; Z < n_pt5; ++Z) {
      if (!keep5[Z]) continue;
      if (share(mX, 5, t5_md + 5 * pt5[2 * Z + 1], 5) >= 2) keepT[X] = 0;
    }
    for (int Z = 0; Z < n_pt3; ++Z) {
      if (!keep3[Z]) continue;
      if (share(mX, 5, t3_md + 3 * pt3[2 * Z + 1], 3) >= 2) keepT[X] = 0;
    }
  }
  /* rule 4: linked seeds */
  for (int i = 0; i < n_pls; ++i) linked[i] = 0;
  for (int X = 0; X < n_pt5; ++X)
    if (keep5[X]) linked[pt5[2 * X]] = 1;
  for (int X = 0; X < n_pt3; ++X)
    if (keep3[X]) linked[pt3[2 * X]] = 1;
}

/* CUTS.md section 10, rule 5: T4 against better T4s (unfiltered set) and against the survivors of rules 1-3 */
void orc_dedup_t4(const int* md_hits, const int* t3_md, const int* t5_md, int n_t5, const int* pt3, int n_pt3,
                  const int* pt5, int n_pt5, const char* keep5, const char* keep3, const char* keepT,
                  const int* t4_md, int n_t4, const float* t4_score, char* keep4) {
  for (int X = 0; X < n_t4; ++X) {
    const int* mX = t4_md + 4 * X;
    keep4[X] = 1;
    for (int Y = 0; Y < n_t4; ++Y) {
      if (Y == X) continue;
      const int* mY = t4_md + 4 * Y;
      if (share(mY, 4, mX, 4) >= 3 && better(md_hits, t4_score[Y], -1, mY, t4_score[X], -1, mX, 4)) keep4[X] = 0;
    }
    for (int Z = 0; Z < n_pt5; ++Z)
      if (keep5[Z] && share(mX, 4, t5_md + 5 * pt5[2 * Z + 1], 5) >= 2) keep4[X] = 0;
    for (int Z = 0; Z < n_pt3; ++Z)
      if (keep3[Z] && share(mX, 4, t3_md + 3 * pt3[2 * Z + 1], 3) >= 2) keep4[X] = 0;
    for (int Z = 0; Z < n_t5; ++Z)
      if (keepT[Z] && share(mX, 4, t5_md + 5 * Z, 5) >= 2) keep4[X] = 0;
  }
}

static void push_tc(orc_event* ev, int type, int pls, int t5, int t3, const int* md, int nmd) {
  ivec* a = &ev->i32[ORC_K_TC];
  ipush(a, type);
  ipush(a, pls);
  ipush(a, t5);
  ipush(a, t3);
  for (int i = 0; i < 6; ++i) {
    if (i < nmd) {
      ipush(a, MD_I(ev, md[i])[0]);
      ipush(a, MD_I(ev, md[i])[1]);
    } else {
      ipush(a, -1);
      ipush(a, -1);
    }
  }
  ev->n[ORC_K_TC]++;
}

orc_event* orc_run_event(const orc_params* p, int n_modules, const int* subdet, const int* conn_off,
                         const int* conn_tgt, int n_hits, const float* x, const float* y,
                         const float* z, const int* sensor, int n_pls, const float* pls_pt,
                         const int* pls_q, const float* x0, const float* y0, const float* z0,
                         const float* x1, const float* y1, const float* z1) {
  /* input checks */
  for (int i = 0; i < n_hits; ++i)
    if (sensor[i] < 0 || sensor[i] >= 2 * n_modules) return 0;
  if (conn_off[0] != 0) return 0;
  for (int m = 0; m < n_modules; ++m) {
    if (conn_off[m + 1] < conn_off[m]) return 0;
    for (int k = conn_off[m]; k < conn_off[m + 1]; ++k)
      if (conn_tgt[k] < 0 || conn_tgt[k] >= n_modules) return 0;
  }

  orc_event* ev = (orc_event*)calloc(1, sizeof(orc_event));
  const int mask = p->stage_mask;

  /* hits of each sensor, in input order (plain bucket lists) */
  int* s_first = (int*)calloc((size_t)(2 * n_modules + 1), sizeof(int));
  int* s_list = (int*)malloc(sizeof(int) * (size_t)(n_hits > 0 ? n_hits : 1));
  for (int i = 0; i < n_hits; ++i) s_first[sensor[i] + 1]++;
  for (int s = 0; s < 2 * n_modules; ++s) s_first[s + 1] += s_first[s];
  {
    int* cur = (int*)malloc(sizeof(int) * (size_t)(2 * n_modules + 1));
    memcpy(cur, s_first, sizeof(int) * (size_t)(2 * n_modules + 1));
    for (int i = 0; i < n_hits; ++i) s_list[cur[sensor[i]]++] = i;
    free(cur);
  }

  /* ---- stage 0: Mini-Doublets (CUTS.md section 3) ---- */
  int* md_first = (int*)calloc((size_t)(n_modules + 1), sizeof(int));
  if (mask & 1) {
    for (int m = 0; m < n_modules; ++m) {
      md_first[m] = ev->n[ORC_K_MD];
      int endcap = subdet[m] != 0;
      for (int ia = s_first[2 * m]; ia < s_first[2 * m + 1]; ++ia) {
        for (int ib = s_first[2 * m + 1]; ib < s_first[2 * m + 2]; ++ib) {
          int a = s_list[ia], b = s_list[ib];
          float vals[8];
          int nr;
          ev->n_tests[ORC_ST_MD]++;
          int acc = orc_md_test(p, endcap, x[a], y[a], z[a], x[b], y[b], z[b], vals, &nr);
          ev->near[ORC_ST_MD] += nr;
          if (!acc) continue;
          ipush(&ev->i32[ORC_K_MD], a);
          ipush(&ev->i32[ORC_K_MD], b);
          ipush(&ev->i32[ORC_K_MD], m);
          fvec* f = &ev->f32[ORC_K_MD];
          fpush(f, x[a]);
          fpush(f, y[a]);
          fpush(f, z[a]);
          fpush(f, sqrtf(x[a] * x[a] + y[a] * y[a]));
          fpush(f, endcap ? 0.0f : vals[6]);
          fpush(f, endcap ? 0.0f : vals[7]);
          ev->n[ORC_K_MD]++;
        }
      }
    }
  }
  md_first[n_modules] = ev->n[ORC_K_MD];
  const int n_md = ev->n[ORC_K_MD];

  /* ---- stage 1: Line Segments (CUTS.md section 4) ---- */
  int* ls_first = (int*)calloc((size_t)(n_md + 1), sizeof(int)); /* LSs whose inner MD is A */
  if (mask & 2) {
    for (int A = 0; A < n_md; ++A) {
      ls_first[A] = ev->n[ORC_K_LS];
      int m = MD_I(ev, A)[2];
      for (int k = conn_off[m]; k < conn_off[m + 1]; ++k) {
        int m2 = conn_tgt[k];
        for (int B = md_first[m2]; B < md_first[m2 + 1]; ++B) {
          float vals[8];
          int nr;
          ev->n_tests[ORC_ST_LS]++;
          int acc = orc_ls_test(p, MD_F(ev, A), subdet[m] != 0, MD_F(ev, B), subdet[m2] != 0, vals, &nr);
          ev->near[ORC_ST_LS] += nr;
          if (!acc) continue;
          ipush(&ev->i32[ORC_K_LS], A);
          ipush(&ev->i32[ORC_K_LS], B);
          fpush(&ev->f32[ORC_K_LS], vals[0]);
          ev->n[ORC_K_LS]++;
        }
      }
    }
  }
  ls_first[n_md] = ev->n[ORC_K_LS];
  const int n_ls = ev->n[ORC_K_LS];

  /* ---- stage 2: T3 (CUTS.md section 5) ---- */
  int* t3_first = (int*)calloc((size_t)(n_md + 1), sizeof(int)); /* T3s whose first MD is A */
  if (mask & 4) {
    int ls = 0;
    for (int A = 0; A < n_md; ++A) {
      t3_first[A] = ev->n[ORC_K_T3];
      for (ls = ls_first[A]; ls < ls_first[A + 1]; ++ls) {
        int B = LS_I(ev, ls)[1];
        for (int ls2 = ls_first[B]; ls2 < ls_first[B + 1]; ++ls2) {
          int C = LS_I(ev, ls2)[1];
          float vals[4];
          int nr;
          ev->n_tests[ORC_ST_T3]++;
          int acc = orc_t3_test(p, MD_F(ev, A), subdet[MD_I(ev, A)[2]] != 0, MD_F(ev, B),
                                subdet[MD_I(ev, B)[2]] != 0, MD_F(ev, C),
                                subdet[MD_I(ev, C)[2]] != 0, vals, &nr);
          ev->near[ORC_ST_T3] += nr;
          if (!acc) continue;
          ivec* a = &ev->i32[ORC_K_T3];
          ipush(a, ls);
          ipush(a, ls2);
          ipush(a, A);
          ipush(a, B);
          ipush(a, C);
          fpush(&ev->f32[ORC_K_T3], vals[0]);
          ev->n[ORC_K_T3]++;
        }
      }
    }
  }
  t3_first[n_md] = ev->n[ORC_K_T3];
  const int n_t3 = ev->n[ORC_K_T3];

  /* ---- stage 3: T5 (CUTS.md section 6) ---- */
  if (mask & 8) {
    for (int t1 = 0; t1 < n_t3; ++t1) {
      const int* a1 = T3_I(ev, t1);
      int C = a1[4];
      for (int t2 = t3_first[C]; t2 < t3_first[C + 1]; ++t2) {
        const int* a2 = T3_I(ev, t2);
        float vals[4];
        int nr;
        ev->n_tests[ORC_ST_T5]++;
        int acc = orc_t5_test(p, ev->f32[ORC_K_T3].v[t1], ev->f32[ORC_K_T3].v[t2], MD_F(ev, a1[3]),
                              MD_F(ev, C), MD_F(ev, a2[3]), vals, &nr);
        ev->near[ORC_ST_T5] += nr;
        if (!acc) continue;
        ivec* a = &ev->i32[ORC_K_T5];
        ipush(a, t1);
        ipush(a, t2);
        ipush(a, a1[2]);
        ipush(a, a1[3]);
        ipush(a, a1[4]);
        ipush(a, a2[3]);
        ipush(a, a2[4]);
        fpush(&ev->f32[ORC_K_T5], vals[2]);
        ev->n[ORC_K_T5]++;
      }
    }
  }
  const int n_t5 = ev->n[ORC_K_T5];

  /* ---- stage 6 (extension): T4 (CUTS.md section 10) ---- */
  if (mask & 64) {
    /* T3s whose FIRST LS is l: T3s are pushed in order of their first LS */
    int* t3_of_ls = (int*)calloc((size_t)(n_ls + 2), sizeof(int));
    for (int t = 0; t < n_t3; ++t) t3_of_ls[T3_I(ev, t)[0] + 1]++;
    for (int l = 0; l < n_ls; ++l) t3_of_ls[l + 1] += t3_of_ls[l];
    for (int t1 = 0; t1 < n_t3; ++t1) {
      const int* a1 = T3_I(ev, t1);
      int l2 = a1[1];
      for (int t2 = t3_of_ls[l2]; t2 < t3_of_ls[l2 + 1]; ++t2) {
        const int* a2 = T3_I(ev, t2);
        float vals[4];
        int nr;
        ev->n_tests[ORC_ST_T4]++;
        int acc = orc_t4_test(p, ev->f32[ORC_K_T3].v[t1], ev->f32[ORC_K_T3].v[t2], vals, &nr);
        ev->near[ORC_ST_T4] += nr;
        if (!acc) continue;
        ivec* a = &ev->i32[ORC_K_T4];
        ipush(a, t1);
        ipush(a, t2);
        ipush(a, a1[2]);
        ipush(a, a1[3]);
        ipush(a, a1[4]);
        ipush(a, a2[4]);
        fpush(&ev->f32[ORC_K_T4], vals[2]);
        ev->n[ORC_K_T4]++;
      }
    }
    free(t3_of_ls);
  }
  const int n_t4 = ev->n[ORC_K_T4];

  /* ---- stages 4, 5: pT3 / pT5 (CUTS.md section 7) ---- */
  if ((mask & 16) && n_pls > 0) {
    for (int ip = 0; ip < n_pls; ++ip) {
      float pls[8] = {pls_pt[ip], (float)pls_q[ip], x0[ip], y0[ip], z0[ip], x1[ip], y1[ip], z1[ip]};
      for (int t = 0; t < n_t3; ++t) {
        const int* a = T3_I(ev, t);
        int A = a[2], L = a[4];
        float kt[1] = {ev->f32[ORC_K_T3].v[t]};
        float vals[8];
        int nr;
        ev->n_tests[ORC_ST_PT3]++;
        int acc = orc_pt_test(p, pls, MD_F(ev, A), subdet[MD_I(ev, A)[2]] != 0, MD_F(ev, L),
                              subdet[MD_I(ev, L)[2]] != 0, kt, 1, 0.0f, vals, &nr);
        ev->near[ORC_ST_PT3] += nr;
        if (!acc) continue;
        ipush(&ev->i32[ORC_K_PT3], ip);
        ipush(&ev->i32[ORC_K_PT3], t);
        fpush(&ev->f32[ORC_K_PT3], vals[7]);
        ev->n[ORC_K_PT3]++;
      }
      for (int t = 0; t < n_t5; ++t) {
        const int* a = T5_I(ev, t);
        int A = a[2], L = a[6];
        float kt[2] = {ev->f32[ORC_K_T3].v[a[0]], ev->f32[ORC_K_T3].v[a[1]]};
        float vals[8];
        int nr;
        ev->n_tests[ORC_ST_PT5]++;
        int acc = orc_pt_test(p, pls, MD_F(ev, A), subdet[MD_I(ev, A)[2]] != 0, MD_F(ev, L),
                              subdet[MD_I(ev, L)[2]] != 0, kt, 2, ev->f32[ORC_K_T5].v[t], vals, &nr);
        ev->near[ORC_ST_PT5] += nr;
        if (!acc) continue;
        ipush(&ev->i32[ORC_K_PT5], ip);
        ipush(&ev->i32[ORC_K_PT5], t);
        fpush(&ev->f32[ORC_K_PT5], vals[7]);
        ev->n[ORC_K_PT5]++;
      }
    }
  }
  const int n_pt3 = ev->n[ORC_K_PT3], n_pt5 = ev->n[ORC_K_PT5];

  /* ---- duplicate removal + track-candidate selection (CUTS.md section 8) ---- */
  if (mask & 32) {
    char* keep5 = (char*)malloc((size_t)(n_pt5 + 1));
    char* keep3 = (char*)malloc((size_t)(n_pt3 + 1));
    char* keepT = (char*)malloc((size_t)(n_t5 + 1));
    char* linked = (char*)calloc((size_t)(n_pls + 1), 1);
    /* repack the records into the plain arrays orc_dedup takes */
    int* md_hits = (int*)malloc(sizeof(int) * (size_t)(2 * n_md + 2));
    int* t3_md = (int*)malloc(sizeof(int) * (size_t)(3 * n_t3 + 3));
    int* t5_md = (int*)malloc(sizeof(int) * (size_t)(5 * n_t5 + 5));
    for (int i = 0; i < n_md; ++i) {
      md_hits[2 * i] = MD_I(ev, i)[0];
      md_hits[2 * i + 1] = MD_I(ev, i)[1];
    }
    for (int i = 0; i < n_t3; ++i)
      for (int k = 0; k < 3; ++k) t3_md[3 * i + k] = T3_I(ev, i)[2 + k];
    for (int i = 0; i < n_t5; ++i)
      for (int k = 0; k < 5; ++k) t5_md[5 * i + k] = T5_I(ev, i)[2 + k];
    orc_dedup(md_hits, t3_md, n_t3, t5_md, n_t5, ev->f32[ORC_K_T5].v, ev->i32[ORC_K_PT3].v, n_pt3,
              ev->f32[ORC_K_PT3].v, ev->i32[ORC_K_PT5].v, n_pt5, ev->f32[ORC_K_PT5].v, n_pls, keep5,
              keep3, keepT, linked);
    /* output in class order pT5, pT3, T5, pLS */
    for (int X = 0; X < n_pt5; ++X)
      if (keep5[X])
        push_tc(ev, 0, PT5_I(ev, X)[0], PT5_I(ev, X)[1], -1, T5_I(ev, PT5_I(ev, X)[1]) + 2, 5);
    for (int X = 0; X < n_pt3; ++X)
      if (keep3[X])
        push_tc(ev, 1, PT3_I(ev, X)[0], -1, PT3_I(ev, X)[1], T3_I(ev, PT3_I(ev, X)[1]) + 2, 3);
    for (int X = 0; X < n_t5; ++X)
      if (keepT[X]) push_tc(ev, 2, -1, X, -1, T5_I(ev, X) + 2, 5);
    for (int ip = 0; ip < n_pls; ++ip)
      if (!linked[ip]) push_tc(ev, 3, ip, -1, -1, 0, 0);
    if (n_t4 > 0) { /* CUTS.md section 10, rule 5 and TC class 4 */
      char* keep4 = (char*)malloc((size_t)n_t4);
      int* t4_md = (int*)malloc(sizeof(int) * (size_t)(4 * n_t4));
      for (int i = 0; i < n_t4; ++i)
        for (int k = 0; k < 4; ++k) t4_md[4 * i + k] = T4_I(ev, i)[2 + k];
      orc_dedup_t4(md_hits, t3_md, t5_md, n_t5, ev->i32[ORC_K_PT3].v, n_pt3, ev->i32[ORC_K_PT5].v, n_pt5, keep5,
                   keep3, keepT, t4_md, n_t4, ev->f32[ORC_K_T4].v, keep4);
      for (int X = 0; X < n_t4; ++X)
        if (keep4[X]) push_tc(ev, 4, -1, -1, T4_I(ev, X)[0], t4_md + 4 * X, 4);
      free(keep4);
      free(t4_md);
    }
    free(keep5);
    free(keep3);
    free(keepT);
    free(linked);
    free(md_hits);
    free(t3_md);
    free(t5_md);
  }

  free(s_first);
  free(s_list);
  free(md_first);
  free(ls_first);
  free(t3_first);
  (void)n_ls;
  return ev;
}
