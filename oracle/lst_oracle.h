/* lst_oracle.h -- CPU oracle of the LST object-building chain.  TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, single-threaded restatement of CUTS.md (the documented stand-in for the selections
 * that PAPER.md:29 defers to its Refs. [4], [5]) and of the object hierarchy of PAPER.md:23, 29-34.
 * It shares no code with the CUDA path (paper_2407_18231_b200/csrc); only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Precision: binary32, fixed operation order, no FMA (north_star fixes the precision; build with
 * -O2 -ffp-contract=off -fno-fast-math).
 *
 * Pins (tests/test_oracle_pins.py, test_oracle_values.py, test_oracle_dedup.py): a hand-built candidate
 * with the expected threshold for every term of every cut (value and accept / reject decision), the
 * near-threshold rule at t (1 +- 0.5e-5) / t (1 +- 2e-5) and the order of the cuts for every stage,
 * closed-form helix values, textbook circumradius for kappa3, asin series for g, hand-computed
 * straight/curved single tracks (tests/golden/), brute-force all-pairs enumeration, structural
 * invariants, monotonicity in the cut windows, every clause of the duplicate removal.
 * tests/test_oracle_mutants.py applies 51 one-line mistakes to a copy of lst_oracle.c: each fails a
 * named pin.  tests/test_oracle_sanitizers.py runs the pins under ASan + UBSan.
 * "parity unpinned" against the paper's own numbers: PAPER.md prints no object counts or
 * intermediate values.
 */
#ifndef LST_ORACLE_H
#define LST_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct orc_params {
  float b_field, pt_min, z0_max;
  float md_b_phi_tol, md_z_tol, md_e_slope, md_e_tol;
  float ls_kappa_max, ls_z_tol, ls_dir_tol;
  float t3_kappa_max, t3_z_tol0, t3_z_tol1;
  float t5_tol0, t5_tol1;
  float pt_gate_tol, pt_k_tol0, pt_k_tol1, pt_z_tol;
  float near_rel;
  int stage_mask;
  /* extensions (CUTS.md sections 10, 11), off unless stage_mask bits 6 / 7 are set */
  float t4_tol0, t4_tol1;
  float t5_mlp_scale, t5_mlp_thr;
  float t5_mlp[65]; /* W1[8][6], b1[8], W2[8], b2 */
} orc_params;

enum { ORC_ST_MD = 0, ORC_ST_LS, ORC_ST_T3, ORC_ST_T5, ORC_ST_PT3, ORC_ST_PT5, ORC_ST_T4, ORC_N_STAGES };

/* CUTS.md section 1 defaults. */
void orc_default_params(orc_params* p);
/* CUTS.md section 1 derived constants: out[0]=KR, out[1]=R_MIN, out[2]=INV_2RMIN. */
void orc_derived(const orc_params* p, float out[3]);

/* ---- single-candidate functions (what the pins and the brute-force tests call) ------------- */
/* CUTS.md section 1: g(u) ~ asin(sqrt(u))/sqrt(u). */
float orc_g(float u);
/* CUTS.md section 5: signed circumcircle curvature; len[0..2] = |PQ|, |QS|, |PS| (may be NULL). */
float orc_kappa3(float xp, float yp, float xq, float yq, float xs, float ys, float* len);

/* Each returns 1 = accept, 0 = reject; *near = near-threshold flag (CUTS.md section 0);
 * vals (may be NULL) receives the named quantities of the spec. */
/* CUTS.md section 3.  vals[8] = dd, dot, crs, lim, zv, zl, ux, uy (barrel)
 *                      vals[8] = crs, lim, rv, rl, 0, 0, 0, 0      (endcap) */
int orc_md_test(const orc_params* p, int endcap, float xa, float ya, float za, float xb, float yb,
                float zb, float* vals, int* near);
/* CUTS.md section 4.  md = x, y, z, r, ux, uy.  vals[8] = kappa, kv, rho, zv, zl, half, dA, dB. */
int orc_ls_test(const orc_params* p, const float* mdA, int endcapA, const float* mdB, int endcapB,
                float* vals, int* near);
/* CUTS.md section 5.  md = x, y, z, r.  vals[4] = k3, ratio, zv, tol. */
int orc_t3_test(const orc_params* p, const float* mdA, int eA, const float* mdB, int eB,
                const float* mdC, int eC, float* vals, int* near);
/* CUTS.md section 6 (section 11 when stage_mask bit 7 is set).  vals[4] = kb, tol, score, s (MLP output, else 0). */
int orc_t5_test(const orc_params* p, float ki, float ko, const float* mdB, const float* mdC,
                const float* mdD, float* vals, int* near);
/* CUTS.md section 10.  vals[4] = d, tol, score, 0. */
int orc_t4_test(const orc_params* p, float k1, float k2, float* vals, int* near);
/* CUTS.md section 7.  pls = pt, q, x0, y0, z0, x1, y1, z1.  kt[0..n_kt) = the stored curvatures
 * compared with kx (1 for a T3, 2 for a T5); base_score added to the score (0 / T5 score).
 * vals[8] = kp, gdot, gcrs, glim, kx, zqA, zqL, score. */
int orc_pt_test(const orc_params* p, const float* pls, const float* mdA, int eA, const float* mdL,
                int eL, const float* kt, int n_kt, float base_score, float* vals, int* near);

/* CUTS.md section 8 rules 1-4 on plain arrays (md_hits [n_md][2], t3_md [n_t3][3], t5_md [n_t5][5],
 * pt3/pt5 [n][2] = (pls, t3|t5)).  Outputs keep5[n_pt5], keep3[n_pt3], keepT[n_t5], linked[n_pls]. */
void orc_dedup(const int* md_hits, const int* t3_md, int n_t3, const int* t5_md, int n_t5,
               const float* t5_score, const int* pt3, int n_pt3, const float* pt3_score,
               const int* pt5, int n_pt5, const float* pt5_score, int n_pls, char* keep5,
               char* keep3, char* keepT, char* linked);
/* CUTS.md section 10 rule 5, after orc_dedup: t4_md [n_t4][4]; output keep4[n_t4]. */
void orc_dedup_t4(const int* md_hits, const int* t3_md, const int* t5_md, int n_t5, const int* pt3, int n_pt3,
                  const int* pt5, int n_pt5, const char* keep5, const char* keep3, const char* keepT,
                  const int* t4_md, int n_t4, const float* t4_score, char* keep4);

/* ---- whole event ------------------------------------------------------------------------------ */
typedef struct orc_event orc_event;

/* Runs the chain selected by p->stage_mask on one event.  Returns NULL on invalid input
 * (sensor id out of range, bad CSR).  pLS arrays may be NULL when n_pls == 0. */
orc_event* orc_run_event(const orc_params* p, int n_modules, const int* subdet, const int* conn_off,
                         const int* conn_tgt, int n_hits, const float* x, const float* y,
                         const float* z, const int* sensor, int n_pls, const float* pls_pt,
                         const int* pls_q, const float* x0, const float* y0, const float* z0,
                         const float* x1, const float* y1, const float* z1);
void orc_free_event(orc_event* ev);

enum {
  ORC_K_MD = 0, /* i32 [n][3]  h_lo, h_hi, module */
  ORC_K_LS,     /* i32 [n][2]  md_in, md_out */
  ORC_K_T3,     /* i32 [n][5]  ls0, ls1, mdA, mdB, mdC */
  ORC_K_T5,     /* i32 [n][7]  t3_0, t3_1, md x5 */
  ORC_K_PT3,    /* i32 [n][2]  pls, t3 */
  ORC_K_PT5,    /* i32 [n][2]  pls, t5 */
  ORC_K_TC,     /* i32 [n][16] type, pls, t5, t3, hit_idx[12] */
  ORC_K_T4,     /* i32 [n][6]  t3_0, t3_1, md x4 (CUTS.md section 10) */
  ORC_N_KINDS
};
int orc_count(const orc_event* ev, int kind);
void orc_copy_i32(const orc_event* ev, int kind, int* dst);
/* f32 payload per object: MD [n][6] x,y,z,r,ux,uy; LS [n] kappa; T3 [n] k3; T5/PT3/PT5/T4 [n] score. */
void orc_copy_f32(const orc_event* ev, int kind, float* dst);
/* per-stage counters: near[ORC_N_STAGES], n_tests[ORC_N_STAGES] (candidates evaluated). */
void orc_counters(const orc_event* ev, long long* near, long long* n_tests);

#ifdef __cplusplus
}
#endif
#endif
