// lst_types.cuh -- device-side data layout of one context (structure of arrays in HBM).
//
// Everything of a batch lives in ONE index space: events are concatenated, a "global module" is
// gm = event * n_mod + module and a "global sensor" gs = 2 * gm + {0,1}.  Because every stage
// stores its objects in owner order (lst_scan.cuh), hits, MDs, LSs, T3s, T5s, pT3s and pT5s of an
// event are contiguous, so per-event ranges follow from the *_begin arrays.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lst_cuts.cuh"

namespace lst {

struct PtEvent;  // lst_pt.cuh

enum Kind { K_MD = 0, K_LS, K_T3, K_T5, K_PT3, K_PT5, K_TC, K_T4, K_NKINDS };
enum Tkt { T_SENS = 0, T_MD, T_LS, T_T3, T_T5, T_PT, T_PP3, T_PP5, T_T4, T_LSE, T_N };

enum ErrBit { E_BAD_SENSOR = 1, E_CAP_MD = 2, E_CAP_LS = 4, E_CAP_T3 = 8, E_CAP_T5 = 16,
              E_CAP_PT3 = 32, E_CAP_PT5 = 64, E_CAP_TC = 128, E_CAP_T4 = 256 };

constexpr int kStages = 7;    // MD, LS, T3, T5, pT3, pT5, T4 (CUTS.md section 2)
constexpr int kEvCnt = 2 * kStages;  // per-event counters: [0, 7) near-threshold candidates, [7, 14) candidates, per stage
constexpr int kTcClasses = 5;        // pT5, pT3, T5, pLS, T4 (CUTS.md section 10)
constexpr int kEvSmem = 64;   // events whose candidate counts a block accumulates in shared memory

// Small control block, zeroed (one memset, together with the tile status words) per batch.
struct Ctl {
  int ticket[T_N];
  int total[K_NKINDS];
  int error;
  int done_rule;                     // blocks of the last rule kernel that have finished (the last one scans tc_cnt)
  int scratch_cur[4];                // accepted objects in the scratch lists: [1] LS, [2] pT3, [3] pT5
  int queue_cur;                     // entries of the exact-evaluation queue of the seed linking
  int ls_tiles_done;                 // scan tiles of k_ls_place that are finished
  int pad[1];
};

// What changes from batch to batch: sizes and input pointers.  Lives in device memory (copied in front of
// every launch sequence), so the kernel arguments -- and with them the CUDA graph of a context -- never change.
struct Batch {
  int n_events, n_hits, n_pls;
  int sensor_u16;  // in_sensor holds unsigned short ids (include/lst.h: lst_hits.sensor_u16)
  const float *in_x, *in_y, *in_z;
  const int* in_sensor;
  const float *p_pt, *p_x0, *p_y0, *p_z0, *p_x1, *p_y1, *p_z1;
  const int* p_q;
};

struct Dev {
  const Batch* batch;  // device copy; load_batch() fills the batch fields below at the top of every kernel
  // ---- geometry (immutable, shared) ----
  int n_mod;
  const int* subdet;    // [n_mod]
  const int* conn_off;  // [n_mod + 1]
  const int* conn_tgt;
  // ---- batch ----
  int n_events, n_hits, n_pls, sensor_u16;
  const int* hit_ev_off;  // [n_events + 1] device copy of the event offsets
  const int* pls_ev_off;  // [n_events + 1]
  const float *in_x, *in_y, *in_z;  // input hits (device), caller order
  const int* in_sensor;
  const float *p_pt, *p_x0, *p_y0, *p_z0, *p_x1, *p_y1, *p_z1;  // pLS (device)
  const int* p_q;
  // ---- control ----
  Ctl* ctl;
  unsigned long long* ev_cnt;       // [n_events][kEvCnt]: near[6] then n_tests[6] of every event (zeroed per batch)
  unsigned long long* tstate[T_N];  // look-back status words per scanning kernel
  // ---- a0: hits binned by global sensor ----
  int* hit_rank;     // [n_hits] rank of input hit i among the hits of its (chunk, sensor) (k_ingest_count)
  int* chunk_cnt;    // [n_events][kIngestChunks][2 * n_mod] hits per (chunk of the event's hits, sensor)
  int* chunk_part;   // [n_events][kIngestChunks][kIngestScanParts] hits of a chunk per part of the sensor range
  int* sens_begin;   // [n_events * 2 * n_mod + 1] first sorted hit of every global sensor
  float4* hit;       // [2 * n_hits] sorted hits, 32 bytes each: (x, y, z, r), (event-local input index, global sensor, -, -)
  // ---- scratch lists of accepted objects in arrival order (LS, then pT3; pT5) ----
  void* ev_scratch;
  void* ev_scratch2;
  // ---- a1: MD (grouped by global module) ----
  int2* md_cnt;       // [n_hits] (MDs owned by a sorted hit: upper-sensor hits only, its global sensor)
  int* md_stash;      // [n_hits][4] sorted positions of the first accepted lower hits
  int* mod_md_begin;  // [n_events * n_mod + 1] first MD of a global module
  int2* md_hit;       // (h_lo, h_hi) event-local input indices
  int* md_info;       // 2 * gm + endcap
  float4* md_a;       // anchor = lower hit (x, y, z, r)
  float2* md_u;       // unit direction (barrel), 0 (endcap)
  // ---- a2: LS (owner = inner MD) ----
  int* md_ls_begin;  // [n_md + 1]
  int *ls_cnt, *ls_cur;  // [n_md] LSs of an inner MD, and the next free slot of its range (both zeroed per batch)
  int2* ls_md;       // (md_in, md_out) batch-global MD indices
  float* ls_kappa;
  // ---- a3: T3 (owner = first LS) ----
  int* ls_t3_begin;  // [n_ls + 1]
  int2* t3_ls;
  int4* t3_md;  // (A, B, C, endcap flags bit0 A, bit1 B, bit2 C)
  float* t3_k;
  float4* t3_l;  // last MD (x, y, z, r | endcap << 31): the operand of the seed linking's pre-filters
  float4* t3_q;  // (x, y of the last MD, k3, |first MD - last MD|^2 in the transverse plane): one load per candidate in k_pt_eval
  // ---- a4: T5 (owner = first T3) ----
  int* t3_t5_begin;  // [n_t3 + 1]
  int2* t5_t3;
  int* t5_md;  // [n_t5][5]
  float* t5_score;
  float4* t5_l;    // last MD, as t3_l
  float2* t5_kio;  // (ki, ko) = k3 of the two T3s
  // ---- extension: T4 (owner = first T3; CUTS.md section 10) ----
  int* t3_t4_begin;  // [n_t3 + 1]
  int2* t4_t3;
  int4* t4_md;
  float* t4_score;
  // ---- a5: pT3 / pT5 (owner = pLS) ----
  float4* seed_a;      // [n_pls] x1, y1, vx, vy           (CUTS.md section 7, computed once per seed)
  float4* seed_b;      // [n_pls] lv, kp, tolk, slope
  float* seed_z1;      // [n_pls]
  float4* seed_g;      // [n_pls] lv INV_2RMIN, lv PT_GATE_TOL, kp, tolk: the per-lane constants of k_pt_eval
  int* seed_perm;      // [n_pls] the seeds of every event in azimuth order (k_anchor_sort)
  PtEvent* pt_ev;      // [n_events + 1] anchor / seed ranges and first tile of every event
  int *anc_bin, *anc_rank;  // [n_md] bin (radial class * 64 + sector, -1 = no anchor) and arrival rank in the event's bin
  int* anc_bin_cnt;    // [n_events * 512] anchors per (event, bin) (zeroed per batch)
  float4* anc_a;       // [n_md] anchor (x, y, z, r | endcap << 31), the anchors of event e from mod_md_begin[e * n_mod] on
  int4* anc_t;         // [n_md] (first T3, number of T3s, first T5, number of T5s) starting at the anchor
  float4* anc_c;       // [5 * (n_md / 32 + n_events + 1)] bounding circle (x, y, h) of every block of 32 sorted anchors, then of its 4 sub-blocks of 8
  int* anc_done;       // [n_events] blocks of k_anchor_sort that have placed their share of the event (zeroed per batch)
  int2* pt_queue;      // candidates for the exact cuts: (seed, T3 / T5 index | T5 flag << 31)
  int *pls_pt3_cnt, *pls_pt5_cnt;  // [n_pls + 1] accepted per seed (zeroed per batch)
  int *pls_pt3_cur, *pls_pt5_cur;  // [n_pls] next free slot of a seed's range (zeroed per batch)
  int* pls_event;      // [n_pls]
  int* pls_pt3_begin;  // [n_pls + 1]
  int* pls_pt5_begin;  // [n_pls + 1]
  int2* pt3;           // (pls, t3) batch-global
  float* pt3_score;
  int2* pt5;
  float* pt5_score;
  // ---- a6: duplicate removal + track candidates ----
  int* idx_head;   // [4 * n_md] objects containing MD m, as linked lists: kind 0 T5, 1 pT5, 2 pT3, 3 T4; 0 = end, else node + 1
  int* idx_next;   // [5 * cap T5 | 5 * cap pT5 | 3 * cap pT3 | 4 * cap T4] node = object * (5, 3 or 4) + position of the MD in it
  unsigned char *keep5, *keep3, *keepT, *keep4, *linked;
#ifdef LST_RULE3_SKIP_COVERED  // reproducer of profiles/r03_rule3_fault.md only
  unsigned char* t5_cov;  // [n_t5] a surviving pT5 is built on this T5 (set by k_rule1; zeroed per batch)
#endif
  int* tc_cnt;    // [n_events * 5 + 1] survivors per (event, class) (zeroed per batch)
  int* tc_begin;  // [n_events * 5 + 1]
  int* tc_cur;    // [n_events * 5] (zeroed per batch)
  int* tc;        // [n_tc][16]
  int* ev_first;  // [K_PT5 + 1][n_events + 1] first object of every event, per kind
  // ---- capacities ----
  int cap[K_NKINDS];
  int cap_queue;
  Cuts cuts;
};

// first statement of every kernel: the batch fields of the by-value argument come from device memory
__device__ __forceinline__ void load_batch(Dev& d) {
  const Batch* __restrict__ b = d.batch;
  d.n_events = b->n_events;  d.n_hits = b->n_hits;  d.n_pls = b->n_pls;  d.sensor_u16 = b->sensor_u16;
  d.in_x = b->in_x;  d.in_y = b->in_y;  d.in_z = b->in_z;  d.in_sensor = b->in_sensor;
  d.p_pt = b->p_pt;  d.p_q = b->p_q;
  d.p_x0 = b->p_x0;  d.p_y0 = b->p_y0;  d.p_z0 = b->p_z0;
  d.p_x1 = b->p_x1;  d.p_y1 = b->p_y1;  d.p_z1 = b->p_z1;
}

}  // namespace lst
