// lst_select.cuh -- step a6: duplicate removal and track-candidate selection (CUTS.md section 8,
// PAPER.md:31-34, 56), and the grouping of the accepted pT3 / pT5 by seed that precedes it.
// Set-defined rules; the candidates that can overlap an object are found through an inverted index
// "objects containing MD m": three linked lists per MD (T5, pT5, pT3), built in ONE pass with an atomic
// exchange per (object, MD) -- node = object * 5 (or 3) + position, so no allocation, no counting pass and
// no scan.  By the pigeonhole principle an object sharing >= 3 of X's 5 MDs contains X.md[0], [2] or [4];
// one sharing >= 2 of 5 contains one of X.md[0..3]; one sharing >= 2 of X's 3 MDs contains X.md[0] or [1].
#pragma once
#include "lst_ls.cuh"
#include "lst_pt.cuh"

namespace lst {

__device__ __forceinline__ int ev_of_md(const Dev& d, int md) { return (d.md_info[md] >> 1) / d.n_mod; }

// offsets of the three node arrays inside idx_next
__device__ __forceinline__ int node_base(const Dev& d, int kind) {
  return kind == 0 ? 0 : (kind == 1 ? 5 * d.cap[K_T5] : (kind == 2 ? 5 * d.cap[K_T5] + 5 * d.cap[K_PT5]
                                                                   : 5 * d.cap[K_T5] + 5 * d.cap[K_PT5] + 3 * d.cap[K_PT3]));
}
__device__ __forceinline__ void idx_link(const Dev& d, int n_md, int kind, int md, int node) {
  d.idx_next[node_base(d, kind) + node] = atomicExch(d.idx_head + kind * n_md + md, node + 1);
}

// After k_scan2 (per-seed counts -> begin offsets): every accepted (seed, T3) / (seed, T5) of the scratch
// lists takes the next free slot of its seed (order inside a seed's range is arrival order: free by the
// spec, reading S9) and is linked into the index of its MDs; the T5s are linked as well.
// Block 0 also writes the first object of every event per kind (what the read-back slices by).
__global__ void __launch_bounds__(kBlock) k_pt_place(Dev d) {
  load_batch(d);
  const int n3 = d.ctl->scratch_cur[2], n5 = d.ctl->scratch_cur[3];
  const int cap3 = d.cap[K_PT3], cap5 = d.cap[K_PT5];
  const bool fit3 = n3 <= cap3, fit5 = n5 <= cap5;
  const int n_t5 = d.ctl->total[K_T5], n_md = d.ctl->total[K_MD];
  const bool sel = (d.cuts.stage_mask & 32) != 0 && fit3 && fit5;
  const int n_t4 = sel ? d.ctl->total[K_T4] : 0;
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const PtAccepted* s3 = reinterpret_cast<const PtAccepted*>(d.ev_scratch);
  const PtAccepted* s5 = reinterpret_cast<const PtAccepted*>(d.ev_scratch2);
  if (i0 == 0) {
    if (!fit3) atomicOr(&d.ctl->error, E_CAP_PT3);
    if (!fit5) atomicOr(&d.ctl->error, E_CAP_PT5);
    d.ctl->total[K_PT3] = fit3 ? n3 : 0;
    d.ctl->total[K_PT5] = fit5 ? n5 : 0;
  }
  const int n_a = fit3 ? n3 : 0, n_b = fit5 ? n5 : 0;
  for (int i = i0; i < n_a + n_b + (sel ? n_t5 : 0) + n_t4; i += stride) {
    if (i < n_a) {
      const PtAccepted a = s3[i];
      const int pos = d.pls_pt3_begin[a.p] + atomicAdd(d.pls_pt3_cur + a.p, 1);
      d.pt3[pos] = make_int2(a.p, a.t);
      d.pt3_score[pos] = a.score;
      if (sel) {
        const int4 m = d.t3_md[a.t];
        idx_link(d, n_md, 2, m.x, 3 * pos);
        idx_link(d, n_md, 2, m.y, 3 * pos + 1);
        idx_link(d, n_md, 2, m.z, 3 * pos + 2);
      }
    } else if (i < n_a + n_b) {
      const PtAccepted a = s5[i - n_a];
      const int pos = d.pls_pt5_begin[a.p] + atomicAdd(d.pls_pt5_cur + a.p, 1);
      d.pt5[pos] = make_int2(a.p, a.t);
      d.pt5_score[pos] = a.score;
      if (sel) {
        const int* md = d.t5_md + 5 * (size_t)a.t;
#pragma unroll
        for (int k = 0; k < 5; ++k) idx_link(d, n_md, 1, md[k], 5 * pos + k);
      }
    } else if (i < n_a + n_b + n_t5) {
      const int t = i - n_a - n_b;
      const int* md = d.t5_md + 5 * (size_t)t;
#pragma unroll
      for (int k = 0; k < 5; ++k) idx_link(d, n_md, 0, md[k], 5 * t + k);
    } else {
      const int t = i - n_a - n_b - n_t5;
      const int4 m = d.t4_md[t];
      idx_link(d, n_md, 3, m.x, 4 * t);
      idx_link(d, n_md, 3, m.y, 4 * t + 1);
      idx_link(d, n_md, 3, m.z, 4 * t + 2);
      idx_link(d, n_md, 3, m.w, 4 * t + 3);
    }
  }
  if (blockIdx.x == 0) {
    const int E1 = d.n_events + 1;
    for (int ev = threadIdx.x; ev < E1; ev += blockDim.x) {
      const int p = d.pls_ev_off[ev];
      const int md = n_md > 0 ? d.mod_md_begin[ev * d.n_mod] : 0;
      const int ls = d.ctl->total[K_LS] > 0 ? d.md_ls_begin[md] : 0;
      const int t3 = d.ctl->total[K_T3] > 0 ? d.ls_t3_begin[ls] : 0;
      const int t5 = n_t5 > 0 ? d.t3_t5_begin[t3] : 0;
      d.ev_first[K_MD * E1 + ev] = md;
      d.ev_first[K_LS * E1 + ev] = ls;
      d.ev_first[K_T3 * E1 + ev] = t3;
      d.ev_first[K_T5 * E1 + ev] = t5;
      d.ev_first[K_PT3 * E1 + ev] = n_a > 0 ? d.pls_pt3_begin[p] : 0;
      d.ev_first[K_PT5 * E1 + ev] = n_b > 0 ? d.pls_pt5_begin[p] : 0;
      d.ev_first[K_T4 * E1 + ev] = d.ctl->total[K_T4] > 0 ? d.t3_t4_begin[t3] : 0;
    }
  }
}

__device__ __forceinline__ int share(const int* a, int na, const int* b, int nb) {
  int s = 0;
  for (int i = 0; i < na; ++i)
    for (int j = 0; j < nb; ++j) s += (a[i] == b[j]);
  return s;
}

// CUTS.md section 8: better(Y, X); key = (pls,) + hit pairs of the MDs in order
__device__ __forceinline__ bool better(const Dev& d, float sY, int pY, const int* mY, float sX, int pX,
                                       const int* mX, int nmd) {
  if (sY < sX) return true;
  if (!(sY == sX)) return false;
  if (pY != pX) return pY < pX;
  for (int i = 0; i < nmd; ++i) {
    const int2 hy = d.md_hit[mY[i]], hx = d.md_hit[mX[i]];
    if (hy.x != hx.x) return hy.x < hx.x;
    if (hy.y != hx.y) return hy.y < hx.y;
  }
  return false;
}

__device__ __forceinline__ void load_t3_md(const Dev& d, int t3, int* m) {
  const int4 v = d.t3_md[t3];
  m[0] = v.x; m[1] = v.y; m[2] = v.z;
}
__device__ __forceinline__ void load_t5_md(const Dev& d, int t5, int* m) {
  const int* p = d.t5_md + 5 * (size_t)t5;
#pragma unroll
  for (int k = 0; k < 5; ++k) m[k] = p[k];
}

// walks the list of objects of `kind` containing MD `md`: for (It it(d, n_md, kind, md); it.obj >= 0; it.next())
struct IdxIt {
  const int* next;
  int node, per, obj;
  __device__ IdxIt(const Dev& d, int n_md, int kind, int md)
      : next(d.idx_next + node_base(d, kind)), node(d.idx_head[kind * n_md + md]), per(kind == 2 ? 3 : (kind == 3 ? 4 : 5)) {
    obj = node ? (node - 1) / per : -1;
  }
  __device__ void advance() {
    node = next[node - 1];
    obj = node ? (node - 1) / per : -1;
  }
};

// The three rules are latency-bound: an object walks a handful of short linked lists, every element a chain of
// dependent loads.  Each object is therefore given a group of 4, 8 or 16 lanes, one list (or the same-seed
// range) per lane; a ballot over the group decides.  Groups are aligned sub-warps.
template <int LANES>
__device__ __forceinline__ bool group_any(bool pred) {
  const unsigned m = __ballot_sync(kFull, pred);
  const int lane = threadIdx.x & 31;
  return ((m >> (lane & ~(LANES - 1))) & ((1u << LANES) - 1u)) != 0u;
}

// rule 1: pT5 X is removed by a better pT5 of the same seed (task 0) or sharing >= 3 MDs (tasks 1..3: the
// lists of X.md[0], [2], [4])
__global__ void __launch_bounds__(kBlock) k_rule1(Dev d) {
  load_batch(d);
  constexpr int kRuleLanes = 4;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_PT5];
  const int task = threadIdx.x & (kRuleLanes - 1);
  const int n_groups = gridDim.x * blockDim.x / kRuleLanes, g0 = (blockIdx.x * blockDim.x + threadIdx.x) / kRuleLanes;
  for (int X0 = 0; X0 < n; X0 += n_groups) {  // all lanes of a warp stay in the loop (ballot)
    const int X = X0 + g0;
    bool rem = false;
    int2 x = make_int2(0, 0);
    if (X < n && task < 4) {
      x = d.pt5[X];
      const float sX = d.pt5_score[X];
      int mX[5], mY[5];
      load_t5_md(d, x.y, mX);
      if (task == 0) {
        for (int Y = d.pls_pt5_begin[x.x]; Y < d.pls_pt5_begin[x.x + 1] && !rem; ++Y) {
          if (Y == X) continue;
          load_t5_md(d, d.pt5[Y].y, mY);
          rem = better(d, d.pt5_score[Y], x.x, mY, sX, x.x, mX, 5);
        }
      } else {
        for (IdxIt it(d, n_md, 1, mX[2 * (task - 1)]); it.obj >= 0 && !rem; it.advance()) {
          const int Y = it.obj;
          if (Y == X) continue;
          const int2 y = d.pt5[Y];
          load_t5_md(d, y.y, mY);
          rem = share(mY, 5, mX, 5) >= 3 && better(d, d.pt5_score[Y], y.x, mY, sX, x.x, mX, 5);
        }
      }
    }
    const bool keep = !group_any<kRuleLanes>(rem);
    if (X < n && task == 0) {
      d.keep5[X] = keep;
      if (keep) {
        d.linked[x.x] = 1;  // one writer per value; rule 4 (k_rule3) completes it with the surviving pT3s
#ifdef LST_RULE3_SKIP_COVERED
        d.t5_cov[x.y] = 1;
#endif
        atomicAdd(d.tc_cnt + kTcClasses * d.pls_event[x.x] + 0, 1);
      }
    }
  }
}

// rule 2: pT3 X is removed by a better pT3 of the same seed (task 0) or sharing >= 2 MDs (tasks 1, 2: lists of
// X.md[0], [1]), or by a SURVIVING pT5 of its seed (task 0) or sharing >= 2 MDs (tasks 3, 4)
__global__ void __launch_bounds__(kBlock) k_rule2(Dev d) {
  load_batch(d);
  constexpr int kRuleLanes = 8;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_PT3], n_pt5 = d.ctl->total[K_PT5];
  const int task = threadIdx.x & (kRuleLanes - 1);
  const int n_groups = gridDim.x * blockDim.x / kRuleLanes, g0 = (blockIdx.x * blockDim.x + threadIdx.x) / kRuleLanes;
  for (int X0 = 0; X0 < n; X0 += n_groups) {
    const int X = X0 + g0;
    bool rem = false;
    int2 x = make_int2(0, 0);
    if (X < n) {
      x = d.pt3[X];
      rem = d.linked[x.x] & 1;  // rule 2b: seed already in a surviving pT5 (about half of the pT3s: the whole group skips its lists)
    }
    if (X < n && task < 5 && !rem) {
      const float sX = d.pt3_score[X];
      int mX[3], mY[5];
      load_t3_md(d, x.y, mX);
      if (task == 0) {
        for (int Y = d.pls_pt3_begin[x.x]; Y < d.pls_pt3_begin[x.x + 1] && !rem; ++Y) {
          if (Y == X) continue;
          load_t3_md(d, d.pt3[Y].y, mY);
          rem = better(d, d.pt3_score[Y], x.x, mY, sX, x.x, mX, 3);
        }
      } else if (task <= 2) {
        for (IdxIt it(d, n_md, 2, mX[task - 1]); it.obj >= 0 && !rem; it.advance()) {
          const int Y = it.obj;
          if (Y == X) continue;
          const int2 y = d.pt3[Y];
          load_t3_md(d, y.y, mY);
          rem = share(mY, 3, mX, 3) >= 2 && better(d, d.pt3_score[Y], y.x, mY, sX, x.x, mX, 3);
        }
      } else if (n_pt5 > 0) {
        for (IdxIt it(d, n_md, 1, mX[task - 3]); it.obj >= 0 && !rem; it.advance()) {
          const int Z = it.obj;
          if (!d.keep5[Z]) continue;
          load_t5_md(d, d.pt5[Z].y, mY);
          rem = share(mX, 3, mY, 5) >= 2;
        }
      }
    }
    const bool keep = !group_any<kRuleLanes>(rem);
    if (X < n && task == 0) {
      d.keep3[X] = keep;
      if (keep) atomicAdd(d.tc_cnt + kTcClasses * d.pls_event[x.x] + 1, 1);
    }
  }
}

// Called by every block at the end of the last rule kernel: the last block to arrive turns the per-(event, class)
// survivor counts into tc_begin (a scan of kTcClasses * n_events + 1 numbers, in chunks of kBlock).
__device__ __forceinline__ void tc_scan_by_last_block(const Dev& d) {
  __shared__ int s_last;
  __shared__ int s_carry;
  __shared__ int s_warp[kWarps];
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    s_last = atomicAdd(&d.ctl->done_rule, 1) == (int)gridDim.x - 1;
    s_carry = 0;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  const int m = kTcClasses * d.n_events;  // tc_begin[0 .. m], tc_begin[m] = total
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int c0 = 0; c0 < m; c0 += kBlock) {
    const int i = c0 + threadIdx.x;
    const int v = i < m ? __ldcg(d.tc_cnt + i) : 0;
    const int incl = warp_incl_scan(v);
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int base = s_carry;
    for (int w = 0; w < warp; ++w) base += s_warp[w];
    if (i < m) d.tc_begin[i] = base + incl - v;
    __syncthreads();
    if (threadIdx.x == kBlock - 1) s_carry = base + incl;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    const int total = s_carry;
    d.tc_begin[m] = total;
    if (total > d.cap[K_TC]) {
      atomicOr(&d.ctl->error, E_CAP_TC);
      d.ctl->total[K_TC] = 0;
    } else {
      d.ctl->total[K_TC] = total;
    }
  }
}

// rule 3: T5 X is removed by a better T5 sharing >= 3 MDs (tasks 0..2: lists of X.md[0], [2], [4]), by a surviving
// pT5 (tasks 3..6) or pT3 (tasks 7..10) sharing >= 2 MDs (lists of X.md[0..3]); rule 4: unlinked pLS.  The last
// block to finish turns the per-(event, class) survivor counts into tc_begin (a scan of 4 * n_events + 1 numbers).
template <bool SCAN>
__global__ void __launch_bounds__(kBlock) k_rule3(Dev d) {
  load_batch(d);
  constexpr int kRuleLanes = 16;
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_T5];
  const int n_pt5 = d.ctl->total[K_PT5], n_pt3 = d.ctl->total[K_PT3];
  const int task = threadIdx.x & (kRuleLanes - 1);
  const int n_groups = stride / kRuleLanes, g0 = i0 / kRuleLanes;
  for (int X0 = 0; X0 < n; X0 += n_groups) {
    const int X = X0 + g0;
#ifdef LST_RULE3_SKIP_COVERED
    // NOT part of the product: the variant that faults (profiles/r03_rule3_fault.md).  A T5 with a surviving pT5 built
    // on it (rule 3b, all five MDs shared) skips its lists.  Same results by the spec; built with this macro the
    // kernel gives wrong survivor sets within a few batches and then hangs or faults -- unless the MD of a lane's
    // list is picked by selects (LST_RULE3_SELECT) instead of mX[2 * task] / mX[task - 3] / mX[task - 7].
    bool rem = X < n && d.t5_cov[X] != 0;
#else
    bool rem = false;
#endif
    int md0 = 0;
    if (X < n && task < 11 && !rem) {
      const float sX = d.t5_score[X];
      int mX[5], mY[5];
      load_t5_md(d, X, mX);
      md0 = mX[0];
#ifdef LST_RULE3_SELECT
      const int t4 = task < 7 ? task - 3 : task - 7;
      const int md_a = task == 0 ? mX[0] : (task == 1 ? mX[2] : mX[4]);
      const int md_b = t4 == 0 ? mX[0] : (t4 == 1 ? mX[1] : (t4 == 2 ? mX[2] : mX[3]));
#define LST_MD_A md_a
#define LST_MD_B md_b
#define LST_MD_C md_b
#else
#define LST_MD_A mX[2 * task]
#define LST_MD_B mX[task - 3]
#define LST_MD_C mX[task - 7]
#endif
      if (task < 3) {
        for (IdxIt it(d, n_md, 0, LST_MD_A); it.obj >= 0 && !rem; it.advance()) {
          const int Y = it.obj;
          if (Y == X) continue;
          load_t5_md(d, Y, mY);
          rem = share(mY, 5, mX, 5) >= 3 && better(d, d.t5_score[Y], -1, mY, sX, -1, mX, 5);
        }
      } else if (task < 7) {
        if (n_pt5 > 0)
          for (IdxIt it(d, n_md, 1, LST_MD_B); it.obj >= 0 && !rem; it.advance()) {
            const int Z = it.obj;
            if (!d.keep5[Z]) continue;
            load_t5_md(d, d.pt5[Z].y, mY);
            rem = share(mX, 5, mY, 5) >= 2;
          }
      } else if (n_pt3 > 0) {
        for (IdxIt it(d, n_md, 2, LST_MD_C); it.obj >= 0 && !rem; it.advance()) {
          const int Z = it.obj;
          if (!d.keep3[Z]) continue;
          load_t3_md(d, d.pt3[Z].y, mY);
          rem = share(mX, 5, mY, 3) >= 2;
        }
      }
    }
    const bool keep = !group_any<kRuleLanes>(rem);
    if (X < n && task == 0) {
      d.keepT[X] = keep;
      if (keep) atomicAdd(d.tc_cnt + kTcClasses * ev_of_md(d, md0) + 2, 1);
    }
  }
  // rule 4: a pLS is linked if it seeds a surviving pT5 (flag set by rule 1) or pT3
  for (int p = i0; p < d.n_pls; p += stride) {
    bool lk = d.linked[p] & 1;
    for (int Y = n_pt3 > 0 ? d.pls_pt3_begin[p] : 0; !lk && n_pt3 > 0 && Y < d.pls_pt3_begin[p + 1]; ++Y)
      lk = d.keep3[Y];
    d.linked[p] = lk;
    if (!lk) atomicAdd(d.tc_cnt + kTcClasses * d.pls_event[p] + 3, 1);
  }
  if (SCAN) tc_scan_by_last_block(d);
}

// rule 5 of CUTS.md section 10 (extension): T4 X is removed by a better T4 sharing >= 3 MDs (tasks 0, 1: lists of
// X.md[0], [1]) or by a surviving pT5 / pT3 / T5 sharing >= 2 MDs (tasks 2..10: lists of X.md[0..2] per kind).
// Launched (after k_rule3<false>) only when T4s are built; ends with the tc_begin scan.
__global__ void __launch_bounds__(kBlock) k_rule_t4(Dev d) {
  load_batch(d);
  constexpr int kRuleLanes = 16;
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_T4];
  const int task = threadIdx.x & (kRuleLanes - 1);
  const int n_groups = stride / kRuleLanes, g0 = i0 / kRuleLanes;
  for (int X0 = 0; X0 < n; X0 += n_groups) {
    const int X = X0 + g0;
    bool rem = false;
    int md0 = 0;
    if (X < n && task < 11) {
      const float sX = d.t4_score[X];
      const int4 m = d.t4_md[X];
      const int mX[4] = {m.x, m.y, m.z, m.w};
      int mY[5];
      md0 = m.x;
      if (task < 2) {
        for (IdxIt it(d, n_md, 3, mX[task]); it.obj >= 0 && !rem; it.advance()) {
          const int Y = it.obj;
          if (Y == X) continue;
          const int4 y = d.t4_md[Y];
          mY[0] = y.x; mY[1] = y.y; mY[2] = y.z; mY[3] = y.w;
          rem = share(mY, 4, mX, 4) >= 3 && better(d, d.t4_score[Y], -1, mY, sX, -1, mX, 4);
        }
      } else {
        const int kind = (task - 2) / 3 == 0 ? 1 : ((task - 2) / 3 == 1 ? 2 : 0);  // pT5, pT3, T5
        for (IdxIt it(d, n_md, kind, mX[(task - 2) % 3]); it.obj >= 0 && !rem; it.advance()) {
          const int Z = it.obj;
          if (kind == 1) {
            if (!d.keep5[Z]) continue;
            load_t5_md(d, d.pt5[Z].y, mY);
            rem = share(mX, 4, mY, 5) >= 2;
          } else if (kind == 2) {
            if (!d.keep3[Z]) continue;
            load_t3_md(d, d.pt3[Z].y, mY);
            rem = share(mX, 4, mY, 3) >= 2;
          } else {
            if (!d.keepT[Z]) continue;
            load_t5_md(d, Z, mY);
            rem = share(mX, 4, mY, 5) >= 2;
          }
        }
      }
    }
    const bool keep = !group_any<kRuleLanes>(rem);
    if (X < n && task == 0) {
      d.keep4[X] = keep;
      if (keep) atomicAdd(d.tc_cnt + kTcClasses * ev_of_md(d, md0) + 4, 1);
    }
  }
  tc_scan_by_last_block(d);
}

// track candidates: (type, pls, t5, t3, hit_idx[12]) per event in class order; event-local indices
__global__ void __launch_bounds__(kBlock) k_tc_emit(Dev d) {
  load_batch(d);
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int E1 = d.n_events + 1;
  const int n_pt5 = d.ctl->total[K_PT5], n_pt3 = d.ctl->total[K_PT3], n_t5 = d.ctl->total[K_T5];
  const int n_t4 = (d.cuts.stage_mask & 64) ? d.ctl->total[K_T4] : 0;
  const int* __restrict__ ev_first = d.ev_first;
  if (d.tc_begin[kTcClasses * d.n_events] > d.cap[K_TC]) return;  // flagged by the scan of the last rule kernel
  for (int i = i0; i < n_pt5 + n_pt3 + n_t5 + d.n_pls + n_t4; i += stride) {
    int cls, ev, pls = -1, t5 = -1, t3 = -1, nmd = 0;
    int md[5];
    if (i < n_pt5) {
      if (!d.keep5[i]) continue;
      cls = 0; pls = d.pt5[i].x; t5 = d.pt5[i].y; ev = d.pls_event[pls];
      load_t5_md(d, t5, md); nmd = 5;
    } else if (i < n_pt5 + n_pt3) {
      const int X = i - n_pt5;
      if (!d.keep3[X]) continue;
      cls = 1; pls = d.pt3[X].x; t3 = d.pt3[X].y; ev = d.pls_event[pls];
      load_t3_md(d, t3, md); nmd = 3;
    } else if (i < n_pt5 + n_pt3 + n_t5) {
      t5 = i - n_pt5 - n_pt3;
      if (!d.keepT[t5]) continue;
      cls = 2; load_t5_md(d, t5, md); nmd = 5; ev = ev_of_md(d, md[0]);
    } else if (i < n_pt5 + n_pt3 + n_t5 + d.n_pls) {
      pls = i - n_pt5 - n_pt3 - n_t5;
      if (d.linked[pls]) continue;
      cls = 3; ev = d.pls_event[pls];
    } else {  // T4 (CUTS.md section 10): t3 = its first T3
      const int X = i - n_pt5 - n_pt3 - n_t5 - d.n_pls;
      if (!d.keep4[X]) continue;
      const int4 m = d.t4_md[X];
      cls = 4; t3 = d.t4_t3[X].x; md[0] = m.x; md[1] = m.y; md[2] = m.z; md[3] = m.w; nmd = 4; ev = ev_of_md(d, m.x);
    }
    const int pos = d.tc_begin[kTcClasses * ev + cls] + atomicAdd(d.tc_cur + kTcClasses * ev + cls, 1);
    int* o = d.tc + 16 * (size_t)pos;
    o[0] = cls;
    o[1] = pls >= 0 ? pls - d.pls_ev_off[ev] : -1;
    o[2] = t5 >= 0 ? t5 - ev_first[K_T5 * E1 + ev] : -1;
    o[3] = t3 >= 0 ? t3 - ev_first[K_T3 * E1 + ev] : -1;
    for (int k = 0; k < 6; ++k) {
      int2 h = make_int2(-1, -1);
      if (k < nmd) h = d.md_hit[md[k]];
      o[4 + 2 * k] = h.x;
      o[5 + 2 * k] = h.y;
    }
  }
}

}  // namespace lst
