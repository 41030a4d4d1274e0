// lst_ls.cuh -- step a2: Line Segments (CUTS.md section 4).
//
// Candidates of an inner MD A: the MDs of every module in conn[module(A)] (the CSR row of the
// precomputed connection map).  A PU200 batch holds 2.1e5 MDs, rows of 7.7 targets on average and
// 1.4 MDs per target: 5e6 candidate pairs in 1.6e6 tiny (MD, target) lists.  Flattening the pairs
// (lst_pairs.cuh) costs more in decoding (pair -> module -> MD -> row edge -> B: ~290 thread
// instructions per pair, ncu) than the cuts themselves (~40), because a 32-pair step crosses a
// module boundary almost every time.  Here the unit is the list:
//   * 8 lanes (a "sub-warp") per inner MD, 4 MDs per warp; lane e walks target e, e + 8, ... of the
//     row, so the CSR walk is done once per (MD, target) and a candidate costs two loads + the cuts;
//   * the lanes of a warp step through their lists together; accepted (B, kappa) pairs are compacted
//     per sub-warp with one ballot per step into shared memory, then copied to a scratch list with
//     one atomic per MD (an MD with more than kLsStage LSs evaluates its row again and writes directly);
//   * k_scan turns the per-MD counts into md_ls_begin; k_ls_place copies each MD's LSs to their slot.
// LSs therefore sit grouped by inner MD (what T3 building looks up); the order inside an MD's range
// is free (reading S9).
#pragma once
#include "lst_stages.cuh"

namespace lst {

constexpr int kLsSub = 8;     // lanes per inner MD
constexpr int kLsStage = 48;  // staged LSs per inner MD

struct LsAccepted {
  int B;
  float kappa;
};

__global__ void __launch_bounds__(kBlock) k_ls_eval(Dev d) {
  __shared__ LsAccepted s_stage[kBlock / kLsSub][kLsStage];
  const int lane = threadIdx.x & 31;
  const int sl = lane & (kLsSub - 1);             // lane inside the sub-warp
  const int sw = lane / kLsSub;                   // sub-warp inside the warp
  const unsigned sub_mask = ((1u << kLsSub) - 1u) << (sw * kLsSub);
  const int sub_id = threadIdx.x / kLsSub;        // sub-warp inside the block
  const int per_block = kBlock / kLsSub;
  const bool on = (d.cuts.stage_mask & 2) != 0;
  const int n_md = d.ctl->total[K_MD];
  const int cap = d.cap[K_LS];
  LsAccepted* scratch = reinterpret_cast<LsAccepted*>(d.ev_scratch);
  unsigned long long near = 0, tests = 0;
  for (int a0 = blockIdx.x * per_block; a0 < n_md; a0 += gridDim.x * per_block) {
    const int A = a0 + sub_id;
    const bool have = A < n_md && on;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    float2 ua = make_float2(0.f, 0.f);
    int eA = 0, k0 = 0, deg = 0, gm_base = 0;
    if (have) {
      const int info = d.md_info[A];
      const int gm = info >> 1;
      const int ev = gm / d.n_mod;
      eA = info & 1;
      a = d.md_a[A];
      ua = d.md_u[A];
      k0 = __ldg(d.conn_off + (gm - ev * d.n_mod));
      deg = __ldg(d.conn_off + (gm - ev * d.n_mod) + 1) - k0;
      gm_base = ev * d.n_mod;
    }
    int cnt = 0;  // accepted so far for this MD (uniform inside the sub-warp)
    // pass 0 stages; pass 1 (only if the stage overflowed) writes directly at the reserved base
    int base = 0;
    for (int pass = 0; pass < 2; ++pass) {
      cnt = 0;
      for (int e0 = 0; __any_sync(kFull, e0 < deg); e0 += kLsSub) {
        const int e = e0 + sl;
        int B = 0, b1 = 0, eB = 0;
        if (e < deg) {
          const int m2 = __ldg(d.conn_tgt + k0 + e);
          B = d.mod_md_begin[gm_base + m2];
          b1 = d.mod_md_begin[gm_base + m2 + 1];
          eB = __ldg(d.subdet + m2) != 0;
          if (pass == 0) tests += (unsigned long long)(b1 - B);
        }
        while (__any_sync(kFull, B < b1)) {
          unsigned r = 0;
          float kappa = 0.0f;
          if (B < b1) r = ls_test(d.cuts, a, ua, eA != 0, d.md_a[B], d.md_u[B], eB != 0, kappa);
          if (pass == 0) near += (r >> 1) & 1u;
          const unsigned m = __ballot_sync(kFull, r & ACC) & sub_mask;
          if (r & ACC) {
            const int pos = cnt + __popc(m & ((1u << lane) - 1u));
            if (pass == 0) {
              if (pos < kLsStage) s_stage[sub_id][pos] = LsAccepted{B, kappa};
            } else if (base + pos < cap) {
              scratch[base + pos] = LsAccepted{B, kappa};
            }
          }
          cnt += __popc(m);
          ++B;
        }
      }
      if (pass == 0) {
        if (sl == 0 && cnt > 0) base = atomicAdd(&d.ctl->scratch_cur[1], cnt);
        base = __shfl_sync(kFull, base, sw * kLsSub);
        if (A < n_md && sl == 0) {
          d.ls_cnt[A] = cnt;
          d.ls_sbase[A] = base;
        }
        __syncwarp();
        if (cnt <= kLsStage)
          for (int k = sl; k < cnt; k += kLsSub)
            if (base + k < cap) scratch[base + k] = s_stage[sub_id][k];
        __syncwarp();  // the staging rows are reused by the next MD
        if (!__any_sync(kFull, cnt > kLsStage)) break;
        if (cnt <= kLsStage) deg = 0;  // only the overflowing sub-warps walk their row again
      }
    }
  }
  near = warp_sum_u64(near);
  tests = warp_sum_u64(tests);
  if (lane == 0) {
    if (near) atomicAdd(&d.ctl->near[1], near);
    if (tests) atomicAdd(&d.ctl->n_tests[1], tests);
  }
}

// After k_scan(ls_cnt -> md_ls_begin): every MD's LSs go from the scratch list to their final slot.
__global__ void __launch_bounds__(kBlock) k_ls_place(Dev d) {
  const int n_md = d.ctl->total[K_MD];
  const int total = d.ctl->scratch_cur[1];
  const int cap = d.cap[K_LS];
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    if (total > cap) {
      atomicOr(&d.ctl->error, E_CAP_LS);
      d.ctl->total[K_LS] = 0;
    } else {
      d.ctl->total[K_LS] = total;
    }
  }
  if (total > cap) return;
  const LsAccepted* scratch = reinterpret_cast<const LsAccepted*>(d.ev_scratch);
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < n_md; A += gridDim.x * blockDim.x) {
    const int n = d.ls_cnt[A], src = d.ls_sbase[A];
    const int dst = d.md_ls_begin[A];
    for (int k = 0; k < n; ++k) {
      const LsAccepted s = scratch[src + k];
      d.ls_md[dst + k] = make_int2(A, s.B);
      d.ls_kappa[dst + k] = s.kappa;
    }
  }
}

}  // namespace lst
