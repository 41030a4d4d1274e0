// lst_pt.cuh -- step a5: pLS x T3 -> pT3 and pLS x T5 -> pT5 (CUTS.md section 7).
// Warp per pLS; lanes stride over the event's T3s / T5s reading the first-MD anchor (float2,
// coalesced) for the gate; the rare gate survivors gather the rest.  Accepted candidates are
// staged in a per-warp shared-memory buffer so the dominant gate loop runs ONCE; only a warp whose
// seed accepts more than kPtBuf candidates re-evaluates.
#pragma once
#include "lst_cuts_pt.cuh"
#include "lst_stages.cuh"

namespace lst {

constexpr int kPtBuf = 96;

template <bool IS5>
struct PtCand {
  // evaluates candidate t for seed s; returns ACC/NEAR bits, score on accept
  static __device__ __forceinline__ unsigned test(const Dev& d, const Seed& s, int t, float& score) {
    const float2 axy = IS5 ? d.t5_axy[t] : d.t3_axy[t];
    unsigned r = pt_gate(d.cuts, s, axy.x, axy.y);
    if (!(r & ACC)) return r;
    r &= NEAR;
    if (IS5) {
      const int* md = d.t5_md + 5 * (size_t)t;
      const int A = md[0], L = md[4];
      const int2 tt = d.t5_t3[t];
      const float kt[2] = {d.t3_k[tt.x], d.t3_k[tt.y]};
      r |= pt_after_gate<2>(d.cuts, s, d.md_a[A], d.md_info[A] & 1, d.md_a[L], d.md_info[L] & 1, kt,
                            d.t5_score[t], score);
    } else {
      const int4 m = d.t3_md[t];
      const float kt[1] = {d.t3_k[t]};
      r |= pt_after_gate<1>(d.cuts, s, d.md_a[m.x], m.w & 1, d.md_a[m.z], (m.w >> 2) & 1, kt, 0.0f,
                            score);
    }
    return r;
  }
};

template <bool IS5>
__global__ void __launch_bounds__(kBlock) k_pt(Dev d) {
  constexpr int kKind = IS5 ? K_PT5 : K_PT3;
  constexpr int kTicket = IS5 ? T_PT5 : T_PT3;
  constexpr int kStage = IS5 ? 5 : 4;
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  __shared__ int s_t[kWarps][kPtBuf];
  __shared__ float s_s[kWarps][kPtBuf];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int n = (d.cuts.stage_mask & 16) ? d.n_pls : 0;
  const int n_tiles = n > 0 ? (n + kWarps - 1) / kWarps : 1;
  const int n_cand_total = d.ctl->total[IS5 ? K_T5 : K_T3];
  int* begin = IS5 ? d.pls_pt5_begin : d.pls_pt3_begin;
  int2* out = IS5 ? d.pt5 : d.pt3;
  float* out_s = IS5 ? d.pt5_score : d.pt3_score;
  const int cap = d.cap[kKind];
  unsigned long long near = 0, tests = 0;
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(d.ctl->ticket + kTicket, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int p = tile * kWarps + warp;
    int cnt = 0, c0 = 0, c1 = 0;
    Seed s;
    if (p < n) {
      if (n_cand_total > 0) {
        const int ev = d.pls_event[p];
        const int md0 = d.mod_md_begin[ev * d.n_mod];
        const int md1 = d.mod_md_begin[(ev + 1) * d.n_mod];
        c0 = d.ls_t3_begin[d.md_ls_begin[md0]];
        c1 = d.ls_t3_begin[d.md_ls_begin[md1]];
        if (IS5) {
          c0 = d.t3_t5_begin[c0];
          c1 = d.t3_t5_begin[c1];
        }
      }
      s = make_seed(d.cuts, __ldg(d.p_pt + p), __ldg(d.p_q + p), __ldg(d.p_x0 + p), __ldg(d.p_y0 + p),
                    __ldg(d.p_z0 + p), __ldg(d.p_x1 + p), __ldg(d.p_y1 + p), __ldg(d.p_z1 + p));
      if (lane == 0) tests += (unsigned long long)(c1 - c0);
      for (int base = c0; base < c1; base += 32) {
        const int t = base + lane;
        unsigned r = 0;
        float score = 0.0f;
        if (t < c1) r = PtCand<IS5>::test(d, s, t, score);
        near += (r >> 1) & 1u;
        const unsigned m = __ballot_sync(kFull, r & ACC);
        if (r & ACC) {
          const int k = cnt + __popc(m & ((1u << lane) - 1u));
          if (k < kPtBuf) {
            s_t[warp][k] = t;
            s_s[warp][k] = score;
          }
        }
        cnt += __popc(m);
      }
    }
    int tb, tt;
    int off = tile_alloc(lane == 0 ? cnt : 0, d.tstate[kTicket], tile, s_scan, tb, tt);
    off = __shfl_sync(kFull, off, 0);
    if (p < n) {
      if (lane == 0) begin[p] = off;
      if (cnt <= kPtBuf) {
        for (int k = lane; k < cnt; k += 32) {
          if (off + k < cap) {
            out[off + k] = make_int2(p, s_t[warp][k]);
            out_s[off + k] = s_s[warp][k];
          }
        }
      } else {  // rare: buffer overflow -> re-evaluate and write directly, same order
        int pos = off;
        for (int base = c0; base < c1; base += 32) {
          const int t = base + lane;
          unsigned r = 0;
          float score = 0.0f;
          if (t < c1) r = PtCand<IS5>::test(d, s, t, score);
          const unsigned m = __ballot_sync(kFull, r & ACC);
          if (r & ACC) {
            const int k = pos + __popc(m & ((1u << lane) - 1u));
            if (k < cap) {
              out[k] = make_int2(p, t);
              out_s[k] = score;
            }
          }
          pos += __popc(m);
        }
      }
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) {
      const int total = tb + tt;
      begin[n] = total;
      if (total > cap) {
        atomicOr(&d.ctl->error, IS5 ? E_CAP_PT5 : E_CAP_PT3);
        d.ctl->total[kKind] = 0;
      } else {
        d.ctl->total[kKind] = total;
      }
    }
    __syncthreads();  // s_t / s_s are reused by the next tile
  }
  near = warp_sum_u64(near);
  tests = warp_sum_u64(tests);
  if (lane == 0) {
    if (near) atomicAdd(&d.ctl->near[kStage], near);
    if (tests) atomicAdd(&d.ctl->n_tests[kStage], tests);
  }
}

}  // namespace lst
