// lst_pt.cuh -- step a5: pLS x T3 -> pT3 and pLS x T5 -> pT5 (CUTS.md section 7).
// Candidates of a seed = every T3 / T5 of its event (CUTS.md section 7; the direction gate of the
// spec replaces the IT->OT connection map): ~1.2e8 (seed, T3) pairs per 16-event PU200 batch, of
// which 8% pass the gate and 0.06% are accepted.  This is the heaviest loop of the chain, so its
// inner step is stripped to the arithmetic of a NECESSARY condition of the gate:
//   * a tile = 256 candidates of one event (one per thread, first/last anchor in registers) x up
//     to kSeedTile seeds of the same event (staged in shared memory, read as broadcasts);
//   * phase 1 (every pair): gdot > 0 exactly as in the spec and gcrs <= glim with |A - P1| from
//     the approximate reciprocal square root and a 1e-4 margin; a survivor costs one store into
//     the thread's own queue -- no ballot, no index arithmetic;
//   * phase 1b (8%): the exact gate (near-threshold accounting of CUTS.md section 0 happens here)
//     and a sqrt-free necessary condition of the curvature match;
//   * phase 2 (<1%): the exact cut list.
// Accepted pairs go to a scratch list (atomics per accepted object, ~4 per 10^4 tests); k_pt_place
// groups them by seed with a counting sort (count in phase 2, generic scan, scatter).  Order
// inside a seed's range is arrival order -- free by the spec (reading S9).
#pragma once
#include "lst_cuts_pt.cuh"
#include "lst_stages.cuh"

namespace lst {

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

// first candidate (T3 or T5) of event ev and one past its last
template <bool IS5>
__device__ __forceinline__ void event_cands(const Dev& d, int ev, int& c0, int& c1) {
  const int md0 = d.mod_md_begin[ev * d.n_mod], md1 = d.mod_md_begin[(ev + 1) * d.n_mod];
  c0 = d.ls_t3_begin[d.md_ls_begin[md0]];
  c1 = d.ls_t3_begin[d.md_ls_begin[md1]];
  if (IS5) {
    c0 = d.t3_t5_begin[c0];
    c1 = d.t3_t5_begin[c1];
  }
}

constexpr int kSeedTile = 128;   // seeds staged per tile
constexpr int kSeedSub = 128;    // seeds between two drains of the survivor queues
constexpr int kQueue = 64;       // survivor queue entries per thread (drained early when one fills up)

// per-event table written by k_pt_tiles: candidate ranges, seed range, first tile (T3 / T5 kernels)
struct PtEvent {
  int c0[2], c1[2];  // [0] T3, [1] T5
  int s0, s1;
  int tile0[2];
};

// One block.  Fills pt_ev[0..n_events) and pt_ev[n_events].tile0 = number of tiles; n_tests.
__global__ void __launch_bounds__(kBlock) k_pt_tiles(Dev d) {
  const int E = d.n_events;
  const bool on = (d.cuts.stage_mask & 16) != 0;
  unsigned long long t3 = 0, t5 = 0;
  for (int e = threadIdx.x; e < E; e += kBlock) {
    PtEvent ev;
    ev.s0 = d.pls_ev_off[e];
    ev.s1 = d.pls_ev_off[e + 1];
    ev.c0[0] = ev.c1[0] = ev.c0[1] = ev.c1[1] = 0;
    if (on && d.ctl->total[K_T3] > 0) event_cands<false>(d, e, ev.c0[0], ev.c1[0]);
    if (on && d.ctl->total[K_T5] > 0) event_cands<true>(d, e, ev.c0[1], ev.c1[1]);
    const int ns = on ? ev.s1 - ev.s0 : 0;
    for (int k = 0; k < 2; ++k)
      ev.tile0[k] = ((ev.c1[k] - ev.c0[k] + kBlock - 1) / kBlock) * ((ns + kSeedTile - 1) / kSeedTile);
    t3 += (unsigned long long)ns * (ev.c1[0] - ev.c0[0]);
    t5 += (unsigned long long)ns * (ev.c1[1] - ev.c0[1]);
    d.pt_ev[e] = ev;
  }
  t3 = warp_sum_u64(t3);
  t5 = warp_sum_u64(t5);
  if ((threadIdx.x & 31) == 0) {
    if (t3) atomicAdd(&d.ctl->n_tests[4], t3);
    if (t5) atomicAdd(&d.ctl->n_tests[5], t5);
  }
  __syncthreads();
  if (threadIdx.x == 0) {  // exclusive prefix of the tile counts (n_events is small)
    int a = 0, b = 0;
    for (int e = 0; e < E; ++e) {
      const int ta = d.pt_ev[e].tile0[0], tb = d.pt_ev[e].tile0[1];
      d.pt_ev[e].tile0[0] = a;
      d.pt_ev[e].tile0[1] = b;
      a += ta;
      b += tb;
    }
    d.pt_ev[E].tile0[0] = a;
    d.pt_ev[E].tile0[1] = b;
  }
}

struct PtAccepted {
  int p, t;
  float score;
};

template <bool IS5>
__global__ void __launch_bounds__(kBlock) k_pt_eval(Dev d) {
  constexpr int K = IS5 ? 1 : 0;
  constexpr int kKind = IS5 ? K_PT5 : K_PT3;
  __shared__ int s_tile, s_ev;
  __shared__ float4 s_seed[kSeedTile];  // x1, y1, vx, vy
  __shared__ float s_lv[kSeedTile];
  __shared__ unsigned short s_q[kQueue][kBlock];  // [entry][thread]: conflict-free per-thread queues
  __shared__ unsigned s_w2[kWarps][64];           // phase-2 list of the warp: source lane << 16 | seed slot
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int E = d.n_events;
  const int n_tiles = d.pt_ev[E].tile0[K];
  const int cap = d.cap[kKind];
  const float2* axy = IS5 ? d.t5_axy : d.t3_axy;
  const float2* lxy = IS5 ? d.t5_lxy : d.t3_lxy;
  int* cnt_p = IS5 ? d.pls_pt5_cnt : d.pls_pt3_cnt;
  PtAccepted* scratch = reinterpret_cast<PtAccepted*>(d.ev_scratch);
  const float inv_2rmin = d.cuts.inv_2rmin * 1.0001f, gate_tol = d.cuts.pt_gate_tol * 1.0001f;
  unsigned long long near = 0;
  for (;;) {
    if (threadIdx.x == 0) {
      const int tile = atomicAdd(d.ctl->ticket + (IS5 ? T_PT5 : T_PT3), 1);
      int lo = 0, hi = E;  // event of the tile: largest e with tile0[e] <= tile
      if (tile < n_tiles)
        while (hi - lo > 1) {
          const int mid = (lo + hi) >> 1;
          if (d.pt_ev[mid].tile0[K] <= tile) lo = mid; else hi = mid;
        }
      s_tile = tile;
      s_ev = lo;
    }
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const PtEvent ev = d.pt_ev[s_ev];
    const int n_cb = (ev.c1[K] - ev.c0[K] + kBlock - 1) / kBlock;
    const int local = tile - ev.tile0[K];
    const int sb = local / n_cb, cb = local - sb * n_cb;
    const int p0 = ev.s0 + sb * kSeedTile;
    const int n_seed = min(kSeedTile, ev.s1 - p0);
    for (int k = threadIdx.x; k < n_seed; k += kBlock) {
      const int p = p0 + k;
      const float x1 = __ldg(d.p_x1 + p), y1 = __ldg(d.p_y1 + p);
      const float vx = x1 - __ldg(d.p_x0 + p), vy = y1 - __ldg(d.p_y0 + p);
      s_seed[k] = make_float4(x1, y1, vx, vy);
      s_lv[k] = sqrtf(vx * vx + vy * vy);
    }
    __syncthreads();
    const int t = ev.c0[K] + cb * kBlock + threadIdx.x;
    const bool valid = t < ev.c1[K];
    float2 A = make_float2(0.0f, 0.0f), L = A;
    if (valid) {
      A = axy[t];
      L = lxy[t];
    }
    // ---- phase 2: the exact cut list for one entry of the warp's list; returns its near flag ----
    const int t_warp = ev.c0[K] + cb * kBlock + warp * 32;
    auto phase2 = [&](unsigned ent) -> unsigned {
      const int ks = ent & 0xffff, tt = t_warp + (int)(ent >> 16);
      const int p = p0 + ks;
      const float4 sd = s_seed[ks];
      const Seed full = make_seed(d.cuts, __ldg(d.p_pt + p), __ldg(d.p_q + p), __ldg(d.p_x0 + p), __ldg(d.p_y0 + p),
                                  __ldg(d.p_z0 + p), sd.x, sd.y, __ldg(d.p_z1 + p));
      float score;
      const unsigned r2 = PtCand<IS5>::test(d, full, tt, score);
      if (r2 & ACC) {
        const int slot = atomicAdd(&d.ctl->scratch_cur[IS5 ? 3 : 2], 1);
        if (slot < cap) scratch[slot] = PtAccepted{p, tt, score};
        atomicAdd(cnt_p + p, 1);
      }
      return (r2 >> 1) & 1u;
    };
    int n2 = 0;
    for (int k0 = 0; k0 < n_seed; k0 += kSeedSub) {
      // ---- phase 1: necessary condition of the gate, survivors into the thread's own queue ----
      int nq = 0;
      const int k1 = min(n_seed, k0 + kSeedSub);
      int k = k0;
      while (k < k1) {
        if (valid) {
#pragma unroll 4
          for (; k < k1 && nq < kQueue; ++k) {
            const float4 sd = s_seed[k];
            const float wx = A.x - sd.x, wy = A.y - sd.y;
            const float gdot = sd.z * wx + sd.w * wy;
            const float lw2 = wx * wx + wy * wy;
            float rl;
            asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rl) : "f"(lw2));
            const float lw = lw2 * rl;
            const float gcrs = fabsf(sd.z * wy - sd.w * wx);
            const float lim = (s_lv[k] * lw) * (lw * inv_2rmin + gate_tol);
            // keep unless surely rejected; out of the approximation's range the exact gate decides
            const bool keep = gdot > 0.0f && (!(gcrs > lim) || !(lw2 >= 1e-30f) || !(lw2 <= 1e30f));
            if (keep) s_q[nq++][threadIdx.x] = (unsigned short)k;
          }
        } else {
          k = k1;
        }
        // a full queue anywhere in the warp: drain now, then go on with the rest of the sub-block
        const bool more = __any_sync(kFull, k < k1);
        // ---- phase 1b over the queues, lanes in lockstep; survivors into the warp's phase-2 list ----
        const int nq_max = __reduce_max_sync(kFull, nq);
        for (int i = 0; i < nq_max; ++i) {
          bool go = false;
          int ks = 0;
          if (i < nq) {
            ks = s_q[i][threadIdx.x];
            const float4 sd = s_seed[ks];
            Seed s;
            s.x1 = sd.x;  s.y1 = sd.y;  s.vx = sd.z;  s.vy = sd.w;  s.lv = s_lv[ks];
            const unsigned r = pt_gate(d.cuts, s, A.x, A.y);  // exact gate (CUTS.md section 7)
            go = (r & ACC) != 0;
            if (!go) near += (r >> 1) & 1u;
            if (go && !(r & NEAR))
              go = pt_curv_possible(d.cuts, __ldg(d.p_pt + p0 + ks), __ldg(d.p_q + p0 + ks), sd.x, sd.y, A, L);
          }
          const unsigned m = __ballot_sync(kFull, go);
          if (go) s_w2[warp][n2 + __popc(m & ((1u << lane) - 1u))] = ((unsigned)lane << 16) | (unsigned)ks;
          n2 += __popc(m);
          if (n2 >= 32) {  // a full warp of phase-2 work
            __syncwarp();
            near += phase2(s_w2[warp][lane]);
            const unsigned rest = (32 + lane < n2) ? s_w2[warp][32 + lane] : 0u;
            __syncwarp();
            s_w2[warp][lane] = rest;
            n2 -= 32;
            __syncwarp();
          }
        }
        nq = 0;
        if (!more) break;
      }
    }
    __syncwarp();
    if (lane < n2) near += phase2(s_w2[warp][lane]);
    __syncthreads();  // the seed tile is reused
  }
  near = warp_sum_u64(near);
  if (lane == 0 && near) atomicAdd(&d.ctl->near[IS5 ? 5 : 4], near);
}

// Groups the accepted pairs by seed: begin = exclusive scan of the per-seed counts (k_scan, before
// this kernel); every scratch entry takes the next free slot of its seed.
template <bool IS5>
__global__ void __launch_bounds__(kBlock) k_pt_place(Dev d) {
  constexpr int kKind = IS5 ? K_PT5 : K_PT3;
  const int n = d.ctl->scratch_cur[IS5 ? 3 : 2];
  const int cap = d.cap[kKind];
  const int* begin = IS5 ? d.pls_pt5_begin : d.pls_pt3_begin;
  int* cur = IS5 ? d.pls_pt5_cur : d.pls_pt3_cur;
  int2* out = IS5 ? d.pt5 : d.pt3;
  float* out_s = IS5 ? d.pt5_score : d.pt3_score;
  const PtAccepted* scratch = reinterpret_cast<const PtAccepted*>(d.ev_scratch);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    if (n > cap) {
      atomicOr(&d.ctl->error, IS5 ? E_CAP_PT5 : E_CAP_PT3);
      d.ctl->total[kKind] = 0;
    } else {
      d.ctl->total[kKind] = n;
    }
  }
  if (n > cap) return;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const PtAccepted a = scratch[i];
    const int pos = begin[a.p] + atomicAdd(cur + a.p, 1);
    out[pos] = make_int2(a.p, a.t);
    out_s[pos] = a.score;
  }
}

}  // namespace lst
