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

constexpr int kSeedTile = 128;  // seeds staged per tile

// ---- anchors: the MDs that start at least one T3 (and therefore every T5) ----------------------
// The gate of CUTS.md section 7 depends only on the seed and on the FIRST MD of the candidate, and
// T3s / T5s are stored grouped by first MD: all candidates of an anchor share one gate evaluation.
// The anchors of an event are sorted into kAncBins = 8 radial classes x 64 azimuthal sectors
// (counting sort: k_anchor counts and keeps the arrival rank, k_scan, k_anchor_sort places), so the
// 32 anchors of a warp of k_pt_eval sit within a few cm of each other and a seed whose gate cone
// misses their bounding circle is skipped for the whole warp.
constexpr int kAncBins = 512;

__device__ __forceinline__ int anchor_bin(float x, float y, float r) {
  const int rc = (r >= 29.5f) + (r >= 43.5f) + (r >= 59.5f) + (r >= 78.0f) + (r >= 98.0f) + (r >= 125.0f);
  const float a = fabsf(x) + fabsf(y);
  const float t = a > 0.0f ? y / a : 0.0f;                                  // diamond angle, monotone in azimuth
  const float ps = x >= 0.0f ? (y >= 0.0f ? t : 4.0f + t) : 2.0f - t;      // [0, 4)
  int sec = (int)(ps * 16.0f);
  sec = sec < 0 ? 0 : (sec > 63 ? 63 : sec);
  return rc * 64 + sec;  // any finite or non-finite input lands in [0, 512): binning never affects results
}

__global__ void __launch_bounds__(kBlock) k_anchor(Dev d) {
  const bool on = (d.cuts.stage_mask & 16) && d.ctl->total[K_T3] > 0;
  const int n = d.ctl->total[K_MD];
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < n; A += gridDim.x * blockDim.x) {
    int bin = -1, rank = 0;
    if (on && d.ls_t3_begin[d.md_ls_begin[A + 1]] > d.ls_t3_begin[d.md_ls_begin[A]]) {
      const float4 a = d.md_a[A];
      const int ev = (d.md_info[A] >> 1) / d.n_mod;
      bin = ev * kAncBins + anchor_bin(a.x, a.y, a.w);
      rank = atomicAdd(d.anc_bin_cnt + bin, 1);
    }
    d.anc_bin[A] = bin;
    d.anc_rank[A] = rank;
  }
}

// after k_scan(anc_bin_cnt -> anc_bin_begin)
__global__ void __launch_bounds__(kBlock) k_anchor_sort(Dev d) {
  const bool on5 = d.ctl->total[K_T5] > 0;
  const int n = d.ctl->total[K_MD];
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < n; A += gridDim.x * blockDim.x) {
    const int bin = d.anc_bin[A];
    if (bin < 0) continue;
    const int pos = d.anc_bin_begin[bin] + d.anc_rank[A];
    const int t0 = d.ls_t3_begin[d.md_ls_begin[A]], t1 = d.ls_t3_begin[d.md_ls_begin[A + 1]];
    const float4 a = d.md_a[A];
    d.anc_axy[pos] = make_float2(a.x, a.y);
    d.anc_t3[pos] = make_int2(t0, t1 - t0);
    const int u0 = on5 ? d.t3_t5_begin[t0] : 0, u1 = on5 ? d.t3_t5_begin[t1] : 0;
    d.anc_t5[pos] = make_int2(u0, u1 - u0);
  }
}

// per-event table written by k_pt_tiles: anchor range, seed range, first tile
struct PtEvent {
  int a0, a1;
  int s0, s1;
  int tile0;
};

// One block.  Fills pt_ev[0..n_events) and pt_ev[n_events].tile0 = number of tiles; n_tests.
__global__ void __launch_bounds__(kBlock) k_pt_tiles(Dev d) {
  const int E = d.n_events;
  const bool on = (d.cuts.stage_mask & 16) != 0;
  for (int e = threadIdx.x; e < E; e += kBlock) {
    PtEvent ev;
    ev.s0 = d.pls_ev_off[e];
    ev.s1 = d.pls_ev_off[e + 1];
    ev.a0 = ev.a1 = 0;
    const int ns = on ? ev.s1 - ev.s0 : 0;
    int c0 = 0, c1 = 0;
    if (on && d.ctl->total[K_T3] > 0) {
      ev.a0 = d.anc_bin_begin[e * kAncBins];
      ev.a1 = d.anc_bin_begin[(e + 1) * kAncBins];
      event_cands<false>(d, e, c0, c1);
      // candidates of CUTS.md section 7: every (seed, T3) of the event
      d.ev_cnt[(size_t)e * kEvCnt + 6 + 4] = (unsigned long long)ns * (c1 - c0);
    }
    if (on && d.ctl->total[K_T5] > 0) {
      event_cands<true>(d, e, c0, c1);
      d.ev_cnt[(size_t)e * kEvCnt + 6 + 5] = (unsigned long long)ns * (c1 - c0);
    }
    ev.tile0 = ((ev.a1 - ev.a0 + 31) / 32) * ((ns + kSeedTile - 1) / kSeedTile);  // warp tiles
    d.pt_ev[e] = ev;
  }
  __syncthreads();
  if (threadIdx.x == 0) {  // exclusive prefix of the tile counts (n_events is small)
    int a = 0;
    for (int e = 0; e < E; ++e) {
      const int ta = d.pt_ev[e].tile0;
      d.pt_ev[e].tile0 = a;
      a += ta;
    }
    d.pt_ev[E].tile0 = a;
  }
}

struct PtAccepted {
  int p, t;
  float score;
};

struct PtWarp {  // per-warp scratch of k_pt_eval (dynamic shared memory: kWarps of these)
  float4 seed[kSeedTile];  // x1, y1, vx, vy of the tile's seeds
  float lv[kSeedTile];
  int2 w2[64];         // phase-2 list: (candidate | T5 flag << 31, seed slot)
  float2 axy[32];      // the warp's anchors
  int2 r3[32], r5[32];  // (first, count) of their T3s / T5s
  unsigned w1[64];     // gate survivors: seed slot | anchor lane << 16 | gate-near << 31
  int pref[33];        // exclusive prefix of the candidate counts of w1[0..32)
  unsigned heads[32];  // head bits of the entries over the first 1024 items
  float kp[32], tolk[32];
};

// pT3 and pT5 of the whole batch.  A tile = 32 anchors of one event (one per lane) x up to kSeedTile
// seeds of the same event (shared memory, read as broadcasts).  Warps take tiles by ticket and never
// wait for one another (with a block-wide tile, a quarter of the warp time was spent at the barrier
// behind the warp whose anchors matched the most seeds; profiles/).
__global__ void __launch_bounds__(kBlock) k_pt_eval(Dev d) {
  extern __shared__ __align__(16) unsigned char s_dyn[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  PtWarp& w = reinterpret_cast<PtWarp*>(s_dyn)[warp];
  float4* const s_seed = w.seed;
  float* const s_lv = w.lv;
  const int E = d.n_events;
  const int n_tiles = d.pt_ev[E].tile0;
  const int cap3 = d.cap[K_PT3], cap5 = d.cap[K_PT5];
  PtAccepted* scratch3 = reinterpret_cast<PtAccepted*>(d.ev_scratch);
  PtAccepted* scratch5 = reinterpret_cast<PtAccepted*>(d.ev_scratch2);
  const float inv_2rmin = d.cuts.inv_2rmin * 1.0001f, gate_tol = d.cuts.pt_gate_tol * 1.0001f;
  for (;;) {
    unsigned near3 = 0, near5 = 0;  // near-threshold candidates of this tile (one event)
    int tile = 0, evi = 0;
    if (lane == 0) {
      tile = atomicAdd(d.ctl->ticket + T_PT3, 1);
      int hi = E;  // event of the tile: largest e with tile0[e] <= tile
      if (tile < n_tiles)
        while (hi - evi > 1) {
          const int mid = (evi + hi) >> 1;
          if (d.pt_ev[mid].tile0 <= tile) evi = mid; else hi = mid;
        }
    }
    tile = __shfl_sync(kFull, tile, 0);
    evi = __shfl_sync(kFull, evi, 0);
    if (tile >= n_tiles) break;
    const PtEvent ev = d.pt_ev[evi];
    const int n_ab = (ev.a1 - ev.a0 + 31) / 32;
    const int local = tile - ev.tile0;
    const int sb = local / n_ab, ab = local - sb * n_ab;
    const int p0 = ev.s0 + sb * kSeedTile;
    const int n_seed = min(kSeedTile, ev.s1 - p0);
    for (int k = lane; k < n_seed; k += 32) {
      const int p = p0 + k;
      const float x1 = __ldg(d.p_x1 + p), y1 = __ldg(d.p_y1 + p);
      const float vx = x1 - __ldg(d.p_x0 + p), vy = y1 - __ldg(d.p_y0 + p);
      s_seed[k] = make_float4(x1, y1, vx, vy);
      s_lv[k] = sqrtf(vx * vx + vy * vy);
    }
    __syncwarp();
    const int anc = ev.a0 + ab * 32 + lane;
    const bool valid = anc < ev.a1;
    float2 A = make_float2(0.0f, 0.0f);
    int2 r3 = make_int2(0, 0), r5 = make_int2(0, 0);  // (first, count) of the anchor's T3s / T5s
    if (valid) {
      A = d.anc_axy[anc];
      r3 = d.anc_t3[anc];
      r5 = d.anc_t5[anc];
    }
    // ---- phase 2: the exact cut list for one entry of the warp's list ----
    auto phase2 = [&](int2 ent) {
      const bool is5 = ent.x < 0;
      const int t = ent.x & 0x7fffffff, ks = ent.y;
      const int p = p0 + ks;
      const float4 sd = s_seed[ks];
      const Seed full = make_seed(d.cuts, __ldg(d.p_pt + p), __ldg(d.p_q + p), __ldg(d.p_x0 + p), __ldg(d.p_y0 + p),
                                  __ldg(d.p_z0 + p), sd.x, sd.y, __ldg(d.p_z1 + p));
      float score;
      const unsigned r2 = is5 ? PtCand<true>::test(d, full, t, score) : PtCand<false>::test(d, full, t, score);
      if (is5) near5 += (r2 >> 1) & 1u; else near3 += (r2 >> 1) & 1u;
      if (r2 & ACC) {
        const int slot = atomicAdd(&d.ctl->scratch_cur[is5 ? 3 : 2], 1);
        if (slot < (is5 ? cap5 : cap3)) (is5 ? scratch5 : scratch3)[slot] = PtAccepted{p, t, score};
        atomicAdd((is5 ? d.pls_pt5_cnt : d.pls_pt3_cnt) + p, 1);
      }
    };
    int n2 = 0;
    // pushes up to one entry per lane onto the warp's phase-2 list; runs phase 2 whenever 32 are waiting
    auto push2 = [&](bool go, int cand, int ks) {
      const unsigned m = __ballot_sync(kFull, go);
      if (m == 0u) return;
      if (go) w.w2[n2 + __popc(m & ((1u << lane) - 1u))] = make_int2(cand, ks);
      n2 += __popc(m);
      if (n2 >= 32) {
        __syncwarp();
        phase2(w.w2[lane]);
        const int2 rest = (32 + lane < n2) ? w.w2[32 + lane] : make_int2(0, 0);
        __syncwarp();
        w.w2[lane] = rest;
        n2 -= 32;
        __syncwarp();
      }
    };
    // The warp's 32 anchors, readable by every lane (a gate survivor is expanded by whichever lane is free).
    w.axy[lane] = A;
    w.r3[lane] = r3;
    w.r5[lane] = r5;
    __syncwarp();
    // ---- expansion of up to 32 gate survivors (seed slot | anchor lane << 16 | gate-near << 31) into
    // their (seed, T3) / (seed, T5) candidates, flattened over the lanes; the curvature pre-filter
    // decides which go on to the exact cuts ----
    auto expand = [&](int n_ent) {
      int n_c = 0;
      if (lane < n_ent) {
        const unsigned ent = w.w1[lane];
        const int src = (ent >> 16) & 31, ks = ent & 0xffff;
        n_c = w.r3[src].y + w.r5[src].y;
        const float kp = (-(float)__ldg(d.p_q + p0 + ks)) / (__ldg(d.p_pt + p0 + ks) * d.cuts.kr);
        w.kp[lane] = kp;
        w.tolk[lane] = d.cuts.pt_k_tol0 + d.cuts.pt_k_tol1 * fabsf(kp);
      }
      const int incl = warp_incl_scan(n_c);
      w.pref[lane] = incl - n_c;
      const int T = __shfl_sync(kFull, incl, 31);
      // item -> entry in O(1): one head bit per entry at the position of its first item; the entry of
      // item `it` = number of head bits at or before it, minus one (falls back to bisection beyond 1024 items)
      w.heads[lane] = 0u;
      __syncwarp();
      if (n_c > 0 && incl - n_c < 1024) atomicOr(&w.heads[(incl - n_c) >> 5], 1u << ((incl - n_c) & 31));
      __syncwarp();
      int heads_before = 0;
      for (int i0 = 0; i0 < T; i0 += 32) {
        const int it = i0 + lane;
        bool go = false;
        int cand = 0, ks = 0;
        const unsigned hw = i0 < 1024 ? w.heads[i0 >> 5] : 0u;
        if (it < T) {
          int lo;
          if (i0 < 1024) {
            lo = heads_before + __popc(hw & (0xffffffffu >> (31 - lane))) - 1;
          } else {
            lo = 0;
            int hi = 32;  // largest e with pref[e] <= it
#pragma unroll
            for (int sft = 0; sft < 5; ++sft) {
              const int mid = (lo + hi) >> 1;
              if (w.pref[mid] <= it) lo = mid; else hi = mid;
            }
          }
          const unsigned ent = w.w1[lo];
          const int src = (ent >> 16) & 31, c = it - w.pref[lo];
          ks = ent & 0xffff;
          const int2 a3 = w.r3[src], a5 = w.r5[src];
          const bool is5 = c >= a3.y;
          const int t = is5 ? a5.x + (c - a3.y) : a3.x + c;
          cand = t | (is5 ? 0x80000000 : 0);
          go = true;
          if (!(ent >> 31)) {
            const float4 sd = s_seed[ks];
            go = pt_curv_possible(w.kp[lo], w.tolk[lo], sd.x, sd.y, w.axy[src], is5 ? d.t5_lxy[t] : d.t3_lxy[t]);
          }
        }
        heads_before += __popc(hw);
        push2(go, cand, ks);
      }
      __syncwarp();
    };
    int n1 = 0;  // gate survivors waiting in w.w1
    // ---- bounding circle of the warp's anchors (sorted by radius class and azimuth: a few cm) ----
    float bx0 = valid ? A.x : 3e38f, bx1 = valid ? A.x : -3e38f, by0 = valid ? A.y : 3e38f, by1 = valid ? A.y : -3e38f;
#pragma unroll
    for (int sh = 16; sh > 0; sh >>= 1) {
      bx0 = fminf(bx0, __shfl_xor_sync(kFull, bx0, sh));
      bx1 = fmaxf(bx1, __shfl_xor_sync(kFull, bx1, sh));
      by0 = fminf(by0, __shfl_xor_sync(kFull, by0, sh));
      by1 = fmaxf(by1, __shfl_xor_sync(kFull, by1, sh));
    }
    const bool warp_has = bx0 <= bx1;
    const float bcx = 0.5f * (bx0 + bx1), bcy = 0.5f * (by0 + by1);
    const float bh = 0.5f * sqrtf((bx1 - bx0) * (bx1 - bx0) + (by1 - by0) * (by1 - by0)) * 1.001f + 1e-3f;
    // ---- phase 1, 32 seeds at a time ----
    for (int kb = 0; kb < n_seed && warp_has; kb += 32) {
      // (a) one seed per lane against the circle: can its gate accept ANY point within bh of the centre?
      //     gdot(A) <= v.wc + lv*bh and gcrs(A) >= |v x wc| - lv*bh, glim(A) <= glim at |wc| + bh; margins
      //     1e-3 cover the rounding of both sides (~1e-6 relative).  Out of range: tested by every lane.
      bool maybe = false;
      if (kb + lane < n_seed) {
        const float4 sd = s_seed[kb + lane];
        const float lv = s_lv[kb + lane];
        const float wx = bcx - sd.x, wy = bcy - sd.y;
        const float lw2 = wx * wx + wy * wy;
        float rl;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rl) : "f"(lw2));
        const float Lw = (lw2 * rl + bh) * 1.001f;
        const float slack = lv * (bh * 1.001f + 1e-4f);
        const float dotc = sd.z * wx + sd.w * wy;
        const float crsc = fabsf(sd.z * wy - sd.w * wx);
        const bool in_range = lw2 >= 1e-30f && lw2 <= 1e30f && lv <= 1e30f;
        maybe = !in_range || (dotc + slack > 0.0f && crsc - slack <= (lv * Lw) * (Lw * inv_2rmin + gate_tol));
      }
      unsigned word = __ballot_sync(kFull, maybe);
      // (b) the seeds that may match: every lane tests its own anchor
      while (word) {
        const int k = kb + __ffs(word) - 1;
        word &= word - 1;
        bool pass = false;
        unsigned ent = 0u;
        if (valid) {
          const float4 sd = s_seed[k];
          const float wx = A.x - sd.x, wy = A.y - sd.y;
          const float gdot = sd.z * wx + sd.w * wy;
          const float lw2 = wx * wx + wy * wy;
          float rl;
          asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rl) : "f"(lw2));
          const float lw = lw2 * rl;
          const float gcrs = fabsf(sd.z * wy - sd.w * wx);
          const float lim = (s_lv[k] * lw) * (lw * inv_2rmin + gate_tol);
          // three outcomes: surely rejected (dropped), surely accepted and not near-threshold (the exact
          // gate is skipped), uncertain = within 2e-4 of the threshold or out of the approximation's
          // range (the exact gate decides)
          const bool in_range = lw2 >= 1e-30f && lw2 <= 1e30f;
          pass = gdot > 0.0f && (!(gcrs > lim) || !in_range);
          if (pass && !(in_range && gcrs <= lim * 0.9998f)) {
            // phase 1b: the exact gate (CUTS.md section 7) decides and flags near-threshold
            Seed s;
            s.x1 = sd.x;  s.y1 = sd.y;  s.vx = sd.z;  s.vy = sd.w;  s.lv = s_lv[k];
            const unsigned r = pt_gate(d.cuts, s, A.x, A.y);
            pass = (r & ACC) != 0;
            if (!pass && (r & NEAR)) {  // every candidate of the anchor fails the gate near its threshold
              near3 += (unsigned)r3.y;
              near5 += (unsigned)r5.y;
            }
            if (r & NEAR) ent = 0x80000000u;
          }
          ent |= (unsigned)k | ((unsigned)lane << 16);
        }
        // gate survivors onto the warp's list, in (seed, lane) order; a full warp of them is expanded at once
        const unsigned m = __ballot_sync(kFull, pass);
        if (m == 0u) continue;
        if (pass) w.w1[n1 + __popc(m & ((1u << lane) - 1u))] = ent;
        n1 += __popc(m);
        if (n1 >= 32) {
          __syncwarp();
          expand(32);
          const unsigned rest = (32 + lane < n1) ? w.w1[32 + lane] : 0u;
          __syncwarp();
          w.w1[lane] = rest;
          n1 -= 32;
          __syncwarp();
        }
      }
    }
    __syncwarp();
    if (n1 > 0) expand(n1);
    if (lane < n2) phase2(w.w2[lane]);
    if (__any_sync(kFull, (near3 | near5) != 0u)) {
      const int s3 = warp_sum((int)near3), s5 = warp_sum((int)near5);
      if (lane == 0) {
        if (s3) atomicAdd(d.ev_cnt + (size_t)evi * kEvCnt + 4, (unsigned long long)s3);
        if (s5) atomicAdd(d.ev_cnt + (size_t)evi * kEvCnt + 5, (unsigned long long)s5);
      }
    }
    __syncwarp();  // the seed tile is reused
  }
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
  const PtAccepted* scratch = reinterpret_cast<const PtAccepted*>(IS5 ? d.ev_scratch2 : d.ev_scratch);
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
