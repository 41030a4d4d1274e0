// lst_pt.cuh -- step a5: pLS x T3 -> pT3 and pLS x T5 -> pT5 (CUTS.md section 7).
// Candidates of a seed = every T3 / T5 of its event (the direction gate of the spec replaces the IT->OT
// connection map): ~1.2e8 (seed, T3) + 2.5e7 (seed, T5) pairs per 16-event PU200 batch, of which 8 % pass
// the gate, 0.9 % the curvature match with the seed and 0.06 % are accepted.  Structure:
//   * anchors: the gate depends only on the seed and the FIRST MD of the candidate, and T3s / T5s are stored
//     grouped by first MD, so the gate is evaluated once per (seed, anchor) and shared by pT3 and pT5;
//     anchors are sorted into radius x azimuth bins (lst_stages.cuh, k_anchor_sort);
//   * k_pt_eval, tile = 32 anchors (one per lane) x 64 seeds of the same event (shared memory, broadcast):
//     (1a) one seed per lane against the bounding circle of the warp's anchors;
//     (1b) every lane tests its anchor against the seeds that may match: a necessary condition of the gate
//          with |A - P1| from rsqrt.approx; only within 1e-4 of the threshold the exact gate decides (and
//          flags near-threshold);
//     (2)  gate survivors are expanded into their (seed, T3 / T5) candidates, flattened over the lanes;
//          kx~ (lst_cuts_pt.cuh) drops those whose curvature match with the seed surely fails;
//     (3)  the rest of the approximate cascade (stored curvatures, r-z at both ends) on full warps;
//     what cannot be rejected for sure goes to a queue;
//   * k_pt_exact runs the exact cut list of CUTS.md section 7 on the queue (1.1 x the accepted objects):
//     accepted pairs go to scratch lists with a count per seed; k_scan2 + k_pt_place group them by seed.
// Objects and both counters are those of the spec: lst_cuts_pt.cuh states why no pre-filter can change them.
#pragma once
#include "lst_cuts_pt.cuh"
#include "lst_stages.cuh"

namespace lst {

__device__ __forceinline__ Seed seed_from_table(const Dev& d, int p) {
  const float4 a = d.seed_a[p], b = d.seed_b[p];
  Seed s;
  s.x1 = a.x;  s.y1 = a.y;  s.z1 = d.seed_z1[p];
  s.vx = a.z;  s.vy = a.w;  s.lv = b.x;
  s.kp = b.y;  s.tolk = b.z;  s.slope = b.w;
  return s;
}

template <bool IS5>
struct PtCand {
  // the exact cut list for seed s and candidate t; returns ACC/NEAR bits, score on accept
  static __device__ __forceinline__ unsigned test(const Dev& d, const Seed& s, int t, float& score) {
    int A, L, eA, eL;
    if (IS5) {
      const int* md = d.t5_md + 5 * (size_t)t;
      A = md[0];  L = md[4];
      eA = d.md_info[A] & 1;  eL = d.md_info[L] & 1;
    } else {
      const int4 m = d.t3_md[t];
      A = m.x;  L = m.z;
      eA = m.w & 1;  eL = (m.w >> 2) & 1;
    }
    const float4 a = d.md_a[A];
    unsigned r = pt_gate(d.cuts, s, a.x, a.y);
    if (!(r & ACC)) return r;
    r &= NEAR;
    if (IS5) {
      const float2 kio = d.t5_kio[t];
      const float kt[2] = {kio.x, kio.y};
      r |= pt_after_gate<2>(d.cuts, s, a, eA, d.md_a[L], eL, kt, d.t5_score[t], score);
    } else {
      const float kt[1] = {d.t3_k[t]};
      r |= pt_after_gate<1>(d.cuts, s, a, eA, d.md_a[L], eL, kt, 0.0f, score);
    }
    return r;
  }
};

constexpr int kSeedTile = 64;           // seeds staged per tile
constexpr int kAncBlocksPerEvent = 8;   // blocks of k_anchor_sort per event

// per-event table written by k_anchor_sort: anchor range, seed range, first tile
struct PtEvent {
  int a0, a1;
  int s0, s1;
  int tile0;
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

// Counting sort of an event's anchors by bin (the counts and arrival ranks come from the T5 kernel's
// prologue).  grid = n_events * kAncBlocksPerEvent; every block scans the 512 bin counts of its event in
// shared memory and places its share of the event's MDs; the anchors of event e start at the event's
// first MD (an event has no more anchors than MDs), so no prefix across events is needed.  Block 0 also
// writes the per-event table of k_pt_eval (ranges, tile prefix) and the candidate counts of stages 4, 5.
__global__ void __launch_bounds__(kBlock) k_anchor_sort(Dev d) {
  load_batch(d);
  __shared__ int s_begin[kAncBins];
  __shared__ int s_warp[kWarps];
  const int E = d.n_events;
  const int e = blockIdx.x / kAncBlocksPerEvent, part = blockIdx.x - e * kAncBlocksPerEvent;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool on = (d.cuts.stage_mask & 16) && d.ctl->total[K_T3] > 0 && d.n_pls > 0;
  const bool on5 = d.ctl->total[K_T5] > 0;
  if (on) {
    // exclusive scan of the event's 512 bin counts: 2 per thread
    const int c0 = d.anc_bin_cnt[e * kAncBins + 2 * threadIdx.x], c1 = d.anc_bin_cnt[e * kAncBins + 2 * threadIdx.x + 1];
    const int incl = warp_incl_scan(c0 + c1);
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    int base = 0;
    for (int w = 0; w < warp; ++w) base += s_warp[w];
    s_begin[2 * threadIdx.x] = base + incl - c0 - c1;
    s_begin[2 * threadIdx.x + 1] = base + incl - c1;
    __syncthreads();
    const int md0 = d.mod_md_begin[e * d.n_mod], md1 = d.mod_md_begin[(e + 1) * d.n_mod];
    for (int A = md0 + part * kBlock + threadIdx.x; A < md1; A += kAncBlocksPerEvent * kBlock) {
      const int bin = d.anc_bin[A];
      if (bin < 0) continue;
      const int pos = md0 + s_begin[bin] + d.anc_rank[A];
      const int t0 = d.ls_t3_begin[d.md_ls_begin[A]], t1 = d.ls_t3_begin[d.md_ls_begin[A + 1]];
      const int u0 = on5 ? d.t3_t5_begin[t0] : 0, u1 = on5 ? d.t3_t5_begin[t1] : 0;
      d.anc_a[pos] = pack_flag(d.md_a[A], d.md_info[A] & 1);
      d.anc_t[pos] = make_int4(t0, t1 - t0, u0, u1 - u0);
    }
  }
  if (blockIdx.x != 0) return;
  __syncthreads();
  // ---- the event table (block 0): anchors = sum of the event's bin counts ----
  for (int ev = warp; ev < E; ev += kWarps) {
    int n_a = 0;
    if (on)
      for (int b = lane; b < kAncBins; b += 32) n_a += d.anc_bin_cnt[ev * kAncBins + b];
    n_a = warp_sum(n_a);
    if (lane == 0) {
      PtEvent pe;
      pe.s0 = d.pls_ev_off[ev];
      pe.s1 = d.pls_ev_off[ev + 1];
      pe.a0 = on ? d.mod_md_begin[ev * d.n_mod] : 0;
      pe.a1 = pe.a0 + n_a;
      const int ns = on ? pe.s1 - pe.s0 : 0;
      pe.tile0 = ((n_a + 31) / 32) * ((ns + kSeedTile - 1) / kSeedTile);  // warp tiles; prefix below
      d.pt_ev[ev] = pe;
      int c0 = 0, c1 = 0;
      if (on) {  // candidates of CUTS.md section 7: every (seed, T3) and (seed, T5) of the event
        event_cands<false>(d, ev, c0, c1);
        d.ev_cnt[(size_t)ev * kEvCnt + kStages + 4] = (unsigned long long)ns * (c1 - c0);
        if (on5) {
          event_cands<true>(d, ev, c0, c1);
          d.ev_cnt[(size_t)ev * kEvCnt + kStages + 5] = (unsigned long long)ns * (c1 - c0);
        }
      }
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {  // exclusive prefix of the tile counts (n_events is small)
    int a = 0;
    for (int ev = 0; ev < E; ++ev) {
      const int ta = d.pt_ev[ev].tile0;
      d.pt_ev[ev].tile0 = a;
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
  float4 sa[kSeedTile];  // x1, y1, vx, vy of the tile's seeds
  float4 sg[kSeedTile];  // gate limit lw (lw c1 + c2), c1 = lv INV_2RMIN, c2 = lv PT_GATE_TOL: upper (c1h, c2h) and lower (c1l, c2l) versions
  float2 sk[kSeedTile];  // kp, tolk
  int2 w2[64];           // candidates behind the curvature pre-filter: (T3 / T5 index | T5 flag << 31, seed slot | anchor lane << 16)
  float4 anc[32];        // the warp's anchors (x, y, z, r | endcap << 31)
  int4 at[32];           // (first T3, number of T3s, first T5, number of T5s) of each
  unsigned w1[64];       // gate survivors: seed slot | anchor lane << 16 | gate-near << 31
  int pref[33];          // exclusive prefix of the candidate counts of w1[0..32)
  unsigned heads[32];    // head bits of the entries over the first 1024 items
};

// pT3 and pT5 candidates of the whole batch -> queue of the exact cuts.  Warps take tiles by ticket and
// never wait for one another.
__global__ void __launch_bounds__(kBlock) k_pt_eval(Dev d) {
  load_batch(d);
  extern __shared__ __align__(16) unsigned char s_dyn[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  PtWarp& w = reinterpret_cast<PtWarp*>(s_dyn)[warp];
  const int E = d.n_events;
  const int n_tiles = d.pt_ev[E].tile0;
  const int cap_q = d.cap_queue;
  const float inv = d.cuts.inv_2rmin, gtol = d.cuts.pt_gate_tol;
  // the circle test of phase 1a bounds the gate limit at |w| + h, which needs a limit growing with |w|
  const bool can_prune = inv >= 0.0f && gtol >= 0.0f;
  // warp-aggregated append to the queue of the exact cuts
  auto push_q = [&](bool go, int p, int cand) {
    const unsigned m = __ballot_sync(kFull, go);
    if (m == 0u) return;
    int base = 0;
    if (lane == __ffs(m) - 1) base = atomicAdd(&d.ctl->queue_cur, __popc(m));
    base = __shfl_sync(kFull, base, __ffs(m) - 1);
    const int pos = base + __popc(m & ((1u << lane) - 1u));
    if (go && pos < cap_q) d.pt_queue[pos] = make_int2(p, cand);
  };
  for (;;) {
    unsigned near3 = 0, near5 = 0;  // candidates failing the gate near its threshold, this tile (one event)
    int tile = 0, evi = 0;
    if (lane == 0) {
      tile = atomicAdd(d.ctl->ticket + T_PT, 1);
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
      const float4 a = d.seed_a[p0 + k], b = d.seed_b[p0 + k];
      const float c1 = b.x * inv, c2 = b.x * gtol;
      w.sa[k] = a;
      w.sg[k] = make_float4(c1 + 1e-4f * fabsf(c1), c2 + 1e-4f * fabsf(c2), c1 - 1e-4f * fabsf(c1), c2 - 1e-4f * fabsf(c2));
      w.sk[k] = make_float2(b.y, b.z);
    }
    const int anc = ev.a0 + ab * 32 + lane;
    const bool valid = anc < ev.a1;
    float4 A = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    int4 at = make_int4(0, 0, 0, 0);
    if (valid) {
      A = d.anc_a[anc];
      at = d.anc_t[anc];
    }
    w.anc[lane] = A;
    w.at[lane] = at;
    __syncwarp();
    // ---- (3) the rest of the approximate cascade for one entry of w2; what survives goes to the queue ----
    auto tail = [&](int2 ent, bool active) {
      bool go = false;
      const int t = ent.x & 0x7fffffff, ks = ent.y & 0xffff, src = (ent.y >> 16) & 31;
      const bool is5 = ent.x < 0;
      if (active) {
        const float4 s = w.sa[ks];
        const float2 kt = w.sk[ks];
        const float4 a = w.anc[src];
        const float4 l = is5 ? d.t5_l[t] : d.t3_l[t];
        bool ok;
        const float kx = kx_approx(s.x, s.y, a.x, a.y, l.x, l.y, ok);
        int c = pt_class_curv(kx, kt.x, kt.y, ok);
        if (c == PT_PASS) {
          if (is5) {
            const float2 kio = d.t5_kio[t];
            c = pt_class_curv(kx, kio.x, kt.y, ok);
            if (c == PT_PASS) c = pt_class_curv(kx, kio.y, kt.y, ok);
          } else {
            c = pt_class_curv(kx, d.t3_k[t], kt.y, ok);
          }
        }
        if (c == PT_PASS) {
          const float z1 = d.seed_z1[p0 + ks], slope = d.seed_b[p0 + ks].w;
          c = pt_class_rz(d.cuts, s.x, s.y, z1, slope, kx, a, ok);
          if (c == PT_PASS) c = pt_class_rz(d.cuts, s.x, s.y, z1, slope, kx, l, ok);
        }
        go = c != PT_FAIL;  // all cuts surely pass, or one of them cannot be decided here: the exact cuts decide
      }
      push_q(go, p0 + ks, ent.x);
    };
    int n2 = 0;
    // pushes up to one entry per lane onto w2; runs the cascade whenever 32 are waiting
    auto push2 = [&](bool go, int cand, int tag) {
      const unsigned m = __ballot_sync(kFull, go);
      if (m == 0u) return;
      if (go) w.w2[n2 + __popc(m & ((1u << lane) - 1u))] = make_int2(cand, tag);
      n2 += __popc(m);
      if (n2 >= 32) {
        __syncwarp();
        tail(w.w2[lane], true);
        const int2 rest = (32 + lane < n2) ? w.w2[32 + lane] : make_int2(0, 0);
        __syncwarp();
        w.w2[lane] = rest;
        n2 -= 32;
        __syncwarp();
      }
    };
    // ---- (2) expansion of up to 32 gate survivors into their (seed, T3) / (seed, T5) candidates, flattened
    // over the lanes; kx~ against the seed's curvature decides which go on ----
    auto expand = [&](int n_ent) {
      int n_c = 0;
      if (lane < n_ent) {
        const int4 a = w.at[(w.w1[lane] >> 16) & 31];
        n_c = a.y + a.w;
      }
      const int incl = warp_incl_scan(n_c);
      const int excl = incl - n_c;
      w.pref[lane] = excl;
      const int T = __shfl_sync(kFull, incl, 31);
      // item -> entry in O(1): one head bit per entry at the position of its first item; the entry of item
      // `it` = number of head bits at or before it, minus one (bisection beyond 1024 items)
      w.heads[lane] = 0u;
      __syncwarp();
      if (n_c > 0 && excl < 1024) atomicOr(&w.heads[excl >> 5], 1u << (excl & 31));
      __syncwarp();
      int heads_before = 0;
      for (int i0 = 0; i0 < T; i0 += 32) {
        const int it = i0 + lane;
        bool go = false, direct = false;
        int cand = 0, tag = 0;
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
          const int src = (ent >> 16) & 31, ks = ent & 0xffff, c = it - w.pref[lo];
          const int4 a = w.at[src];
          const bool is5 = c >= a.y;
          const int t = is5 ? a.z + (c - a.y) : a.x + c;
          cand = t | (is5 ? 0x80000000 : 0);
          tag = ks | (src << 16);
          if (ent >> 31) {
            direct = true;  // the gate was near its threshold: every candidate of the pair is flagged by the exact cuts
          } else {
            const float4 s = w.sa[ks];
            const float2 kt = w.sk[ks];
            const float4 an = w.anc[src];
            const float2 l = *reinterpret_cast<const float2*>(is5 ? d.t5_l + t : d.t3_l + t);
            bool ok;
            const float kx = kx_approx(s.x, s.y, an.x, an.y, l.x, l.y, ok);
            go = pt_class_curv(kx, kt.x, kt.y, ok) != PT_FAIL;
          }
        }
        heads_before += __popc(hw);
        push_q(direct, p0 + (tag & 0xffff), cand);
        push2(go, cand, tag);
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
    // ---- (1) 32 seeds at a time ----
    for (int kb = 0; kb < n_seed && warp_has; kb += 32) {
      // (1a) one seed per lane against the circle: can its gate accept ANY point within bh of the centre?
      //      gdot(A) <= v.wc + lv bh, gcrs(A) >= |v x wc| - lv bh, glim(A) <= glim at |wc| + bh (c1h, c2h >= 0
      //      here); the 1e-4 inflation of c1h, c2h and the 1.001 factors cover the rounding of both sides.
      //      Out of range: tested by every lane.
      bool maybe = false;
      if (kb + lane < n_seed) {
        const float4 s = w.sa[kb + lane];
        const float4 g = w.sg[kb + lane];
        const float wx = bcx - s.x, wy = bcy - s.y;
        const float lw2 = wx * wx + wy * wy;
        const float Lw = (lw2 * rsqrt_approx(lw2) + bh) * 1.001f;
        const float lv2 = s.z * s.z + s.w * s.w;
        const float lvh = lv2 * rsqrt_approx(lv2) * 1.001f;
        const float slack = lvh * (bh * 1.001f + 1e-4f);
        const float dotc = s.z * wx + s.w * wy;
        const float crsc = fabsf(s.z * wy - s.w * wx);
        const bool in_range = lw2 >= 1e-30f && lw2 <= 1e30f && lv2 >= 1e-30f && lv2 <= 1e30f;
        maybe = !can_prune || !in_range || (dotc + slack > 0.0f && crsc - slack <= Lw * (Lw * g.x + g.y));
      }
      unsigned word = __ballot_sync(kFull, maybe);
      // (1b) the seeds that may match: every lane tests its own anchor
      while (word) {
        const int k = kb + __ffs(word) - 1;
        word &= word - 1;
        bool pass = false;
        unsigned ent = 0u;
        if (valid) {
          const float4 s = w.sa[k];
          const float4 g = w.sg[k];
          const float wx = A.x - s.x, wy = A.y - s.y;
          const float gdot = s.z * wx + s.w * wy;          // exactly the spec's gdot and gcrs (no FMA)
          const float gcrs = fabsf(s.z * wy - s.w * wx);
          const float lw2 = fmaf(wx, wx, wy * wy);
          const float lw = lw2 * rsqrt_approx(lw2);
          // three outcomes: surely rejected (dropped), surely accepted and not near-threshold (the exact gate
          // is skipped), uncertain = within 1e-4 of the threshold or out of the approximation's range (NaN
          // limits compare false both ways): the exact gate decides
          pass = gdot > 0.0f && !(gcrs > lw * fmaf(lw, g.x, g.y));
          if (pass && !(gcrs <= lw * fmaf(lw, g.z, g.w) && lw2 >= 1e-30f && lw2 <= 1e30f)) {
            Seed sd;
            sd.x1 = s.x;  sd.y1 = s.y;  sd.vx = s.z;  sd.vy = s.w;  sd.lv = d.seed_b[p0 + k].x;
            const unsigned r = pt_gate(d.cuts, sd, A.x, A.y);
            pass = (r & ACC) != 0;
            if (!pass && (r & NEAR)) {  // every candidate of the anchor fails the gate near its threshold
              near3 += (unsigned)at.y;
              near5 += (unsigned)at.w;
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
    if (n2 > 0) {
      __syncwarp();
      tail(lane < n2 ? w.w2[lane] : make_int2(0, 0), lane < n2);
    }
    if (__any_sync(kFull, (near3 | near5) != 0u)) {
      const int s3 = warp_sum((int)near3), s5 = warp_sum((int)near5);
      if (lane == 0) {
        if (s3) atomicAdd(d.ev_cnt + (size_t)evi * kEvCnt + 4, (unsigned long long)s3);
        if (s5) atomicAdd(d.ev_cnt + (size_t)evi * kEvCnt + 5, (unsigned long long)s5);
      }
    }
    __syncwarp();  // the tile's tables are reused
  }
}

// The exact cut list of CUTS.md section 7 on the queue.  Accepted pairs go to scratch lists (one atomic per
// accepted object) with a count per seed; near-threshold flags are counted here (and, for pairs failing the
// gate near its threshold, in k_pt_eval).
__global__ void __launch_bounds__(kBlock) k_pt_exact(Dev d) {
  load_batch(d);
  const int n_q = d.ctl->queue_cur;
  const int cap3 = d.cap[K_PT3], cap5 = d.cap[K_PT5];
  PtAccepted* scratch3 = reinterpret_cast<PtAccepted*>(d.ev_scratch);
  PtAccepted* scratch5 = reinterpret_cast<PtAccepted*>(d.ev_scratch2);
  if (n_q > d.cap_queue) {  // the queue holds the accepted pairs and the few undecided ones: capacity error
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(&d.ctl->error, E_CAP_PT3 | E_CAP_PT5);
    return;
  }
  const int lane = threadIdx.x & 31;
  for (int i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; i0 < n_q; i0 += gridDim.x * blockDim.x) {
    const int i = i0 + lane;  // whole warps stay in the loop: the scratch slots are taken with one atomic per warp and class
    bool is5 = false;
    unsigned r = 0;
    PtAccepted acc{0, 0, 0.0f};
    if (i < n_q) {
      const int2 q = d.pt_queue[i];
      acc.p = q.x;
      acc.t = q.y & 0x7fffffff;
      is5 = q.y < 0;
      const Seed s = seed_from_table(d, acc.p);
      r = is5 ? PtCand<true>::test(d, s, acc.t, acc.score) : PtCand<false>::test(d, s, acc.t, acc.score);
      if (r & NEAR) count_near(d.ev_cnt, d.pls_event[acc.p], is5 ? 5 : 4);
    }
    const unsigned m3 = __ballot_sync(kFull, (r & ACC) && !is5), m5 = __ballot_sync(kFull, (r & ACC) && is5);
    int b3 = 0, b5 = 0;
    if (lane == 0) {
      if (m3) b3 = atomicAdd(&d.ctl->scratch_cur[2], __popc(m3));
      if (m5) b5 = atomicAdd(&d.ctl->scratch_cur[3], __popc(m5));
    }
    b3 = __shfl_sync(kFull, b3, 0);
    b5 = __shfl_sync(kFull, b5, 0);
    if (r & ACC) {
      const unsigned below = (1u << lane) - 1u;
      const int slot = is5 ? b5 + __popc(m5 & below) : b3 + __popc(m3 & below);
      if (slot < (is5 ? cap5 : cap3)) (is5 ? scratch5 : scratch3)[slot] = acc;
      atomicAdd((is5 ? d.pls_pt5_cnt : d.pls_pt3_cnt) + acc.p, 1);
    }
  }
}

}  // namespace lst
