// lst_pt.cuh -- step a5: pLS x T3 -> pT3 and pLS x T5 -> pT5 (CUTS.md section 7).
// Candidates of a seed = every T3 / T5 of its event (the direction gate of the spec replaces the IT->OT
// connection map): ~1.2e8 (seed, T3) + 2.5e7 (seed, T5) pairs per 16-event PU200 batch, of which 8 % pass
// the gate, 0.9 % the curvature match with the seed and 0.06 % are accepted.  Structure:
//   * anchors: the gate depends only on the seed and the FIRST MD of the candidate, and T3s / T5s are stored
//     grouped by first MD, so the gate is evaluated once per (seed, anchor) and shared by pT3 and pT5;
//     anchors are sorted into radius x azimuth bins (lst_stages.cuh, k_anchor_sort), which also writes the
//     bounding circle of every block of 32 sorted anchors and of its four sub-blocks of 8, and the seeds of
//     every event in azimuth order (seed_perm);
//   * k_pt_eval, tile = 32 seeds consecutive in azimuth (one per LANE, their constants in registers) x
//     kPtBlocks anchor blocks:
//     (1a) every lane tests its seed against the bounding circle of the block, then of each sub-block;
//     (1b) the anchors of a surviving sub-block are walked one by one (broadcast from shared memory): a
//          necessary condition of the gate with |A - P1| from rsqrt.approx; only within 1e-4 of the threshold
//          the exact gate decides (and flags near-threshold);
//     (2)  the anchor's T3s and T5s in a warp-uniform loop -- one broadcast load per candidate, no index
//          decoding: kx~ (lst_cuts_pt.cuh) against the seed's curvature and, behind a sure pass of that cut,
//          against the candidate's stored curvature(s);
//     (3)  the rest of the approximate cascade (r-z at both ends) on full warps of survivors;
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

constexpr int kPtBlocks = 2;           // anchor blocks (of 32 sorted anchors) per tile; 1 when that leaves fewer than kPtMinTiles tiles
constexpr int kPtMinTiles = 12288;     // about two tiles per resident warp of k_pt_eval
constexpr int kSeedSectors = 128;       // azimuth sectors of the seed sort
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

// azimuth sector of the point where the straight line through the seed's two pixel hits reaches r ~ 35 cm
// (diamond angle, as anchor_bin): only the ORDER of the seeds in k_pt_eval depends on it, never a result
__device__ __forceinline__ int seed_sector(float4 sa) {
  const float x = sa.x + 7.0f * sa.z, y = sa.y + 7.0f * sa.w;
  const float a = fabsf(x) + fabsf(y);
  const float t = a > 0.0f ? y / a : 0.0f;
  const float ps = x >= 0.0f ? (y >= 0.0f ? t : 4.0f + t) : 2.0f - t;  // [0, 4)
  int sec = (int)(ps * (kSeedSectors / 4));
  return sec < 0 ? 0 : (sec > kSeedSectors - 1 ? kSeedSectors - 1 : sec);
}

// Counting sort of an event's anchors by bin (the counts and arrival ranks come from the T5 kernel's
// prologue).  grid = n_events * kAncBlocksPerEvent; every block scans the 512 bin counts of its event in
// shared memory and places its share of the event's MDs; the anchors of event e start at the event's
// first MD (an event has no more anchors than MDs), so no prefix across events is needed.  The last block
// of an event also sorts the event's seeds by azimuth sector (seed_perm).  Block 0 also writes the
// per-event table of k_pt_eval (ranges, tile prefix) and the candidate counts of stages 4, 5.
__global__ void __launch_bounds__(kBlock) k_anchor_sort(Dev d) {
  load_batch(d);
  __shared__ int s_begin[kAncBins];
  __shared__ int s_warp[kWarps];
  __shared__ int s_sec[kSeedSectors];
  __shared__ int s_secw[kSeedSectors / 32];
  __shared__ int s_last;
  const int E = d.n_events;
  const int e = blockIdx.x / kAncBlocksPerEvent, part = blockIdx.x - e * kAncBlocksPerEvent;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool on = (d.cuts.stage_mask & 16) && d.ctl->total[K_T3] > 0 && d.n_pls > 0;
  const bool on5 = d.ctl->total[K_T5] > 0;
  if (on && e < E) {
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
    // ---- the last of the event's blocks to get here: bounding circles (x, y, h) of every block of 32 sorted
    // anchors and of its four sub-blocks of 8, at anc_c[5 * ((md0 >> 5) + e + block)] (ranges of different
    // events cannot overlap: an event has no more anchors than MDs) ----
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(d.anc_done + e, 1) == kAncBlocksPerEvent - 1;
    __syncthreads();
    if (s_last) {
      __threadfence();
      const int n_a = s_begin[kAncBins - 1] + d.anc_bin_cnt[e * kAncBins + kAncBins - 1];
      const int n_blk = (n_a + 31) / 32;
      float4* out = d.anc_c + 5 * (size_t)((md0 >> 5) + e);
      auto circ_of = [](float x0, float x1, float y0, float y1) {
        return make_float4(0.5f * (x0 + x1), 0.5f * (y0 + y1),
                           0.5f * sqrtf((x1 - x0) * (x1 - x0) + (y1 - y0) * (y1 - y0)) * 1.001f + 1e-3f, 0.0f);
      };
      constexpr int U = 4;  // blocks in flight per warp (independent load + shuffle chains)
      for (int b0 = warp * U; b0 < n_blk; b0 += kWarps * U) {
        float x0[U], x1[U], y0[U], y1[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
          const bool valid = (b0 + u) * 32 + lane < n_a;
          float4 A = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
          if (valid) A = __ldcg(d.anc_a + md0 + (b0 + u) * 32 + lane);
          x0[u] = valid ? A.x : 3e38f;  x1[u] = valid ? A.x : -3e38f;
          y0[u] = valid ? A.y : 3e38f;  y1[u] = valid ? A.y : -3e38f;
        }
#pragma unroll
        for (int sh = 1; sh < 32; sh <<= 1) {
#pragma unroll
          for (int u = 0; u < U; ++u) {
            if (sh == 8 && (lane & 7) == 0 && b0 + u < n_blk)
              out[5 * (b0 + u) + 1 + (lane >> 3)] = circ_of(x0[u], x1[u], y0[u], y1[u]);
            x0[u] = fminf(x0[u], __shfl_xor_sync(kFull, x0[u], sh));
            x1[u] = fmaxf(x1[u], __shfl_xor_sync(kFull, x1[u], sh));
            y0[u] = fminf(y0[u], __shfl_xor_sync(kFull, y0[u], sh));
            y1[u] = fmaxf(y1[u], __shfl_xor_sync(kFull, y1[u], sh));
          }
        }
#pragma unroll
        for (int u = 0; u < U; ++u)
          if (lane == 0 && b0 + u < n_blk) out[5 * (b0 + u)] = circ_of(x0[u], x1[u], y0[u], y1[u]);
      }
    }
    if (part == kAncBlocksPerEvent - 1) {
      // ---- the event's seeds in azimuth order: counting sort over kSeedSectors sectors ----
      const int s0 = d.pls_ev_off[e], s1 = d.pls_ev_off[e + 1];
      if (threadIdx.x < kSeedSectors) s_sec[threadIdx.x] = 0;
      __syncthreads();
      for (int p = s0 + threadIdx.x; p < s1; p += kBlock) atomicAdd(&s_sec[seed_sector(d.seed_a[p])], 1);
      __syncthreads();
      int cs = 0, is = 0;
      if (threadIdx.x < kSeedSectors) {
        cs = s_sec[threadIdx.x];
        is = warp_incl_scan(cs);
        if (lane == 31) s_secw[warp] = is;
      }
      __syncthreads();
      if (threadIdx.x < kSeedSectors) {
        int base2 = 0;
        for (int w = 0; w < warp; ++w) base2 += s_secw[w];
        s_sec[threadIdx.x] = base2 + is - cs;
      }
      __syncthreads();
      for (int p = s0 + threadIdx.x; p < s1; p += kBlock)
        d.seed_perm[s0 + atomicAdd(&s_sec[seed_sector(d.seed_a[p])], 1)] = p;
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
      pe.tile0 = 0;  // first tile: prefix below
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
  if (threadIdx.x == 0) {  // blocks per tile, and the exclusive prefix of the tile counts (n_events is small)
    auto tiles_of = [&](int ev, int K) {
      const PtEvent pe = d.pt_ev[ev];
      const int n_blk = (pe.a1 - pe.a0 + 31) / 32, ns = on ? pe.s1 - pe.s0 : 0;
      return ((n_blk + K - 1) / K) * ((ns + 31) / 32);
    };
    long long t2 = 0;
    for (int ev = 0; ev < E; ++ev) t2 += tiles_of(ev, kPtBlocks);
    const int K = t2 >= kPtMinTiles ? kPtBlocks : 1;  // a small batch: shorter tiles, more warps busy
    int a = 0;
    for (int ev = 0; ev < E; ++ev) {
      const int ta = tiles_of(ev, K);
      d.pt_ev[ev].tile0 = a;
      a += ta;
    }
    d.pt_ev[E].tile0 = a;
    d.pt_ev[E].a0 = K;
  }
}

struct PtAccepted {
  int p, t;
  float score;
};

struct PtWarp {  // per-warp scratch of k_pt_eval (dynamic shared memory: kWarps of these)
  float4 anc[32];  // the anchors of the current block (x, y, z, r | endcap << 31)
  int4 at[32];     // (first T3, number of T3s, first T5, number of T5s) of each
  int4 w2[64];     // candidates behind the curvature pre-filter: (T3 / T5 index | T5 flag << 31, seed, anchor position in anc_a, 0)
};

// pT3 and pT5 candidates of the whole batch -> queue of the exact cuts.  tile = 32 seeds of one event
// (consecutive in azimuth order, one per LANE, their constants in registers) x kPtBlocks blocks of 32
// sorted anchors; warps take tiles by ticket and never wait for one another.  Per block: every lane tests
// its seed against the bounding circle of the block's anchors; if any lane may match, the block's anchors
// are walked one by one (anchor data broadcast from shared memory): gate per lane, then the anchor's T3s
// and T5s in a warp-uniform loop (one broadcast load per candidate, no index decoding) with kx~ against
// the seed's and the candidate's stored curvatures.
__global__ void __launch_bounds__(kBlock) k_pt_eval(Dev d) {
  load_batch(d);
  extern __shared__ __align__(16) unsigned char s_dyn[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  PtWarp& w = reinterpret_cast<PtWarp*>(s_dyn)[warp];
  const int E = d.n_events;
  const int n_tiles = d.pt_ev[E].tile0;
  const int K = d.pt_ev[E].a0;  // anchor blocks per tile (k_anchor_sort)
  const int cap_q = d.cap_queue;
  const float inv = d.cuts.inv_2rmin, gtol = d.cuts.pt_gate_tol;
  // the circle test bounds the gate limit at |w| + h, which needs a limit growing with |w|
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
  // ---- (3) the rest of the approximate cascade for one entry of w2; what survives goes to the queue ----
  auto tail = [&](int4 ent, bool active) {
    bool go = false;
    if (active) {
      const int t = ent.x & 0x7fffffff;
      const bool is5 = ent.x < 0;
      const float4 s = d.seed_a[ent.y], sb = d.seed_b[ent.y];  // sb = lv, kp, tolk, slope
      const float4 a = d.anc_a[ent.z];
      const float4 l = is5 ? d.t5_l[t] : d.t3_l[t];
      bool ok;
      const float kx = kx_approx(s.x, s.y, a.x, a.y, l.x, l.y, ok);
      int c = pt_class_curv(kx, sb.y, sb.z, ok);
      if (c == PT_PASS) {
        if (is5) {
          const float2 kio = d.t5_kio[t];
          c = pt_class_curv(kx, kio.x, sb.z, ok);
          if (c == PT_PASS) c = pt_class_curv(kx, kio.y, sb.z, ok);
        } else {
          c = pt_class_curv(kx, d.t3_k[t], sb.z, ok);
        }
      }
      if (c == PT_PASS) {
        const float z1 = d.seed_z1[ent.y];
        c = pt_class_rz(d.cuts, s.x, s.y, z1, sb.w, kx, a, ok);
        if (c == PT_PASS) c = pt_class_rz(d.cuts, s.x, s.y, z1, sb.w, kx, l, ok);
      }
      go = c != PT_FAIL;  // all cuts surely pass, or one of them cannot be decided here: the exact cuts decide
    }
    push_q(go, ent.y, ent.x);
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
    const int n_blk = (ev.a1 - ev.a0 + 31) / 32;
    const int n_ch = (n_blk + K - 1) / K;
    const int local = tile - ev.tile0;
    const int sg = local / n_ch, ch = local - sg * n_ch;
    const int cbase = (ev.a0 >> 5) + evi;  // first bounding circle of the event's anchor blocks (k_anchor_sort)
    // ---- this lane's seed (CUTS.md section 7: the per-seed quantities) ----
    const int si = ev.s0 + sg * 32 + lane;
    const bool has_seed = si < ev.s1;
    const int p = d.seed_perm[has_seed ? si : ev.s1 - 1];
    const float4 sa = d.seed_a[p], sgc = d.seed_g[p];
    const float x1 = sa.x, y1 = sa.y, vx = sa.z, vy = sa.w;
    // gate limit glim = lw (lw c1 + c2), c1 = lv INV_2RMIN, c2 = lv PT_GATE_TOL (both >= 0 when can_prune);
    // loaded, not computed here, so that they stay in registers
    const float c1 = sgc.x, c2 = sgc.y, kp = sgc.z, tolk = sgc.w;
    const float lv2 = vx * vx + vy * vy;
    const float lvh = lv2 * rsqrt_approx(lv2) * 1.001f;
    const bool v_in_range = lv2 >= 1e-30f && lv2 <= 1e30f;
    const float tband = 1.2e-5f * fabsf(tolk);  // pt_class_curv's band = tband + 4e-6 |kx~|
    int n2 = 0;
    // pushes up to one entry per lane onto w2; runs the cascade whenever 32 are waiting
    auto push2 = [&](bool go, int cand, int anc_pos) {
      const unsigned m = __ballot_sync(kFull, go);
      if (m == 0u) return;
      if (go) w.w2[n2 + __popc(m & ((1u << lane) - 1u))] = make_int4(cand, p, anc_pos, 0);
      n2 += __popc(m);
      if (n2 >= 32) {
        __syncwarp();
        tail(w.w2[lane], true);
        const int4 rest = (32 + lane < n2) ? w.w2[32 + lane] : make_int4(0, 0, 0, 0);
        __syncwarp();
        w.w2[lane] = rest;
        n2 -= 32;
        __syncwarp();
      }
    };
    const int b_end = min(n_blk, (ch + 1) * K);
    for (int b = ch * K; b < b_end; ++b) {
      const int anc0 = ev.a0 + b * 32;
      const int nb = min(32, ev.a1 - anc0);
      // ---- (1a) lanes as seeds: can this seed's gate accept ANY point within h of the centre (cx, cy)?
      //      gdot(A) <= v.wc + lv h, gcrs(A) >= |v x wc| - lv h, glim(A) <= glim at |wc| + h (c1, c2 >= 0
      //      here); the 1e-4 inflation of the limit and the 1.001 factors cover the rounding of both sides.
      //      Out of range: every anchor is tested.  First the bounding circle of the block (k_anchor_sort),
      //      then those of its four sub-blocks of 8 consecutive anchors. ----
      auto circle = [&](float4 c) {
        const float wx = c.x - x1, wy = c.y - y1;
        const float lw2 = wx * wx + wy * wy;
        const float Lw = (lw2 * rsqrt_approx(lw2) + c.z) * 1.001f;
        const float slack = lvh * (c.z * 1.001f + 1e-4f);
        const float dotc = vx * wx + vy * wy;
        const float crsc = fabsf(vx * wy - vy * wx);
        const bool in_range = lw2 >= 1e-30f && lw2 <= 1e30f && v_in_range;
        return !can_prune || !in_range || (dotc + slack > 0.0f && crsc - slack <= (Lw * (Lw * c1 + c2)) * 1.0001f);
      };
      const float4* __restrict__ circ = d.anc_c + 5 * (size_t)(cbase + b);
      const bool maybe_b = has_seed && circle(__ldg(circ));
      if (!__any_sync(kFull, maybe_b)) continue;
      __syncwarp();
      if (lane < nb) {  // lanes as anchors: the block goes to shared memory
        w.anc[lane] = d.anc_a[anc0 + lane];
        w.at[lane] = d.anc_t[anc0 + lane];
      }
      __syncwarp();
      // ---- (1b) the block's anchors one by one: gate of CUTS.md section 7 for this lane's seed ----
      for (int j0 = 0; j0 < nb; j0 += 8) {
        // a sub-block is skipped if no seed of the warp can match any of its anchors
        const bool maybe = maybe_b && circle(__ldg(circ + 1 + (j0 >> 3)));
        if (!__any_sync(kFull, maybe)) continue;
        const int j1 = min(nb, j0 + 8);
        for (int j = j0; j < j1; ++j) {
          const float4 Aj = w.anc[j];
          const int4 tj = w.at[j];
          const float wx = Aj.x - x1, wy = Aj.y - y1;
          const float gdot = vx * wx + vy * wy;          // exactly the spec's gdot and gcrs (no FMA)
          const float gcrs = fabsf(vx * wy - vy * wx);
          const float lw2 = fmaf(wx, wx, wy * wy);
          const float lw = lw2 * rsqrt_approx(lw2);
          // three outcomes: surely rejected (dropped), surely accepted and not near-threshold (the exact gate
          // is skipped), uncertain = within 1e-4 of the threshold or out of the approximation's range (NaN
          // limits compare false both ways): the exact gate decides
          const float G = lw * fmaf(lw, c1, c2);  // >= 0 when can_prune; within 1e-6 of the spec's glim
          bool pass = maybe && gdot > 0.0f && !(can_prune && gcrs > G * 1.0001f);
          const bool sure = can_prune && gcrs <= G * 0.9999f && lw2 >= 1e-30f && lw2 <= 1e30f;
          if (!__any_sync(kFull, pass)) continue;
          bool gnear = false;
          if (__any_sync(kFull, pass && !sure)) {
            if (pass && !sure) {
              Seed sd;
              sd.x1 = x1;  sd.y1 = y1;  sd.vx = vx;  sd.vy = vy;  sd.lv = d.seed_b[p].x;
              const unsigned r = pt_gate(d.cuts, sd, Aj.x, Aj.y);
              pass = (r & ACC) != 0;
              gnear = (r & NEAR) != 0;
              if (!pass && gnear) {  // every candidate of the anchor fails the gate near its threshold
                near3 += (unsigned)tj.y;
                near5 += (unsigned)tj.w;
              }
            }
            // the gate passed near its threshold: every candidate of the pair is flagged by the exact cuts
            unsigned dm = __ballot_sync(kFull, pass && gnear);
            while (dm) {
              const int src = __ffs(dm) - 1;
              dm &= dm - 1;
              const int pp = __shfl_sync(kFull, p, src);
              for (int c0 = 0; c0 < tj.y + tj.w; c0 += 32) {
                const int c = c0 + lane;
                const bool in = c < tj.y + tj.w;
                push_q(in, pp, c < tj.y ? tj.x + c : (tj.z + (c - tj.y)) | 0x80000000);
              }
            }
          }
          const bool active = pass && !gnear;
          // ---- (2) the anchor's T3s, then its T5s: kx~ (lst_cuts_pt.cuh) with a = A - P1 and |a|^2 from the
          // gate, one broadcast load per candidate.  A candidate is dropped if its curvature match with the seed
          // surely fails, or -- behind a sure pass of that cut -- the match with its own stored curvature(s)
          // surely fails (pt_class_curv's bands, written out as predicates); NaNs drop nothing. ----
          const float4* __restrict__ q3 = d.t3_q + tj.x;
          for (int c = 0; c < tj.y; ++c, ++q3) {
            const float4 q = __ldg(q3);  // last MD x, y; k3; |AL|^2
            const float cx = q.x - x1, cy = q.y - y1;
            const float crs = wx * cy - wy * cx;  // the spec's crs (no FMA contraction in this translation unit)
            const float prod = (lw2 * q.w) * fmaf(cx, cx, cy * cy);
            const float kx = (crs + crs) * rsqrt_approx(prod);
            const float band = fmaf(fabsf(kx), 4e-6f, tband);
            const float hi = tolk + band, lo = tolk - band;
            const float dp = fabsf(kx - kp), dt = fabsf(kx - q.z);
            const bool ok = prod >= 1e-30f && prod <= 1e30f;
            const bool drop = ok && (dp > hi || (dp < lo && dt > hi));
            push2(active && !drop, tj.x + c, anc0 + j);
          }
          const float4* __restrict__ l5 = d.t5_l + tj.z;
          const float2* __restrict__ k5 = d.t5_kio + tj.z;
          for (int c = 0; c < tj.w; ++c, ++l5, ++k5) {
            const float2 l = __ldg(reinterpret_cast<const float2*>(l5));
            const float2 kio = __ldg(k5);
            const float bx = l.x - Aj.x, by = l.y - Aj.y;
            const float cx = l.x - x1, cy = l.y - y1;
            const float crs = wx * cy - wy * cx;
            const float prod = (lw2 * fmaf(bx, bx, by * by)) * fmaf(cx, cx, cy * cy);
            const float kx = (crs + crs) * rsqrt_approx(prod);
            const float band = fmaf(fabsf(kx), 4e-6f, tband);
            const float hi = tolk + band, lo = tolk - band;
            const float dp = fabsf(kx - kp), di = fabsf(kx - kio.x), dq = fabsf(kx - kio.y);
            const bool ok = prod >= 1e-30f && prod <= 1e30f;
            const bool drop = ok && (dp > hi || (dp < lo && (di > hi || (di < lo && dq > hi))));
            push2(active && !drop, (tj.z + c) | 0x80000000, anc0 + j);
          }
        }
      }
    }
    if (n2 > 0) {
      __syncwarp();
      tail(lane < n2 ? w.w2[lane] : make_int4(0, 0, 0, 0), lane < n2);
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
