// lst_md.cuh -- step a1: Mini-Doublets (CUDA transcription of CUTS.md section 3).
//
// Candidates of an upper-sensor hit b: the hits of the lower sensor of the same module (a contiguous
// range of the sorted hits, just before the module's upper range).  1.4e7 hit pairs per PU200 batch,
// 1.5 % accepted.  One LANE per upper hit, the lower hits are walked in a plain loop: no pair
// decoding, no ballot per step (the even-split pair engine spent 100 of its 151 instructions per 32
// pairs on those; profiles/).  Lanes of a warp hold consecutive upper hits, i.e. hits of the same or
// neighbouring modules, so their loops have similar lengths (the hot layer-1 modules fill whole warps)
// and their loads hit the same cache lines.
//   * k_md_eval: a warp takes windows of 64 sorted hits, queues the upper-sensor ones (ballot), and
//     whenever 32 are waiting every lane tests one against its module's lower hits; the positions of the first
//     kMdStash accepted lower hits are stashed per upper hit, the count is exact;
//   * k_md_place scans the counts (fused, look-back) and writes each upper hit's MDs (re-evaluating only
//     the rare hit with more than kMdStash MDs) and the first MD of every module.
#pragma once
#include "lst_stages.cuh"

namespace lst {

constexpr int kMdStash = 4;  // stashed MDs per upper hit

__global__ void __launch_bounds__(kBlock) k_md_eval(Dev d) {
  load_batch(d);
  __shared__ int s_own[kWarps][96];
  __shared__ unsigned s_tests[2 * kEvSmem];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int n = (d.cuts.stage_mask & 1) ? d.n_hits : 0;
  EvTests tbl;
  tbl.init(s_tests, d.ev_cnt, 0, d.n_events);
  // candidates of CUTS.md section 3 per event: (lower hits) x (upper hits) of every module (consecutive
  // threads take consecutive modules, i.e. one event: one shared-memory update per warp)
  if (n > 0) {
    const int n_gm = d.n_events * d.n_mod;
    for (int g0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31; g0 < n_gm; g0 += gridDim.x * blockDim.x) {
      const int gm = g0 + lane;
      unsigned t = 0u;
      if (gm < n_gm) {
        const int s0 = __ldg(d.sens_begin + 2 * gm), s1 = __ldg(d.sens_begin + 2 * gm + 1), s2 = __ldg(d.sens_begin + 2 * gm + 2);
        const unsigned long long t64 = (unsigned long long)(s1 - s0) * (unsigned long long)(s2 - s1);
        if (t64 < (1ull << 26)) {
          t = (unsigned)t64;
        } else {  // a module with > 6.7e7 hit pairs: straight to global memory (the warp sum above stays < 2^32)
          atomicAdd(d.ev_cnt + (size_t)(gm / d.n_mod) * kEvCnt + kStages, t64);
        }
      }
      tbl.warp_add(min(gm, n_gm - 1) / d.n_mod, t);
    }
  }
  // one round: up to 32 queued upper hits, one per lane, each against its module's lower hits
  auto round = [&](int n_now) {
    int i = -1, a = 0, a1 = 0, endcap = 0, ev = 0;
    float4 hb = make_float4(0.f, 0.f, 0.f, 0.f);
    if (lane < n_now) {
      i = s_own[warp][lane];
      const int gs = hit_ig(d, i).y;
      const int gm = gs >> 1;
      ev = gm / d.n_mod;
      a = __ldg(d.sens_begin + gs - 1);
      a1 = __ldg(d.sens_begin + gs);
      endcap = __ldg(d.subdet + (gm - ev * d.n_mod)) != 0;
      hb = hit_xyzr(d, i);
    }
    int cnt = 0, near = 0;
    int stash[kMdStash];
#pragma unroll
    for (int k = 0; k < kMdStash; ++k) stash[k] = 0;
    for (; a < a1; ++a) {
      const float4 ha = hit_xyzr(d, a);
      int cl = md_class(d.cuts, endcap, ha, hb);  // sqrt- and division-free; the exact cuts only where it cannot decide
      if (cl == PT_UNSURE) {
        float ux, uy;
        const unsigned r = md_test(d.cuts, endcap, ha, hb, ux, uy);
        near += (r >> 1) & 1u;
        cl = (r & ACC) ? PT_PASS : PT_FAIL;
      }
      if (cl == PT_PASS) {
#pragma unroll
        for (int k = 0; k < kMdStash; ++k)
          if (cnt == k) stash[k] = a;
        ++cnt;
      }
    }
    if (near) atomicAdd(d.ev_cnt + (size_t)ev * kEvCnt + 0, (unsigned long long)near);
    if (i >= 0) {
      d.md_cnt[i].x = cnt;
      reinterpret_cast<int4*>(d.md_stash)[i] = make_int4(stash[0], stash[1], stash[2], stash[3]);
    }
  };
  int n_q = 0;  // upper hits waiting in s_own (always < 32 between windows, so 96 slots suffice)
  for (int w0 = (blockIdx.x * kWarps + warp) * 64; w0 < d.n_hits; w0 += gridDim.x * kWarps * 64) {
    // ---- the upper-sensor hits of the window join the queue, in order ----
    const int i0 = w0 + lane, i1 = w0 + 32 + lane;
    const int gs0 = i0 < n ? hit_ig(d, i0).y : 0, gs1 = i1 < n ? hit_ig(d, i1).y : 0;
    const unsigned m0 = __ballot_sync(kFull, gs0 & 1), m1 = __ballot_sync(kFull, gs1 & 1);
    const int n0 = __popc(m0);
    if (gs0 & 1) s_own[warp][n_q + __popc(m0 & ((1u << lane) - 1u))] = i0;
    if (gs1 & 1) s_own[warp][n_q + n0 + __popc(m1 & ((1u << lane) - 1u))] = i1;
    // (MDs owned, global sensor) of every hit, for k_md_place: lower-sensor hits own no MD, the count of an
    // upper-sensor hit follows from its round
    if (i0 < d.n_hits) d.md_cnt[i0] = make_int2(0, gs0);
    if (i1 < d.n_hits) d.md_cnt[i1] = make_int2(0, gs1);
    n_q += n0 + __popc(m1);
    __syncwarp();
    while (n_q >= 32) {  // full rounds only; the remainder waits for the next window
      round(32);
      const int r0 = (32 + lane < n_q) ? s_own[warp][32 + lane] : 0;
      const int r1 = (64 + lane < n_q) ? s_own[warp][64 + lane] : 0;
      __syncwarp();
      s_own[warp][lane] = r0;
      s_own[warp][32 + lane] = r1;
      n_q -= 32;
      __syncwarp();
    }
  }
  if (n_q > 0) round(n_q);
  tbl.flush();
}

// Placement with the exclusive scan of md_cnt fused in (tiles of kBlock * kMdPlaceItems sorted hits taken
// by ticket, block scan + decoupled look-back): the MDs of upper hit i go to the running offset, in
// lower-hit order, so MDs end up grouped by module.  The thread of the FIRST hit after a module boundary
// also writes mod_md_begin for the modules that start there (empty modules in between included); gaps
// longer than kMdGapSerial modules (sparse batches) are filled by the whole block.
constexpr int kMdPlaceItems = 4;
constexpr int kMdGapSerial = 16;
constexpr int kMdBigGaps = 16;

__global__ void __launch_bounds__(kBlock) k_md_place(Dev d) {
  load_batch(d);
  static_assert(kMdStash == 4, "the stash is stored as one int4 per hit");
  constexpr int kTile = kBlock * kMdPlaceItems;
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  __shared__ int s_nbig;
  __shared__ int s_big[kMdBigGaps][3];  // (first module, one past the last, offset)
  const bool on = (d.cuts.stage_mask & 1) != 0;
  const int n = on ? d.n_hits : 0;
  const int cap = d.cap[K_MD];
  const int n_gm = d.n_events * d.n_mod;
  const int n_tiles = n > 0 ? (n + kTile - 1) / kTile : 1;
  // mod_md_begin[g0 .. g1) = off
  auto fill = [&](int g0, int g1, int off) {
    if (g1 - g0 <= kMdGapSerial) {
      for (int g = g0; g < g1; ++g) d.mod_md_begin[g] = off;
      return;
    }
    const int slot = atomicAdd(&s_nbig, 1);
    if (slot < kMdBigGaps) {
      s_big[slot][0] = g0;  s_big[slot][1] = g1;  s_big[slot][2] = off;
    } else {
      for (int g = g0; g < g1; ++g) d.mod_md_begin[g] = off;
    }
  };
  for (;;) {
    if (threadIdx.x == 0) {
      s_tile = atomicAdd(d.ctl->ticket + T_MD, 1);
      s_nbig = 0;
    }
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int i0 = tile * kTile + threadIdx.x * kMdPlaceItems;
    int cnt[kMdPlaceItems], gsv[kMdPlaceItems], sum = 0;
#pragma unroll
    for (int k = 0; k < kMdPlaceItems; ++k) {
      const int2 cg = (i0 + k < n) ? d.md_cnt[i0 + k] : make_int2(0, 0);
      cnt[k] = cg.x;
      gsv[k] = cg.y;
      sum += cnt[k];
    }
    int tb, tt;
    int pos = tile_alloc(sum, d.tstate[T_MD], tile, s_scan, tb, tt);
    int gm_prev = (i0 > 0 && i0 <= n) ? (d.md_cnt[i0 - 1].y >> 1) : -1;
#pragma unroll
    for (int k = 0; k < kMdPlaceItems; ++k) {
      const int i = i0 + k;
      if (i >= n) break;
      const int gs = gsv[k], gm = gs >> 1;
      if (gm != gm_prev) fill(gm_prev + 1, gm + 1, pos);  // the modules that begin at hit i
      gm_prev = gm;
      if (cnt[k] == 0) continue;
      const int2 ib = hit_ig(d, i);
      const int endcap = __ldg(d.subdet + (gm - (gm / d.n_mod) * d.n_mod)) != 0;
      const float4 hb = hit_xyzr(d, i);
      auto emit = [&](int a) {  // unit direction exactly as in md_test (CUTS.md section 3)
        if (pos < cap) {
          const float4 ha = hit_xyzr(d, a);
          float ux = 0.0f, uy = 0.0f;
          if (!endcap) {
            const float dx = hb.x - ha.x, dy = hb.y - ha.y;
            const float dd = sqrtf(dx * dx + dy * dy);
            ux = dx / dd;
            uy = dy / dd;
          }
          d.md_hit[pos] = make_int2(hit_ig(d, a).x, ib.x);
          d.md_info[pos] = (gs - 1) | endcap;
          d.md_a[pos] = ha;
          d.md_u[pos] = make_float2(ux, uy);
        }
        ++pos;
      };
      if (cnt[k] <= kMdStash) {
        const int4 st = reinterpret_cast<const int4*>(d.md_stash)[i];
        emit(st.x);
        if (cnt[k] > 1) emit(st.y);
        if (cnt[k] > 2) emit(st.z);
        if (cnt[k] > 3) emit(st.w);
      } else {  // rare: more MDs than the stash holds -> evaluate this hit's candidates again
        const int a1 = __ldg(d.sens_begin + gs);
        for (int a = __ldg(d.sens_begin + gs - 1); a < a1; ++a) {
          float ux, uy;
          if (md_test(d.cuts, endcap, hit_xyzr(d, a), hb, ux, uy) & ACC) emit(a);
        }
      }
    }
    const int total = tb + tt;
    if (tile == n_tiles - 1) {
      // the modules after the last hit (all of them when there is no hit), and the totals
      const int last = n - 1 - tile * kTile;  // position of the last hit in this tile, -1 = no hit at all
      if (n == 0 ? threadIdx.x == 0 : (last / kMdPlaceItems == threadIdx.x)) fill(n == 0 ? 0 : gm_prev + 1, n_gm + 1, total);
      if (threadIdx.x == 0) {
        if (total > cap) {
          atomicOr(&d.ctl->error, E_CAP_MD);
          d.ctl->total[K_MD] = 0;
        } else {
          d.ctl->total[K_MD] = total;
        }
      }
    }
    __syncthreads();
    const int nbig = min(s_nbig, kMdBigGaps);
    for (int b = 0; b < nbig; ++b)
      for (int g = s_big[b][0] + threadIdx.x; g < s_big[b][1]; g += kBlock) d.mod_md_begin[g] = s_big[b][2];
    __syncthreads();  // s_nbig / s_big are reset by the next tile
  }
}

}  // namespace lst
