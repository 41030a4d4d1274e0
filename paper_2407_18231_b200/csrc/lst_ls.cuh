// lst_ls.cuh -- step a2: Line Segments (CUTS.md section 4).
//
// Candidates of an inner MD A: the MDs of every module in conn[module(A)] (the CSR row of the
// precomputed connection map).  A PU200 batch holds 2.1e5 MDs, rows of 7.7 targets on average and
// 1.4 MDs per target: 5e6 candidate pairs in 1.6e6 tiny (MD, target) lists.  Flattening the pairs of
// the whole batch (an earlier engine, profiles/r01_v2_even_split.md) costs more in decoding (pair -> module -> MD -> row edge -> B: ~290 thread
// instructions per pair, ncu) than the cuts themselves (~40), because a 32-pair step crosses a
// module boundary almost every time.  Here the unit is the list:
//   * a warp takes 8 consecutive inner MDs and builds, once, the table of their (MD, target) lists
//     in shared memory (first candidate, length prefix): the CSR walk is done once per list;
//   * the ~180 candidate pairs of the 8 MDs are then taken 32 at a time (pair -> list through a
//     bit mask of list starts, inner-MD operands from shared memory), so lanes stay busy
//     whatever the list lengths; accepted (B, kappa) pairs are compacted in pair order with one
//     ballot per step and copied to a scratch list with one atomic per warp pass (a pass with more
//     than kLsStage LSs evaluates its pairs again and writes directly);
//   * k_ls_place scans the per-MD counts into md_ls_begin (fused, look-back) and copies each MD's LSs to their slot.
// LSs therefore sit grouped by inner MD (what T3 building looks up); the order inside an MD's range
// is free (reading S9).
#pragma once
#include "lst_md.cuh"

namespace lst {

constexpr int kLsOwners = 8;    // inner MDs per warp
constexpr int kLsRanges = 256;  // (MD, target) lists per warp pass; also the longest row supported
constexpr int kLsStage = 96;    // staged LSs per warp pass
constexpr int kLsHeadWords = 64;

struct LsAccepted {
  int B;
  float kappa;
};

struct LsWarp {  // per-warp scratch in shared memory
  float4 a[kLsOwners];
  float2 u[kLsOwners];
  int e[kLsOwners];
  int cnt[kLsOwners];
  int dex[kLsOwners + 1];  // exclusive prefix of the row lengths
  int k0[kLsOwners];
  int gb[kLsOwners];       // event * n_mod
  int pref[kLsRanges + 1];  // exclusive prefix of the list lengths
  int b0[kLsRanges];        // first MD of the list | endcap(target) << 27 | owner slot << 28
  unsigned heads[kLsHeadWords];  // bit p set = a list starts at pair p (pairs below 32 * kLsHeadWords)
  int2 cq[64];                   // pairs the pre-filter could not reject: (B, owner slot | endcap(B) << 8), in pair order
  LsAccepted stage[kLsStage];
};

__global__ void __launch_bounds__(kBlock) k_ls_eval(Dev d) {
  load_batch(d);
  __shared__ LsWarp s_w[kWarps];
  __shared__ unsigned s_tests[2 * kEvSmem];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  LsWarp& w = s_w[warp];
  EvTests tbl;
  tbl.init(s_tests, d.ev_cnt, 1, d.n_events);
  const bool on = (d.cuts.stage_mask & 2) != 0;
  const int n_md = d.ctl->total[K_MD];
  const int cap = d.cap[K_LS];
  LsAccepted* scratch = reinterpret_cast<LsAccepted*>(d.ev_scratch);
  for (int A0 = (blockIdx.x * kWarps + warp) * kLsOwners; A0 < n_md; A0 += gridDim.x * kWarps * kLsOwners) {
    // ---- lanes 0..7: one inner MD each ----
    const int A = A0 + lane;
    int k0 = 0, deg = 0, gm_base = 0;
    if (lane < kLsOwners && A < n_md && on) {
      const int info = d.md_info[A];
      const int gm = info >> 1;
      const int ev = gm / d.n_mod;
      w.a[lane] = d.md_a[A];
      w.u[lane] = d.md_u[A];
      w.e[lane] = info & 1;
      k0 = __ldg(d.conn_off + (gm - ev * d.n_mod));
      deg = __ldg(d.conn_off + (gm - ev * d.n_mod) + 1) - k0;
      gm_base = ev * d.n_mod;
    }
    const int dincl = warp_incl_scan(deg);  // rows of the 8 MDs, concatenated
    if (lane < kLsOwners) {
      w.dex[lane] = dincl - deg;
      w.k0[lane] = k0;
      w.gb[lane] = gm_base;
    }
    if (lane == kLsOwners - 1) w.dex[kLsOwners] = dincl;
    __syncwarp();
    int first = 0;                          // MDs [first, first + take) are handled per pass
    while (first < kLsOwners) {
      const int d_first = w.dex[first];
      // as many MDs as fit the range table (a single row always fits: lst_load_geometry checks)
      const unsigned fit = __ballot_sync(kFull, lane >= first && lane < kLsOwners && dincl - d_first <= kLsRanges);
      const int take = __popc(fit >> first & ~((fit >> first) + 1u)) ;  // length of the run of ones starting at `first`
      const int last = first + take;  // exclusive
      const int R = w.dex[last] - d_first;
      const bool one_event = w.gb[first] == w.gb[last - 1];  // the MDs of the pass belong to one event (nearly always)
      if (lane < kLsOwners) w.cnt[lane] = 0;
      // ---- table of the non-empty lists (owner, target e) in row order, and their head bits ----
      for (int k = lane; k < kLsHeadWords; k += 32) w.heads[k] = 0u;
      __syncwarp();
      int carry = 0, Rn = 0;
      for (int r0 = 0; r0 < R; r0 += 32) {
        const int r = r0 + lane;
        int n_t = 0, ent = 0;
        if (r < R) {
          int o = first;  // owner slot of list r: last o with (dex[o] - d_first) <= r
          for (int k = first + 1; k < last; ++k)
            if (w.dex[k] - d_first <= r) o = k;
          const int e = r - (w.dex[o] - d_first);
          const int m2 = __ldg(d.conn_tgt + w.k0[o] + e);
          const int gb = w.gb[o];
          const int B0 = d.mod_md_begin[gb + m2];
          n_t = d.mod_md_begin[gb + m2 + 1] - B0;
          ent = B0 | ((__ldg(d.subdet + m2) != 0) << 27) | (o << 28);
          if (!one_event) tbl.add(gb / d.n_mod, (unsigned)n_t);
        }
        const int incl = warp_incl_scan(n_t);
        const unsigned nz = __ballot_sync(kFull, n_t > 0);
        if (n_t > 0) {
          const int idx = Rn + __popc(nz & ((1u << lane) - 1u));
          const int start = carry + incl - n_t;
          w.pref[idx] = start;
          w.b0[idx] = ent;
          if (start < 32 * kLsHeadWords) atomicOr(&w.heads[start >> 5], 1u << (start & 31));
        }
        Rn += __popc(nz);
        carry += __shfl_sync(kFull, incl, 31);
      }
      const int P = carry;
      if (lane == 0) w.pref[Rn] = P;
      __syncwarp();
      if (one_event && lane == 0) tbl.add(w.gb[first] / d.n_mod, (unsigned)P);
      // ---- pairs of the pass, 32 at a time: the approximate cut list (ls_class) drops 95 % of them; the rest
      // queue up in pair order and take the exact cuts of CUTS.md section 4 on full warps.  Pass 1 runs only
      // if the stage overflowed: it evaluates the pairs again and writes straight to the scratch list. ----
      int base = 0, run = 0;
      for (int pass = 0; pass < 2; ++pass) {
        run = 0;
        int heads_before = 0, n_c = 0;
        auto exact = [&](int n_now) {  // lanes below n_now take one queued pair each
          unsigned res = 0;
          LsAccepted acc;
          int o = 0;
          if (lane < n_now) {
            const int2 q = w.cq[lane];
            o = q.y & 0xff;
            acc.B = q.x;
            res = ls_test(d.cuts, w.a[o], w.u[o], w.e[o] != 0, d.md_a[acc.B], d.md_u[acc.B], (q.y >> 8) & 1, acc.kappa);
          }
          if (pass == 0 && (res & NEAR)) count_near(d.ev_cnt, w.gb[o] / d.n_mod, 1);
          const unsigned m = __ballot_sync(kFull, res & ACC);
          if (res & ACC) {
            const int pos = run + __popc(m & ((1u << lane) - 1u));
            if (pass == 0) {
              if (pos < kLsStage) w.stage[pos] = acc;
              atomicAdd(&w.cnt[o], 1);
            } else if (base + pos < cap) {
              scratch[base + pos] = acc;
            }
          }
          run += __popc(m);
        };
        for (int p0 = 0; p0 < P; p0 += 32) {
          const int p = p0 + lane;
          bool go = false;
          int2 q = make_int2(0, 0);
          const unsigned hw = p0 < 32 * kLsHeadWords ? w.heads[p0 >> 5] : 0u;
          if (p < P) {
            int lo;  // list of pair p: the last list starting at or before p
            if (p0 < 32 * kLsHeadWords) {
              lo = heads_before + __popc(hw & (0xffffffffu >> (31 - lane))) - 1;
            } else {
              lo = 0;
              int hi = Rn;
              while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (w.pref[mid] <= p) lo = mid; else hi = mid;
              }
            }
            const int ent = w.b0[lo];
            const int o = (unsigned)ent >> 28, eB = (ent >> 27) & 1;
            q.x = (ent & 0x7ffffff) + (p - w.pref[lo]);
            q.y = o | (eB << 8);
            go = ls_class(d.cuts, w.a[o], w.u[o], w.e[o] != 0, d.md_a[q.x], d.md_u[q.x], eB != 0) != PT_FAIL;
          }
          heads_before += __popc(hw);
          const unsigned m = __ballot_sync(kFull, go);
          if (m == 0u) continue;
          if (go) w.cq[n_c + __popc(m & ((1u << lane) - 1u))] = q;
          n_c += __popc(m);
          if (n_c >= 32) {
            __syncwarp();
            exact(32);
            const int2 rest = (32 + lane < n_c) ? w.cq[32 + lane] : make_int2(0, 0);
            __syncwarp();
            w.cq[lane] = rest;
            n_c -= 32;
            __syncwarp();
          }
        }
        if (n_c > 0) {
          __syncwarp();
          exact(n_c);
        }
        if (pass == 1) break;
        // ---- one atomic for the pass; per-MD count and scratch position ----
        if (lane == 0 && run > 0) base = atomicAdd(&d.ctl->scratch_cur[1], run);
        base = __shfl_sync(kFull, base, 0);
        __syncwarp();
        const int c = (lane >= first && lane < last) ? w.cnt[lane] : 0;
        const int cincl = warp_incl_scan(c);
        if (lane >= first && lane < last && A < n_md) {
          d.ls_cnt[A] = c;
          d.ls_sbase[A] = base + cincl - c;
        }
        if (run <= kLsStage) {
          for (int k = lane; k < run; k += 32)
            if (base + k < cap) scratch[base + k] = w.stage[k];
          break;
        }
      }
      __syncwarp();  // the tables are reused by the next pass
      first = last;
    }
  }
  tbl.flush();
}

// Placement with the exclusive scan of ls_cnt fused in (tiles of kBlock inner MDs by ticket, block scan +
// look-back): every MD's LSs go from the scratch list to their final slot, md_ls_begin is written on the
// way.  Rides along: the four list heads of every MD of the duplicate-removal index are cleared.
__global__ void __launch_bounds__(kBlock) k_ls_place(Dev d) {
  load_batch(d);
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  const int n_md = d.ctl->total[K_MD];
  const int total = d.ctl->scratch_cur[1];
  const int cap = d.cap[K_LS];
  const bool fits = total <= cap;
  const int n_tiles = n_md > 0 ? (n_md + kBlock - 1) / kBlock : 1;
  const LsAccepted* scratch = reinterpret_cast<const LsAccepted*>(d.ev_scratch);
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(d.ctl->ticket + T_LS, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int A = tile * kBlock + threadIdx.x;
    const int n = (A < n_md && fits) ? d.ls_cnt[A] : 0;
    int tb, tt;
    const int dst = tile_alloc(n, d.tstate[T_LS], tile, s_scan, tb, tt);
    if (A < n_md) {
      d.md_ls_begin[A] = dst;
      d.idx_head[A] = 0;
      d.idx_head[n_md + A] = 0;
      d.idx_head[2 * n_md + A] = 0;
      d.idx_head[3 * n_md + A] = 0;
      const int src = d.ls_sbase[A];
      for (int k = 0; k < n; ++k) {
        const LsAccepted s = scratch[src + k];
        d.ls_md[dst + k] = make_int2(A, s.B);
        d.ls_kappa[dst + k] = s.kappa;
      }
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) {
      d.md_ls_begin[n_md] = tb + tt;
      if (!fits) {
        atomicOr(&d.ctl->error, E_CAP_LS);
        d.ctl->total[K_LS] = 0;
      } else {
        d.ctl->total[K_LS] = total;
      }
    }
  }
}

}  // namespace lst
