// lst_ls.cuh -- step a2: Line Segments (CUTS.md section 4).
//
// Candidates of an inner MD A: the MDs of every module in conn[module(A)] (the CSR row of the
// precomputed connection map).  A PU200 batch holds 2.1e5 MDs, rows of 7.7 targets on average and
// 1.4 MDs per target: 5e6 candidate pairs.  All inner MDs of a module share the same candidates, so the
// unit of work is the MODULE (the "thread group per module" of north_star, here a warp):
//   * a warp takes kLsModules modules by ticket and handles the non-empty ones one by one;
//   * the module's row is walked ONCE: lanes = targets, their MD ranges are concatenated (prefix sum) and
//     taken 32 at a time, one candidate B per lane, its operands loaded into registers;
//   * the module's inner MDs are then a warp-uniform loop (A broadcast, no pair decoding): the first cut
//     of the approximate list (ls_class: curvature) runs here and drops 73 % of the pairs;
//   * survivors queue up (across modules) and take the rest of ls_class, then the exact cuts of CUTS.md
//     section 4, on full warps; accepted (A, B, kappa) go to a scratch list with one atomic per 32 LSs and
//     a count per inner MD;
//   * k_ls_place scans the per-MD counts into md_ls_begin (tiles by ticket + look-back), waits until every
//     tile is done, and moves the LSs to their slot (one cursor per inner MD).
// LSs therefore sit grouped by inner MD (what T3 building looks up); the order inside an MD's range
// is free (reading S9).
#pragma once
#include "lst_md.cuh"

namespace lst {

constexpr int kLsRanges = 256;  // longest connection-map row accepted by lst_load_geometry
constexpr int kLsModules = 4;   // modules per ticket (the non-empty ones are handled one after the other); fewer in small batches
constexpr int kLsStride = 1187; // module-index distance between the modules of a ticket

struct LsAccepted {
  int A, B;
  float kappa;
};

struct LsWarp {    // per-warp scratch in shared memory
  int pref[33];    // exclusive prefix of the MD counts of the round's 32 targets
  int b0[32];      // first MD of each target | endcap(target) << 30
  int2 q1[64];     // pairs behind the curvature cut: (A, B | endcap(B) << 30)
  int2 q2[64];     // pairs the approximate list could not reject
  LsAccepted acc[64];
};

__global__ void __launch_bounds__(kBlock) k_ls_eval(Dev d) {
  load_batch(d);
  __shared__ LsWarp s_w[kWarps];
  __shared__ unsigned s_tests[2 * kEvSmem];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned below = (1u << lane) - 1u;
  LsWarp& w = s_w[warp];
  EvTests tbl;
  tbl.init(s_tests, d.ev_cnt, 1, d.n_events);
  const bool on = (d.cuts.stage_mask & 2) != 0;
  const int n_gm = on && d.ctl->total[K_MD] > 0 ? d.n_events * d.n_mod : 0;
  const int cap = d.cap[K_LS];
  LsAccepted* scratch = reinterpret_cast<LsAccepted*>(d.ev_scratch);
  int n1 = 0, n2 = 0, n3 = 0;  // entries waiting in q1, q2, acc
  // ---- accepted LSs -> scratch list (one atomic per flush) and the count of their inner MD ----
  auto flush = [&](int n_now) {
    int base = 0;
    if (lane == 0) base = atomicAdd(&d.ctl->scratch_cur[1], n_now);
    base = __shfl_sync(kFull, base, 0);
    if (lane < n_now) {
      const LsAccepted a = w.acc[lane];
      if (base + lane < cap) scratch[base + lane] = a;
      atomicAdd(d.ls_cnt + a.A, 1);
    }
  };
  // ---- the exact cuts of CUTS.md section 4 on up to 32 queued pairs ----
  auto exact = [&](int n_now) {
    unsigned res = 0;
    LsAccepted a{0, 0, 0.0f};
    if (lane < n_now) {
      const int2 q = w.q2[lane];
      a.A = q.x;
      a.B = q.y & 0x3fffffff;
      const int infoA = d.md_info[a.A];
      res = ls_test(d.cuts, d.md_a[a.A], d.md_u[a.A], infoA & 1, d.md_a[a.B], d.md_u[a.B], (q.y >> 30) & 1, a.kappa);
      if (res & NEAR) count_near(d.ev_cnt, (infoA >> 1) / d.n_mod, 1);
    }
    const unsigned m = __ballot_sync(kFull, res & ACC);
    if (m == 0u) return;
    if (res & ACC) w.acc[n3 + __popc(m & below)] = a;
    n3 += __popc(m);
    __syncwarp();
    if (n3 >= 32) {
      flush(32);
      const LsAccepted rest = (32 + lane < n3) ? w.acc[32 + lane] : a;
      __syncwarp();
      w.acc[lane] = rest;
      n3 -= 32;
      __syncwarp();
    }
  };
  // ---- the approximate cut list (ls_class) on up to 32 pairs behind the curvature cut ----
  auto second = [&](int n_now) {
    bool go = false;
    int2 q = make_int2(0, 0);
    if (lane < n_now) {
      q = w.q1[lane];
      const int B = q.y & 0x3fffffff;
      go = ls_class(d.cuts, d.md_a[q.x], d.md_u[q.x], d.md_info[q.x] & 1, d.md_a[B], d.md_u[B], (q.y >> 30) & 1) != PT_FAIL;
    }
    const unsigned m = __ballot_sync(kFull, go);
    if (m == 0u) return;
    if (go) w.q2[n2 + __popc(m & below)] = q;
    n2 += __popc(m);
    __syncwarp();
    if (n2 >= 32) {
      exact(32);
      const int2 rest = (32 + lane < n2) ? w.q2[32 + lane] : q;
      __syncwarp();
      w.q2[lane] = rest;
      n2 -= 32;
      __syncwarp();
    }
  };
  // modules per ticket: kLsModules, fewer when that leaves less than two tickets per warp (a small batch)
  const int mpt = max(1, min(kLsModules, n_gm / (2 * (int)gridDim.x * kWarps)));
  const int n_tickets = (n_gm + mpt - 1) / mpt;
  for (;;) {
    int ticket = 0;
    if (lane == 0) ticket = atomicAdd(d.ctl->ticket + T_LSE, 1);
    ticket = __shfl_sync(kFull, ticket, 0);
    if (ticket >= n_tickets) break;
    // ---- kLsModules modules, one per lane, from different parts of the module table (neighbouring modules,
    // and the same module in different events, are equally busy: a ticket gets a mix); the non-empty ones
    // are handled one by one ----
    const int gm_l = lane * n_tickets + (int)(((long long)ticket + (long long)lane * kLsStride) % n_tickets);
    int A0_l = 0, A1_l = 0;
    if (lane < mpt && gm_l < n_gm) {
      A0_l = d.mod_md_begin[gm_l];
      A1_l = d.mod_md_begin[gm_l + 1];
    }
    unsigned todo = __ballot_sync(kFull, A1_l > A0_l);
    while (todo) {
      const int src = __ffs(todo) - 1;
      todo &= todo - 1;
      const int gm = __shfl_sync(kFull, gm_l, src);
      const int A0 = __shfl_sync(kFull, A0_l, src), A1 = __shfl_sync(kFull, A1_l, src);
      const int ev = gm / d.n_mod, gb = ev * d.n_mod, mod = gm - gb;
      const int k0 = __ldg(d.conn_off + mod), deg = __ldg(d.conn_off + mod + 1) - k0;
      for (int r0 = 0; r0 < deg; r0 += 32) {
        // ---- the row, 32 targets at a time: lanes = targets, their MD ranges concatenated ----
        int n_t = 0, ent = 0;
        if (r0 + lane < deg) {
          const int m2 = __ldg(d.conn_tgt + k0 + r0 + lane);
          const int B0 = d.mod_md_begin[gb + m2];
          n_t = d.mod_md_begin[gb + m2 + 1] - B0;
          ent = B0 | ((__ldg(d.subdet + m2) != 0) << 30);
        }
        const int incl = warp_incl_scan(n_t);
        const int NB = __shfl_sync(kFull, incl, 31);
        if (NB == 0) continue;
        __syncwarp();
        w.pref[lane] = incl - n_t;
        w.b0[lane] = ent;
        if (lane == 31) w.pref[32] = NB;
        __syncwarp();
        if (lane == 0) {  // candidates of CUTS.md section 4: (MDs of the module) x (MDs of its targets)
          const unsigned long long t64 = (unsigned long long)(A1 - A0) * (unsigned long long)NB;
          if (t64 < (1ull << 32)) tbl.add(ev, (unsigned)t64);
          else atomicAdd(d.ev_cnt + (size_t)ev * kEvCnt + kStages + 1, t64);
        }
        for (int c0 = 0; c0 < NB; c0 += 32) {
          // ---- one candidate B per lane: target = the last list starting at or before c0 + lane ----
          const int i = c0 + lane;
          const bool has = i < NB;
          int lo = 0;
#pragma unroll
          for (int step = 16; step > 0; step >>= 1)
            if (w.pref[lo + step] <= i) lo += step;
          const int e = w.b0[lo];
          const int B = has ? (e & 0x3fffffff) + (i - w.pref[lo]) : A0;
          const int tagB = B | (e & 0x40000000);
          const float4 b = d.md_a[B];
          // ---- the module's inner MDs, warp-uniform: first cut of ls_class (|kappa| R_MIN <= LS_KAPPA_MAX), same
          // arithmetic and band; a pair is dropped only if that cut surely fails ----
          for (int A = A0; A < A1; ++A) {
            const float4 a = __ldg(d.md_a + A);
            const float ex = b.x - a.x, ey = b.y - a.y;
            const float c2 = fmaf(ex, ex, ey * ey);
            const float crs = a.x * b.y - a.y * b.x;
            const float rr = a.w * b.w;
            const float den2 = (rr * rr) * c2;
            const bool ok = den2 >= 1e-30f && den2 <= 1e30f && c2 >= 1e-30f && c2 <= 1e30f && rr >= 0.0f;
            const float kv = fabsf((2.0f * crs) * rsqrt_approx(den2)) * d.cuts.r_min;
            const bool go = has && classify(kv, d.cuts.ls_kappa_max, 2e-5f * fabsf(d.cuts.ls_kappa_max) + 3e-6f * kv, ok) != PT_FAIL;
            const unsigned m = __ballot_sync(kFull, go);
            if (m == 0u) continue;
            if (go) w.q1[n1 + __popc(m & below)] = make_int2(A, tagB);
            n1 += __popc(m);
            __syncwarp();
            if (n1 >= 32) {
              second(32);
              const int2 rest = (32 + lane < n1) ? w.q1[32 + lane] : make_int2(0, 0);
              __syncwarp();
              w.q1[lane] = rest;
              n1 -= 32;
              __syncwarp();
            }
          }
        }
      }
    }
  }
  // ---- drain the queues ----
  if (n1 > 0) second(n1);
  if (n2 > 0) exact(n2);
  if (n3 > 0) flush(n3);
  tbl.flush();
}

// Placement.  Phase 1: exclusive scan of ls_cnt into md_ls_begin (tiles of kBlock inner MDs by ticket, block
// scan + look-back); rides along: the four list heads of every MD of the duplicate-removal index are
// cleared.  Phase 2, once every tile is done (all tiles are taken by running blocks before any block gets
// here, so the wait cannot deadlock): every LS of the scratch list goes to the next free slot of its inner MD.
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
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) atomicAdd(&d.ctl->ls_tiles_done, 1);
  }
  if (!fits) return;
  if (threadIdx.x == 0) {
    while (atomicAdd(&d.ctl->ls_tiles_done, 0) < n_tiles) __nanosleep(64);
    __threadfence();
  }
  __syncthreads();
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
    const LsAccepted s = scratch[i];
    const int pos = __ldcg(d.md_ls_begin + s.A) + atomicAdd(d.ls_cur + s.A, 1);
    d.ls_md[pos] = make_int2(s.A, s.B);
    d.ls_kappa[pos] = s.kappa;
  }
}

}  // namespace lst
