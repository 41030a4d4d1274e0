// lst_pairs.cuh -- the evenly split candidate-pair engine of the MD and LS stages.
//
// A stage is "group -> (owners x candidates) -> accepted subset": for Mini-Doublets the group is a
// module of one event (upper hits x lower hits), for Line Segments a module (its MDs x the MDs of
// the modules its connection-map row lists).  Pair counts per group differ by 100x (a layer-1
// barrel module holds ~1000 hit pairs, an outer endcap module a handful), so neither
// thread-per-owner nor warp-per-group keeps the machine busy (profiles/r01_v1_first_path.md: 10 of
// 32 lanes active; r01 notes: warp-per-module stalls the look-back chain behind hot modules).
//
// Here the candidate pairs of the whole batch form ONE index space: a pre-pass scans the pair
// counts of the groups (k_scan_f) and records, for every chunk of kChunk = 256 pairs, the group
// its first pair falls in.  k_even gives every warp exactly one chunk (8 steps of 32 consecutive
// pairs; lanes walk pair -> group -> (owner, candidate) with a division by the group's row
// length), so all warps do the same amount of work whatever the occupancy pattern.  Accepted
// pairs are compacted in pair order with one ballot per step into the warp's shared-memory
// staging area, which holds a full chunk: every pair is evaluated exactly once and nothing can
// overflow.  A tile (8 chunks) gets its output slots from the decoupled look-back of
// lst_scan.cuh, so objects stay in (group, owner, candidate) order -- deterministic and
// contiguous per owner, module and event -- with no global atomics on the data path.  The
// begin-offsets of groups and owners ("first object of module m / of MD A") are ranks of pair
// indices, answered from the staged pair numbers by the tile that holds the pair.
#pragma once
#include "lst_ingest.cuh"

namespace lst {

constexpr int kChunk = 256;                  // pairs per warp
constexpr int kTilePairs = kChunk * kWarps;  // pairs per block-tile

// Exclusive scan of a computed sequence: out[i] = sum_{j<i} F.count(j), i in [0, n]; out[n] =
// total.  For every chunk c whose first pair c * kChunk lies in item i's range, chunk_g0[c] =
// F.group(i).  The 64-bit sum of all counts goes to *total64 (overflow check of the consumer).
// F.count() must not exceed d.cap_pairs (a larger group count is an overflow: F flags it, returns 0).
template <class F>
__global__ void __launch_bounds__(kBlock) k_scan_f(Dev d, int* __restrict__ out, int* __restrict__ chunk_g0,
                                                   unsigned long long* total64, int ticket_id) {
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  F f(d);
  const int n = f.n_items();
  const int n_tiles = (n + kScanTile - 1) / kScanTile > 0 ? (n + kScanTile - 1) / kScanTile : 1;
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(d.ctl->ticket + ticket_id, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int base_i = tile * kScanTile + threadIdx.x * kScanItems;
    int v[kScanItems];
    int sum = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
      v[k] = (base_i + k < n) ? f.count(base_i + k) : 0;
      sum += v[k];
    }
    int tb, tt;
    int off = tile_alloc(sum, d.tstate[ticket_id], tile, s_scan, tb, tt);
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
      if (base_i + k < n) {
        out[base_i + k] = off;
        if (v[k] > 0) {
          const int grp = f.group(base_i + k);
          const int c_end = min((off + v[k] + kChunk - 1) / kChunk, d.cap_pairs / kChunk + 1);
          for (int c = (off + kChunk - 1) / kChunk; c < c_end; ++c) chunk_g0[c] = grp;
        }
      }
      off += v[k];
    }
    const unsigned long long s64 = warp_sum_u64((unsigned long long)sum);  // exact even if the int scan wrapped
    if ((threadIdx.x & 31) == 0 && s64) atomicAdd(total64, s64);
    if (tile == n_tiles - 1 && threadIdx.x == 0) out[n] = tb + tt;
  }
}

// p = o * n_c + j with 0 <= j < n_c (float reciprocal + integer fix-up below 2^24)
__device__ __forceinline__ void split_pair(int p, int n_c, int& o, int& j) {
  if (p >= (1 << 24)) {
    o = p / n_c;
    j = p - o * n_c;
    return;
  }
  o = __float2int_rz(__fdividef(__int2float_rn(p), __int2float_rn(n_c)));
  j = p - o * n_c;
  if (j < 0) { --o; j += n_c; }
  if (j >= n_c) { ++o; j -= n_c; }
}

// Answers "how many accepted pairs of the batch have a pair index < x" for x inside this tile.
struct TileRank {
  const int* woff;                         // [kWarps + 1] global slot of each warp's first object
  const int* run;                          // [kWarps] accepted pairs per warp
  const unsigned short (*q)[kChunk];       // staged pair numbers relative to the tile start
  int ts;
  __device__ int operator()(int x) const {
    const int rel = x - ts;
    const int w = rel / kChunk;
    if (w >= kWarps) return woff[kWarps];
    int lo = 0, hi = run[w];  // first staged entry with q >= rel
    while (lo < hi) {
      const int mid = (lo + hi) >> 1;
      if ((int)q[w][mid] < rel) lo = mid + 1; else hi = mid;
    }
    return woff[w] + lo;
  }
};

// Stage concept (StageMD / StageLS in lst_stages.cuh):
//   static constexpr int kTicket, kKind, kErr, kStage, kPairSlot;
//   struct Group { int gbase, gend; ... };  struct Payload;
//   int  n_groups() const;  const int* chunk_g0() const;
//   int  pp(int g) const;                         // exclusive pair prefix of group g, g in [0, n]
//   void load_group(int g, Group&) const;         // per lane: row length n_c and what test() needs
//   unsigned test(const Group&, int o, int j, Payload&) const;     // ACC | NEAR bits
//   void emit(int pos, const Payload&) const;
//   void boundaries(int tile, bool only_tile, int g_lo, int g_hi, int ts, int te, const TileRank&) const;
//   void finish_total(int total) const;
template <class S>
__global__ void __launch_bounds__(kBlock) k_even(Dev d) {
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  __shared__ int s_woff[kWarps + 1];
  __shared__ int s_run[kWarps];
  __shared__ unsigned short s_q[kWarps][kChunk];
  __shared__ typename S::Payload s_stage[kWarps][kChunk];
  S st(d);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int n = st.n_groups();
  const unsigned long long tp64 = n > 0 ? d.ctl->pair_total[S::kPairSlot] : 0ull;
  const bool too_many = tp64 > (unsigned long long)d.cap_pairs;
  const int TP = too_many ? 0 : (int)tp64;
  const int n_tiles = TP > 0 ? (TP + kTilePairs - 1) / kTilePairs : 1;
  const int cap = d.cap[S::kKind];
  unsigned long long near = 0;
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(d.ctl->ticket + S::kTicket, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int ts = tile * kTilePairs, te = min(TP, ts + kTilePairs);
    const int cs = ts + warp * kChunk;
    // ---- this warp's chunk: every pair once, accepted pairs staged in pair order ----
    int run = 0;
    if (cs < te) {
      typename S::Group G;
      int g = st.chunk_g0()[tile * kWarps + warp];  // group holding pair cs
      G.gbase = st.pp(g);
      G.gend = st.pp(g + 1);
      st.load_group(g, G);
#pragma unroll 1
      for (int s = 0; s < kChunk / 32; ++s) {
        const int q = cs + 32 * s + lane;
        unsigned r = 0;
        typename S::Payload pay;
        if (q < te) {
          if (q >= G.gend) {  // walk to the group holding q (short linear walk, then bisection)
            int steps = 0;
            do {
              ++g;
              G.gbase = G.gend;
              G.gend = st.pp(g + 1);
            } while (q >= G.gend && ++steps < 4);
            if (q >= G.gend) {
              int lo = g, hi = n;  // invariant: pp(lo) <= q < pp(hi)
              while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (st.pp(mid) <= q) lo = mid; else hi = mid;
              }
              g = lo;
              G.gbase = st.pp(g);
              G.gend = st.pp(g + 1);
            }
            st.load_group(g, G);
          }
          int o, j;
          split_pair(q - G.gbase, G.n_c, o, j);
          r = st.test(G, o, j, pay);
        }
        near += (r >> 1) & 1u;
        const unsigned m = __ballot_sync(kFull, r & ACC);
        if (r & ACC) {
          const int k = run + __popc(m & ((1u << lane) - 1u));
          s_stage[warp][k] = pay;
          s_q[warp][k] = (unsigned short)(q - ts);
        }
        run += __popc(m);
      }
    }
    // ---- output slots of the tile; objects out of the staging area ----
    int tb, tt;
    int off = tile_alloc(lane == 0 ? run : 0, d.tstate[S::kTicket], tile, s_scan, tb, tt);
    off = __shfl_sync(kFull, off, 0);
    if (lane == 0) {
      s_woff[warp] = off;
      s_run[warp] = run;
    }
    if (threadIdx.x == 0) s_woff[kWarps] = tb + tt;
    __syncthreads();
    for (int k = lane; k < run; k += 32)
      if (off + k < cap) st.emit(off + k, s_stage[warp][k]);
    // ---- begin offsets owned by this tile: groups in (g_lo, g_hi], tile 0 also [0, g_lo] ----
    {
      const bool last = tile == n_tiles - 1;
      const int g_lo = TP > 0 ? st.chunk_g0()[tile * kWarps] : n;
      const int g_hi = last ? n : st.chunk_g0()[(tile + 1) * kWarps];
      const TileRank rank{s_woff, s_run, s_q, ts};
      st.boundaries(tile, TP == 0, g_lo, g_hi, ts, te, rank);
      if (last && threadIdx.x == 0) {
        const int total = tb + tt;
        st.finish_total(total);
        if (total > cap || too_many) {
          atomicOr(&d.ctl->error, S::kErr);
          d.ctl->total[S::kKind] = 0;
        } else {
          d.ctl->total[S::kKind] = total;
        }
        d.ctl->n_tests[S::kStage] = (unsigned long long)TP;
      }
    }
    __syncthreads();  // staging and s_woff are reused by the next tile
  }
  near = warp_sum_u64(near);
  if (lane == 0 && near) atomicAdd(&d.ctl->near[S::kStage], near);
}

}  // namespace lst
