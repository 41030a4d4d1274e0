// lst_pairs.cuh -- the evenly split candidate-pair engine (used by the MD stage).
//
// A stage is "group -> (owners x candidates) -> accepted subset": for Mini-Doublets the group is a
// module of one event (upper hits x lower hits).  (Line Segments used this engine too until their
// tiny lists made the pair decoding dearer than the cuts; see lst_ls.cuh.)  Pair counts per group
// differ by 100x (a layer-1
// barrel module holds ~1000 hit pairs, an outer endcap module a handful), so neither
// thread-per-owner nor warp-per-group keeps the machine busy (profiles/r01_v1_first_path.md: 10 of
// 32 lanes active; r01 notes: warp-per-module stalls the look-back chain behind hot modules).
//
// Here the candidate pairs of the whole batch form ONE index space: a pre-pass scans the pair
// counts of the groups (k_scan_f) and records, for every chunk of kChunk = 256 pairs, the group
// its first pair falls in.  k_eval gives every warp whole chunks (8 steps of 32 consecutive pairs;
// lanes walk pair -> group -> (owner, candidate) with a division by the group's row length), so
// all warps do the same amount of work whatever the occupancy pattern, and no warp ever waits for
// another: accepted pairs are compacted in pair order (one ballot per step) into the warp's
// staging area, then moved to a scratch list with ONE atomic per chunk; the 8 ballot words and the
// count of the chunk are kept.  k_place then scans the chunk counts (decoupled look-back over
// tiny uniform tiles) and moves every object to its final slot, so objects end up in (group,
// owner, candidate) order -- contiguous per owner, module and event (the order is a function of
// the sorted-hit order; hits of one sensor are sorted in arrival order, lst_ingest.cuh).  The
// begin-offsets of groups and owners ("first object of module m / of MD A") are ranks of pair
// indices: chunk offset + popcount of the ballot words below the pair.
// (A first version kept the look-back inside the evaluating kernel; its tiles then retire in
// ticket order and every block waits for the slowest chunk in flight -- measured 380 us for the MD
// stage against 127 us with the wait removed, profiles/r01_v2_even_split.md.)
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

// p = o * n_c + j with 0 <= j < n_c.  inv_nc ~ 1 / n_c (computed once per group); the float quotient
// is off by at most one below 2^24, which the integer fix-up repairs.
__device__ __forceinline__ void split_pair(int p, int n_c, float inv_nc, int& o, int& j) {
  if (p >= (1 << 24)) {
    o = p / n_c;
    j = p - o * n_c;
    return;
  }
  o = __float2int_rz(__int2float_rn(p) * inv_nc);
  j = p - o * n_c;
  if (j < 0) { --o; j += n_c; }
  if (j >= n_c) { ++o; j -= n_c; }
}


// Stage concept (StageMD in lst_stages.cuh):
//   static constexpr int kTicket, kKind, kErr, kStage, kPairSlot;
//   struct Group { int gbase, gend, n_c; float inv_nc; ... };  struct Payload;
//   int  n_groups() const;
//   int  pp(int g) const;                         // exclusive pair prefix of group g, g in [0, n]
//   void load_group(int g, Group&) const;         // per lane: row length n_c and what test() needs
//   unsigned test(const Group&, int o, int j, Payload&) const;     // ACC | NEAR bits
//   void emit(int pos, const Payload&) const;
//   template <class R> void boundaries(int tile, bool no_pairs, int g_lo, int g_hi, int ts, int te, const R& rank)
//   void finish_total(int total) const;

// total candidate pairs of the stage (0 if disabled or beyond the bookkeeping capacity)
template <class S>
__device__ __forceinline__ int stage_pairs(const Dev& d, const S& st, bool& too_many) {
  const unsigned long long tp64 = st.n_groups() > 0 ? d.ctl->pair_total[S::kPairSlot] : 0ull;
  too_many = tp64 > (unsigned long long)d.cap_pairs;
  return too_many ? 0 : (int)tp64;
}

// Evaluates every candidate pair of the stage once.  Warp per chunk, grid-stride, no block barrier.
template <class S>
__global__ void __launch_bounds__(kBlock) k_eval(Dev d) {
  __shared__ typename S::Payload s_stage[kWarps][kChunk];
  S st(d);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int n = st.n_groups();
  bool too_many;
  const int TP = stage_pairs(d, st, too_many);
  const int n_chunks = (TP + kChunk - 1) / kChunk;
  const int cap = d.cap[S::kKind];
  typename S::Payload* scratch = reinterpret_cast<typename S::Payload*>(d.ev_scratch);
  unsigned long long near = 0;
  for (int c = blockIdx.x * kWarps + warp; c < n_chunks; c += gridDim.x * kWarps) {
    const int cs = c * kChunk;
    typename S::Group G;
    int g = d.ev_cg0[c];  // group holding pair cs
    G.gbase = st.pp(g);
    G.gend = st.pp(g + 1);
    st.load_group(g, G);
    int run = 0;
    unsigned my_mask = 0;
#pragma unroll 1
    for (int s = 0; s < kChunk / 32; ++s) {
      const int q = cs + 32 * s + lane;
      unsigned r = 0;
      typename S::Payload pay;
      if (q < TP) {
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
        split_pair(q - G.gbase, G.n_c, G.inv_nc, o, j);
        r = st.test(G, o, j, pay);
      }
      near += (r >> 1) & 1u;
      const unsigned m = __ballot_sync(kFull, r & ACC);
      if (r & ACC) s_stage[warp][run + __popc(m & ((1u << lane) - 1u))] = pay;
      if (lane == s) my_mask = m;
      run += __popc(m);
    }
    int base = 0;
    if (lane == 0 && run > 0) base = atomicAdd(&d.ctl->scratch_cur[S::kPairSlot], run);
    base = __shfl_sync(kFull, base, 0);
    __syncwarp();
    if (base + run <= cap)  // beyond the capacity the stage reports E_CAP (k_place), nothing is placed
      for (int k = lane; k < run; k += 32) scratch[base + k] = s_stage[warp][k];
    if (lane < kChunk / 32) d.ev_mask[c * (kChunk / 32) + lane] = my_mask;
    if (lane == 0) d.ev_cnt[c] = make_int2(run, base);
    __syncwarp();  // the staging area is reused by the warp's next chunk
  }
  near = warp_sum_u64(near);
  if (lane == 0 && near) atomicAdd(&d.ctl->near[S::kStage], near);
}

// Rank of pair index x among the accepted pairs of the batch, for x inside the placing tile.
constexpr int kPlaceChunks = 64;  // chunks per placing tile: small tiles, many blocks (the work is latency-bound)

struct PlaceRank {
  const int* s_off;      // [kPlaceChunks + 1] slot offsets of the tile's chunks relative to tile_base
  const unsigned* mask;  // ballot words of all chunks
  int c0, tile_base;
  __device__ int operator()(int x) const {
    const int ci = (x >> 8) - c0;
    if (ci >= kPlaceChunks) return tile_base + s_off[kPlaceChunks];
    const int r = x & (kChunk - 1);
    const unsigned* m = mask + (size_t)(x >> 8) * (kChunk / 32);
    int cnt = 0;
    for (int w = 0; w < (r >> 5); ++w) cnt += __popc(m[w]);
    if (r & 31) cnt += __popc(m[r >> 5] & ((1u << (r & 31)) - 1u));
    return tile_base + s_off[ci] + cnt;
  }
};

// Scans the chunk counts and moves every accepted object from the scratch list to its final slot;
// fills the begin-offset arrays.  Tile = kPlaceChunks chunks.
template <class S>
__global__ void __launch_bounds__(kBlock) k_place(Dev d) {
  static_assert(kChunk == 256, "PlaceRank shifts by 8");
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  __shared__ int s_off[kPlaceChunks + 1];
  __shared__ int s_base[kPlaceChunks];
  S st(d);
  const int n = st.n_groups();
  bool too_many;
  const int TP = stage_pairs(d, st, too_many);
  const int n_chunks = (TP + kChunk - 1) / kChunk;
  const int n_tiles = n_chunks > 0 ? (n_chunks + kPlaceChunks - 1) / kPlaceChunks : 1;
  const int cap = d.cap[S::kKind];
  const bool fits = d.ctl->scratch_cur[S::kPairSlot] <= cap;  // final: k_eval has completed
  const typename S::Payload* scratch = reinterpret_cast<const typename S::Payload*>(d.ev_scratch);
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(d.ctl->ticket + S::kTicket, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int c0 = tile * kPlaceChunks, c = c0 + threadIdx.x;
    int2 cb = make_int2(0, 0);
    if (threadIdx.x < kPlaceChunks && c < n_chunks) cb = d.ev_cnt[c];
    int tb, tt;
    const int off = tile_alloc(cb.x, d.tstate[S::kTicket], tile, s_scan, tb, tt);
    if (threadIdx.x < kPlaceChunks) {
      s_off[threadIdx.x] = off - tb;
      s_base[threadIdx.x] = cb.y;
    }
    if (threadIdx.x == 0) s_off[kPlaceChunks] = tt;
    __syncthreads();
    if (fits) {
      for (int e = threadIdx.x; e < tt; e += kBlock) {
        int lo = 0, hi = kPlaceChunks;  // chunk of entry e: largest ci with s_off[ci] <= e
        while (hi - lo > 1) {
          const int mid = (lo + hi) >> 1;
          if (s_off[mid] <= e) lo = mid; else hi = mid;
        }
        st.emit(tb + e, scratch[s_base[lo] + (e - s_off[lo])]);
      }
    }
    {
      const bool last = tile == n_tiles - 1;
      const int ts = c0 * kChunk;
      const int te = last ? TP : ts + kPlaceChunks * kChunk;
      const int g_lo = TP > 0 ? d.ev_cg0[c0] : n;
      const int g_hi = last ? n : d.ev_cg0[c0 + kPlaceChunks];
      const PlaceRank rank{s_off, d.ev_mask, c0, tb};
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
    __syncthreads();  // s_off / s_base are reused by the next tile
  }
}

}  // namespace lst
