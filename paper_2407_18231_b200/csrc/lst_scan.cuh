// lst_scan.cuh -- single-pass allocation primitives: warp/block scans and decoupled look-back.
//
// Every object-building stage is "owner -> variable number of accepted candidates".  Output slots
// are assigned by an exclusive prefix sum over the owners, computed INSIDE the producing kernel:
// tiles of owners take a ticket (so lower tiles always started earlier), scan their counts in
// shared memory, publish the tile aggregate in a 64-bit status word and look back over the
// predecessors' words for their prefix.  Result: objects are stored in owner order (contiguous per owner,
// per module and per event) with one kernel launch per stage and no atomics
// on the data path.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lst {

constexpr int kBlock = 256;  // threads per block of every stage kernel
constexpr int kWarps = kBlock / 32;
constexpr unsigned kFull = 0xffffffffu;

__device__ __forceinline__ int warp_incl_scan(int v) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int t = __shfl_up_sync(kFull, v, d);
    if (lane >= d) v += t;
  }
  return v;
}

__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
  return v;
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(kFull, v, d);
  return v;
}

// ---- per-event counters (CUTS.md section 0: near-threshold candidates and candidates per stage) ----
// Near-threshold candidates are rare (a few per million): one global atomic where it happens.
__device__ __forceinline__ void count_near(unsigned long long* ev_cnt, int ev, int stage) {
  atomicAdd(ev_cnt + (size_t)ev * 14 + stage, 1ull);  // 14 = kEvCnt (lst_types.cuh)
}

// Candidate counts are accumulated per block in a shared-memory table indexed by event (events beyond
// the table go straight to global memory) and flushed once at the end of the kernel.  The table holds
// 64-bit counts as two 32-bit words (shared-memory atomics are native for 32 bits only; a 64-bit add is a
// compare-and-swap loop): the low word is added atomically, a wrap-around carries into the high word.
struct EvTests {
  unsigned* s;            // [2][64] shared: low words, high words
  unsigned long long* g;  // ev_cnt
  int stage, n_events;
  __device__ __forceinline__ void init(unsigned* smem, unsigned long long* ev_cnt, int st, int n_ev) {
    s = smem;  g = ev_cnt;  stage = st;  n_events = n_ev;
    for (int i = threadIdx.x; i < 128; i += blockDim.x) smem[i] = 0u;
    __syncthreads();
  }
  // n < 2^32 per call
  __device__ __forceinline__ void add(int ev, unsigned n) const {
    if (n == 0u) return;
    if (ev < 64) {
      const unsigned old = atomicAdd(s + ev, n);
      if (old + n < old) atomicAdd(s + 64 + ev, 1u);
    } else {
      atomicAdd(g + (size_t)ev * 14 + 7 + stage, (unsigned long long)n);
    }
  }
  // called by all 32 lanes: lanes of the leader's event are summed into one update (the common case:
  // consecutive work items belong to one event), the others add their own.  Sum over the warp < 2^32.
  __device__ __forceinline__ void warp_add(int ev, unsigned n) const {
    const unsigned act = __ballot_sync(kFull, n != 0u);
    if (act == 0u) return;
    const int lane = threadIdx.x & 31, lead = __ffs(act) - 1;
    const int ev0 = __shfl_sync(kFull, ev, lead);
    const bool same = n != 0u && ev == ev0;
    const unsigned sum = (unsigned)warp_sum((int)(same ? n : 0u));
    if (lane == lead) add(ev0, sum);
    else if (n != 0u && !same) add(ev, n);
  }
  __device__ __forceinline__ void flush() const {  // all threads of the block
    __syncthreads();
    for (int e = threadIdx.x; e < 64 && e < n_events; e += blockDim.x) {
      const unsigned long long v = ((unsigned long long)s[64 + e] << 32) | s[e];
      if (v) atomicAdd(g + (size_t)e * 14 + 7 + stage, v);
    }
  }
};

// tile status word: [63:32] flag (0 empty, 1 aggregate, 2 inclusive prefix), [31:0] value
__device__ __forceinline__ void st_state(unsigned long long* p, unsigned flag, int v) {
  unsigned long long w = ((unsigned long long)flag << 32) | (unsigned)v;
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(w) : "memory");
}
__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p) {
  unsigned long long w;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(p) : "memory");
  return w;
}

// Called by ONE full warp.  Publishes `aggregate` of tile `tile`, looks back, publishes the
// inclusive prefix and returns the exclusive prefix of the tile.
__device__ __forceinline__ int lookback_exclusive(unsigned long long* state, int tile, int aggregate) {
  const int lane = threadIdx.x & 31;
  if (tile == 0) {
    if (lane == 0) st_state(state, 2u, aggregate);
    return 0;
  }
  if (lane == 0) st_state(state + tile, 1u, aggregate);
  int excl = 0;
  int t = tile - 1;
  for (;;) {
    const int idx = t - lane;
    unsigned long long w = (idx >= 0) ? ld_state(state + idx) : (2ull << 32);
    while (__any_sync(kFull, (unsigned)(w >> 32) == 0u)) {
      if ((unsigned)(w >> 32) == 0u) w = ld_state(state + idx);
    }
    const unsigned incl_mask = __ballot_sync(kFull, (unsigned)(w >> 32) == 2u);
    const int val = (int)(unsigned)(w & 0xffffffffull);
    if (incl_mask) {
      const int first = __ffs(incl_mask) - 1;  // nearest predecessor holding an inclusive prefix
      excl += warp_sum(lane <= first ? val : 0);
      break;
    }
    excl += warp_sum(val);
    t -= 32;
  }
  if (lane == 0) st_state(state + tile, 2u, excl + aggregate);
  return excl;
}

// Block-wide exclusive scan of one int per thread + look-back.  Returns the GLOBAL exclusive
// offset of this thread's count; tile_total/tile_base are block-uniform.  Must be called by all
// kBlock threads.  smem: kWarps + 2 ints.
__device__ __forceinline__ int tile_alloc(int cnt, unsigned long long* state, int tile, int* smem,
                                          int& tile_base, int& tile_total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int incl = warp_incl_scan(cnt);
  if (lane == 31) smem[warp] = incl;
  __syncthreads();
  if (warp == 0) {
    int w = (lane < kWarps) ? smem[lane] : 0;
    const int wincl = warp_incl_scan(w);
    const int total = __shfl_sync(kFull, wincl, kWarps - 1);
    const int base = lookback_exclusive(state, tile, total);
    if (lane < kWarps) smem[lane] = wincl - w;  // exclusive warp offsets
    if (lane == 0) {
      smem[kWarps] = base;
      smem[kWarps + 1] = total;
    }
  }
  __syncthreads();
  tile_base = smem[kWarps];
  tile_total = smem[kWarps + 1];
  const int off = tile_base + smem[warp] + incl - cnt;
  __syncthreads();  // smem is reused by the caller's next tile
  return off;
}

}  // namespace lst
