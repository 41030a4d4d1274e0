// lst_ingest.cuh -- step a0: hit ingestion and module binning (counting sort by global sensor, k_ingest),
// plus the generic single-pass exclusive scan kernel (used for the per-seed counts of the seed linking).  PAPER.md:23 ("uses as input the hits of the
// ... outer tracker"); SURVEY.md section 8(a) row a0.
#pragma once
#include "lst_cuts_pt.cuh"
#include "lst_scan.cuh"
#include "lst_types.cuh"

namespace lst {

// a0: counting sort of the hits by global sensor, three small kernels, no global atomic.  The hits of an event are a
// contiguous range of the input (event offsets) and stay one after the sort (global sensor = event * n_sens +
// sensor), so counts and scan are local to the event.  Block (e, c) owns chunk c (of kIngestChunks) of the
// event's hits and keeps one counter per sensor in shared memory (sensors are taken kIngestMaxBins at a time:
// one round for any realistic geometry):
//   k_ingest_count: shared-memory atomic per hit of the chunk; the returned value is the hit's rank among the
//                   chunk's hits of that sensor (hit_rank); the chunk's counters go to chunk_cnt[e][c][sensor];
//   k_ingest_scan:  one block per event: totals over the chunks, exclusive scan over the event's sensors ->
//                   sens_begin, and the first slot of every chunk's hits of every sensor;
//   k_scatter:      every hit of the batch (all SMs: the scattered 16- and 8-byte stores are the cost) is written
//                   at slot + rank: (x, y, z, r), r = sqrtf(x*x + y*y), and (event-local input index, global sensor).
// The order inside a sensor is chunk order, then arrival order: free.  Invalid sensor ids raise E_BAD_SENSOR
// (-> LST_ERR_ARG) and count as sensor 0.  k_ingest_count's block (e, 0) also fills the per-seed table of event e
// (CUTS.md section 7: the quantities that do not depend on the candidate).
constexpr int kIngestThreads = 1024;
constexpr int kIngestMaxBins = 40960;  // counters per round (160 KB of shared memory)
constexpr int kIngestChunks = 4;       // blocks per event
constexpr int kIngestBatch = 8;        // sensor ids a thread has in flight
constexpr int kIngestScanParts = 4;    // blocks per event of k_ingest_scan

__device__ __forceinline__ int load_sensor(const Dev& d, int i) {
  return d.sensor_u16 ? (int)__ldg(reinterpret_cast<const unsigned short*>(d.in_sensor) + i) : __ldg(d.in_sensor + i);
}

struct IngestChunk {  // what block (e, c) works on
  int e, c, h0, i_lo, i_hi, n_sens, R;
  __device__ __forceinline__ bool init(const Dev& d) {
    e = blockIdx.x / kIngestChunks;
    c = blockIdx.x - e * kIngestChunks;
    if (e >= d.n_events) return false;
    h0 = d.hit_ev_off[e];
    const int h1 = d.hit_ev_off[e + 1];
    const int per = (h1 - h0 + kIngestChunks - 1) / kIngestChunks;
    i_lo = min(h1, h0 + c * per);
    i_hi = min(h1, i_lo + per);
    n_sens = 2 * d.n_mod;
    R = min(n_sens, kIngestMaxBins);
    return true;
  }
};

__global__ void __launch_bounds__(kIngestThreads) k_ingest_count(Dev d) {
  load_batch(d);
  extern __shared__ int s_bin[];  // R counters
  IngestChunk k;
  if (!k.init(d)) return;
  if (k.c == 0) {
    // the per-seed quantities of CUTS.md section 7, computed once per seed exactly as written there
    for (int p = d.pls_ev_off[k.e] + threadIdx.x; p < d.pls_ev_off[k.e + 1]; p += kIngestThreads) {
      d.pls_event[p] = k.e;
      const Seed s = make_seed(d.cuts, __ldg(d.p_pt + p), __ldg(d.p_q + p), __ldg(d.p_x0 + p), __ldg(d.p_y0 + p),
                               __ldg(d.p_z0 + p), __ldg(d.p_x1 + p), __ldg(d.p_y1 + p), __ldg(d.p_z1 + p));
      d.seed_a[p] = make_float4(s.x1, s.y1, s.vx, s.vy);
      d.seed_b[p] = make_float4(s.lv, s.kp, s.tolk, s.slope);
      d.seed_z1[p] = s.z1;
      // what k_pt_eval keeps per lane: the coefficients of the gate limit glim = lw (lw c1 + c2), and kp, tolk
      d.seed_g[p] = make_float4(s.lv * d.cuts.inv_2rmin, s.lv * d.cuts.pt_gate_tol, s.kp, s.tolk);
    }
  }
  int* __restrict__ row = d.chunk_cnt + ((size_t)k.e * kIngestChunks + k.c) * k.n_sens;
  __shared__ int s_part[kIngestScanParts];
  if (threadIdx.x < kIngestScanParts) s_part[threadIdx.x] = 0;
  const int plen = (k.n_sens + kIngestScanParts - 1) / kIngestScanParts;  // sensors per block of k_ingest_scan
  int part_sum[kIngestScanParts];
#pragma unroll
  for (int q = 0; q < kIngestScanParts; ++q) part_sum[q] = 0;
  bool bad = false;
  for (int r_lo = 0; r_lo < k.n_sens; r_lo += k.R) {
    const int r_n = min(k.R, k.n_sens - r_lo);
    for (int j = threadIdx.x; j < r_n; j += kIngestThreads) s_bin[j] = 0;
    __syncthreads();
    for (int i0 = k.i_lo + threadIdx.x; i0 < k.i_hi; i0 += kIngestBatch * kIngestThreads) {
      int sv[kIngestBatch];
#pragma unroll
      for (int u = 0; u < kIngestBatch; ++u) {  // kIngestBatch independent loads in flight
        const int i = i0 + u * kIngestThreads;
        sv[u] = i < k.i_hi ? load_sensor(d, i) : 0;
      }
#pragma unroll
      for (int u = 0; u < kIngestBatch; ++u) {
        const int i = i0 + u * kIngestThreads;
        if (i >= k.i_hi) break;
        int s = sv[u];
        if (s < 0 || s >= k.n_sens) {
          bad = true;
          s = 0;
        }
        if (s >= r_lo && s < r_lo + r_n) d.hit_rank[i] = atomicAdd(&s_bin[s - r_lo], 1);
      }
    }
    __syncthreads();
    for (int j = threadIdx.x; j < r_n; j += kIngestThreads) {
      const int v = s_bin[j];
      row[r_lo + j] = v;
#pragma unroll
      for (int q = 0; q < kIngestScanParts; ++q) part_sum[q] += (r_lo + j) / plen == q ? v : 0;
    }
    __syncthreads();
  }
  // the chunk's hits per part of the sensor range: where the blocks of k_ingest_scan start
#pragma unroll
  for (int q = 0; q < kIngestScanParts; ++q) {
    const int v = warp_sum(part_sum[q]);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(&s_part[q], v);
  }
  __syncthreads();
  if (threadIdx.x < kIngestScanParts)
    d.chunk_part[((size_t)k.e * kIngestChunks + k.c) * kIngestScanParts + threadIdx.x] = s_part[threadIdx.x];
  if (bad) atomicOr(&d.ctl->error, E_BAD_SENSOR);
}

// kIngestScanParts blocks per event, each a part of the sensor range: totals over the chunks, exclusive scan over
// the sensors -> sens_begin; the chunk counters are replaced, in place, by the first slot of the chunk's hits of
// every sensor.
__global__ void __launch_bounds__(kIngestThreads) k_ingest_scan(Dev d) {
  load_batch(d);
  __shared__ int s_warp[2][kIngestThreads / 32];
  const int e = blockIdx.x / kIngestScanParts, part = blockIdx.x - e * kIngestScanParts;
  if (e >= d.n_events) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int n_all = 2 * d.n_mod;
  const int plen = (n_all + kIngestScanParts - 1) / kIngestScanParts;
  const int n_sens = min(n_all, (part + 1) * plen);  // this block: sensors [part * plen, n_sens)
  int* __restrict__ rows = d.chunk_cnt + (size_t)e * kIngestChunks * n_all;
  int* __restrict__ begin = d.sens_begin + (size_t)e * n_all;
  constexpr int T = 4;  // tiles of kIngestThreads consecutive sensors whose loads are in flight together
  int carry = d.hit_ev_off[e];  // + the event's hits on the sensors of the lower parts (k_ingest_count)
  for (int c = 0; c < kIngestChunks; ++c)
    for (int q = 0; q < part; ++q) carry += d.chunk_part[((size_t)e * kIngestChunks + c) * kIngestScanParts + q];
  int par = 0;
  for (int t0 = part * plen; t0 < n_sens; t0 += T * kIngestThreads) {
    int v[T][kIngestChunks];
#pragma unroll
    for (int t = 0; t < T; ++t) {
      const int j = t0 + t * kIngestThreads + threadIdx.x;  // coalesced: consecutive threads, consecutive sensors
#pragma unroll
      for (int c = 0; c < kIngestChunks; ++c) v[t][c] = j < n_sens ? rows[(size_t)c * n_all + j] : 0;
    }
#pragma unroll
    for (int t = 0; t < T; ++t) {
      const int j = t0 + t * kIngestThreads + threadIdx.x;
      if (t0 + t * kIngestThreads >= n_sens) break;
      int tot = 0;
#pragma unroll
      for (int c = 0; c < kIngestChunks; ++c) tot += v[t][c];
      const int incl = warp_incl_scan(tot);
      if (lane == 31) s_warp[par][warp] = incl;
      __syncthreads();
      const int wv = s_warp[par][lane];           // every warp scans the 32 warp totals itself
      const int wi = warp_incl_scan(wv);
      const int wbase = __shfl_sync(kFull, wi - wv, warp);
      const int tile_total = __shfl_sync(kFull, wi, 31);
      int run = carry + wbase + incl - tot;
      if (j < n_sens) {
        begin[j] = run;
#pragma unroll
        for (int c = 0; c < kIngestChunks; ++c) {
          rows[(size_t)c * n_all + j] = run;
          run += v[t][c];
        }
      }
      carry += tile_total;
      par ^= 1;  // the other buffer: no second barrier per tile
    }
  }
  if (e == d.n_events - 1 && part == kIngestScanParts - 1 && threadIdx.x == 0) d.sens_begin[(size_t)d.n_events * n_all] = carry;
}

// Every hit goes to (first slot of its chunk's hits of its sensor) + (its rank among them): sorted SoA
// (float4 x, y, z, r + int2 event-local input index, global sensor), r = sqrtf(x*x + y*y).
constexpr int kIngestUnroll = 4;

// sorted hit `i`: one 32-byte record = one sector, (x, y, z, r) then (event-local input index, global sensor, -, -)
__device__ __forceinline__ float4 hit_xyzr(const Dev& d, int i) { return d.hit[2 * (size_t)i]; }
__device__ __forceinline__ int2 hit_ig(const Dev& d, int i) {
  return *reinterpret_cast<const int2*>(d.hit + 2 * (size_t)i + 1);
}

__global__ void __launch_bounds__(kBlock) k_scatter(Dev d) {  // grid (blocks per event, max_events)
  load_batch(d);
  const int e = blockIdx.y;
  if (e >= d.n_events) return;
  const int stride = gridDim.x * blockDim.x;
  const int n_sens = 2 * d.n_mod;
  const int h0 = d.hit_ev_off[e], h1 = d.hit_ev_off[e + 1];
  const int per = (h1 - h0 + kIngestChunks - 1) / kIngestChunks;  // as IngestChunk::init
  const int* __restrict__ slots = d.chunk_cnt + (size_t)e * kIngestChunks * n_sens;
  const int gs0 = e * n_sens;
  for (int i0 = h0 + blockIdx.x * blockDim.x + threadIdx.x; i0 < h1; i0 += kIngestUnroll * stride) {
    int slot[kIngestUnroll], rk[kIngestUnroll], sv[kIngestUnroll];
    float x[kIngestUnroll], y[kIngestUnroll], z[kIngestUnroll];
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      const bool ok = i < h1;
      int s = ok ? load_sensor(d, i) : 0;
      if (s < 0 || s >= n_sens) s = 0;
      const int k = i - h0;
      int c = 0;  // chunk of hit i: k / per
#pragma unroll
      for (int cc = 1; cc < kIngestChunks; ++cc) c += k >= cc * per;
      sv[u] = s;
      slot[u] = ok ? slots[(size_t)c * n_sens + s] : 0;
      rk[u] = ok ? d.hit_rank[i] : 0;
      x[u] = ok ? __ldg(d.in_x + i) : 0.0f;
      y[u] = ok ? __ldg(d.in_y + i) : 0.0f;
      z[u] = ok ? __ldg(d.in_z + i) : 0.0f;
    }
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      if (i < h1) {
        const int pos = slot[u] + rk[u];
        d.hit[2 * (size_t)pos] = make_float4(x[u], y[u], z[u], sqrtf(x[u] * x[u] + y[u] * y[u]));
        d.hit[2 * (size_t)pos + 1] = make_float4(__int_as_float(i - h0), __int_as_float(gs0 + sv[u]), 0.0f, 0.0f);
      }
    }
  }
}

// Generic exclusive scan out[i] = sum_{j<i} in[j], i in [0, n], n = (*n_ptr) * n_mul + n_add
// (n_ptr may be NULL -> n = n_add).  in[n] is not read; out[n] = total.  Persistent blocks take
// tile tickets; ITEMS consecutive items per thread (16 for the million-item scans: the cost of a scan
// is its number of tiles, i.e. look-back round trips).
constexpr int kScanItems = 4;
constexpr int kScanTile = kBlock * kScanItems;

struct ScanJob {
  const int* in;
  int* out;
  const int* n_ptr;
  int n_mul, n_add;
  int* ticket;
  unsigned long long* state;
};

template <int ITEMS>
__device__ __forceinline__ void scan_body(const ScanJob& j) {
  constexpr int kTile = kBlock * ITEMS;
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  const int* __restrict__ in = j.in;
  int* __restrict__ out = j.out;
  const int n = (j.n_ptr ? (*j.n_ptr) * j.n_mul : 0) + j.n_add;
  const int n_tiles = (n + kTile - 1) / kTile > 0 ? (n + kTile - 1) / kTile : 1;
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(j.ticket, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int base_i = tile * kTile + threadIdx.x * ITEMS;
    int v[ITEMS];
    int sum = 0;
    if (ITEMS % 4 == 0 && base_i + ITEMS <= n) {  // full thread: 16-byte loads (arrays are 256-byte aligned)
#pragma unroll
      for (int k = 0; k < ITEMS; k += 4) {
        const int4 q = *reinterpret_cast<const int4*>(in + base_i + k);
        v[k] = q.x;  v[k + 1] = q.y;  v[k + 2] = q.z;  v[k + 3] = q.w;
      }
    } else {
#pragma unroll
      for (int k = 0; k < ITEMS; ++k) v[k] = (base_i + k < n) ? in[base_i + k] : 0;
    }
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) sum += v[k];
    int tb, tt;
    int off = tile_alloc(sum, j.state, tile, s_scan, tb, tt);
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      if (base_i + k < n) out[base_i + k] = off;
      off += v[k];
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) out[n] = tb + tt;
  }
}

template <int ITEMS>
__global__ void __launch_bounds__(kBlock)
k_scan_t(const int* __restrict__ in, int* __restrict__ out, const int* n_ptr, int n_mul, int n_add,
         int* ticket, unsigned long long* state) {
  scan_body<ITEMS>(ScanJob{in, out, n_ptr, n_mul, n_add, ticket, state});
}

// two independent scans in one launch (blockIdx.y picks the job)
__global__ void __launch_bounds__(kBlock) k_scan2(ScanJob j0, ScanJob j1) {
  scan_body<kScanItems>(blockIdx.y ? j1 : j0);
}

#define k_scan k_scan_t<kScanItems>

}  // namespace lst
