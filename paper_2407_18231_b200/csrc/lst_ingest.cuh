// lst_ingest.cuh -- step a0: hit ingestion and module binning (counting sort by global sensor),
// plus the generic single-pass exclusive scan kernel.  PAPER.md:23 ("uses as input the hits of the
// ... outer tracker"); SURVEY.md section 8(a) row a0.
#pragma once
#include "lst_cuts_pt.cuh"
#include "lst_scan.cuh"
#include "lst_types.cuh"

namespace lst {

// event of a batch-global index, from the (<= a few dozen entries) offsets array
__device__ __forceinline__ int event_of(const int* __restrict__ off, int n_events, int i) {
  int lo = 0, hi = n_events;  // invariant: off[lo] <= i < off[hi]
  while (hi - lo > 1) {
    int mid = (lo + hi) >> 1;
    if (__ldg(off + mid) <= i) lo = mid; else hi = mid;
  }
  return lo;
}

// a0.1 histogram: one atomic per hit on its sensor counter; the returned rank is kept so that the
// scatter pass needs no second atomic.  Invalid sensor ids raise E_BAD_SENSOR (-> LST_ERR_ARG).
// kIngestUnroll hits per thread are in flight at once (the kernel is latency-bound: every hit is a
// chain load -> atomic -> store).
constexpr int kIngestUnroll = 4;

__global__ void __launch_bounds__(kBlock) k_hist(Dev d) {
  load_batch(d);
  const int stride = gridDim.x * blockDim.x;
  const int n_sens = 2 * d.n_mod;
  for (int i0 = blockIdx.x * blockDim.x + threadIdx.x; i0 < d.n_hits; i0 += kIngestUnroll * stride) {
    int s[kIngestUnroll], gs[kIngestUnroll];
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      s[u] = i >= d.n_hits ? 0 : (d.sensor_u16 ? (int)__ldg(reinterpret_cast<const unsigned short*>(d.in_sensor) + i)
                                                 : __ldg(d.in_sensor + i));
    }
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      if (i < d.n_hits && (s[u] < 0 || s[u] >= n_sens)) {
        atomicOr(&d.ctl->error, E_BAD_SENSOR);
        s[u] = 0;
      }
      gs[u] = (i < d.n_hits ? event_of(d.hit_ev_off, d.n_events, i) : 0) * n_sens + s[u];
    }
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      if (i < d.n_hits) {
        d.hit_gs_in[i] = gs[u];
        d.hit_rank[i] = atomicAdd(d.sens_cnt + gs[u], 1);
      }
    }
  }
  // pLS -> event, and the per-seed quantities of CUTS.md section 7 (computed once per seed, exactly as
  // written there: lv, kp, tolk, slope); tiny, rides along
  for (int p = blockIdx.x * blockDim.x + threadIdx.x; p < d.n_pls; p += stride) {
    d.pls_event[p] = event_of(d.pls_ev_off, d.n_events, p);
    const Seed s = make_seed(d.cuts, __ldg(d.p_pt + p), __ldg(d.p_q + p), __ldg(d.p_x0 + p), __ldg(d.p_y0 + p),
                             __ldg(d.p_z0 + p), __ldg(d.p_x1 + p), __ldg(d.p_y1 + p), __ldg(d.p_z1 + p));
    d.seed_a[p] = make_float4(s.x1, s.y1, s.vx, s.vy);
    d.seed_b[p] = make_float4(s.lv, s.kp, s.tolk, s.slope);
    d.seed_z1[p] = s.z1;
    // what k_pt_eval keeps per lane: the coefficients of the gate limit glim = lw (lw c1 + c2), and kp, tolk
    d.seed_g[p] = make_float4(s.lv * d.cuts.inv_2rmin, s.lv * d.cuts.pt_gate_tol, s.kp, s.tolk);
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

// a0.3 scatter: sorted SoA (float4 x,y,z,r + int2 input index, global sensor), r = sqrtf(x*x + y*y)
__global__ void __launch_bounds__(kBlock) k_scatter(Dev d) {
  load_batch(d);
  const int stride = gridDim.x * blockDim.x;
  const int n_sens = 2 * d.n_mod;
  for (int i0 = blockIdx.x * blockDim.x + threadIdx.x; i0 < d.n_hits; i0 += kIngestUnroll * stride) {
    int gs[kIngestUnroll], pos[kIngestUnroll];
    float x[kIngestUnroll], y[kIngestUnroll], z[kIngestUnroll];
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      const bool ok = i < d.n_hits;
      gs[u] = ok ? d.hit_gs_in[i] : 0;
      pos[u] = ok ? d.hit_rank[i] : 0;
      x[u] = ok ? __ldg(d.in_x + i) : 0.0f;
      y[u] = ok ? __ldg(d.in_y + i) : 0.0f;
      z[u] = ok ? __ldg(d.in_z + i) : 0.0f;
    }
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) pos[u] += __ldg(d.sens_begin + gs[u]);
#pragma unroll
    for (int u = 0; u < kIngestUnroll; ++u) {
      const int i = i0 + u * stride;
      if (i < d.n_hits) {
        d.hit[pos[u]] = make_float4(x[u], y[u], z[u], sqrtf(x[u] * x[u] + y[u] * y[u]));
        const int ev = gs[u] / n_sens;
        d.hit_ig[pos[u]] = make_int2(i - __ldg(d.hit_ev_off + ev), gs[u]);
      }
    }
  }
}

}  // namespace lst
