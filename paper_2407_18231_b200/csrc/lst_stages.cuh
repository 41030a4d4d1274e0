// lst_stages.cuh -- steps a3, a4: T3 and T5.  One launch per stage: thread per owner;
// pass 1 counts the accepted candidates of the owner, tile_alloc() turns the counts into output
// offsets (shared-memory scan + decoupled look-back), pass 2 re-evaluates and writes.  T3s therefore
// sit grouped by first LS (= by first MD), T5s by first T3.  (MD: lst_md.cuh, LS: lst_ls.cuh.)
#pragma once
#include "lst_ingest.cuh"

namespace lst {

template <class Stage>
__global__ void __launch_bounds__(kBlock) k_stage(Dev d) {
  load_batch(d);
  __shared__ int s_tile;
  __shared__ int s_scan[kWarps + 2];
  __shared__ unsigned s_tests[2 * kEvSmem];
  Stage st(d);
  st.prologue();
  const int n = st.n_owners();
  const int n_tiles = n > 0 ? (n + kBlock - 1) / kBlock : 1;
  EvTests tbl;
  tbl.init(s_tests, d.ev_cnt, Stage::kStage, d.n_events);
  for (;;) {
    if (threadIdx.x == 0) s_tile = atomicAdd(d.ctl->ticket + Stage::kTicket, 1);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const int owner = tile * kBlock + threadIdx.x;
    int cnt = 0, ev = 0;
    unsigned tests = 0;
    if (owner < n) cnt = st.template visit<false>(owner, 0, ev, tests);
    tbl.warp_add(ev, tests);
    int tb, tt;
    const int off = tile_alloc(cnt, d.tstate[Stage::kTicket], tile, s_scan, tb, tt);
    if (owner < n) st.begin()[owner] = off;
    if (cnt > 0) {
      unsigned t0 = 0;
      st.template visit<true>(owner, off, ev, t0);
    }
    if (tile == n_tiles - 1 && threadIdx.x == 0) {
      const int total = tb + tt;
      st.begin()[n] = total;
      if (total > d.cap[Stage::kKind]) {
        atomicOr(&d.ctl->error, Stage::kErr);
        d.ctl->total[Stage::kKind] = 0;
      } else {
        d.ctl->total[Stage::kKind] = total;
      }
    }
  }
  tbl.flush();
}

// position (x, y, z, r) of an MD with its endcap flag in the sign bit of r (r >= 0): what the seed linking reads
__device__ __forceinline__ float4 pack_flag(float4 a, int endcap) {
  a.w = __int_as_float(__float_as_int(a.w) | (endcap ? 0x80000000 : 0));
  return a;
}

// ---- anchors of the seed linking (lst_pt.cuh): the MDs that start at least one T3 ----
// The anchors of an event are sorted into kAncBins = 8 radial classes x 64 azimuthal sectors (counting sort:
// the T5 kernel's prologue counts and keeps the arrival rank, k_anchor_sort scans the event's bins and
// places), so the 32 anchors of a warp of k_pt_eval sit within a few cm of each other.
constexpr int kAncBins = 512;

__device__ __forceinline__ int anchor_bin(float x, float y, float r) {
  const int rc = (r >= 29.5f) + (r >= 43.5f) + (r >= 59.5f) + (r >= 78.0f) + (r >= 98.0f) + (r >= 125.0f);
  const float a = fabsf(x) + fabsf(y);
  const float t = a > 0.0f ? y / a : 0.0f;                                  // diamond angle, monotone in azimuth
  const float ps = x >= 0.0f ? (y >= 0.0f ? t : 4.0f + t) : 2.0f - t;      // [0, 4)
  int sec = (int)(ps * 16.0f);
  sec = sec < 0 ? 0 : (sec > 63 ? 63 : sec);
  return rc * 64 + sec;  // any finite or non-finite input lands in [0, 512): binning never affects results
}

// ---- a1: Mini-Doublets: lst_md.cuh ----
// ---- a2: Line Segments: lst_ls.cuh ----

// ---- a3: T3 (CUTS.md section 5).  owner = LS (A->B); candidates = the LSs whose inner MD is B.
struct StageT3 {
  static constexpr int kTicket = T_T3, kKind = K_T3, kErr = E_CAP_T3, kStage = 2;
  const Dev& d;
  __device__ explicit StageT3(const Dev& dd) : d(dd) {}
  __device__ void prologue() const {}
  __device__ int n_owners() const { return (d.cuts.stage_mask & 4) ? d.ctl->total[K_LS] : 0; }
  __device__ int* begin() const { return d.ls_t3_begin; }
  template <bool FILL>
  __device__ int visit(int l, int pos, int& ev, unsigned& tests) const {
    const int2 ab = d.ls_md[l];
    const int l0 = d.md_ls_begin[ab.y], l1 = d.md_ls_begin[ab.y + 1];
    if (l0 == l1) return 0;
    const float4 a = d.md_a[ab.x], b = d.md_a[ab.y];
    const int infoA = d.md_info[ab.x];
    const int eAB = (infoA & 1) | ((d.md_info[ab.y] & 1) << 1);
    if (!FILL) {
      ev = (infoA >> 1) / d.n_mod;
      tests = (unsigned)(l1 - l0);
    }
    const int cap = d.cap[K_T3];
    int cnt = 0;
    for (int l2 = l0; l2 < l1; ++l2) {
      const int C = d.ls_md[l2].y;
      const float4 c = d.md_a[C];
      const int eC = d.md_info[C] & 1;
      float k3;
      const unsigned r = t3_test(d.cuts, a, b, c, (eAB | eC) != 0, k3);
      if (!FILL && (r & NEAR)) count_near(d.ev_cnt, ev, 2);
      if (r & ACC) {
        if (FILL && pos < cap) {
          d.t3_ls[pos] = make_int2(l, l2);
          d.t3_md[pos] = make_int4(ab.x, ab.y, C, eAB | (eC << 2));
          d.t3_k[pos] = k3;
          d.t3_l[pos] = pack_flag(c, eC);
          d.t3_q[pos] = make_float4(c.x, c.y, k3, fmaf(c.x - a.x, c.x - a.x, (c.y - a.y) * (c.y - a.y)));
        }
        ++pos;
        ++cnt;
      }
    }
    return cnt;
  }
};

// ---- a4: T5 (CUTS.md section 6).  owner = T3 (A,B,C); candidates = the T3s whose first MD is C,
// i.e. the T3 range of the LSs whose inner MD is C.
struct StageT5 {
  static constexpr int kTicket = T_T5, kKind = K_T5, kErr = E_CAP_T5, kStage = 3;
  const Dev& d;
  __device__ explicit StageT5(const Dev& dd) : d(dd) {}
  // Rides along (needs the finished T3s only): which MDs are anchors of the seed linking, their bin and
  // their arrival rank in it.
  __device__ void prologue() const {
    const bool on = (d.cuts.stage_mask & 16) && d.ctl->total[K_T3] > 0 && d.n_pls > 0;
    const int n = d.ctl->total[K_MD];
    for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < n; A += gridDim.x * blockDim.x) {
      int bin = -1, rank = 0;
      if (on && d.ls_t3_begin[d.md_ls_begin[A + 1]] > d.ls_t3_begin[d.md_ls_begin[A]]) {
        const float4 a = d.md_a[A];
        const int ev = (d.md_info[A] >> 1) / d.n_mod;
        bin = anchor_bin(a.x, a.y, a.w);
        rank = atomicAdd(d.anc_bin_cnt + ev * kAncBins + bin, 1);
      }
      d.anc_bin[A] = bin;
      d.anc_rank[A] = rank;
    }
  }
  __device__ int n_owners() const { return (d.cuts.stage_mask & 8) ? d.ctl->total[K_T3] : 0; }
  __device__ int* begin() const { return d.t3_t5_begin; }
  template <bool FILL>
  __device__ int visit(int t1, int pos, int& ev, unsigned& tests) const {
    const int4 m1 = d.t3_md[t1];
    const int u0 = d.ls_t3_begin[d.md_ls_begin[m1.z]], u1 = d.ls_t3_begin[d.md_ls_begin[m1.z + 1]];
    if (u0 == u1) return 0;
    if (!FILL) {
      ev = (d.md_info[m1.x] >> 1) / d.n_mod;
      tests = (unsigned)(u1 - u0);
    }
    const float ki = d.t3_k[t1];
    const float4 b = d.md_a[m1.y], c = d.md_a[m1.z];
    const int cap = d.cap[K_T5];
    int cnt = 0;
    for (int t2 = u0; t2 < u1; ++t2) {
      const int4 m2 = d.t3_md[t2];
      float score;
      const unsigned r = t5_test(d.cuts, ki, d.t3_k[t2], b, c, d.md_a[m2.y], score);
      if (!FILL && (r & NEAR)) count_near(d.ev_cnt, ev, 3);
      if (r & ACC) {
        if (FILL && pos < cap) {
          d.t5_t3[pos] = make_int2(t1, t2);
          int* md = d.t5_md + 5 * (size_t)pos;
          md[0] = m1.x; md[1] = m1.y; md[2] = m1.z; md[3] = m2.y; md[4] = m2.z;
          d.t5_score[pos] = score;
          d.t5_l[pos] = d.t3_l[t2];
          d.t5_kio[pos] = make_float2(ki, d.t3_k[t2]);
        }
        ++pos;
        ++cnt;
      }
    }
    return cnt;
  }
};

// ---- extension: T4 (CUTS.md section 10).  owner = T3 (LS1, LS2); candidates = the T3s whose FIRST LS is LS2.
struct StageT4 {
  static constexpr int kTicket = T_T4, kKind = K_T4, kErr = E_CAP_T4, kStage = 6;
  const Dev& d;
  __device__ explicit StageT4(const Dev& dd) : d(dd) {}
  __device__ void prologue() const {}
  __device__ int n_owners() const { return (d.cuts.stage_mask & 64) ? d.ctl->total[K_T3] : 0; }
  __device__ int* begin() const { return d.t3_t4_begin; }
  template <bool FILL>
  __device__ int visit(int t1, int pos, int& ev, unsigned& tests) const {
    const int l2 = d.t3_ls[t1].y;
    const int u0 = d.ls_t3_begin[l2], u1 = d.ls_t3_begin[l2 + 1];
    if (u0 == u1) return 0;
    const int4 m1 = d.t3_md[t1];
    if (!FILL) {
      ev = (d.md_info[m1.x] >> 1) / d.n_mod;
      tests = (unsigned)(u1 - u0);
    }
    const float k1 = d.t3_k[t1];
    const int cap = d.cap[K_T4];
    int cnt = 0;
    for (int t2 = u0; t2 < u1; ++t2) {
      float score;
      const unsigned r = t4_test(d.cuts, k1, d.t3_k[t2], score);
      if (!FILL && (r & NEAR)) count_near(d.ev_cnt, ev, 6);
      if (r & ACC) {
        if (FILL && pos < cap) {
          d.t4_t3[pos] = make_int2(t1, t2);
          d.t4_md[pos] = make_int4(m1.x, m1.y, m1.z, d.t3_md[t2].z);
          d.t4_score[pos] = score;
        }
        ++pos;
        ++cnt;
      }
    }
    return cnt;
  }
};

}  // namespace lst
