// lst_pt.cuh -- step a5: pLS x T3 -> pT3 and pLS x T5 -> pT5 (CUTS.md section 7).
// Candidates of a seed = every T3 / T5 of its event (CUTS.md section 7; the direction gate of the
// spec replaces the IT->OT connection map).  The pairs (pLS, candidate) of the batch are split
// evenly over warps (lst_pairs.cuh, k_eval2): phase 1 reads the first-MD anchor (float2,
// coalesced) and applies a conservative, sqrt-free form of the gate; phase 2 evaluates the exact
// cut list on the ~8% that survive, with full warps.
#pragma once
#include "lst_cuts_pt.cuh"
#include "lst_stages.cuh"

namespace lst {

template <bool IS5>
struct PtCand {
  // evaluates candidate t for seed s; returns ACC/NEAR bits, score on accept
  static __device__ __forceinline__ unsigned test(const Dev& d, const Seed& s, int t, float& score) {
    const float2 axy = IS5 ? d.t5_axy[t] : d.t3_axy[t];
    unsigned r = pt_gate(d.cuts, s, axy.x, axy.y);
    if (!(r & ACC)) return r;
    r &= NEAR;
    if (IS5) {
      const int* md = d.t5_md + 5 * (size_t)t;
      const int A = md[0], L = md[4];
      const int2 tt = d.t5_t3[t];
      const float kt[2] = {d.t3_k[tt.x], d.t3_k[tt.y]};
      r |= pt_after_gate<2>(d.cuts, s, d.md_a[A], d.md_info[A] & 1, d.md_a[L], d.md_info[L] & 1, kt,
                            d.t5_score[t], score);
    } else {
      const int4 m = d.t3_md[t];
      const float kt[1] = {d.t3_k[t]};
      r |= pt_after_gate<1>(d.cuts, s, d.md_a[m.x], m.w & 1, d.md_a[m.z], (m.w >> 2) & 1, kt, 0.0f,
                            score);
    }
    return r;
  }
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

template <bool IS5>
struct PairsPT {  // pre-pass: candidates per seed
  const Dev& d;
  __device__ explicit PairsPT(const Dev& dd) : d(dd) {}
  __device__ int n_items() const {
    return ((d.cuts.stage_mask & 16) && d.ctl->total[IS5 ? K_T5 : K_T3] > 0) ? d.n_pls : 0;
  }
  __device__ int count(int p) const {
    int c0, c1;
    event_cands<IS5>(d, d.pls_event[p], c0, c1);
    return c1 - c0;  // <= capacity of the T3 / T5 array
  }
  __device__ int group(int p) const { return p; }
};

template <bool IS5>
struct StagePT {
  static constexpr int kTicket = IS5 ? T_PT5 : T_PT3, kKind = IS5 ? K_PT5 : K_PT3;
  static constexpr int kErr = IS5 ? E_CAP_PT5 : E_CAP_PT3, kStage = IS5 ? 5 : 4, kPairSlot = IS5 ? 3 : 2;
  struct Group {
    int gbase, gend, n_c;
    int c0;                        // first candidate of the seed's event
    float x1, y1, vx, vy, lv;      // outer pixel hit and P1 - P0 (CUTS.md section 7)
  };
  struct Pre {
    int t_q;  // candidate (22 bits; lst_ctx_create bounds max_t3 / max_t5) | pair number inside the super-chunk << 22
    int p;    // seed
  };
  struct Payload {
    int p, t;
    float score;
  };
  const Dev& d;
  __device__ explicit StagePT(const Dev& dd) : d(dd) {}
  __device__ bool enabled() const { return (d.cuts.stage_mask & 16) && d.ctl->total[IS5 ? K_T5 : K_T3] > 0; }
  __device__ int n_groups() const { return enabled() ? d.n_pls : 0; }
  __device__ int pp(int g) const { return d.pp_pt[g]; }
  __device__ void load_group(int p, Group& G) const {
    int c1;
    event_cands<IS5>(d, d.pls_event[p], G.c0, c1);
    G.n_c = c1 - G.c0;
    const float x0 = __ldg(d.p_x0 + p), y0 = __ldg(d.p_y0 + p);
    G.x1 = __ldg(d.p_x1 + p);
    G.y1 = __ldg(d.p_y1 + p);
    G.vx = G.x1 - x0;
    G.vy = G.y1 - y0;
    G.lv = sqrtf(G.vx * G.vx + G.vy * G.vy);
  }
  // Necessary condition of the gate (CUTS.md section 7): gdot > 0 exactly as in the spec, and the
  // gcrs <= glim cut with |A - P1| from the approximate reciprocal square root and a 1e-4 margin
  // (the exact glim differs by < 1e-6 relative; near-threshold candidates lie within 1e-5).
  __device__ bool prefilter(const Group& G, int p, int j, int qrel, Pre& pre) const {
    const int t = G.c0 + j;
    const float2 a = IS5 ? d.t5_axy[t] : d.t3_axy[t];
    const float wx = a.x - G.x1, wy = a.y - G.y1;
    const float gdot = G.vx * wx + G.vy * wy;
    if (!(gdot > 0.0f)) return false;
    pre.t_q = t | (qrel << 22);
    pre.p = p;
    const float lw2 = wx * wx + wy * wy;
    if (!(lw2 >= 1e-30f) || !(lw2 <= 1e30f)) return true;  // out of the approximation's range: exact path decides
    float rl;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rl) : "f"(lw2));
    const float lw = lw2 * rl;
    const float gcrs = fabsf(G.vx * wy - G.vy * wx);
    const float lim = (G.lv * lw) * (lw * d.cuts.inv_2rmin + d.cuts.pt_gate_tol);
    return !(gcrs > lim * 1.0001f);
  }
  // Necessary condition of the curvature match |kx - kp| <= tolk, kx = kappa3(P1, A, L): compares
  // kx^2 = 4 crs^2 / (|P1A|^2 |AL|^2 |P1L|^2) with (|kp| -+ tolk)^2 without sqrt or division.  crs is
  // formed exactly as in kappa3 (same operands, same order), so cancellation affects both alike;
  // everything else differs by ~1e-6 relative and the bounds carry a 1e-3 margin.
  // The exact gate comes first: a candidate it rejects is final (its near-threshold flag is counted
  // here), one it flags near-threshold goes on to the exact cut list whatever its curvature.
  __device__ bool midfilter(const Pre& pre, unsigned long long& near) const {
    const int p = pre.p, t = pre.t_q & 0x3fffff;
    const float x1 = __ldg(d.p_x1 + p), y1 = __ldg(d.p_y1 + p);
    const float2 A = IS5 ? d.t5_axy[t] : d.t3_axy[t];
    {
      Seed s;
      s.x1 = x1;
      s.y1 = y1;
      s.vx = x1 - __ldg(d.p_x0 + p);
      s.vy = y1 - __ldg(d.p_y0 + p);
      s.lv = sqrtf(s.vx * s.vx + s.vy * s.vy);
      const unsigned r = pt_gate(d.cuts, s, A.x, A.y);
      if (!(r & ACC)) {
        near += (r >> 1) & 1u;
        return false;
      }
      if (r & NEAR) return true;
    }
    const float kp = (-(float)__ldg(d.p_q + p)) / (__ldg(d.p_pt + p) * d.cuts.kr);
    const float tolk = d.cuts.pt_k_tol0 + d.cuts.pt_k_tol1 * fabsf(kp);
    const float2 L = IS5 ? d.t5_lxy[t] : d.t3_lxy[t];
    const float ax = A.x - x1, ay = A.y - y1;
    const float bx = L.x - A.x, by = L.y - A.y;
    const float cx = L.x - x1, cy = L.y - y1;
    const float crs = ax * cy - ay * cx;
    const float prod = ((ax * ax + ay * ay) * (bx * bx + by * by)) * (cx * cx + cy * cy);
    const float k2 = 4.0f * (crs * crs);
    const float hi = (fabsf(kp) + tolk) * 1.001f;
    if (k2 > (hi * hi) * prod) return false;
    const float lo = (fabsf(kp) - tolk) * 0.999f;
    if (lo > 0.0f) {
      if (k2 < (lo * lo) * prod) return false;
      if ((crs > 0.0f) != (kp > 0.0f)) return false;  // |kx| >= lo > 0 with the wrong sign: |kx - kp| > tolk
    }
    return true;
  }
  __device__ int qrel(const Pre& pre) const { return (unsigned)pre.t_q >> 22; }
  __device__ unsigned test_pre(const Pre& pre, Payload& pay) const {
    const int p = pre.p, t = pre.t_q & 0x3fffff;
    const Seed s = make_seed(d.cuts, __ldg(d.p_pt + p), __ldg(d.p_q + p), __ldg(d.p_x0 + p), __ldg(d.p_y0 + p),
                             __ldg(d.p_z0 + p), __ldg(d.p_x1 + p), __ldg(d.p_y1 + p), __ldg(d.p_z1 + p));
    pay.p = p;
    pay.t = t;
    return PtCand<IS5>::test(d, s, t, pay.score);
  }
  __device__ void emit(int pos, const Payload& pay) const {
    (IS5 ? d.pt5 : d.pt3)[pos] = make_int2(pay.p, pay.t);
    (IS5 ? d.pt5_score : d.pt3_score)[pos] = pay.score;
  }
  // first pT object of every seed: rank of the seed's first pair
  template <class R>
  __device__ void boundaries(int tile, bool no_pairs, int g_lo, int g_hi, int, int, const R& rank) const {
    int* begin = IS5 ? d.pls_pt5_begin : d.pls_pt3_begin;
    if (no_pairs) {
      const int n = (d.cuts.stage_mask & 16) ? d.n_pls : 0;
      for (int g = threadIdx.x; g <= n; g += kBlock) begin[g] = 0;
      return;
    }
    for (int g = (tile == 0 ? 0 : g_lo + 1) + threadIdx.x; g <= g_hi; g += kBlock) begin[g] = rank(pp(g));
  }
  __device__ void finish_total(int) const {}
};

}  // namespace lst
