// lst_audit.cuh -- brute-force re-evaluation of the stages that sit behind an approximate cut cascade.
//
// MD, LS and the seed linking (pT3 / pT5) drop or accept most of their candidates on cheaper arithmetic
// (rsqrt.approx, approximate division, FMA, bounding circles) with hand-derived error bands: md_class, ls_class
// and the inline predicates of k_ls_eval / k_pt_eval (lst_cuts.cuh, lst_cuts_pt.cuh).  The claim is that no such
// decision differs from the exact cut list of CUTS.md sections 3, 4, 7 and that none hides a near-threshold
// candidate.  The kernels here test that claim on the batch a context has just run, without any of that
// machinery: EVERY candidate of the stage (all hit pairs of a module; all MD pairs along the connection map; all
// (seed, T3) and (seed, T5) pairs of an event) goes through the exact test -- the same md_test / ls_test /
// PtCand::test the chain uses when it cannot decide, which the parity tests check against the oracle -- and
// three numbers per stage are accumulated: candidates, accepted, near-threshold, plus an order-independent
// 64-bit hash of the accepted candidates' identities.  A second set of kernels hashes what the chain stored.
// Any wrong decision of a pre-filter shows:
//   dropped, but the exact cuts accept        -> an accepted candidate is missing from the chain's objects (count, hash)
//   accepted without the exact cuts (MD only), but they reject -> an object too many (count, hash)
//   decided either way, but the exact cuts flag it near        -> the chain's near counter is lower
// (the chain never raises a near flag without the exact cuts, so two errors cannot cancel in that counter).
// T3, T5 and T4 have no pre-filter (k_stage runs the exact cuts on every candidate) and are not re-evaluated.
// Never part of a timed path: called only through lst_ctx_audit.
#pragma once
#include "lst_pt.cuh"

namespace lst {

enum AuditStage { AU_MD = 0, AU_LS, AU_PT3, AU_PT5, AU_N };

struct AuditAcc {  // device accumulator of lst_ctx_audit
  unsigned long long cand[AU_N], acc[AU_N], near[AU_N], hash_exact[AU_N], hash_chain[AU_N];
};

__device__ __forceinline__ unsigned long long audit_mix(unsigned long long a, unsigned long long b,
                                                        unsigned long long c) {
  unsigned long long z = a * 0x9e3779b97f4a7c15ull + b * 0xc2b2ae3d27d4eb4full + c * 0x165667b19e3779f9ull + 1ull;
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  return z ^ (z >> 31);
}

// every thread of the block calls this once at the end of a kernel
__device__ __forceinline__ void audit_flush(AuditAcc* out, int stage, unsigned long long cand, unsigned long long acc,
                                            unsigned long long near, unsigned long long hash) {
  cand = warp_sum_u64(cand);
  acc = warp_sum_u64(acc);
  near = warp_sum_u64(near);
  hash = warp_sum_u64(hash);
  if ((threadIdx.x & 31) == 0) {
    if (cand) atomicAdd(&out->cand[stage], cand);
    if (acc) atomicAdd(&out->acc[stage], acc);
    if (near) atomicAdd(&out->near[stage], near);
    if (hash) atomicAdd(&out->hash_exact[stage], hash);
  }
}

// CUTS.md section 3: every (lower hit, upper hit) pair of every module of every event; one upper hit per thread
__global__ void __launch_bounds__(kBlock) k_audit_md(Dev d, AuditAcc* out) {
  load_batch(d);
  unsigned long long cand = 0, acc = 0, near = 0, hash = 0;
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < d.n_hits; i += gridDim.x * blockDim.x) {
    const int2 ig = hit_ig(d, i);
    if (!(ig.y & 1)) continue;  // lower-sensor hit
    const int gm = ig.y >> 1, ev = gm / d.n_mod;
    const bool endcap = d.subdet[gm - ev * d.n_mod] != 0;
    const float4 hb = hit_xyzr(d, i);
    for (int a = d.sens_begin[ig.y - 1]; a < d.sens_begin[ig.y]; ++a) {
      float ux, uy;
      const unsigned r = md_test(d.cuts, endcap, hit_xyzr(d, a), hb, ux, uy);
      ++cand;
      near += (r >> 1) & 1u;
      if (r & ACC) {
        ++acc;
        hash += audit_mix((unsigned long long)ev, (unsigned long long)hit_ig(d, a).x, (unsigned long long)ig.x);
      }
    }
  }
  audit_flush(out, AU_MD, cand, acc, near, hash);
}

// CUTS.md section 4: every MD A with every MD of every module its module's row of the connection map names
__global__ void __launch_bounds__(kBlock) k_audit_ls(Dev d, AuditAcc* out) {
  load_batch(d);
  const int n_md = d.ctl->total[K_MD];
  unsigned long long cand = 0, acc = 0, near = 0, hash = 0;
  for (int A = blockIdx.x * blockDim.x + threadIdx.x; A < n_md; A += gridDim.x * blockDim.x) {
    const int info = d.md_info[A];
    const int gm = info >> 1, ev = gm / d.n_mod, gb = ev * d.n_mod, mod = gm - gb;
    const float4 a = d.md_a[A];
    const float2 ua = d.md_u[A];
    for (int k = d.conn_off[mod]; k < d.conn_off[mod + 1]; ++k) {
      const int m2 = d.conn_tgt[k];
      const bool eB = d.subdet[m2] != 0;
      for (int B = d.mod_md_begin[gb + m2]; B < d.mod_md_begin[gb + m2 + 1]; ++B) {
        float kappa;
        const unsigned r = ls_test(d.cuts, a, ua, info & 1, d.md_a[B], d.md_u[B], eB, kappa);
        ++cand;
        near += (r >> 1) & 1u;
        if (r & ACC) {
          ++acc;
          hash += audit_mix(1ull, (unsigned long long)A, (unsigned long long)B);
        }
      }
    }
  }
  audit_flush(out, AU_LS, cand, acc, near, hash);
}

// CUTS.md section 7: every seed of an event with every T3 (IS5: T5) of that event.  grid (x, events)
template <bool IS5>
__global__ void __launch_bounds__(kBlock) k_audit_pt(Dev d, AuditAcc* out) {
  load_batch(d);
  const int ev = blockIdx.y;
  unsigned long long cand = 0, acc = 0, near = 0, hash = 0;
  if (ev < d.n_events) {
    int c0, c1;
    event_cands<IS5>(d, ev, c0, c1);
    const int p0 = d.pls_ev_off[ev], p1 = d.pls_ev_off[ev + 1];
    const long long n_c = c1 - c0, total = (long long)(p1 - p0) * n_c;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
      const int p = p0 + (int)(i / n_c), t = c0 + (int)(i % n_c);
      float score;
      const unsigned r = PtCand<IS5>::test(d, seed_from_table(d, p), t, score);
      ++cand;
      near += (r >> 1) & 1u;
      if (r & ACC) {
        ++acc;
        hash += audit_mix(IS5 ? 3ull : 2ull, (unsigned long long)p, (unsigned long long)t);
      }
    }
  }
  audit_flush(out, IS5 ? AU_PT5 : AU_PT3, cand, acc, near, hash);
}

// what the chain stored: the same identities, hashed the same way
__global__ void __launch_bounds__(kBlock) k_audit_chain(Dev d, AuditAcc* out, int do_md, int do_ls, int do_pt) {
  load_batch(d);
  const int n_md = d.ctl->total[K_MD], n_ls = d.ctl->total[K_LS], n_p3 = d.ctl->total[K_PT3], n_p5 = d.ctl->total[K_PT5];
  unsigned long long h[AU_N] = {0, 0, 0, 0};
  const int stride = gridDim.x * blockDim.x, first = blockIdx.x * blockDim.x + threadIdx.x;
  if (do_md)
    for (int m = first; m < n_md; m += stride) {
      const int2 hh = d.md_hit[m];
      h[AU_MD] += audit_mix((unsigned long long)((d.md_info[m] >> 1) / d.n_mod), (unsigned long long)hh.x, (unsigned long long)hh.y);
    }
  if (do_ls)
    for (int l = first; l < n_ls; l += stride) {
      const int2 ab = d.ls_md[l];
      h[AU_LS] += audit_mix(1ull, (unsigned long long)ab.x, (unsigned long long)ab.y);
    }
  if (do_pt) {
    for (int i = first; i < n_p3; i += stride) {
      const int2 pt = d.pt3[i];
      h[AU_PT3] += audit_mix(2ull, (unsigned long long)pt.x, (unsigned long long)pt.y);
    }
    for (int i = first; i < n_p5; i += stride) {
      const int2 pt = d.pt5[i];
      h[AU_PT5] += audit_mix(3ull, (unsigned long long)pt.x, (unsigned long long)pt.y);
    }
  }
#pragma unroll
  for (int s = 0; s < AU_N; ++s) {
    const unsigned long long v = warp_sum_u64(h[s]);
    if ((threadIdx.x & 31) == 0 && v) atomicAdd(&out->hash_chain[s], v);
  }
}

}  // namespace lst
