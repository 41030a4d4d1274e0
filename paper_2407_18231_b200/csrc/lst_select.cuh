// lst_select.cuh -- step a6: duplicate removal and track-candidate selection (CUTS.md section 8,
// PAPER.md:31-34, 56).  Set-defined rules; the candidates that can overlap an object are found
// through an inverted index "objects containing MD m" (three lists per MD: T5, pT5, pT3), built
// with one counting pass, the generic scan and one fill pass.  By the pigeonhole principle an
// object sharing >= 3 of X's 5 MDs contains X.md[0], [2] or [4]; one sharing >= 2 of 5 contains one
// of X.md[0..3]; one sharing >= 2 of X's 3 MDs contains X.md[0] or [1].
#pragma once
#include "lst_ls.cuh"
#include "lst_pt.cuh"

namespace lst {

__device__ __forceinline__ int ev_of_md(const Dev& d, int md) { return (d.md_info[md] >> 1) / d.n_mod; }

// first object index of every event, per kind: ev_first[kind * (n_events + 1) + ev]
__global__ void k_event_ranges(Dev d, int* ev_first) {
  const int E1 = d.n_events + 1;
  for (int ev = threadIdx.x; ev < E1; ev += blockDim.x) {
    const int p = d.pls_ev_off[ev];
    const int md = d.ctl->total[K_MD] > 0 ? d.mod_md_begin[min(ev, d.n_events) * d.n_mod] : 0;
    const int ls = d.ctl->total[K_LS] > 0 ? d.md_ls_begin[md] : 0;
    const int t3 = d.ctl->total[K_T3] > 0 ? d.ls_t3_begin[ls] : 0;
    const int t5 = d.ctl->total[K_T5] > 0 ? d.t3_t5_begin[t3] : 0;
    ev_first[K_MD * E1 + ev] = md;
    ev_first[K_LS * E1 + ev] = ls;
    ev_first[K_T3 * E1 + ev] = t3;
    ev_first[K_T5 * E1 + ev] = t5;
    ev_first[K_PT3 * E1 + ev] = d.ctl->total[K_PT3] > 0 ? d.pls_pt3_begin[p] : 0;
    ev_first[K_PT5 * E1 + ev] = d.ctl->total[K_PT5] > 0 ? d.pls_pt5_begin[p] : 0;
  }
}

__global__ void __launch_bounds__(kBlock) k_sel_prepare(Dev d) {
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_slots = 3 * d.ctl->total[K_MD];
  for (int i = i0; i <= n_slots; i += stride) {
    d.idx_cnt[i] = 0;
    d.idx_cur[i] = 0;
  }
  for (int i = i0; i <= 4 * d.n_events; i += stride) {
    d.tc_cnt[i] = 0;
    d.tc_cur[i] = 0;
  }
  for (int i = i0; i < d.n_pls; i += stride) d.linked[i] = 0;
}

// FILL = false: count list lengths; FILL = true: write the lists (order inside a list is free)
template <bool FILL>
__global__ void __launch_bounds__(kBlock) k_index(Dev d) {
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_md = d.ctl->total[K_MD];
  const int n_t5 = d.ctl->total[K_T5], n_pt5 = d.ctl->total[K_PT5], n_pt3 = d.ctl->total[K_PT3];
  for (int i = i0; i < n_t5 + n_pt5 + n_pt3; i += stride) {
    int obj, base, nmd;
    const int* md;
    int tmp[3];
    if (i < n_t5) {
      obj = i; base = 0; nmd = 5; md = d.t5_md + 5 * (size_t)obj;
    } else if (i < n_t5 + n_pt5) {
      obj = i - n_t5; base = n_md; nmd = 5; md = d.t5_md + 5 * (size_t)d.pt5[obj].y;
    } else {
      obj = i - n_t5 - n_pt5; base = 2 * n_md; nmd = 3;
      const int4 m = d.t3_md[d.pt3[obj].y];
      tmp[0] = m.x; tmp[1] = m.y; tmp[2] = m.z;
      md = tmp;
    }
    for (int k = 0; k < nmd; ++k) {
      const int slot = base + md[k];
      if (!FILL) {
        atomicAdd(d.idx_cnt + slot, 1);
      } else {
        const int pos = d.idx_begin[slot] + atomicAdd(d.idx_cur + slot, 1);
        if (pos < d.cap_idx) d.idx_list[pos] = obj;
      }
    }
  }
}

__device__ __forceinline__ int share(const int* a, int na, const int* b, int nb) {
  int s = 0;
  for (int i = 0; i < na; ++i)
    for (int j = 0; j < nb; ++j) s += (a[i] == b[j]);
  return s;
}

// CUTS.md section 8: better(Y, X); key = (pls,) + hit pairs of the MDs in order
__device__ __forceinline__ bool better(const Dev& d, float sY, int pY, const int* mY, float sX, int pX,
                                       const int* mX, int nmd) {
  if (sY < sX) return true;
  if (!(sY == sX)) return false;
  if (pY != pX) return pY < pX;
  for (int i = 0; i < nmd; ++i) {
    const int2 hy = d.md_hit[mY[i]], hx = d.md_hit[mX[i]];
    if (hy.x != hx.x) return hy.x < hx.x;
    if (hy.y != hx.y) return hy.y < hx.y;
  }
  return false;
}

__device__ __forceinline__ void load_t3_md(const Dev& d, int t3, int* m) {
  const int4 v = d.t3_md[t3];
  m[0] = v.x; m[1] = v.y; m[2] = v.z;
}
__device__ __forceinline__ void load_t5_md(const Dev& d, int t5, int* m) {
  const int* p = d.t5_md + 5 * (size_t)t5;
#pragma unroll
  for (int k = 0; k < 5; ++k) m[k] = p[k];
}

// rule 1: pT5 vs pT5
__global__ void __launch_bounds__(kBlock) k_rule1(Dev d) {
  const int stride = gridDim.x * blockDim.x;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_PT5];
  for (int X = blockIdx.x * blockDim.x + threadIdx.x; X < n; X += stride) {
    const int2 x = d.pt5[X];
    const float sX = d.pt5_score[X];
    int mX[5], mY[5];
    load_t5_md(d, x.y, mX);
    bool keep = true;
    for (int Y = d.pls_pt5_begin[x.x]; Y < d.pls_pt5_begin[x.x + 1] && keep; ++Y) {
      if (Y == X) continue;
      load_t5_md(d, d.pt5[Y].y, mY);
      if (better(d, d.pt5_score[Y], x.x, mY, sX, x.x, mX, 5)) keep = false;
    }
    for (int k = 0; k < 5 && keep; k += 2) {
      const int slot = n_md + mX[k];
      for (int j = d.idx_begin[slot]; j < d.idx_begin[slot + 1] && keep; ++j) {
        const int Y = d.idx_list[j];
        if (Y == X) continue;
        const int2 y = d.pt5[Y];
        load_t5_md(d, y.y, mY);
        if (share(mY, 5, mX, 5) >= 3 && better(d, d.pt5_score[Y], y.x, mY, sX, x.x, mX, 5)) keep = false;
      }
    }
    d.keep5[X] = keep;
    if (keep) {
      d.linked[x.x] = 1;  // one writer per value; pT3 survivors OR in 2 (rule 2)
      atomicAdd(d.tc_cnt + 4 * d.pls_event[x.x] + 0, 1);
    }
  }
}

// rule 2: pT3 vs pT3, then vs surviving pT5
__global__ void __launch_bounds__(kBlock) k_rule2(Dev d) {
  const int stride = gridDim.x * blockDim.x;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_PT3], n_pt5 = d.ctl->total[K_PT5];
  for (int X = blockIdx.x * blockDim.x + threadIdx.x; X < n; X += stride) {
    const int2 x = d.pt3[X];
    const float sX = d.pt3_score[X];
    int mX[3], mY[5];
    load_t3_md(d, x.y, mX);
    bool keep = !(d.linked[x.x] & 1);  // rule 2b: seed already in a surviving pT5
    for (int Y = d.pls_pt3_begin[x.x]; Y < d.pls_pt3_begin[x.x + 1] && keep; ++Y) {
      if (Y == X) continue;
      load_t3_md(d, d.pt3[Y].y, mY);
      if (better(d, d.pt3_score[Y], x.x, mY, sX, x.x, mX, 3)) keep = false;
    }
    for (int k = 0; k < 2 && keep; ++k) {
      int slot = 2 * n_md + mX[k];
      for (int j = d.idx_begin[slot]; j < d.idx_begin[slot + 1] && keep; ++j) {
        const int Y = d.idx_list[j];
        if (Y == X) continue;
        const int2 y = d.pt3[Y];
        load_t3_md(d, y.y, mY);
        if (share(mY, 3, mX, 3) >= 2 && better(d, d.pt3_score[Y], y.x, mY, sX, x.x, mX, 3)) keep = false;
      }
      if (n_pt5 > 0) {
        slot = n_md + mX[k];
        for (int j = d.idx_begin[slot]; j < d.idx_begin[slot + 1] && keep; ++j) {
          const int Z = d.idx_list[j];
          if (!d.keep5[Z]) continue;
          load_t5_md(d, d.pt5[Z].y, mY);
          if (share(mX, 3, mY, 5) >= 2) keep = false;
        }
      }
    }
    d.keep3[X] = keep;
    if (keep) atomicAdd(d.tc_cnt + 4 * d.pls_event[x.x] + 1, 1);
  }
}

// rule 3: T5 vs T5, vs surviving pT5, vs surviving pT3; rule 4: unlinked pLS
__global__ void __launch_bounds__(kBlock) k_rule3(Dev d) {
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_md = d.ctl->total[K_MD], n = d.ctl->total[K_T5];
  const int n_pt5 = d.ctl->total[K_PT5], n_pt3 = d.ctl->total[K_PT3];
  for (int X = i0; X < n; X += stride) {
    const float sX = d.t5_score[X];
    int mX[5], mY[5];
    load_t5_md(d, X, mX);
    bool keep = true;
    for (int k = 0; k < 5 && keep; k += 2) {
      const int slot = mX[k];
      for (int j = d.idx_begin[slot]; j < d.idx_begin[slot + 1] && keep; ++j) {
        const int Y = d.idx_list[j];
        if (Y == X) continue;
        load_t5_md(d, Y, mY);
        if (share(mY, 5, mX, 5) >= 3 && better(d, d.t5_score[Y], -1, mY, sX, -1, mX, 5)) keep = false;
      }
    }
    for (int k = 0; k < 4 && keep; ++k) {
      if (n_pt5 > 0) {
        const int slot = n_md + mX[k];
        for (int j = d.idx_begin[slot]; j < d.idx_begin[slot + 1] && keep; ++j) {
          const int Z = d.idx_list[j];
          if (!d.keep5[Z]) continue;
          load_t5_md(d, d.pt5[Z].y, mY);
          if (share(mX, 5, mY, 5) >= 2) keep = false;
        }
      }
      if (n_pt3 > 0) {
        const int slot = 2 * n_md + mX[k];
        for (int j = d.idx_begin[slot]; j < d.idx_begin[slot + 1] && keep; ++j) {
          const int Z = d.idx_list[j];
          if (!d.keep3[Z]) continue;
          load_t3_md(d, d.pt3[Z].y, mY);
          if (share(mX, 5, mY, 3) >= 2) keep = false;
        }
      }
    }
    d.keepT[X] = keep;
    if (keep) atomicAdd(d.tc_cnt + 4 * ev_of_md(d, mX[0]) + 2, 1);
  }
  // rule 4: a pLS is linked if it seeds a surviving pT5 (flag set by rule 1) or pT3
  for (int p = i0; p < d.n_pls; p += stride) {
    bool lk = d.linked[p] & 1;
    for (int Y = n_pt3 > 0 ? d.pls_pt3_begin[p] : 0; !lk && n_pt3 > 0 && Y < d.pls_pt3_begin[p + 1]; ++Y)
      lk = d.keep3[Y];
    d.linked[p] = lk;
    if (!lk) atomicAdd(d.tc_cnt + 4 * d.pls_event[p] + 3, 1);
  }
}

// track candidates: (type, pls, t5, t3, hit_idx[12]) per event in class order; event-local indices
__global__ void __launch_bounds__(kBlock) k_tc_emit(Dev d, const int* __restrict__ ev_first) {
  const int stride = gridDim.x * blockDim.x, i0 = blockIdx.x * blockDim.x + threadIdx.x;
  const int E1 = d.n_events + 1;
  const int n_pt5 = d.ctl->total[K_PT5], n_pt3 = d.ctl->total[K_PT3], n_t5 = d.ctl->total[K_T5];
  const int total = d.tc_begin[4 * d.n_events];
  const bool fits = total <= d.cap[K_TC];
  if (i0 == 0) {
    if (!fits) atomicOr(&d.ctl->error, E_CAP_TC);
    d.ctl->total[K_TC] = fits ? total : 0;
  }
  if (!fits) return;
  for (int i = i0; i < n_pt5 + n_pt3 + n_t5 + d.n_pls; i += stride) {
    int cls, ev, pls = -1, t5 = -1, t3 = -1, nmd = 0;
    int md[5];
    if (i < n_pt5) {
      if (!d.keep5[i]) continue;
      cls = 0; pls = d.pt5[i].x; t5 = d.pt5[i].y; ev = d.pls_event[pls];
      load_t5_md(d, t5, md); nmd = 5;
    } else if (i < n_pt5 + n_pt3) {
      const int X = i - n_pt5;
      if (!d.keep3[X]) continue;
      cls = 1; pls = d.pt3[X].x; t3 = d.pt3[X].y; ev = d.pls_event[pls];
      load_t3_md(d, t3, md); nmd = 3;
    } else if (i < n_pt5 + n_pt3 + n_t5) {
      t5 = i - n_pt5 - n_pt3;
      if (!d.keepT[t5]) continue;
      cls = 2; load_t5_md(d, t5, md); nmd = 5; ev = ev_of_md(d, md[0]);
    } else {
      pls = i - n_pt5 - n_pt3 - n_t5;
      if (d.linked[pls]) continue;
      cls = 3; ev = d.pls_event[pls];
    }
    const int pos = d.tc_begin[4 * ev + cls] + atomicAdd(d.tc_cur + 4 * ev + cls, 1);
    int* o = d.tc + 16 * (size_t)pos;
    o[0] = cls;
    o[1] = pls >= 0 ? pls - d.pls_ev_off[ev] : -1;
    o[2] = t5 >= 0 ? t5 - ev_first[K_T5 * E1 + ev] : -1;
    o[3] = t3 >= 0 ? t3 - ev_first[K_T3 * E1 + ev] : -1;
    for (int k = 0; k < 6; ++k) {
      int2 h = make_int2(-1, -1);
      if (k < nmd) h = d.md_hit[md[k]];
      o[4 + 2 * k] = h.x;
      o[5 + 2 * k] = h.y;
    }
  }
}

}  // namespace lst
