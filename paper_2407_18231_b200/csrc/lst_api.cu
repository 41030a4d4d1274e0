// lst_api.cu -- the C ABI of include/lst.h: geometry upload, contexts (workspace + stream), the
// launch sequence of one batch, result read-back.  Host code only marshals; every step of the
// chain runs in the kernels of lst_ingest/lst_stages/lst_pt/lst_select.cuh.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/lst.h"
#include "lst_select.cuh"
#include "lst_audit.cuh"

using namespace lst;

namespace {

constexpr uint64_t MAGIC_GEOM = 0x4c535447454f4d31ull;  // "LSTGEOM1"
constexpr uint64_t MAGIC_CTX = 0x4c53544354583031ull;
constexpr uint64_t MAGIC_OUT = 0x4c53544f55543031ull;
constexpr int kMaxKernels = 32;

#define CK(call)                                  \
  do {                                            \
    cudaError_t e_ = (call);                      \
    if (e_ != cudaSuccess) return LST_ERR_CUDA;   \
  } while (0)

}  // namespace

struct lst_geometry {
  uint64_t magic;
  int n_mod, n_edges, max_deg;
  int *d_subdet, *d_conn_off, *d_conn_tgt;
  lst_params params;
  Cuts cuts;
  lst_ctx* default_ctx;   // lst_run_event's context, created on first use under default_mu
  std::mutex default_mu;  // serialises lst_run_event on one geometry
  int n_sm;
};

struct lst_ctx {
  uint64_t magic;
  lst_geometry* g;
  lst_caps caps;
  cudaStream_t stream;
  Dev dev;                    // pointer table (inputs patched per run)
  std::vector<void*> allocs;  // device allocations
  size_t bytes;
  void* zero_region;
  size_t zero_bytes;
  // device staging of host inputs
  float *in_x, *in_y, *in_z;
  int* in_sensor;
  float *p_pt, *p_x0, *p_y0, *p_z0, *p_x1, *p_y1, *p_z1;
  int* p_q;
  int *d_hit_ev_off, *d_pls_ev_off;
  Batch* d_batch;
  cudaStream_t owned_stream;  // non-null: created by the library (lst_run_event's context), destroyed with the context
  cudaGraphExec_t graph;   // the launch sequence of one batch, captured on first use (kernel arguments never change)
  bool use_graph;
  // pinned host mirrors
  Ctl* h_ctl;
  unsigned long long* h_ev_cnt;  // [max_events][kEvCnt]
  int* h_ev_first;  // [K_NKINDS][max_events + 1]
  int* h_tc_begin;  // [kTcClasses * max_events + 1] first track candidate of every (event, class)
  int h_pls_off[2];
  std::vector<int> last_hit_off, last_pls_off;
  int last_n_events;
  bool synced;
  int occ_md, occ_ls, occ_pt;  // resident blocks per SM of the three heavy kernels (occupancy)
  int blocks_per_sm;           // lst_ctx_set_blocks_per_sm (default 8 = fill the GPU)
  // timing
  bool timing;
  cudaEvent_t ev[kMaxKernels + 1];
  const char* kname[kMaxKernels];
  int n_kernels;
};

extern "C" const char* lst_strerror(int s) {
  switch (s) {
    case LST_OK: return "ok";
    case LST_ERR_ARG: return "invalid argument (null pointer, bad size, sensor id or event offsets out of range)";
    case LST_ERR_CUDA: return "CUDA runtime error (no device, out of memory or launch failure)";
    case LST_ERR_CAPACITY: return "object array capacity of the context exceeded (nothing was truncated)";
    case LST_ERR_GEOMETRY: return "malformed module table or connection map";
    case LST_ERR_LIMIT: return "size beyond the fixed maximum of a non-allocating entry point (LST_SCAN_STATIC_MAX_N)";
    default: return "unknown status";
  }
}

extern "C" void lst_default_params(lst_params* p) {  // CUTS.md section 1
  if (!p) return;
  p->b_field = 3.8f;  p->pt_min = 0.8f;  p->z0_max = 15.0f;
  p->md_b_phi_tol = 0.06f;  p->md_z_tol = 0.9f;  p->md_e_slope = 1.15f;  p->md_e_tol = 0.015f;
  p->ls_kappa_max = 1.05f;  p->ls_z_tol = 1.0f;  p->ls_dir_tol = 0.05f;
  p->t3_kappa_max = 1.10f;  p->t3_z_tol0 = 1.0f;  p->t3_z_tol1 = 0.6f;
  p->t5_tol0 = 4e-4f;  p->t5_tol1 = 0.05f;
  p->pt_gate_tol = 0.05f;  p->pt_k_tol0 = 5e-4f;  p->pt_k_tol1 = 0.10f;  p->pt_z_tol = 2.0f;
  p->near_rel = 1e-5f;
  p->stage_mask = 0x3f;
  p->t4_tol0 = 4e-4f;  p->t4_tol1 = 0.05f;              // CUTS.md section 10
  p->t5_mlp_scale = 100.0f;  p->t5_mlp_thr = 1.0f;      // CUTS.md section 11; the weights are inputs (default 0)
  for (int i = 0; i < 65; ++i) p->t5_mlp[i] = 0.0f;
}

extern "C" void lst_default_caps(lst_caps* c) {
  if (!c) return;
  c->max_events = 16;
  c->max_hits = 4 << 20;
  c->max_pls = 64 << 10;
  c->max_md = 1 << 20;
  c->max_ls = 2 << 20;
  c->max_t3 = 2 << 20;
  c->max_t5 = 1 << 20;
  c->max_pt3 = 1 << 20;
  c->max_pt5 = 1 << 20;
  c->max_tc = 256 << 10;
  c->max_t4 = 2 << 20;
}

static Cuts make_cuts(const lst_params& p) {  // CUTS.md section 1, derived constants in binary32
  Cuts c;
  c.z0_max = p.z0_max;
  c.md_b_phi_tol = p.md_b_phi_tol;  c.md_z_tol = p.md_z_tol;
  c.md_e_slope = p.md_e_slope;  c.md_e_tol = p.md_e_tol;
  c.ls_kappa_max = p.ls_kappa_max;  c.ls_z_tol = p.ls_z_tol;  c.ls_dir_tol = p.ls_dir_tol;
  c.t3_kappa_max = p.t3_kappa_max;  c.t3_z_tol0 = p.t3_z_tol0;  c.t3_z_tol1 = p.t3_z_tol1;
  c.t5_tol0 = p.t5_tol0;  c.t5_tol1 = p.t5_tol1;
  c.pt_gate_tol = p.pt_gate_tol;  c.pt_k_tol0 = p.pt_k_tol0;  c.pt_k_tol1 = p.pt_k_tol1;
  c.pt_z_tol = p.pt_z_tol;
  c.near_rel = p.near_rel;
  volatile float kr = 100.0f / (0.3f * p.b_field);
  volatile float r_min = p.pt_min * kr;
  volatile float inv = 1.0f / (2.0f * r_min);
  c.kr = kr;  c.r_min = r_min;  c.inv_2rmin = inv;
  c.stage_mask = p.stage_mask;
  c.t4_tol0 = p.t4_tol0;  c.t4_tol1 = p.t4_tol1;
  c.t5_mlp_scale = p.t5_mlp_scale;  c.t5_mlp_thr = p.t5_mlp_thr;
  for (int i = 0; i < 65; ++i) c.t5_mlp[i] = p.t5_mlp[i];
  return c;
}

extern "C" int lst_load_geometry(const lst_module* modules, int32_t n_modules, const int32_t* conn_offsets,
                                 const int32_t* conn_targets, const lst_params* params, lst_geometry** out) {
  if (!out) return LST_ERR_ARG;
  *out = nullptr;
  if (!modules || n_modules <= 0 || !conn_offsets) return LST_ERR_ARG;
  // The approximate pre-filters in front of the exact cuts (lst_cuts.cuh, lst_cuts_pt.cuh, lst_ls.cuh, lst_pt.cuh)
  // leave every candidate within NEAR_REL = 1e-5 of a threshold to the exact cut; their bands are constants sized
  // for that value.  A wider near window would be classified by them and never counted: refused, not mis-counted.
  if (params && !(params->near_rel >= 0.0f && params->near_rel <= 1e-5f)) return LST_ERR_ARG;
  if (conn_offsets[0] != 0) return LST_ERR_GEOMETRY;
  for (int m = 0; m < n_modules; ++m) {
    if (conn_offsets[m + 1] < conn_offsets[m]) return LST_ERR_GEOMETRY;
    if (modules[m].subdet != 0 && modules[m].subdet != 1) return LST_ERR_GEOMETRY;
  }
  const int n_edges = conn_offsets[n_modules];
  int max_deg = 0;
  for (int m = 0; m < n_modules; ++m)
    if (conn_offsets[m + 1] - conn_offsets[m] > max_deg) max_deg = conn_offsets[m + 1] - conn_offsets[m];
  if (n_edges > 0 && !conn_targets) return LST_ERR_ARG;
  if (max_deg > kLsRanges) return LST_ERR_GEOMETRY;  // longest connection-map row the LS stage's tables hold
  for (int k = 0; k < n_edges; ++k)
    if (conn_targets[k] < 0 || conn_targets[k] >= n_modules) return LST_ERR_GEOMETRY;

  int dev = 0;
  CK(cudaGetDevice(&dev));
  lst_geometry* g = new (std::nothrow) lst_geometry();
  if (!g) return LST_ERR_CUDA;
  g->magic = MAGIC_GEOM;
  g->n_mod = n_modules;
  g->n_edges = n_edges;
  g->max_deg = max_deg;
  g->default_ctx = nullptr;
  if (params) g->params = *params; else lst_default_params(&g->params);
  g->cuts = make_cuts(g->params);
  if (cudaDeviceGetAttribute(&g->n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    delete g;
    return LST_ERR_CUDA;
  }
  std::vector<int> sub(n_modules);
  for (int m = 0; m < n_modules; ++m) sub[m] = modules[m].subdet;
  bool ok = cudaMalloc(&g->d_subdet, sizeof(int) * n_modules) == cudaSuccess &&
            cudaMalloc(&g->d_conn_off, sizeof(int) * (n_modules + 1)) == cudaSuccess &&
            cudaMalloc(&g->d_conn_tgt, sizeof(int) * (n_edges > 0 ? n_edges : 1)) == cudaSuccess;
  ok = ok && cudaMemcpy(g->d_subdet, sub.data(), sizeof(int) * n_modules, cudaMemcpyHostToDevice) == cudaSuccess;
  ok = ok && cudaMemcpy(g->d_conn_off, conn_offsets, sizeof(int) * (n_modules + 1), cudaMemcpyHostToDevice) == cudaSuccess;
  if (ok && n_edges > 0)
    ok = cudaMemcpy(g->d_conn_tgt, conn_targets, sizeof(int) * n_edges, cudaMemcpyHostToDevice) == cudaSuccess;
  if (!ok) {
    cudaFree(g->d_subdet);  cudaFree(g->d_conn_off);  cudaFree(g->d_conn_tgt);
    delete g;
    return LST_ERR_CUDA;
  }
  *out = g;
  return LST_OK;
}

// ---- workspace layout: one device allocation, carved by a bump pointer -------------------------
namespace {

struct Bump {
  char* base;
  size_t off;
  template <class T>
  T* take(size_t n) {
    off = (off + 255) & ~size_t(255);
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += sizeof(T) * (n ? n : 1);
    return p;
  }
};

inline int tiles_of(long long n, int tile) { return (int)((n + tile - 1) / tile) + 2; }

// Fills the pointer table of `dev` (pointers are offsets from `base`; base == nullptr only sizes).
// Rule: everything a kernel reads before a kernel of the SAME batch has written it -- counters, cursors, tickets,
// status words, flags that are only ever set (linked) -- lives in the leading region that is cleared per batch.
// An array outside it still holds the previous batch of this context.
// Returns total bytes; *zero_bytes = size of the leading region that is memset per batch.
size_t layout(const lst_caps& c, int n_mod, char* base, Dev& d, lst_ctx* ctx, size_t* zero_bytes) {
  Bump b{base, 0};
  const long long n_sens = (long long)c.max_events * 2 * n_mod;
  // --- zeroed per batch ---
  d.ctl = b.take<Ctl>(1);
  d.ev_cnt = b.take<unsigned long long>((size_t)c.max_events * kEvCnt);
  d.tstate[T_SENS] = nullptr;  // unused (the sensor scan is local to k_ingest)
  d.tstate[T_MD] = b.take<unsigned long long>(tiles_of((long long)c.max_hits + 1, kBlock * kMdPlaceItems));
  d.tstate[T_LS] = b.take<unsigned long long>(tiles_of((long long)c.max_md + 1, kBlock));
  d.tstate[T_T3] = b.take<unsigned long long>(tiles_of(c.max_ls, kBlock));
  d.tstate[T_T5] = b.take<unsigned long long>(tiles_of(c.max_t3, kBlock));
  d.tstate[T_PT] = nullptr;  // ticket only
  d.tstate[T_PP3] = b.take<unsigned long long>(tiles_of((long long)c.max_pls + 1, kScanTile));
  d.tstate[T_PP5] = b.take<unsigned long long>(tiles_of((long long)c.max_pls + 1, kScanTile));
  d.tstate[T_T4] = b.take<unsigned long long>(tiles_of(c.max_t3, kBlock));
  d.tstate[T_LSE] = nullptr;  // ticket only
  d.anc_bin_cnt = b.take<int>((size_t)c.max_events * kAncBins);
  d.anc_done = b.take<int>(c.max_events);
  d.pls_pt3_cnt = b.take<int>((size_t)c.max_pls + 1);
  d.pls_pt5_cnt = b.take<int>((size_t)c.max_pls + 1);
  d.pls_pt3_cur = b.take<int>(c.max_pls);
  d.pls_pt5_cur = b.take<int>(c.max_pls);
  d.tc_cnt = b.take<int>(kTcClasses * (size_t)c.max_events + 1);
  d.tc_cur = b.take<int>(kTcClasses * (size_t)c.max_events + 1);
  d.linked = b.take<unsigned char>(c.max_pls);
#ifdef LST_RULE3_SKIP_COVERED
  d.t5_cov = b.take<unsigned char>(c.max_t5);
#endif
  d.ls_cnt = b.take<int>(c.max_md);
  d.ls_cur = b.take<int>(c.max_md);
  b.off = (b.off + 255) & ~size_t(255);
  if (zero_bytes) *zero_bytes = b.off;
  // --- a0 ---
  d.sens_begin = b.take<int>(n_sens + 1);
  d.hit_rank = b.take<int>(c.max_hits);
  d.chunk_cnt = b.take<int>((size_t)n_sens * kIngestChunks);
  d.chunk_part = b.take<int>((size_t)c.max_events * kIngestChunks * kIngestScanParts);
  d.hit = b.take<float4>(2 * (size_t)c.max_hits);
  // --- a1..a4 ---
  {
    size_t sz = sizeof(LsAccepted) * (size_t)c.max_ls;
    const size_t other = sizeof(PtAccepted) * (size_t)c.max_pt3;
    sz = other > sz ? other : sz;
    d.ev_scratch = b.take<char>(sz);
    d.ev_scratch2 = b.take<char>(sizeof(PtAccepted) * (size_t)c.max_pt5);
  }
  d.md_cnt = b.take<int2>(c.max_hits);
  d.md_stash = b.take<int>(4 * (size_t)c.max_hits);
  d.mod_md_begin = b.take<int>(n_sens / 2 + 1);
  d.md_hit = b.take<int2>(c.max_md);
  d.md_info = b.take<int>(c.max_md);
  d.md_a = b.take<float4>(c.max_md);
  d.md_u = b.take<float2>(c.max_md);
  d.md_ls_begin = b.take<int>((size_t)c.max_md + 1);
  d.ls_md = b.take<int2>(c.max_ls);
  d.ls_kappa = b.take<float>(c.max_ls);
  d.ls_t3_begin = b.take<int>((size_t)c.max_ls + 1);
  d.t3_ls = b.take<int2>(c.max_t3);
  d.t3_md = b.take<int4>(c.max_t3);
  d.t3_k = b.take<float>(c.max_t3);
  d.t3_l = b.take<float4>(c.max_t3);
  d.t3_q = b.take<float4>(c.max_t3);
  d.t3_t5_begin = b.take<int>((size_t)c.max_t3 + 1);
  d.t5_t3 = b.take<int2>(c.max_t5);
  d.t5_md = b.take<int>(5 * (size_t)c.max_t5);
  d.t5_score = b.take<float>(c.max_t5);
  d.t5_l = b.take<float4>(c.max_t5);
  d.t5_kio = b.take<float2>(c.max_t5);
  d.t3_t4_begin = b.take<int>((size_t)c.max_t3 + 1);
  d.t4_t3 = b.take<int2>(c.max_t4);
  d.t4_md = b.take<int4>(c.max_t4);
  d.t4_score = b.take<float>(c.max_t4);
  // --- a5 ---
  d.seed_a = b.take<float4>(c.max_pls);
  d.seed_b = b.take<float4>(c.max_pls);
  d.seed_z1 = b.take<float>(c.max_pls);
  d.seed_g = b.take<float4>(c.max_pls);
  d.seed_perm = b.take<int>(c.max_pls);
  d.pls_event = b.take<int>(c.max_pls);
  d.pt_ev = b.take<PtEvent>((size_t)c.max_events + 1);
  d.anc_bin = b.take<int>(c.max_md);
  d.anc_rank = b.take<int>(c.max_md);
  d.anc_a = b.take<float4>(c.max_md);
  d.anc_t = b.take<int4>(c.max_md);
  d.anc_c = b.take<float4>(5 * ((size_t)c.max_md / 32 + c.max_events + 2));
  d.cap_queue = (int)(2LL * ((long long)c.max_pt3 + c.max_pt5) < 0x7fffffffLL ? 2LL * ((long long)c.max_pt3 + c.max_pt5)
                                                                             : 0x7fffffffLL);
  d.pt_queue = b.take<int2>(d.cap_queue);
  d.pls_pt3_begin = b.take<int>((size_t)c.max_pls + 1);
  d.pls_pt5_begin = b.take<int>((size_t)c.max_pls + 1);
  d.pt3 = b.take<int2>(c.max_pt3);
  d.pt3_score = b.take<float>(c.max_pt3);
  d.pt5 = b.take<int2>(c.max_pt5);
  d.pt5_score = b.take<float>(c.max_pt5);
  // --- a6 ---
  d.idx_head = b.take<int>(4 * (size_t)c.max_md);
  d.idx_next = b.take<int>(5 * (size_t)c.max_t5 + 5 * (size_t)c.max_pt5 + 3 * (size_t)c.max_pt3 + 4 * (size_t)c.max_t4);
  d.keep4 = b.take<unsigned char>(c.max_t4);
  d.keep5 = b.take<unsigned char>(c.max_pt5);
  d.keep3 = b.take<unsigned char>(c.max_pt3);
  d.keepT = b.take<unsigned char>(c.max_t5);
  d.tc_begin = b.take<int>(kTcClasses * (size_t)c.max_events + 1);
  d.tc = b.take<int>(16 * (size_t)c.max_tc);
  d.ev_first = b.take<int>((size_t)K_NKINDS * (c.max_events + 1));
  // --- staging of host inputs + per-event tables + the batch record ---
  float* fx = b.take<float>(c.max_hits);
  float* fy = b.take<float>(c.max_hits);
  float* fz = b.take<float>(c.max_hits);
  int* is = b.take<int>(c.max_hits);
  float* pf[7];
  for (int k = 0; k < 7; ++k) pf[k] = b.take<float>(c.max_pls);
  int* pq = b.take<int>(c.max_pls);
  int* ho = b.take<int>((size_t)c.max_events + 1);
  int* po = b.take<int>((size_t)c.max_events + 1);
  Batch* bt = b.take<Batch>(1);
  d.batch = bt;
  d.hit_ev_off = ho;
  d.pls_ev_off = po;
  if (ctx) {
    ctx->in_x = fx;  ctx->in_y = fy;  ctx->in_z = fz;  ctx->in_sensor = is;
    ctx->p_pt = pf[0];  ctx->p_x0 = pf[1];  ctx->p_y0 = pf[2];  ctx->p_z0 = pf[3];
    ctx->p_x1 = pf[4];  ctx->p_y1 = pf[5];  ctx->p_z1 = pf[6];  ctx->p_q = pq;
    ctx->d_hit_ev_off = ho;  ctx->d_pls_ev_off = po;  ctx->d_batch = bt;
  }
  d.cap[K_MD] = c.max_md;  d.cap[K_LS] = c.max_ls;  d.cap[K_T3] = c.max_t3;  d.cap[K_T5] = c.max_t5;
  d.cap[K_PT3] = c.max_pt3;  d.cap[K_PT5] = c.max_pt5;  d.cap[K_TC] = c.max_tc;  d.cap[K_T4] = c.max_t4;
  return (b.off + 255) & ~size_t(255);
}

bool caps_ok(const lst_caps& c) {
  // max_md: the LS stage packs an MD index into 27 bits (lst_ls.cuh); max_pls: a seed slot into 16 bits per tile
  return c.max_events > 0 && c.max_hits > 0 && c.max_pls > 0 && c.max_md > 0 && c.max_ls > 0 && c.max_t3 > 0 &&
         c.max_t5 > 0 && c.max_pt3 > 0 && c.max_pt5 > 0 && c.max_tc > 0 && c.max_t4 > 0 && c.max_md <= LST_MAX_MD &&
         5LL * c.max_t5 + 5LL * c.max_pt5 + 3LL * c.max_pt3 + 4LL * c.max_t4 < 0x7fffffffLL &&
         16LL * c.max_tc < 0x7fffffffLL;
}

}  // namespace

extern "C" size_t lst_workspace_bytes(const lst_caps* caps, int32_t n_modules) {
  lst_caps c;
  if (caps) c = *caps; else lst_default_caps(&c);
  if (!caps_ok(c) || n_modules <= 0) return 0;
  Dev d;
  return layout(c, n_modules, nullptr, d, nullptr, nullptr);
}

static void ctx_destroy(lst_ctx* ctx) {
  if (!ctx) return;
  if (ctx->graph) cudaGraphExecDestroy(ctx->graph);
  if (ctx->owned_stream) {
    cudaStreamSynchronize(ctx->owned_stream);
    cudaStreamDestroy(ctx->owned_stream);
  }
  for (void* p : ctx->allocs) cudaFree(p);
  if (ctx->h_ctl) cudaFreeHost(ctx->h_ctl);
  if (ctx->h_ev_cnt) cudaFreeHost(ctx->h_ev_cnt);
  if (ctx->h_ev_first) cudaFreeHost(ctx->h_ev_first);
  if (ctx->h_tc_begin) cudaFreeHost(ctx->h_tc_begin);
  for (int i = 0; i <= kMaxKernels; ++i)
    if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
  ctx->magic = 0;
  delete ctx;
}

extern "C" int lst_ctx_create(lst_geometry* g, const lst_caps* caps, void* cuda_stream, lst_ctx** out) {
  if (!out) return LST_ERR_ARG;
  *out = nullptr;
  if (!g || g->magic != MAGIC_GEOM) return LST_ERR_ARG;
  lst_caps c;
  if (caps) c = *caps; else lst_default_caps(&c);
  if (!caps_ok(c)) return LST_ERR_ARG;
  if ((long long)c.max_events * 2 * g->n_mod + 1 > 0x7fffffffLL) return LST_ERR_ARG;
  lst_ctx* ctx = new (std::nothrow) lst_ctx();
  if (!ctx) return LST_ERR_CUDA;
  ctx->magic = MAGIC_CTX;
  ctx->g = g;
  ctx->caps = c;
  ctx->stream = (cudaStream_t)cuda_stream;
  ctx->h_ctl = nullptr;
  ctx->h_ev_cnt = nullptr;
  ctx->h_ev_first = nullptr;
  ctx->h_tc_begin = nullptr;
  for (int i = 0; i <= kMaxKernels; ++i) ctx->ev[i] = nullptr;
  ctx->timing = false;
  ctx->graph = nullptr;
  ctx->owned_stream = nullptr;
  ctx->use_graph = cuda_stream != nullptr;  // lst_ctx_set_graph;  // the legacy default stream cannot be captured
  ctx->n_kernels = 0;
  ctx->last_n_events = 0;
  ctx->synced = true;
  Dev probe;
  ctx->bytes = layout(c, g->n_mod, nullptr, probe, nullptr, nullptr);
  char* base = nullptr;
  if (cudaMalloc(&base, ctx->bytes) != cudaSuccess) {
    cudaGetLastError();
    ctx_destroy(ctx);
    return LST_ERR_CUDA;
  }
  ctx->allocs.push_back(base);
  memset(&ctx->dev, 0, sizeof(Dev));
  layout(c, g->n_mod, base, ctx->dev, ctx, &ctx->zero_bytes);
  ctx->zero_region = base;
  ctx->dev.n_mod = g->n_mod;
  ctx->dev.subdet = g->d_subdet;
  ctx->dev.conn_off = g->d_conn_off;
  ctx->dev.conn_tgt = g->d_conn_tgt;
  ctx->dev.cuts = g->cuts;
  bool ok = cudaMallocHost(&ctx->h_ctl, sizeof(Ctl)) == cudaSuccess &&
            cudaMallocHost(&ctx->h_ev_cnt, sizeof(unsigned long long) * kEvCnt * c.max_events) == cudaSuccess &&
            cudaMallocHost(&ctx->h_ev_first, sizeof(int) * K_NKINDS * (c.max_events + 1)) == cudaSuccess &&
            cudaMallocHost(&ctx->h_tc_begin, sizeof(int) * (kTcClasses * (size_t)c.max_events + 1)) == cudaSuccess;
  for (int i = 0; ok && i <= kMaxKernels; ++i) ok = cudaEventCreate(&ctx->ev[i]) == cudaSuccess;
  if (!ok) {
    ctx_destroy(ctx);
    return LST_ERR_CUDA;
  }
  // grid-stride kernels are launched with exactly the blocks that fit the GPU at once
  int occ_md = 0, occ_ls = 0, occ_pt = 0;
  const size_t pt_smem = sizeof(PtWarp) * kWarps;
  // the limit is a property of the function, shared by every geometry and context of the process: the largest a launch can ask for
  const int ingest_smem = (int)sizeof(int) * kIngestMaxBins;
  if (cudaFuncSetAttribute(k_ingest_count, cudaFuncAttributeMaxDynamicSharedMemorySize, ingest_smem) != cudaSuccess ||
      cudaFuncSetAttribute(k_pt_eval, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pt_smem) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_md, k_md_eval, kBlock, 0) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_ls, k_ls_eval, kBlock, 0) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_pt, k_pt_eval, kBlock, pt_smem) != cudaSuccess ||
      occ_md < 1 || occ_ls < 1 || occ_pt < 1) {
    ctx_destroy(ctx);
    return LST_ERR_CUDA;
  }
  ctx->occ_md = occ_md;
  ctx->occ_ls = occ_ls;
  ctx->occ_pt = occ_pt;
  ctx->blocks_per_sm = 8;
  *out = ctx;
  return LST_OK;
}

#include "lst_api_run.inl"
#include "lst_api_fetch.inl"
#include "lst_api_static.inl"
#include "lst_api_audit.inl"
