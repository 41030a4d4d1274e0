// lst_api_fetch.inl -- included by lst_api.cu: result read-back, lst_run_event, lst_free.

namespace {

void out_destroy(lst_event_out* o) {
  if (!o) return;
  free(o->md_hits);  free(o->md_module);  free(o->md_f);
  free(o->ls_md);  free(o->ls_kappa);
  free(o->t3_ls);  free(o->t3_md);  free(o->t3_k);
  free(o->t5_t3);  free(o->t5_md);  free(o->t5_score);
  free(o->pt3);  free(o->pt3_score);  free(o->pt5);  free(o->pt5_score);
  free(o->tc);
  free(o->t4_t3);  free(o->t4_md);  free(o->t4_score);
  o->magic = 0;
  free(o);
}

template <class T>
T* halloc(size_t n) { return static_cast<T*>(malloc(sizeof(T) * (n ? n : 1))); }

// device slice -> host buffer, enqueued on the context's stream (the caller synchronises once)
struct D2H {
  cudaStream_t st;
  template <class T>
  bool operator()(T* dst, const T* src, size_t first, size_t n) const {
    if (n == 0) return true;
    return cudaMemcpyAsync(dst, src + first, sizeof(T) * n, cudaMemcpyDeviceToHost, st) == cudaSuccess;
  }
};

}  // namespace

extern "C" int lst_ctx_fetch_event(lst_ctx* ctx, int32_t ev, lst_event_out** out) {
  if (!out) return LST_ERR_ARG;
  *out = nullptr;
  if (!ctx || ctx->magic != MAGIC_CTX || !ctx->synced || ev < 0 || ev >= ctx->last_n_events) return LST_ERR_ARG;
  const Ctl& h = *ctx->h_ctl;
  if (h.error) return (h.error & E_BAD_SENSOR) ? LST_ERR_ARG : LST_ERR_CAPACITY;
  const Dev& d = ctx->dev;
  const int E1 = ctx->last_n_events + 1;
  auto first = [&](int kind, int e) { return ctx->h_ev_first[kind * E1 + e]; };
  const int f_md = first(K_MD, ev), f_ls = first(K_LS, ev), f_t3 = first(K_T3, ev), f_t5 = first(K_T5, ev);
  const int f_p3 = first(K_PT3, ev), f_p5 = first(K_PT5, ev);
  const int f_pls = ctx->last_pls_off[ev];
  const D2H d2h{ctx->stream};

  lst_event_out* o = static_cast<lst_event_out*>(calloc(1, sizeof(lst_event_out)));
  if (!o) return LST_ERR_CUDA;
  o->magic = MAGIC_OUT;
  o->n_md = first(K_MD, ev + 1) - f_md;
  o->n_ls = first(K_LS, ev + 1) - f_ls;
  o->n_t3 = first(K_T3, ev + 1) - f_t3;
  o->n_t5 = first(K_T5, ev + 1) - f_t5;
  o->n_pt3 = first(K_PT3, ev + 1) - f_p3;
  o->n_pt5 = first(K_PT5, ev + 1) - f_p5;
  const bool has_tc = (ctx->g->cuts.stage_mask & 32) != 0;
  const int tc0 = has_tc ? ctx->h_tc_begin[kTcClasses * (size_t)ev] : 0;
  o->n_tc = has_tc ? ctx->h_tc_begin[kTcClasses * (size_t)(ev + 1)] - tc0 : 0;
  const bool has_t4 = (ctx->g->cuts.stage_mask & 64) != 0;
  const int f_t4 = has_t4 ? first(K_T4, ev) : 0;
  o->n_t4 = has_t4 ? first(K_T4, ev + 1) - f_t4 : 0;
  for (int k = 0; k < LST_N_STAGES; ++k) {  // counters of THIS event
    o->near[k] = (int64_t)ctx->h_ev_cnt[(size_t)ev * kEvCnt + k];
    o->n_tests[k] = (int64_t)ctx->h_ev_cnt[(size_t)ev * kEvCnt + kStages + k];
  }
  const int n_md = o->n_md, n_ls = o->n_ls, n_t3 = o->n_t3, n_t5 = o->n_t5;
  o->md_hits = halloc<int32_t>(2 * (size_t)n_md);
  o->md_module = halloc<int32_t>(n_md);
  o->md_f = halloc<float>(6 * (size_t)n_md);
  o->ls_md = halloc<int32_t>(2 * (size_t)n_ls);
  o->ls_kappa = halloc<float>(n_ls);
  o->t3_ls = halloc<int32_t>(2 * (size_t)n_t3);
  o->t3_md = halloc<int32_t>(3 * (size_t)n_t3);
  o->t3_k = halloc<float>(n_t3);
  o->t5_t3 = halloc<int32_t>(2 * (size_t)n_t5);
  o->t5_md = halloc<int32_t>(5 * (size_t)n_t5);
  o->t5_score = halloc<float>(n_t5);
  o->pt3 = halloc<int32_t>(2 * (size_t)o->n_pt3);
  o->pt3_score = halloc<float>(o->n_pt3);
  o->pt5 = halloc<int32_t>(2 * (size_t)o->n_pt5);
  o->pt5_score = halloc<float>(o->n_pt5);
  o->tc = halloc<int32_t>(16 * (size_t)o->n_tc);
  o->t4_t3 = halloc<int32_t>(2 * (size_t)o->n_t4);
  o->t4_md = halloc<int32_t>(4 * (size_t)o->n_t4);
  o->t4_score = halloc<float>(o->n_t4);
  // host memory: a failed allocation is an error code, never a NULL destination or an exception across the ABI
  const void* const bufs[] = {o->md_hits, o->md_module, o->md_f, o->ls_md, o->ls_kappa, o->t3_ls, o->t3_md, o->t3_k,
                              o->t5_t3, o->t5_md, o->t5_score, o->pt3, o->pt3_score, o->pt5, o->pt5_score, o->tc,
                              o->t4_t3, o->t4_md, o->t4_score};
  bool have = true;
  for (const void* b : bufs) have = have && b != nullptr;
  std::vector<int> info;
  std::vector<float4> a;
  std::vector<float2> u;
  std::vector<int4> m3;
  try {
    info.resize(n_md);  a.resize(n_md);  u.resize(n_md);  m3.resize(n_t3);
  } catch (const std::bad_alloc&) {
    have = false;
  }
  if (!have) {
    out_destroy(o);
    return LST_ERR_CUDA;
  }
  // every copy goes to the context's stream; one synchronisation, then the index shifts on the host
  bool ok = d2h(reinterpret_cast<int2*>(o->md_hits), d.md_hit, f_md, n_md) &&
            d2h(info.data(), d.md_info, f_md, n_md) && d2h(a.data(), d.md_a, f_md, n_md) &&
            d2h(u.data(), d.md_u, f_md, n_md) &&
            d2h(reinterpret_cast<int2*>(o->ls_md), d.ls_md, f_ls, n_ls) && d2h(o->ls_kappa, d.ls_kappa, f_ls, n_ls) &&
            d2h(reinterpret_cast<int2*>(o->t3_ls), d.t3_ls, f_t3, n_t3) && d2h(m3.data(), d.t3_md, f_t3, n_t3) &&
            d2h(o->t3_k, d.t3_k, f_t3, n_t3) &&
            d2h(reinterpret_cast<int2*>(o->t5_t3), d.t5_t3, f_t5, n_t5) &&
            d2h(o->t5_md, d.t5_md, 5 * (size_t)f_t5, 5 * (size_t)n_t5) && d2h(o->t5_score, d.t5_score, f_t5, n_t5) &&
            d2h(reinterpret_cast<int2*>(o->pt3), d.pt3, f_p3, o->n_pt3) &&
            d2h(o->pt3_score, d.pt3_score, f_p3, o->n_pt3) &&
            d2h(reinterpret_cast<int2*>(o->pt5), d.pt5, f_p5, o->n_pt5) &&
            d2h(o->pt5_score, d.pt5_score, f_p5, o->n_pt5) &&
            d2h(o->tc, d.tc, 16 * (size_t)tc0, 16 * (size_t)o->n_tc) &&
            d2h(reinterpret_cast<int2*>(o->t4_t3), d.t4_t3, f_t4, o->n_t4) &&
            d2h(reinterpret_cast<int4*>(o->t4_md), d.t4_md, f_t4, o->n_t4) && d2h(o->t4_score, d.t4_score, f_t4, o->n_t4);
  ok = (cudaStreamSynchronize(ctx->stream) == cudaSuccess) && ok;
  if (!ok) {
    out_destroy(o);
    return LST_ERR_CUDA;
  }
  for (int i = 0; i < n_md; ++i) {
    o->md_module[i] = (info[i] >> 1) - ev * d.n_mod;
    float* f = o->md_f + 6 * (size_t)i;
    f[0] = a[i].x;  f[1] = a[i].y;  f[2] = a[i].z;  f[3] = a[i].w;  f[4] = u[i].x;  f[5] = u[i].y;
  }
  for (size_t i = 0; i < 2 * (size_t)n_ls; ++i) o->ls_md[i] -= f_md;
  for (int i = 0; i < n_t3; ++i) {
    o->t3_ls[2 * i] -= f_ls;  o->t3_ls[2 * i + 1] -= f_ls;
    o->t3_md[3 * i] = m3[i].x - f_md;  o->t3_md[3 * i + 1] = m3[i].y - f_md;  o->t3_md[3 * i + 2] = m3[i].z - f_md;
  }
  for (size_t i = 0; i < 2 * (size_t)n_t5; ++i) o->t5_t3[i] -= f_t3;
  for (size_t i = 0; i < 5 * (size_t)n_t5; ++i) o->t5_md[i] -= f_md;
  for (int i = 0; i < o->n_pt3; ++i) { o->pt3[2 * i] -= f_pls;  o->pt3[2 * i + 1] -= f_t3; }
  for (int i = 0; i < o->n_pt5; ++i) { o->pt5[2 * i] -= f_pls;  o->pt5[2 * i + 1] -= f_t5; }
  for (size_t i = 0; i < 2 * (size_t)o->n_t4; ++i) o->t4_t3[i] -= f_t3;
  for (size_t i = 0; i < 4 * (size_t)o->n_t4; ++i) o->t4_md[i] -= f_md;
  *out = o;
  return LST_OK;
}

extern "C" int lst_ctx_fetch_tc(lst_ctx* ctx, int32_t* tc, int32_t cap_tc, int32_t* tc_event_offsets) {
  if (!ctx || ctx->magic != MAGIC_CTX || !ctx->synced || !tc || !tc_event_offsets || cap_tc < 0) return LST_ERR_ARG;
  const Ctl& h = *ctx->h_ctl;
  if (h.error) return (h.error & E_BAD_SENSOR) ? LST_ERR_ARG : LST_ERR_CAPACITY;
  const int n = h.total[K_TC], E = ctx->last_n_events;
  if (n > cap_tc) return LST_ERR_CAPACITY;
  if (!(ctx->g->cuts.stage_mask & 32)) {
    for (int e = 0; e <= E; ++e) tc_event_offsets[e] = 0;
    return LST_OK;
  }
  if (n > 0) {
    CK(cudaMemcpyAsync(tc, ctx->dev.tc, sizeof(int) * 16 * (size_t)n, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
  }
  for (int e = 0; e <= E; ++e) tc_event_offsets[e] = ctx->h_tc_begin[kTcClasses * (size_t)e];  // read back by lst_ctx_run
  return LST_OK;
}

extern "C" int lst_run_event(lst_geometry* g, const lst_hits* hits, const lst_pls* seeds, lst_event_out** out) {
  if (!out) return LST_ERR_ARG;
  *out = nullptr;
  if (!g || g->magic != MAGIC_GEOM || !hits) return LST_ERR_ARG;
  if (hits->event_offsets || (seeds && seeds->event_offsets)) return LST_ERR_ARG;
  std::lock_guard<std::mutex> lock(g->default_mu);  // one internal context per geometry: calls are serialised
  if (!g->default_ctx) {
    lst_caps c;
    lst_default_caps(&c);
    c.max_events = 1;
    // a stream of its own (a blocking one: ordered after the caller's work on the legacy default stream),
    // so that the launch sequence can run as a CUDA graph
    cudaStream_t own = nullptr;
    if (cudaStreamCreate(&own) != cudaSuccess) return LST_ERR_CUDA;
    int rc = lst_ctx_create(g, &c, own, &g->default_ctx);
    if (rc != LST_OK) {
      cudaStreamDestroy(own);
      return rc;
    }
    g->default_ctx->owned_stream = own;
  }
  int rc = lst_ctx_run(g->default_ctx, 1, hits, seeds);
  if (rc != LST_OK) return rc;
  rc = lst_ctx_sync(g->default_ctx, nullptr);
  if (rc != LST_OK) return rc;
  return lst_ctx_fetch_event(g->default_ctx, 0, out);
}

extern "C" void lst_free(void* p) {
  if (!p) return;
  const uint64_t magic = *static_cast<const uint64_t*>(p);
  if (magic == MAGIC_OUT) {
    out_destroy(static_cast<lst_event_out*>(p));
  } else if (magic == MAGIC_CTX) {
    ctx_destroy(static_cast<lst_ctx*>(p));
  } else if (magic == MAGIC_GEOM) {
    lst_geometry* g = static_cast<lst_geometry*>(p);
    if (g->default_ctx) ctx_destroy(g->default_ctx);
    cudaFree(g->d_subdet);  cudaFree(g->d_conn_off);  cudaFree(g->d_conn_tgt);
    g->magic = 0;
    delete g;
  }
}
