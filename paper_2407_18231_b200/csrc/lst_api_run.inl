// lst_api_run.inl -- included by lst_api.cu: the launch sequence of one batch and its sync.

namespace {

inline int grid_for(const lst_geometry* g, long long n, int per_sm) {
  long long blocks = (n + kBlock - 1) / kBlock;
  const long long maxb = (long long)g->n_sm * per_sm;
  if (blocks > maxb) blocks = maxb;
  if (blocks < 1) blocks = 1;
  return (int)blocks;
}

struct Launcher {
  lst_ctx* ctx;
  int k = 0;
  void mark(const char* name) {
    if (ctx->timing && k < kMaxKernels) {
      cudaEventRecord(ctx->ev[k], ctx->stream);
      ctx->kname[k] = name;
    }
    ++k;
  }
  void finish() {
    if (ctx->timing && k <= kMaxKernels) cudaEventRecord(ctx->ev[k < kMaxKernels ? k : kMaxKernels], ctx->stream);
    ctx->n_kernels = k;
  }
};

bool offsets_ok(const int32_t* off, int n_events, int n) {
  if (off[0] != 0 || off[n_events] != n) return false;
  for (int e = 0; e < n_events; ++e)
    if (off[e + 1] < off[e]) return false;
  return true;
}

}  // namespace

extern "C" int lst_ctx_run(lst_ctx* ctx, int32_t n_events, const lst_hits* hits, const lst_pls* seeds) {
  if (!ctx || ctx->magic != MAGIC_CTX || !hits) return LST_ERR_ARG;
  const lst_caps& c = ctx->caps;
  if (n_events <= 0 || n_events > c.max_events) return n_events > c.max_events ? LST_ERR_CAPACITY : LST_ERR_ARG;
  if (hits->n < 0 || (hits->n > 0 && (!hits->x || !hits->y || !hits->z || !hits->sensor))) return LST_ERR_ARG;
  if (hits->n > c.max_hits) return LST_ERR_CAPACITY;
  const int n_pls = seeds ? seeds->n : 0;
  if (n_pls < 0) return LST_ERR_ARG;
  if (n_pls > c.max_pls) return LST_ERR_CAPACITY;
  if (n_pls > 0 && (!seeds->pt || !seeds->q || !seeds->x0 || !seeds->y0 || !seeds->z0 || !seeds->x1 ||
                    !seeds->y1 || !seeds->z1))
    return LST_ERR_ARG;
  if (n_events > 1 && (!hits->event_offsets || (n_pls > 0 && !seeds->event_offsets))) return LST_ERR_ARG;

  // event offsets (host) -> kept for fetch, copied to the device
  ctx->last_hit_off.assign(n_events + 1, 0);
  ctx->last_pls_off.assign(n_events + 1, 0);
  if (hits->event_offsets) {
    if (!offsets_ok(hits->event_offsets, n_events, hits->n)) return LST_ERR_ARG;
    ctx->last_hit_off.assign(hits->event_offsets, hits->event_offsets + n_events + 1);
  } else {
    ctx->last_hit_off[n_events] = hits->n;
  }
  if (n_pls > 0 && seeds->event_offsets) {
    if (!offsets_ok(seeds->event_offsets, n_events, n_pls)) return LST_ERR_ARG;
    ctx->last_pls_off.assign(seeds->event_offsets, seeds->event_offsets + n_events + 1);
  } else {
    for (int e = 1; e <= n_events; ++e) ctx->last_pls_off[e] = (e == n_events) ? n_pls : 0;
    if (n_events > 1 && n_pls > 0) return LST_ERR_ARG;
  }
  cudaStream_t st = ctx->stream;
  const size_t eo = sizeof(int) * (n_events + 1);
  CK(cudaMemcpyAsync(ctx->d_hit_ev_off, ctx->last_hit_off.data(), eo, cudaMemcpyHostToDevice, st));
  CK(cudaMemcpyAsync(ctx->d_pls_ev_off, ctx->last_pls_off.data(), eo, cudaMemcpyHostToDevice, st));

  Dev d = ctx->dev;
  d.n_events = n_events;
  d.n_hits = hits->n;
  d.n_pls = n_pls;
  d.hit_ev_off = ctx->d_hit_ev_off;
  d.pls_ev_off = ctx->d_pls_ev_off;
  if (hits->on_device || hits->n == 0) {
    d.in_x = hits->x;  d.in_y = hits->y;  d.in_z = hits->z;  d.in_sensor = hits->sensor;
  } else {
    const size_t nb = sizeof(float) * hits->n;
    CK(cudaMemcpyAsync(ctx->in_x, hits->x, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->in_y, hits->y, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->in_z, hits->z, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->in_sensor, hits->sensor, nb, cudaMemcpyHostToDevice, st));
    d.in_x = ctx->in_x;  d.in_y = ctx->in_y;  d.in_z = ctx->in_z;  d.in_sensor = ctx->in_sensor;
  }
  if (n_pls > 0) {
    if (seeds->on_device) {
      d.p_pt = seeds->pt;  d.p_q = seeds->q;
      d.p_x0 = seeds->x0;  d.p_y0 = seeds->y0;  d.p_z0 = seeds->z0;
      d.p_x1 = seeds->x1;  d.p_y1 = seeds->y1;  d.p_z1 = seeds->z1;
    } else {
      const size_t nb = sizeof(float) * n_pls;
      const float* src[7] = {seeds->pt, seeds->x0, seeds->y0, seeds->z0, seeds->x1, seeds->y1, seeds->z1};
      float* dst[7] = {ctx->p_pt, ctx->p_x0, ctx->p_y0, ctx->p_z0, ctx->p_x1, ctx->p_y1, ctx->p_z1};
      for (int k = 0; k < 7; ++k) CK(cudaMemcpyAsync(dst[k], src[k], nb, cudaMemcpyHostToDevice, st));
      CK(cudaMemcpyAsync(ctx->p_q, seeds->q, nb, cudaMemcpyHostToDevice, st));
      d.p_pt = ctx->p_pt;  d.p_q = ctx->p_q;
      d.p_x0 = ctx->p_x0;  d.p_y0 = ctx->p_y0;  d.p_z0 = ctx->p_z0;
      d.p_x1 = ctx->p_x1;  d.p_y1 = ctx->p_y1;  d.p_z1 = ctx->p_z1;
    }
  }

  const lst_geometry* g = ctx->g;
  const int mask = g->cuts.stage_mask;
  const int n_sens = n_events * 2 * g->n_mod;
  const int gp = g->n_sm * 4;  // persistent ticket kernels
  Launcher L{ctx};

  CK(cudaMemsetAsync(ctx->zero_region, 0, ctx->zero_bytes, st));
  L.mark("hist");
  k_hist<<<grid_for(g, hits->n > n_pls ? hits->n : n_pls, 8), kBlock, 0, st>>>(d);
  L.mark("scan_sensors");
  k_scan<<<grid_for(g, (n_sens + kScanItems) / kScanItems, 4), kBlock, 0, st>>>(
      d.sens_cnt, d.sens_begin, nullptr, 0, n_sens, d.ctl->ticket + T_SENS, d.tstate[T_SENS]);
  L.mark("scatter");
  k_scatter<<<grid_for(g, hits->n, 8), kBlock, 0, st>>>(d);
  L.mark("md");
  k_md_eval<<<ctx->grid_md, kBlock, 0, st>>>(d);
  L.mark("md_scan");
  k_scan_t<16><<<grid_for(g, (hits->n + 16) / 16, 4), kBlock, 0, st>>>(
      d.md_cnt, d.hit_md_begin, nullptr, 0, hits->n, d.ctl->ticket + T_MD, d.tstate[T_MD]);
  L.mark("md_place");
  k_md_place<<<grid_for(g, hits->n, 8), kBlock, 0, st>>>(d);
  L.mark("ls");
  k_ls_eval<<<ctx->grid_ls, kBlock, 0, st>>>(d);
  L.mark("ls_scan");
  k_scan<<<gp, kBlock, 0, st>>>(d.ls_cnt, d.md_ls_begin, d.ctl->total + K_MD, 1, 0, d.ctl->ticket + T_LS, d.tstate[T_LS]);
  L.mark("ls_place");
  k_ls_place<<<gp, kBlock, 0, st>>>(d);
  L.mark("t3");
  k_stage<StageT3><<<gp, kBlock, 0, st>>>(d);
  L.mark("t5");
  k_stage<StageT5><<<gp, kBlock, 0, st>>>(d);
  L.mark("anchors");
  k_anchor<<<gp, kBlock, 0, st>>>(d);
  L.mark("anchor_scan");
  k_scan<<<grid_for(g, (n_events * kAncBins + kScanItems) / kScanItems, 4), kBlock, 0, st>>>(
      d.anc_bin_cnt, d.anc_bin_begin, nullptr, 0, n_events * kAncBins, d.ctl->ticket + T_ANC, d.tstate[T_ANC]);
  L.mark("anchor_sort");
  k_anchor_sort<<<gp, kBlock, 0, st>>>(d);
  L.mark("pt_tiles");
  k_pt_tiles<<<1, kBlock, 0, st>>>(d);
  L.mark("pt");
  k_pt_eval<<<ctx->grid_pt, kBlock, sizeof(PtWarp) * kWarps, st>>>(d);
  L.mark("pt3_scan");
  k_scan<<<grid_for(g, (n_pls + kScanItems) / kScanItems, 4), kBlock, 0, st>>>(
      d.pls_pt3_cnt, d.pls_pt3_begin, nullptr, 0, n_pls, d.ctl->ticket + T_PP3, d.tstate[T_PP3]);
  L.mark("pt3_place");
  k_pt_place<false><<<gp, kBlock, 0, st>>>(d);
  L.mark("pt5_scan");
  k_scan<<<grid_for(g, (n_pls + kScanItems) / kScanItems, 4), kBlock, 0, st>>>(
      d.pls_pt5_cnt, d.pls_pt5_begin, nullptr, 0, n_pls, d.ctl->ticket + T_PP5, d.tstate[T_PP5]);
  L.mark("pt5_place");
  k_pt_place<true><<<gp, kBlock, 0, st>>>(d);
  L.mark("event_ranges");
  k_event_ranges<<<1, 64, 0, st>>>(d, ctx->d_ev_first);
  if (mask & 32) {
    L.mark("sel_prepare");
    k_sel_prepare<<<gp, kBlock, 0, st>>>(d);
    L.mark("index_count");
    k_index<false><<<gp, kBlock, 0, st>>>(d);
    L.mark("scan_index");
    k_scan<<<gp, kBlock, 0, st>>>(d.idx_cnt, d.idx_begin, d.ctl->total + K_MD, 3, 0, d.ctl->ticket + T_IDX,
                                  d.tstate[T_IDX]);
    L.mark("index_fill");
    k_index<true><<<gp, kBlock, 0, st>>>(d);
    L.mark("rule1_pt5");
    k_rule1<<<gp, kBlock, 0, st>>>(d);
    L.mark("rule2_pt3");
    k_rule2<<<gp, kBlock, 0, st>>>(d);
    L.mark("rule3_t5");
    k_rule3<<<gp, kBlock, 0, st>>>(d);
    L.mark("scan_tc");
    k_scan<<<1, kBlock, 0, st>>>(d.tc_cnt, d.tc_begin, nullptr, 0, 4 * n_events, d.ctl->ticket + T_TC,
                                 d.tstate[T_TC]);
    L.mark("tc_emit");
    k_tc_emit<<<gp, kBlock, 0, st>>>(d, ctx->d_ev_first);
  }
  L.finish();
  CK(cudaGetLastError());
  CK(cudaMemcpyAsync(ctx->h_ctl, d.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(ctx->h_ev_cnt, d.ev_cnt, sizeof(unsigned long long) * kEvCnt * n_events, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(ctx->h_ev_first, ctx->d_ev_first, sizeof(int) * (K_PT5 + 1) * (n_events + 1),
                     cudaMemcpyDeviceToHost, st));
  if (mask & 32)
    CK(cudaMemcpyAsync(ctx->h_tc_begin, d.tc_begin, sizeof(int) * (4 * (size_t)n_events + 1), cudaMemcpyDeviceToHost, st));
  ctx->dev.n_events = n_events;
  ctx->dev.n_hits = hits->n;
  ctx->dev.n_pls = n_pls;
  ctx->last_n_events = n_events;
  ctx->synced = false;
  return LST_OK;
}

extern "C" int lst_ctx_sync(lst_ctx* ctx, lst_batch_summary* s) {
  if (!ctx || ctx->magic != MAGIC_CTX) return LST_ERR_ARG;
  if (ctx->last_n_events == 0) return LST_ERR_ARG;
  CK(cudaStreamSynchronize(ctx->stream));
  ctx->synced = true;
  const Ctl& h = *ctx->h_ctl;
  if (s) {
    s->n_events = ctx->last_n_events;
    s->n_hits = ctx->dev.n_hits;
    s->n_pls = ctx->dev.n_pls;
    s->n_md = h.total[K_MD];  s->n_ls = h.total[K_LS];  s->n_t3 = h.total[K_T3];  s->n_t5 = h.total[K_T5];
    s->n_pt3 = h.total[K_PT3];  s->n_pt5 = h.total[K_PT5];  s->n_tc = h.total[K_TC];
    for (int k = 0; k < LST_N_STAGES; ++k) {  // batch totals = sums of the per-event counters
      s->near[k] = 0;
      s->n_tests[k] = 0;
      for (int e = 0; e < ctx->last_n_events; ++e) {
        s->near[k] += (int64_t)ctx->h_ev_cnt[(size_t)e * kEvCnt + k];
        s->n_tests[k] += (int64_t)ctx->h_ev_cnt[(size_t)e * kEvCnt + 6 + k];
      }
    }
  }
  if (h.error & E_BAD_SENSOR) return LST_ERR_ARG;
  if (h.error) return LST_ERR_CAPACITY;
  return LST_OK;
}

extern "C" int lst_ctx_set_timing(lst_ctx* ctx, int32_t enable) {
  if (!ctx || ctx->magic != MAGIC_CTX) return LST_ERR_ARG;
  ctx->timing = enable != 0;
  return LST_OK;
}

extern "C" int lst_ctx_kernel_times(lst_ctx* ctx, float* ms, const char** names, int32_t cap) {
  if (!ctx || ctx->magic != MAGIC_CTX || !ms) return LST_ERR_ARG;
  if (!ctx->timing || !ctx->synced) return LST_ERR_ARG;
  const int n = ctx->n_kernels < kMaxKernels ? ctx->n_kernels : kMaxKernels;
  for (int i = 0; i < n && i < cap; ++i) {
    CK(cudaEventElapsedTime(&ms[i], ctx->ev[i], ctx->ev[i + 1]));
    if (names) names[i] = ctx->kname[i];
  }
  return n < cap ? n : cap;
}

extern "C" int lst_ctx_launch_count(lst_ctx* ctx) {
  if (!ctx || ctx->magic != MAGIC_CTX) return LST_ERR_ARG;
  return ctx->n_kernels;
}
