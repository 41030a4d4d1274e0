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
  bool capturing = false;
  void mark(const char* name) {
#ifdef LST_DEBUG_SYNC  // debugging build only: wait for everything launched so far and say which kernel comes next
    if (!capturing) {
      const cudaError_t e = cudaStreamSynchronize(ctx->stream);
      fprintf(stderr, "[lst] before %s: %s\n", name, cudaGetErrorString(e));
    }
#endif
    if (ctx->timing && !capturing && k < kMaxKernels) {
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

// The launch sequence of one batch on stream st.  Grids do not depend on the batch (every kernel is a
// grid-stride or ticket loop over sizes read from device memory), so the sequence can be captured once.
int enqueue(lst_ctx* ctx, cudaStream_t st, Launcher* Lp) {
  Launcher& L = *Lp;
  const lst_geometry* g = ctx->g;
  const Dev& d = ctx->dev;
  const int mask = g->cuts.stage_mask;
  // resident blocks per SM a kernel of this context may take (lst_ctx_set_blocks_per_sm): the streaming
  // kernels take all of them, the ticket kernels half, the three heavy kernels what their occupancy allows
  const int bps = ctx->blocks_per_sm;
  const int gw = g->n_sm * bps;
  const int gp = g->n_sm * (bps > 1 ? bps / 2 : 1);
  const int g_md = g->n_sm * (ctx->occ_md < bps ? ctx->occ_md : bps);
  const int g_ls = g->n_sm * (ctx->occ_ls < bps ? ctx->occ_ls : bps);
  const int g_pt = g->n_sm * (ctx->occ_pt < bps ? ctx->occ_pt : bps);
  CK(cudaMemsetAsync(ctx->zero_region, 0, ctx->zero_bytes, st));
  const size_t ingest_smem = sizeof(int) * (size_t)(2 * g->n_mod < kIngestMaxBins ? 2 * g->n_mod : kIngestMaxBins);
  L.mark("ingest_count");
  k_ingest_count<<<ctx->caps.max_events * kIngestChunks, kIngestThreads, ingest_smem, st>>>(d);
  L.mark("ingest_scan");
  k_ingest_scan<<<ctx->caps.max_events * kIngestScanParts, kIngestThreads, 0, st>>>(d);
  L.mark("scatter");
  k_scatter<<<dim3(gw / ctx->caps.max_events > 0 ? gw / ctx->caps.max_events : 1, ctx->caps.max_events), kBlock, 0, st>>>(d);
  L.mark("md");
  k_md_eval<<<g_md, kBlock, 0, st>>>(d);
  L.mark("md_place");
  k_md_place<<<gw, kBlock, 0, st>>>(d);
  L.mark("ls");
  k_ls_eval<<<g_ls, kBlock, 0, st>>>(d);
  L.mark("ls_place");
  k_ls_place<<<gp, kBlock, 0, st>>>(d);
  L.mark("t3");
  k_stage<StageT3><<<gp, kBlock, 0, st>>>(d);
  L.mark("t5");
  k_stage<StageT5><<<gp, kBlock, 0, st>>>(d);
  if (mask & 64) {  // extension: T4 (CUTS.md section 10)
    L.mark("t4");
    k_stage<StageT4><<<gp, kBlock, 0, st>>>(d);
  }
  L.mark("anchor_sort");
  k_anchor_sort<<<ctx->caps.max_events * kAncBlocksPerEvent, kBlock, 0, st>>>(d);
  L.mark("pt");
  k_pt_eval<<<g_pt, kBlock, sizeof(PtWarp) * kWarps, st>>>(d);
  L.mark("pt_exact");
  k_pt_exact<<<gp, kBlock, 0, st>>>(d);
  L.mark("pt_scan");
  k_scan2<<<dim3(g->n_sm, 2), kBlock, 0, st>>>(
      ScanJob{d.pls_pt3_cnt, d.pls_pt3_begin, &d.batch->n_pls, 1, 0, d.ctl->ticket + T_PP3, d.tstate[T_PP3]},
      ScanJob{d.pls_pt5_cnt, d.pls_pt5_begin, &d.batch->n_pls, 1, 0, d.ctl->ticket + T_PP5, d.tstate[T_PP5]});
  L.mark("pt_place");
  k_pt_place<<<gp, kBlock, 0, st>>>(d);
  if (mask & 32) {
    L.mark("rule1_pt5");
    k_rule1<<<gw, kBlock, 0, st>>>(d);
    L.mark("rule2_pt3");
    k_rule2<<<gw, kBlock, 0, st>>>(d);
    L.mark("rule3_t5");
    if (mask & 64) {
      k_rule3<false><<<gw, kBlock, 0, st>>>(d);
      L.mark("rule_t4");
      k_rule_t4<<<gw, kBlock, 0, st>>>(d);
    } else {
      k_rule3<true><<<gw, kBlock, 0, st>>>(d);
    }
    L.mark("tc_emit");
    k_tc_emit<<<gp, kBlock, 0, st>>>(d);
  }
  CK(cudaGetLastError());
  return LST_OK;
}

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
  if (hits->sensor_u16 && 2LL * ctx->g->n_mod > 65536) return LST_ERR_ARG;
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

  Batch bt;
  memset(&bt, 0, sizeof(bt));
  bt.n_events = n_events;
  bt.n_hits = hits->n;
  bt.n_pls = n_pls;
  bt.sensor_u16 = hits->sensor_u16 != 0;
  if (hits->on_device || hits->n == 0) {
    bt.in_x = hits->x;  bt.in_y = hits->y;  bt.in_z = hits->z;  bt.in_sensor = hits->sensor;
  } else {
    const size_t nb = sizeof(float) * hits->n;
    CK(cudaMemcpyAsync(ctx->in_x, hits->x, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->in_y, hits->y, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->in_z, hits->z, nb, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(ctx->in_sensor, hits->sensor, hits->sensor_u16 ? nb / 2 : nb, cudaMemcpyHostToDevice, st));
    bt.in_x = ctx->in_x;  bt.in_y = ctx->in_y;  bt.in_z = ctx->in_z;  bt.in_sensor = ctx->in_sensor;
  }
  if (n_pls > 0) {
    if (seeds->on_device) {
      bt.p_pt = seeds->pt;  bt.p_q = seeds->q;
      bt.p_x0 = seeds->x0;  bt.p_y0 = seeds->y0;  bt.p_z0 = seeds->z0;
      bt.p_x1 = seeds->x1;  bt.p_y1 = seeds->y1;  bt.p_z1 = seeds->z1;
    } else {
      const size_t nb = sizeof(float) * n_pls;
      const float* src[7] = {seeds->pt, seeds->x0, seeds->y0, seeds->z0, seeds->x1, seeds->y1, seeds->z1};
      float* dst[7] = {ctx->p_pt, ctx->p_x0, ctx->p_y0, ctx->p_z0, ctx->p_x1, ctx->p_y1, ctx->p_z1};
      for (int k = 0; k < 7; ++k) CK(cudaMemcpyAsync(dst[k], src[k], nb, cudaMemcpyHostToDevice, st));
      CK(cudaMemcpyAsync(ctx->p_q, seeds->q, nb, cudaMemcpyHostToDevice, st));
      bt.p_pt = ctx->p_pt;  bt.p_q = ctx->p_q;
      bt.p_x0 = ctx->p_x0;  bt.p_y0 = ctx->p_y0;  bt.p_z0 = ctx->p_z0;
      bt.p_x1 = ctx->p_x1;  bt.p_y1 = ctx->p_y1;  bt.p_z1 = ctx->p_z1;
    }
  }
  // the batch record (pageable source: staged by the runtime before this call returns)
  CK(cudaMemcpyAsync(ctx->d_batch, &bt, sizeof(Batch), cudaMemcpyHostToDevice, st));

  // ---- the launch sequence: memset + 18 kernels (12 without the selection), as a CUDA graph ----
  const int mask = ctx->g->cuts.stage_mask;
  if (ctx->timing || !ctx->use_graph) {
    Launcher L{ctx};
    int rc = enqueue(ctx, st, &L);
    if (rc != LST_OK) return rc;
    L.finish();
  } else {
    if (!ctx->graph) {
      cudaGraph_t graph = nullptr;
      CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
      Launcher L{ctx};
      L.capturing = true;
      const int rc = enqueue(ctx, st, &L);
      const cudaError_t ce = cudaStreamEndCapture(st, &graph);
      if (rc != LST_OK || ce != cudaSuccess || !graph) {
        if (graph) cudaGraphDestroy(graph);
        cudaGetLastError();
        return LST_ERR_CUDA;
      }
      const cudaError_t ie = cudaGraphInstantiate(&ctx->graph, graph, 0);
      cudaGraphDestroy(graph);
      if (ie != cudaSuccess) {
        ctx->graph = nullptr;
        return LST_ERR_CUDA;
      }
      ctx->n_kernels = L.k;
    }
    CK(cudaGraphLaunch(ctx->graph, st));
  }
  CK(cudaGetLastError());
  const Dev& d = ctx->dev;
  CK(cudaMemcpyAsync(ctx->h_ctl, d.ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(ctx->h_ev_cnt, d.ev_cnt, sizeof(unsigned long long) * kEvCnt * n_events, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(ctx->h_ev_first, d.ev_first, sizeof(int) * K_NKINDS * (n_events + 1), cudaMemcpyDeviceToHost, st));
  if (mask & 32)
    CK(cudaMemcpyAsync(ctx->h_tc_begin, d.tc_begin, sizeof(int) * (kTcClasses * (size_t)n_events + 1),
                       cudaMemcpyDeviceToHost, st));
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
    s->n_t4 = (ctx->g->cuts.stage_mask & 64) ? h.total[K_T4] : 0;
    for (int k = 0; k < LST_N_STAGES; ++k) {  // batch totals = sums of the per-event counters
      s->near[k] = 0;
      s->n_tests[k] = 0;
      for (int e = 0; e < ctx->last_n_events; ++e) {
        s->near[k] += (int64_t)ctx->h_ev_cnt[(size_t)e * kEvCnt + k];
        s->n_tests[k] += (int64_t)ctx->h_ev_cnt[(size_t)e * kEvCnt + kStages + k];
      }
    }
  }
  if (h.error & E_BAD_SENSOR) return LST_ERR_ARG;
  if (h.error) return LST_ERR_CAPACITY;
  return LST_OK;
}

extern "C" int lst_ctx_set_blocks_per_sm(lst_ctx* ctx, int32_t blocks) {
  if (!ctx || ctx->magic != MAGIC_CTX || blocks < 0 || blocks > 8) return LST_ERR_ARG;
  const int b = blocks == 0 ? 8 : blocks;
  if (b != ctx->blocks_per_sm && ctx->graph) {  // the captured launch sequence holds the old grids
    if (!ctx->synced) CK(cudaStreamSynchronize(ctx->stream));  // a batch still in flight finishes on the old grids first
    cudaGraphExecDestroy(ctx->graph);
    ctx->graph = nullptr;
  }
  ctx->blocks_per_sm = b;
  return LST_OK;
}

extern "C" int lst_ctx_set_graph(lst_ctx* ctx, int32_t enable) {
  if (!ctx || ctx->magic != MAGIC_CTX) return LST_ERR_ARG;
  if (enable && !ctx->stream) return LST_ERR_ARG;  // the legacy default stream cannot be captured
  ctx->use_graph = enable != 0;
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

extern "C" int64_t lst_ctx_stat(lst_ctx* ctx, int32_t which) {
  if (!ctx || ctx->magic != MAGIC_CTX) return LST_ERR_ARG;
  switch (which) {
    case LST_STAT_PT_QUEUE: return ctx->synced ? (int64_t)ctx->h_ctl->queue_cur : (int64_t)LST_ERR_ARG;
    case LST_STAT_WORKSPACE_MB: return (int64_t)(ctx->bytes >> 20);
    default: return LST_ERR_ARG;
  }
}
