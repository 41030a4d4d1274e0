// lst_api_audit.inl -- included by lst_api.cu: lst_ctx_audit (lst_audit.cuh), a debugging call outside every timed path.

extern "C" int lst_ctx_audit(lst_ctx* ctx, lst_audit_report* rep) {
  if (!ctx || ctx->magic != MAGIC_CTX || !rep) return LST_ERR_ARG;
  if (!ctx->synced || ctx->last_n_events == 0) return LST_ERR_ARG;
  const Ctl& h = *ctx->h_ctl;
  if (h.error) return (h.error & E_BAD_SENSOR) ? LST_ERR_ARG : LST_ERR_CAPACITY;
  memset(rep, 0, sizeof(*rep));
  const int mask = ctx->g->cuts.stage_mask;
  const int do_md = (mask & 1) != 0, do_ls = (mask & 3) == 3, do_pt = (mask & 31) == 31 && ctx->dev.n_pls > 0;
  AuditAcc* acc = nullptr;
  if (cudaMalloc(&acc, sizeof(AuditAcc)) != cudaSuccess) {
    cudaGetLastError();
    return LST_ERR_CUDA;
  }
  cudaStream_t st = ctx->stream;
  const Dev& d = ctx->dev;
  const int grid = ctx->g->n_sm * 8;
  bool ok = cudaMemsetAsync(acc, 0, sizeof(AuditAcc), st) == cudaSuccess;
  if (ok) {
    if (do_md) k_audit_md<<<grid, kBlock, 0, st>>>(d, acc);
    if (do_ls) k_audit_ls<<<grid, kBlock, 0, st>>>(d, acc);
    if (do_pt) {
      const dim3 g2(ctx->g->n_sm * 2, ctx->last_n_events);
      k_audit_pt<false><<<g2, kBlock, 0, st>>>(d, acc);
      k_audit_pt<true><<<g2, kBlock, 0, st>>>(d, acc);
    }
    k_audit_chain<<<grid, kBlock, 0, st>>>(d, acc, do_md, do_ls, do_pt);
  }
  AuditAcc host;
  ok = ok && cudaGetLastError() == cudaSuccess &&
       cudaMemcpyAsync(&host, acc, sizeof(AuditAcc), cudaMemcpyDeviceToHost, st) == cudaSuccess &&
       cudaStreamSynchronize(st) == cudaSuccess;
  cudaFree(acc);
  if (!ok) return LST_ERR_CUDA;
  const int kind[AU_N] = {K_MD, K_LS, K_PT3, K_PT5};
  const int stage[AU_N] = {LST_ST_MD, LST_ST_LS, LST_ST_PT3, LST_ST_PT5};
  const bool on[AU_N] = {do_md != 0, do_ls != 0, do_pt != 0, do_pt != 0};
  for (int s = 0; s < AU_N; ++s) {
    if (!on[s]) continue;
    rep->candidates[s] = (int64_t)host.cand[s];
    rep->accepted[s] = (int64_t)host.acc[s];
    rep->near[s] = (int64_t)host.near[s];
    rep->hash_exact[s] = host.hash_exact[s];
    rep->hash_chain[s] = host.hash_chain[s];
    rep->chain_objects[s] = h.total[kind[s]];
    for (int e = 0; e < ctx->last_n_events; ++e) {
      rep->chain_near[s] += (int64_t)ctx->h_ev_cnt[(size_t)e * kEvCnt + stage[s]];
      rep->chain_candidates[s] += (int64_t)ctx->h_ev_cnt[(size_t)e * kEvCnt + kStages + stage[s]];
    }
    rep->mismatches += (rep->candidates[s] != rep->chain_candidates[s]) + (rep->accepted[s] != rep->chain_objects[s]) +
                       (rep->near[s] != rep->chain_near[s]) + (rep->hash_exact[s] != rep->hash_chain[s]);
  }
  return LST_OK;
}
