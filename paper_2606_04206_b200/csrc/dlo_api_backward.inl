// dlo_api_backward.inl — dlo_backward and the host-buffer convenience calls (included by dlo_api.cu)

template <int VPL> static cudaError_t launch_adjoint_t(dlo_sim* s, const KParams& P, int t0, int t1) {
  cudaError_t e = cudaFuncSetAttribute(k_adjoint<VPL>, cudaFuncAttributeMaxDynamicSharedMemorySize, s->smem_adj > 48 * 1024 ? s->smem_adj : 48 * 1024);
  if (e != cudaSuccess) return e;
  const int grid = (P.B + s->wpb_adj - 1) / s->wpb_adj;
  {
    LaunchTimer lt(s, 2, s->stream, (int64_t)P.B * (t1 - t0));
    k_adjoint<VPL><<<grid, s->wpb_adj * 32, s->smem_adj, s->stream>>>(P, t0, t1);
  }
  s->launches += 1;
  return cudaGetLastError();
}
static cudaError_t launch_adjoint(dlo_sim* s, const KParams& P, int t0, int t1) {
  switch (s->VPL) {
#ifdef DLO_VPL_ONLY   /* development builds: one instantiation only */
    default: return launch_adjoint_t<DLO_VPL_ONLY>(s, P, t0, t1);
#else
    case 2: return launch_adjoint_t<2>(s, P, t0, t1);
    case 4: return launch_adjoint_t<4>(s, P, t0, t1);
    case 6: return launch_adjoint_t<6>(s, P, t0, t1);
    default: return launch_adjoint_t<8>(s, P, t0, t1);
#endif
  }
}

extern "C" {

dlo_status dlo_backward(dlo_sim* s, const float* gxT, const float* gvT, float* g_actions, float* g_x0, float* g_v0, float* g_material) {
  ENTER(s);
  if (s->stride <= 0 || s->H_done <= 0) return fail(DLO_ERR_BAD_STATE, "dlo_backward needs a rollout with checkpoint_stride > 0");
  const int H = s->H_done, stride = s->stride, B = s->P.B;
  const size_t blk = s->blk;
  {
    dlo_status st = ensure_tape(s, H, stride);
    if (st) return st;
  }
  s->have_adj = false;
  // each buffer on its own: a failed allocation leaves the others (and the handle) usable, and is retried by the next call
  if (!s->adj) CU(dalloc(&s->adj, (size_t)B * blk));
  if (!s->replay) CU(dalloc(&s->replay, (size_t)B * blk));
  if (!s->gmat) CU(dalloc(&s->gmat, (size_t)B * 5));
  if (s->P.self_contact && !s->acc_tape) CU(dalloc(&s->acc_tape, (size_t)B * s->P.N_C * 3 * 33 * s->VPL));
  const size_t nadj = (size_t)B * blk;
  k_seed_adjoint<<<(unsigned)((nadj + 255) / 256), 256, 0, s->stream>>>(B, s->P.N, s->P.NS, gxT, gvT, s->adj);
  s->launches += 1;
  CU(cudaGetLastError());
  CU(cudaMemsetAsync(s->gmat, 0, (size_t)B * 5 * sizeof(float), s->stream));
  if (g_actions && s->P.G > 0) CU(cudaMemsetAsync(g_actions, 0, (size_t)H * B * s->P.G * 6 * sizeof(float), s->stream));
  const int nseg = (H + stride - 1) / stride;
  // K tape buffers, segment g in buffer g % K.  The forward rollout left its last K segments on tape; every other segment
  // is replayed from its checkpoint first.  With K > 1 the replays run on a second stream: the replay of segment r goes
  // into the buffer the adjoint of segment r + K has just finished with, K - 1 adjoints before its records are needed.
  const int K = s->n_tape;
  const bool overlap = nseg > 1 && K > 1;
  if (overlap && !s->aux) {
    CU(cudaStreamCreateWithFlags(&s->aux, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&s->ev_fwd, cudaEventDisableTiming));
  }
  if (overlap)
    for (int k = 0; k < K; ++k) {
      if (!s->ev_rep[k]) CU(cudaEventCreateWithFlags(&s->ev_rep[k], cudaEventDisableTiming));
      if (!s->ev_adj[k]) CU(cudaEventCreateWithFlags(&s->ev_adj[k], cudaEventDisableTiming));
    }
  cudaStream_t rs = overlap ? s->aux : s->stream;        // stream of the replays
  // the forward rollout chose the buffers of its taped segments with the buffers it had THEN; if the set has changed since
  // (a buffer that could not be allocated before), its records are not where this pass looks
  const int tape_lo = (s->tape_K == K) ? s->tape_lo : nseg;
  s->tape_lo = 1 << 30;   // the buffers are overwritten below
  std::vector<char> issued(nseg, 0);
  auto replay = [&](int g) -> dlo_status {
    const int t0 = g * stride, t1 = (t0 + stride < H) ? t0 + stride : H, buf = g % K;
    // the buffer's last user is segment g + K, whose adjoint has been launched on the main stream by now
    if (overlap && g + K <= nseg - 1) CU(cudaStreamWaitEvent(s->aux, s->ev_adj[buf], 0));
    CU(cudaMemcpyAsync(s->replay, s->ckpt + (size_t)g * B * blk, nadj * sizeof(float), cudaMemcpyDeviceToDevice, rs));
    KParams Pf = s->P;
    Pf.state = s->replay; Pf.tape = s->tapes[buf]; Pf.tape_flag = s->tape_flags[buf];
    if (s->side[buf]) {
      CU(cudaMemsetAsync(s->side_count[buf], 0, sizeof(int), rs));
      Pf.side = s->side[buf]; Pf.side_count = s->side_count[buf]; Pf.tape_slot = s->tape_slot[buf]; Pf.side_cap = s->side_cap; Pf.side_floats = s->side_floats;
    }
    if (s->sort_mode) {   // envs in the order of the work the segment after this one took (its tape was written earlier on this stream, or before ev_fwd)
      const int src = (g + 1) % K;
      if ((s->sort_mode & 2) && g + 1 < nseg && s->stat_rep_valid[src]) { CU(sort_envs(s, s->stat_rep[src], 0, 4, s->perm_rep, rs)); Pf.perm = s->perm_rep; }
      Pf.stat = s->stat_rep[buf];
    }
    CU(launch_forward(s, Pf, t0, t1, 0, true, rs));
    s->stat_rep_valid[buf] = s->sort_mode != 0;
    if (overlap) CU(cudaEventRecord(s->ev_rep[buf], rs));
    issued[g] = 1;
    return DLO_OK;
  };
  if (overlap) {   // the replays read the checkpoints the forward rollout wrote on the main stream
    CU(cudaEventRecord(s->ev_fwd, s->stream));
    CU(cudaStreamWaitEvent(s->aux, s->ev_fwd, 0));
  }
  dlo_status rst = DLO_OK;
  for (int g = nseg - 1; g >= 0; --g) {
    const int t0 = g * stride, t1 = (t0 + stride < H) ? t0 + stride : H, buf = g % K;
    // replays that can be on their way now: this segment's own (if the forward did not tape it) and those of the K - 1 before it
    for (int r = g; r >= 0 && r > g - K; --r)
      if (r < tape_lo && !issued[r] && (r == g || overlap) && (rst = replay(r))) return rst;
    if (overlap && issued[g]) CU(cudaStreamWaitEvent(s->stream, s->ev_rep[buf], 0));
    KParams Pa = s->P;
    smem_layout(Pa, s->VPL, true);
    Pa.tape = s->tapes[buf]; Pa.tape_flag = s->tape_flags[buf]; Pa.adj = s->adj; Pa.acc_tape = s->acc_tape; Pa.gmat = s->gmat; Pa.g_actions = (s->P.G > 0) ? g_actions : nullptr;
    if (s->side[buf]) { Pa.side = s->side[buf]; Pa.tape_slot = s->tape_slot[buf]; Pa.side_floats = s->side_floats; Pa.side_cap = s->side_cap; }
    if ((s->sort_mode & 4) && s->stat_rep_valid[buf]) {   // envs whose substeps must be recomputed (self-contact corrections) share CTAs
      CU(sort_envs(s, s->stat_rep[buf], 1, 0, s->perm_main, s->stream));
      Pa.perm = s->perm_main;
    }
    CU(launch_adjoint(s, Pa, t0, t1));
    if (overlap) CU(cudaEventRecord(s->ev_adj[buf], s->stream));
  }
  if (g_x0 || g_v0) {
    const size_t n = (size_t)B * STATE_ROWS * s->P.N;
    k_get_state<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(B, s->P.N, s->P.NS, s->adj, g_x0, g_v0, nullptr, nullptr, nullptr);
    s->launches += 1;
    CU(cudaGetLastError());
  }
  if (g_material) CU(cudaMemcpyAsync(g_material, s->gmat, (size_t)B * 5 * sizeof(float), cudaMemcpyDeviceToDevice, s->stream));
  s->have_adj = true;
  return DLO_OK;
}

dlo_status dlo_get_state_adjoint(dlo_sim* s, float* g_x, float* g_v, float* g_d1, float* g_kb) {
  ENTER(s);
  if (!s->have_adj) return fail(DLO_ERR_BAD_STATE, "dlo_get_state_adjoint needs a completed dlo_backward");
  const size_t n = (size_t)s->P.B * STATE_ROWS * s->P.N;
  k_get_state<<<(unsigned)((n + 255) / 256), 256, 0, s->stream>>>(s->P.B, s->P.N, s->P.NS, s->adj, g_x, g_v, g_d1, g_kb, nullptr);
  s->launches += 1;
  CU(cudaGetLastError());
  return DLO_OK;
}

// staging of the *_host calls lives in the handle: grow-only buffers, freed by dlo_destroy
static dlo_status stage_host(float** pinned, size_t n) {
  if (*pinned) { cudaFreeHost(*pinned); *pinned = nullptr; }
  CU(cudaMallocHost((void**)pinned, (n ? n : 1) * sizeof(float)));
  return DLO_OK;
}
static dlo_status stage_dev(dlo_sim* s, float** p, size_t n) {
  if (*p) { CU(cudaStreamSynchronize(s->stream)); cudaFree(*p); *p = nullptr; }
  CU(dalloc(p, n));
  return DLO_OK;
}

dlo_status dlo_rollout_forward_host(dlo_sim* s, const float* x0, const float* v0, const float* kb0, const float* actions,
                                    int32_t horizon, int32_t stride, float* x_T, float* v_T) {
  ENTER(s);
  if (!x0 || !v0) return fail(DLO_ERR_INVALID_ARG, "NULL argument");
  if (horizon < 0 || stride < 0) return fail(DLO_ERR_INVALID_ARG, "horizon < 0 or checkpoint_stride < 0");
  const KParams& P = s->P;
  const size_t nx = (size_t)P.B * 3 * P.N, nk = (size_t)P.B * 2 * P.N, na = (size_t)horizon * P.B * P.G * 6;
  if (P.G > 0 && horizon > 0 && !actions) return fail(DLO_ERR_INVALID_ARG, "actions is NULL");
  dlo_status st;
  {   // the fixed-size buffers (sizes depend on the config only), each checked on its own
    float** hp[] = {&s->hx0, &s->hv0, &s->hxT, &s->hvT};
    float** dp[] = {&s->dx0, &s->dv0, &s->dxT, &s->dvT};
    for (int k = 0; k < 4; ++k) { if (!*hp[k] && (st = stage_host(hp[k], nx))) return st; if (!*dp[k] && (st = stage_dev(s, dp[k], nx))) return st; }
  }
  if (!s->hkb && (st = stage_host(&s->hkb, nk))) return st;
  if (!s->dkb && (st = stage_dev(s, &s->dkb, nk))) return st;
  if (na > s->hact_n) { if ((st = stage_host(&s->hact, na))) { s->hact_n = 0; return st; } s->hact_n = na; }
  if (na > s->dact_n) {
    if (s->actions == s->dact) { s->actions = nullptr; s->P.actions = nullptr; s->H_actions = 0; }   // about to be freed
    if ((st = stage_dev(s, &s->dact, na))) { s->dact_n = 0; return st; }
    s->dact_n = na;
  }
  memcpy(s->hx0, x0, nx * sizeof(float));
  memcpy(s->hv0, v0, nx * sizeof(float));
  CU(cudaMemcpyAsync(s->dx0, s->hx0, nx * sizeof(float), cudaMemcpyHostToDevice, s->stream));
  CU(cudaMemcpyAsync(s->dv0, s->hv0, nx * sizeof(float), cudaMemcpyHostToDevice, s->stream));
  if (kb0) { memcpy(s->hkb, kb0, nk * sizeof(float)); CU(cudaMemcpyAsync(s->dkb, s->hkb, nk * sizeof(float), cudaMemcpyHostToDevice, s->stream)); }
  if (na > 0) { memcpy(s->hact, actions, na * sizeof(float)); CU(cudaMemcpyAsync(s->dact, s->hact, na * sizeof(float), cudaMemcpyHostToDevice, s->stream)); }
  if ((st = dlo_set_state(s, s->dx0, s->dv0, kb0 ? s->dkb : nullptr))) return st;
  if ((st = dlo_set_actions(s, s->dact, horizon))) return st;   // the handle's own copy: stays valid for dlo_backward
  if ((st = dlo_rollout_forward(s, horizon, stride))) return st;
  if ((st = dlo_get_state(s, x_T ? s->dxT : nullptr, v_T ? s->dvT : nullptr, nullptr, nullptr))) return st;
  if (x_T) CU(cudaMemcpyAsync(s->hxT, s->dxT, nx * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
  if (v_T) CU(cudaMemcpyAsync(s->hvT, s->dvT, nx * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  if (x_T) memcpy(x_T, s->hxT, nx * sizeof(float));
  if (v_T) memcpy(v_T, s->hvT, nx * sizeof(float));
  return DLO_OK;
}

dlo_status dlo_backward_host(dlo_sim* s, const float* gxT, const float* gvT, float* g_actions, float* g_x0, float* g_v0, float* g_material) {
  ENTER(s);
  if (s->stride <= 0 || s->H_done <= 0) return fail(DLO_ERR_BAD_STATE, "dlo_backward needs a rollout with checkpoint_stride > 0");
  const KParams& P = s->P;
  const size_t nx = (size_t)P.B * 3 * P.N, na = (size_t)s->H_done * P.B * P.G * 6, nm = (size_t)P.B * DLO_N_MATERIAL_GRADS;
  dlo_status st;
  float** dp[] = {&s->dsx, &s->dsv, &s->dgx, &s->dgv};
  for (float** q : dp) if (!*q && (st = stage_dev(s, q, nx))) return st;
  if (!s->dgm && (st = stage_dev(s, &s->dgm, nm))) return st;
  if (na > s->dga_n) { if ((st = stage_dev(s, &s->dga, na))) { s->dga_n = 0; return st; } s->dga_n = na; }
  if (gxT) CU(cudaMemcpyAsync(s->dsx, gxT, nx * sizeof(float), cudaMemcpyHostToDevice, s->stream));
  if (gvT) CU(cudaMemcpyAsync(s->dsv, gvT, nx * sizeof(float), cudaMemcpyHostToDevice, s->stream));
  st = dlo_backward(s, gxT ? s->dsx : nullptr, gvT ? s->dsv : nullptr, (g_actions && na) ? s->dga : nullptr, g_x0 ? s->dgx : nullptr,
                    g_v0 ? s->dgv : nullptr, g_material ? s->dgm : nullptr);
  if (st) return st;
  if (g_actions && na) CU(cudaMemcpyAsync(g_actions, s->dga, na * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
  if (g_x0) CU(cudaMemcpyAsync(g_x0, s->dgx, nx * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
  if (g_v0) CU(cudaMemcpyAsync(g_v0, s->dgv, nx * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
  if (g_material) CU(cudaMemcpyAsync(g_material, s->dgm, nm * sizeof(float), cudaMemcpyDeviceToHost, s->stream));
  CU(cudaStreamSynchronize(s->stream));
  return DLO_OK;
}

}  // extern "C"
