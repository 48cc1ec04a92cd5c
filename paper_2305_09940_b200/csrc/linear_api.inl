// linear_api.inl — the split Linear operator (include/osdp.h "Linear operator").
// Included at the end of osdp_api.cu: same translation unit, same GEMM instantiations as the MLP path.
//
// Y = X W + b; dX = dY W^T; dW = X^T dY; db = colsum(dY), over k slices of the contraction axis (the
// paper's own split) or of the token axis.  Slices run in order on the caller's stream; results that span slices are
// summed in fp32 in fixed slice order.

namespace osdp {
namespace {

inline int64_t lin_unit(const osdp_linear_desc* d) { return 16 / (int64_t)elem_size(d->dtype); }
int check_linear_desc(const osdp_linear_desc* d) {
  if (!d) return OSDP_ERR_NULL;
  if (d->dtype != OSDP_F32 && d->dtype != OSDP_BF16) return OSDP_ERR_DTYPE;
  const int64_t u = lin_unit(d);
  if (d->tokens < 1 || d->in_features < 1 || d->out_features < 1) return OSDP_ERR_SHAPE;
  if (d->in_features % u || d->out_features % u) return OSDP_ERR_SHAPE;
  if (d->tokens > (1ll << 30) || d->in_features > (1ll << 30) || d->out_features > (1ll << 30)) return OSDP_ERR_SHAPE;
  if (d->axis != OSDP_SPLIT_TOKENS && d->axis != OSDP_SPLIT_CONTRACTION) return OSDP_ERR_ARG;
  if (d->has_bias != 0 && d->has_bias != 1) return OSDP_ERR_ARG;
  const int64_t kmax = d->axis == OSDP_SPLIT_TOKENS ? d->tokens : d->in_features / u;
  if (d->k < 1 || (int64_t)d->k > kmax) return OSDP_ERR_K;
  return OSDP_OK;
}
// slice s of the contraction axis: whole 16-byte groups of input features
inline int64_t lin_lo(const osdp_linear_desc* d, int64_t s) {
  const int64_t u = lin_unit(d), units = d->in_features / u;
  return (s * units / d->k) * u;
}
size_t linear_workspace_bytes(const osdp_linear_desc* d, int pass) {
  if (pass == OSDP_FWD)
    return (d->axis == OSDP_SPLIT_CONTRACTION && d->k > 1) ? align_up((size_t)d->tokens * (size_t)d->out_features * 4, 256) : 0;
  return d->has_bias ? align_up((size_t)kReduceRowChunks * (size_t)d->out_features * 4, 256) : 0;
}

}  // namespace
}  // namespace osdp

extern "C" {

int osdp_split_linear_workspace_bytes(const osdp_linear_desc* desc, int pass, size_t* bytes) {
  if (!bytes) return OSDP_ERR_NULL;
  OSDP_TRY(check_linear_desc(desc));
  if (pass != OSDP_FWD && pass != OSDP_BWD) return OSDP_ERR_ARG;
  *bytes = linear_workspace_bytes(desc, pass);
  return OSDP_OK;
}

int osdp_linear_op_cost(const osdp_linear_desc* desc, int pass, osdp_op_cost* out) {
  if (!out) return OSDP_ERR_NULL;
  OSDP_TRY(check_linear_desc(desc));
  if (pass != OSDP_FWD && pass != OSDP_BWD) return OSDP_ERR_ARG;
  const uint64_t T = desc->tokens, in = desc->in_features, of = desc->out_features, e = elem_size(desc->dtype);
  const uint64_t params = in * of + (desc->has_bias ? of : 0);
  osdp_op_cost c = {};
  c.S = (double)(params * e);
  c.model_bytes = params * e + (pass == OSDP_BWD ? params * 4 : 0);
  c.act_bytes = (pass == OSDP_FWD ? T * (in + of) : T * (2 * in + of)) * e;
  c.extra_fixed = linear_workspace_bytes(desc, pass);
  *out = c;
  return OSDP_OK;
}

int osdp_split_linear_forward(const osdp_linear_desc* desc, const void* X, const void* W, const void* b, void* Y,
                              void* workspace, size_t workspace_bytes_given, void* stream) {
  g_launches = 0;
  OSDP_TRY(check_linear_desc(desc));
  if (!X || !W || !Y || (desc->has_bias && !b)) return OSDP_ERR_NULL;
  if (misaligned(X, 16) || misaligned(W, 16) || misaligned(Y, 16) || (desc->has_bias && misaligned(b, 16))) return OSDP_ERR_ALIGN;
  const size_t need = linear_workspace_bytes(desc, OSDP_FWD);
  if (need > 0 && (!workspace || misaligned(workspace, 256) || workspace_bytes_given < need)) return OSDP_ERR_WORKSPACE;
  if (desc->dtype == OSDP_BF16) OSDP_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t T = desc->tokens, in = desc->in_features, of = desc->out_features;
  const size_t e = elem_size(desc->dtype);
  const int dt = desc->dtype, k = desc->k;
  const void* bias = desc->has_bias ? b : nullptr;
  trace_set_step(11);

  if (desc->axis == OSDP_SPLIT_TOKENS) {
    for (int s = 0; s < k; ++s) {
      const int64_t lo = (int64_t)s * T / k, hi = (int64_t)(s + 1) * T / k;
      const int Ts = (int)(hi - lo);
      if (Ts == 0) continue;
      const char* Xs = (const char*)X + (size_t)lo * in * e;
      char* Ys = (char*)Y + (size_t)lo * of * e;
      EpiParams ep = {bias, Ys, nullptr, nullptr, of, 0};
      if (bias) OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS>(dt, Xs, in, W, of, GemmShape{Ts, (int)of, (int)in}, ep, st)));
      else      OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_PLAIN>(dt, Xs, in, W, of, GemmShape{Ts, (int)of, (int)in}, ep, st)));
    }
    return OSDP_OK;
  }
  // contraction axis: Y (+)= X[:, lo:hi] W[lo:hi, :]   (partial products summed)
  float* Yacc = (float*)workspace;
  for (int s = 0; s < k; ++s) {
    const int64_t lo = lin_lo(desc, s), hi = lin_lo(desc, s + 1);
    const int ks = (int)(hi - lo);
    if (ks == 0) continue;
    const char* Xs = (const char*)X + (size_t)lo * e;            // X[:, lo:hi], leading dimension in
    const char* Ws = (const char*)W + (size_t)lo * of * e;       // W[lo:hi, :]
    if (k == 1) {
      EpiParams ep = {bias, Y, nullptr, nullptr, of, 0};
      if (bias) OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS>(dt, Xs, in, Ws, of, GemmShape{(int)T, (int)of, ks}, ep, st)));
      else      OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_PLAIN>(dt, Xs, in, Ws, of, GemmShape{(int)T, (int)of, ks}, ep, st)));
    } else {
      EpiParams ep = {nullptr, Yacc, nullptr, nullptr, of, s == 0 ? 0 : 1};
      OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_ACCUM_F32>(dt, Xs, in, Ws, of, GemmShape{(int)T, (int)of, ks}, ep, st)));
    }
  }
  if (k > 1) {   // Y = storage(Yacc + b)
    trace_set_step(10);
    sm100::DeviceInfo dev;
    OSDP_TRY(sm100::current_device(&dev));
    OSDP_TRY(launch_acc_to_out(dt, Yacc, bias, Y, T, (int)of, dev.sms, st));
  }
  return OSDP_OK;
}

int osdp_split_linear_backward(const osdp_linear_desc* desc, const void* X, const void* W, const void* dY, void* dX,
                               float* dW, float* db, void* workspace, size_t workspace_bytes_given, void* stream) {
  g_launches = 0;
  OSDP_TRY(check_linear_desc(desc));
  if (!X || !W || !dY || !dX || !dW || (desc->has_bias && !db)) return OSDP_ERR_NULL;
  if (misaligned(X, 16) || misaligned(W, 16) || misaligned(dY, 16) || misaligned(dX, 16) || misaligned(dW, 16) ||
      (desc->has_bias && misaligned(db, 16)))
    return OSDP_ERR_ALIGN;
  const size_t need = linear_workspace_bytes(desc, OSDP_BWD);
  if (need > 0 && (!workspace || misaligned(workspace, 256) || workspace_bytes_given < need)) return OSDP_ERR_WORKSPACE;
  if (desc->dtype == OSDP_BF16) OSDP_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t T = desc->tokens, in = desc->in_features, of = desc->out_features;
  const size_t e = elem_size(desc->dtype);
  const int dt = desc->dtype, k = desc->k;
  float* scratch = (float*)workspace;

  if (desc->axis == OSDP_SPLIT_TOKENS) {
    // dX_s, dW (+)=, db (+)= only share inputs: side by side on small slices (helper streams, osdp_api.cu)
    const int64_t ts_max = (T + k - 1) / k;
    const int64_t fork_max = sm100::tuning().fork_max_tiles.load();
    const bool fork = fork_max > 0 && tiles_256(in, of) <= fork_max && tiles_256(ts_max, in) <= fork_max;
    ForkCtx* fc = nullptr;
    if (fork) {
      OSDP_TRY(fork_ctx(&fc));
      OSDP_TRY(fork_from(fc, st));
    }
    int first = 1;
    for (int s = 0; s < k; ++s) {
      const int64_t lo = (int64_t)s * T / k, hi = (int64_t)(s + 1) * T / k;
      const int Ts = (int)(hi - lo);
      if (Ts == 0) continue;
      const int beta = first ? 0 : 1;
      first = 0;
      const char* Xs = (const char*)X + (size_t)lo * in * e;
      const char* dYs = (const char*)dY + (size_t)lo * of * e;
      char* dXs = (char*)dX + (size_t)lo * in * e;
      trace_set_step(12);   // dX_s = dY_s W^T
      EpiParams e1 = {nullptr, dXs, nullptr, nullptr, in, 0};
      OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_PLAIN>(dt, dYs, of, W, of, GemmShape{Ts, (int)in, (int)of}, e1, st)));
      trace_set_step(13);   // dW (+)= X_s^T dY_s   (slices of dW in order on ONE stream: fixed summation order)
      EpiParams e2 = {nullptr, dW, nullptr, nullptr, of, beta};
      OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, Xs, in, dYs, of, GemmShape{(int)in, (int)of, Ts}, e2,
                                                        fork ? fc->side[0] : st)));
      if (desc->has_bias) {
        trace_set_step(8);  // db (+)= colsum(dY_s)
        OSDP_TRY(colsum_rows(dt, dYs, (int)of, db, Ts, scratch, beta, fork ? fc->side[1] : st));
      }
    }
    if (fork) OSDP_TRY(join_into(fc, st));
    return OSDP_OK;
  }
  // contraction axis: every slice writes its own columns of dX and rows of dW; db once
  if (desc->has_bias) {
    trace_set_step(8);
    OSDP_TRY(colsum_rows(dt, dY, (int)of, db, (int)T, scratch, 0, st));
  }
  for (int s = 0; s < k; ++s) {
    const int64_t lo = lin_lo(desc, s), hi = lin_lo(desc, s + 1);
    const int ks = (int)(hi - lo);
    if (ks == 0) continue;
    const char* Ws = (const char*)W + (size_t)lo * of * e;       // W[lo:hi, :]  = (W[lo:hi, :]^T)^T: K-major B with N = ks
    trace_set_step(12);   // dX[:, lo:hi] = dY W[lo:hi, :]^T
    EpiParams e1 = {nullptr, (char*)dX + (size_t)lo * e, nullptr, nullptr, in, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_PLAIN>(dt, dY, of, Ws, of, GemmShape{(int)T, ks, (int)of}, e1, st)));
    trace_set_step(13);   // dW[lo:hi, :] = X[:, lo:hi]^T dY
    EpiParams e2 = {nullptr, dW + (size_t)lo * of, nullptr, nullptr, of, 0};
    OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, (const char*)X + (size_t)lo * e, in, dY, of,
                                                      GemmShape{ks, (int)of, (int)T}, e2, st)));
  }
  return OSDP_OK;
}

}  // extern "C"
