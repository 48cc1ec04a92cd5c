// zdp_api.inl — ZDP execution of the ffn-axis split MLP with weight-slice gathering (include/osdp.h "ZDP mode";
// SURVEY.md section 8(f2)).  Included at the end of osdp_api.cu.
//
// Per slice: all-gather the slice's parameters (comm stream) -> the ffn-split slice computation on the gathered buffer
// (compute stream) -> reduce-scatter the slice's weight gradients (comm stream).  Two gathered buffers and two gradient
// staging buffers let the collectives of neighbouring slices overlap the GEMMs.

namespace osdp {
namespace {

struct ZdpGeom {
  int64_t T, h, f, N, rank, k, unit, groups;   // groups = f / (N unit)
  size_t e;
  int dt;
  int64_t lo(int64_t s) const { return (s * groups / k) * N * unit; }
  int64_t fs_max() const { return ((groups + k - 1) / k) * N * unit; }
};
int zdp_geom(const osdp_zdp_desc* d, ZdpGeom* g) {
  if (!d) return OSDP_ERR_NULL;
  const osdp_mlp_desc* m = &d->mlp;
  if (m->dtype != OSDP_F32 && m->dtype != OSDP_BF16) return OSDP_ERR_DTYPE;
  if (d->world < 1 || d->world > 4096 || d->rank < 0 || d->rank >= d->world) return OSDP_ERR_ARG;
  const int64_t unit = 16 / (int64_t)elem_size(m->dtype);
  if (m->tokens < 1 || m->hidden < 1 || m->ffn < 1) return OSDP_ERR_SHAPE;
  if (m->tokens > (1ll << 30) || m->hidden > (1ll << 30) || m->ffn > (1ll << 30)) return OSDP_ERR_SHAPE;
  if (m->hidden % (d->world * unit) || m->ffn % (d->world * unit)) return OSDP_ERR_SHAPE;
  const int64_t groups = m->ffn / (d->world * unit);
  if (m->k < 1 || (int64_t)m->k > groups) return OSDP_ERR_K;
  *g = ZdpGeom{m->tokens, m->hidden, m->ffn, d->world, d->rank, m->k, unit, groups, elem_size(m->dtype), m->dtype};
  return OSDP_OK;
}
void zdp_slice(const ZdpGeom& g, int64_t s, osdp_zdp_slice* out) {
  int64_t off = 0;
  for (int64_t i = 0; i <= s && i <= g.k; ++i) {
    osdp_zdp_slice sl = {};
    if (i < g.k) {
      sl.lo = g.lo(i);
      sl.hi = g.lo(i + 1);
      const int64_t fs = sl.hi - sl.lo;
      sl.w1_off = off;                 sl.w1_elems = (g.h / g.N) * fs;
      sl.b1_off = sl.w1_off + sl.w1_elems;   sl.b1_elems = fs / g.N;
      sl.w2_off = sl.b1_off + sl.b1_elems;   sl.w2_elems = (fs / g.N) * g.h;
      off = sl.w2_off + sl.w2_elems;
    } else {   // the b2 piece at the tail
      sl.lo = sl.hi = g.f;
      sl.b1_off = off;
      sl.b1_elems = g.h / g.N;
      sl.w1_off = sl.w2_off = off;
      off += sl.b1_elems;
    }
    if (i == s) *out = sl;
  }
}
inline int64_t zdp_shard_elems(const ZdpGeom& g) { return (g.h * g.f * 2 + g.f + g.h) / g.N; }

// gathered slice buffer: W1g [h x fs_max] | b1g [fs_max] | W2g [fs_max x h], each part 256-byte aligned
struct ZdpBuf {
  size_t w1, b1, w2, total;
};
ZdpBuf zdp_buf(const ZdpGeom& g, size_t e) {
  ZdpBuf b;
  const size_t fm = (size_t)g.fs_max();
  b.w1 = 0;
  b.b1 = align_up((size_t)g.h * fm * e, 256);
  b.w2 = b.b1 + align_up(fm * e, 256);
  b.total = b.w2 + align_up(fm * (size_t)g.h * e, 256);
  return b;
}
struct ZdpWs {
  size_t gbuf[2], b2g, rbuf[2], db2s, zs, hs, acc, scratch1, scratch2, total;
};
ZdpWs zdp_ws(const ZdpGeom& g, int pass) {
  ZdpWs w = {};
  const ZdpBuf gb = zdp_buf(g, g.e), rb = zdp_buf(g, 4);
  size_t off = 0;
  w.gbuf[0] = off; off += gb.total;
  w.gbuf[1] = off; off += gb.total;
  const size_t slice_buf = align_up((size_t)g.T * (size_t)g.fs_max() * g.e, 256);
  const size_t acc = g.k == 1 ? 0 : align_up((size_t)g.T * (size_t)g.h * 4, 256);
  if (pass == OSDP_FWD) {
    w.b2g = off; off += align_up((size_t)g.h * g.e, 256);
    w.hs = off; off += slice_buf;
    w.acc = off; off += acc;
  } else {
    w.rbuf[0] = off; off += rb.total;
    w.rbuf[1] = off; off += rb.total;
    w.db2s = off; off += align_up((size_t)g.h * 4, 256);
    w.zs = off; off += slice_buf;
    w.hs = off; off += slice_buf;
    w.acc = off; off += acc;
    w.scratch1 = off; off += db1_scratch_bytes(g.T, g.fs_max());
    w.scratch2 = off; off += db2_scratch_bytes(g.h);
  }
  w.total = off;
  return w;
}

// The steps of one call in enqueue order.  Forward: gather b2, gather slice 0, then for every slice: gather the next one,
// compute this one.  Backward: gather slice 0, then for every slice: gather the next one, compute this one,
// reduce-scatter its gradients; last, reduce-scatter db2.
void zdp_steps(const ZdpGeom& g, int pass, std::vector<osdp_zdp_step>* out) {
  auto piece_bytes = [&](int64_t s, size_t e) {
    osdp_zdp_slice sl;
    zdp_slice(g, s, &sl);
    return (uint64_t)(sl.w1_elems + sl.b1_elems + sl.w2_elems) * e;
  };
  if (pass == OSDP_FWD) out->push_back({OSDP_ZDP_GATHER, (int32_t)g.k, 0, 1, piece_bytes(g.k, g.e)});
  out->push_back({OSDP_ZDP_GATHER, 0, 0, 1, piece_bytes(0, g.e)});
  for (int64_t s = 0; s < g.k; ++s) {
    if (s + 1 < g.k) out->push_back({OSDP_ZDP_GATHER, (int32_t)(s + 1), (int32_t)((s + 1) % 2), 1, piece_bytes(s + 1, g.e)});
    out->push_back({OSDP_ZDP_COMPUTE, (int32_t)s, (int32_t)(s % 2), 0, 0});
    if (pass == OSDP_BWD) out->push_back({OSDP_ZDP_REDUCE_SCATTER, (int32_t)s, (int32_t)(s % 2), 1, piece_bytes(s, 4)});
  }
  if (pass == OSDP_BWD) out->push_back({OSDP_ZDP_REDUCE_SCATTER, (int32_t)g.k, 0, 1, piece_bytes(g.k, 4)});
}

// events of one call (per host thread and device, created on first use)
struct ZdpEvents {
  cudaEvent_t entry = nullptr, gathered[2] = {}, freed[2] = {}, grads[2] = {}, scattered[2] = {}, b2 = nullptr, tail = nullptr;
  bool ready = false;
};
int zdp_events(ZdpEvents** out) {
  static thread_local ZdpEvents evs[sm100::kMaxDevices];
  sm100::DeviceInfo dev;
  const int rc = sm100::current_device(&dev);
  if (rc != OSDP_OK) return rc;
  ZdpEvents& e = evs[dev.ordinal];
  if (!e.ready) {
    cudaEvent_t* all[] = {&e.entry, &e.gathered[0], &e.gathered[1], &e.freed[0], &e.freed[1], &e.grads[0], &e.grads[1],
                          &e.scattered[0], &e.scattered[1], &e.b2, &e.tail};
    for (cudaEvent_t* p : all) OSDP_CUDA_TRY(cudaEventCreateWithFlags(p, cudaEventDisableTiming));
    e.ready = true;
  }
  *out = &e;
  return OSDP_OK;
}

int zdp_all_gather(const osdp_comm* comm, const void* send, void* recv, size_t bytes, cudaStream_t st) {
  if (bytes == 0) return OSDP_OK;
  if (!comm) {   // world == 1
    OSDP_CUDA_TRY(cudaMemcpyAsync(recv, send, bytes, cudaMemcpyDeviceToDevice, st));
    return OSDP_OK;
  }
  return comm->all_gather(comm->ctx, send, recv, bytes, (void*)st) == 0 ? OSDP_OK : OSDP_ERR_COMM;
}
int zdp_reduce_scatter(const osdp_comm* comm, const float* send, float* recv, size_t floats, cudaStream_t st) {
  if (floats == 0) return OSDP_OK;
  if (!comm) {
    OSDP_CUDA_TRY(cudaMemcpyAsync(recv, send, floats * 4, cudaMemcpyDeviceToDevice, st));
    return OSDP_OK;
  }
  return comm->reduce_scatter_f32(comm->ctx, send, recv, floats, (void*)st) == 0 ? OSDP_OK : OSDP_ERR_COMM;
}

// An error return after comm_stream was forked from compute_stream (a failed collective, a failed launch) still joins
// it back, so a stream capture the call was part of is not left with an unjoined stream.  Disarmed on the normal path.
struct ZdpJoin {
  cudaStream_t cs, ms;
  cudaEvent_t tail;
  bool armed;
  ~ZdpJoin() {
    if (armed && cudaEventRecord(tail, ms) == cudaSuccess) cudaStreamWaitEvent(cs, tail, 0);
  }
};

int zdp_check_call(const osdp_zdp_desc* desc, ZdpGeom* g, int pass, const void* workspace, size_t given, const osdp_comm* comm) {
  OSDP_TRY(zdp_geom(desc, g));
  if (g->N > 1 && (!comm || !comm->all_gather || !comm->reduce_scatter_f32)) return OSDP_ERR_NULL;
  if (!workspace) return OSDP_ERR_NULL;
  if (misaligned(workspace, 256) || given < zdp_ws(*g, pass).total) return OSDP_ERR_WORKSPACE;
  if (g->dt == OSDP_BF16) OSDP_TRY(check_arch());
  return OSDP_OK;
}

}  // namespace
}  // namespace osdp

extern "C" {

int osdp_zdp_shard_elems(const osdp_zdp_desc* desc, int64_t* elems) {
  if (!elems) return OSDP_ERR_NULL;
  ZdpGeom g;
  OSDP_TRY(zdp_geom(desc, &g));
  *elems = zdp_shard_elems(g);
  return OSDP_OK;
}

int osdp_zdp_slice_layout(const osdp_zdp_desc* desc, int32_t s, osdp_zdp_slice* out) {
  if (!out) return OSDP_ERR_NULL;
  ZdpGeom g;
  OSDP_TRY(zdp_geom(desc, &g));
  if (s < 0 || s > g.k) return OSDP_ERR_ARG;
  zdp_slice(g, s, out);
  return OSDP_OK;
}

int64_t osdp_zdp_schedule(const osdp_zdp_desc* desc, int pass, int64_t max_steps, osdp_zdp_step* steps) {
  ZdpGeom g;
  const int rc = zdp_geom(desc, &g);
  if (rc != OSDP_OK) return -(int64_t)rc;
  if (pass != OSDP_FWD && pass != OSDP_BWD) return -(int64_t)OSDP_ERR_ARG;
  std::vector<osdp_zdp_step> v;
  zdp_steps(g, pass, &v);
  for (int64_t i = 0; steps && i < (int64_t)v.size() && i < max_steps; ++i) steps[i] = v[(size_t)i];
  return (int64_t)v.size();
}

int osdp_zdp_ffn_split_mlp_workspace_bytes(const osdp_zdp_desc* desc, int pass, size_t* bytes) {
  if (!bytes) return OSDP_ERR_NULL;
  ZdpGeom g;
  OSDP_TRY(zdp_geom(desc, &g));
  if (pass != OSDP_FWD && pass != OSDP_BWD) return OSDP_ERR_ARG;
  *bytes = zdp_ws(g, pass).total;
  return OSDP_OK;
}

int osdp_zdp_ffn_split_mlp_op_cost(const osdp_zdp_desc* desc, int pass, osdp_op_cost* out) {
  if (!out) return OSDP_ERR_NULL;
  ZdpGeom g;
  OSDP_TRY(zdp_geom(desc, &g));
  if (pass != OSDP_FWD && pass != OSDP_BWD) return OSDP_ERR_ARG;
  const uint64_t T = g.T, h = g.h, f = g.f, e = g.e, params = 2 * h * f + f + h;
  osdp_op_cost c = {};
  c.S = (double)(params * e);
  c.model_bytes = params * e + (pass == OSDP_BWD ? params * 4 : 0);       // sharded: osdp_cost_eval divides by N in ZDP mode
  c.act_bytes = (pass == OSDP_FWD ? 2 : 3) * T * h * e;
  // sliceable: two gathered parameter slices, in the backward also two fp32 gradient staging slices, the
  // db1 band partials and the slice activations - all proportional to the slice width, stated per ffn column
  const uint64_t per_col = 2 * (2 * h + 1) * e + (pass == OSDP_BWD ? 2 * (2 * h + 1) * 4 + ((T + kBandRows - 1) / kBandRows) * 4 : 0) +
                           (pass == OSDP_FWD ? 1 : 2) * T * e;
  c.extra_transient = per_col * f;
  // fixed: the fp32 accumulator of Y / dX (charged at k = 1 too, where the call needs none), the b2 / db2 pieces, and
  // what makes the estimate an UPPER bound of osdp_zdp_ffn_split_mlp_workspace_bytes for every (N, k): a slice is whole
  // groups of N x 16 bytes of columns, so the widest slice has up to one group more than f / k, and each of the at
  // most 24 parts of the workspace is padded to 256 B (the planner's M_limit check must not pass a plan that does not fit)
  const uint64_t group_cols = (uint64_t)g.N * (uint64_t)g.unit;
  c.extra_fixed = align_up((size_t)T * h * 4, 256) + (pass == OSDP_BWD ? db2_scratch_bytes(h) + h * 4 : h * e) +
                  group_cols * per_col + 24 * 256;
  *out = c;
  return OSDP_OK;
}

int osdp_zdp_ffn_split_mlp_forward(const osdp_zdp_desc* desc, const void* param_shard, const void* X, void* Y,
                                   void* workspace, size_t workspace_bytes_given, const osdp_comm* comm,
                                   void* compute_stream, void* comm_stream) {
  g_launches = 0;
  ZdpGeom g;
  OSDP_TRY(zdp_check_call(desc, &g, OSDP_FWD, workspace, workspace_bytes_given, comm));
  if (!param_shard || !X || !Y) return OSDP_ERR_NULL;
  if (misaligned(param_shard, 16) || misaligned(X, 16) || misaligned(Y, 16)) return OSDP_ERR_ALIGN;
  cudaStream_t cs = (cudaStream_t)compute_stream, ms = (cudaStream_t)comm_stream;
  const bool two = ms != cs;
  const ZdpWs w = zdp_ws(g, OSDP_FWD);
  const ZdpBuf gb = zdp_buf(g, g.e);
  char* ws = (char*)workspace;
  const char* shard = (const char*)param_shard;
  ZdpEvents* ev = nullptr;
  OSDP_TRY(zdp_events(&ev));
  if (two) {   // the collectives may read what earlier work on the compute stream produced (an optimizer step, say)
    OSDP_CUDA_TRY(cudaEventRecord(ev->entry, cs));
    OSDP_CUDA_TRY(cudaStreamWaitEvent(ms, ev->entry, 0));
  }
  ZdpJoin join{cs, ms, ev->tail, two};
  std::vector<osdp_zdp_step> steps;
  zdp_steps(g, OSDP_FWD, &steps);
  int used[2] = {0, 0};   // how many computes have used each gathered buffer so far
  for (const osdp_zdp_step& stp : steps) {
    osdp_zdp_slice sl;
    zdp_slice(g, stp.slice, &sl);
    const int b = stp.buffer;
    if (stp.op == OSDP_ZDP_GATHER) {
      if (stp.slice == g.k) {   // b2, once
        OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.b1_off * g.e, ws + w.b2g, (size_t)sl.b1_elems * g.e, ms));
        if (two) OSDP_CUDA_TRY(cudaEventRecord(ev->b2, ms));
        continue;
      }
      if (two && used[b] > 0) OSDP_CUDA_TRY(cudaStreamWaitEvent(ms, ev->freed[b], 0));   // the slice that used this buffer is done
      char* G = ws + w.gbuf[b];
      OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.w1_off * g.e, G + gb.w1, (size_t)sl.w1_elems * g.e, ms));
      OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.b1_off * g.e, G + gb.b1, (size_t)sl.b1_elems * g.e, ms));
      OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.w2_off * g.e, G + gb.w2, (size_t)sl.w2_elems * g.e, ms));
      if (two) OSDP_CUDA_TRY(cudaEventRecord(ev->gathered[b], ms));
    } else if (stp.op == OSDP_ZDP_COMPUTE) {
      if (two) {
        OSDP_CUDA_TRY(cudaStreamWaitEvent(cs, ev->gathered[b], 0));
        if (stp.slice == 0) OSDP_CUDA_TRY(cudaStreamWaitEvent(cs, ev->b2, 0));
      }
      const char* G = ws + w.gbuf[b];
      const int fs = (int)(sl.hi - sl.lo);
      const FfnSliceW sw = {G + gb.w1, fs, G + gb.b1, G + gb.w2};
      OSDP_TRY(ffn_slice_forward(g.dt, g.T, g.h, fs, X, sw, ws + w.b2g, Y, ws + w.hs, (float*)(ws + w.acc), g.k == 1,
                                 stp.slice == 0, cs));
      if (two) OSDP_CUDA_TRY(cudaEventRecord(ev->freed[b], cs));
      ++used[b];
    }
  }
  if (g.k > 1) {   // Y = storage(Yacc + b2)
    trace_set_step(10);
    sm100::DeviceInfo dev;
    OSDP_TRY(sm100::current_device(&dev));
    OSDP_TRY(launch_acc_to_out(g.dt, (const float*)(ws + w.acc), ws + w.b2g, Y, g.T, (int)g.h, dev.sms, cs));
  }
  join.armed = false;
  return OSDP_OK;   // every gather was waited for by a compute step: comm_stream has joined compute_stream
}

int osdp_zdp_ffn_split_mlp_backward(const osdp_zdp_desc* desc, const void* param_shard, const void* X, const void* dY,
                                    void* dX, float* grad_shard, void* workspace, size_t workspace_bytes_given,
                                    const osdp_comm* comm, void* compute_stream, void* comm_stream) {
  g_launches = 0;
  ZdpGeom g;
  OSDP_TRY(zdp_check_call(desc, &g, OSDP_BWD, workspace, workspace_bytes_given, comm));
  if (!param_shard || !X || !dY || !dX || !grad_shard) return OSDP_ERR_NULL;
  if (misaligned(param_shard, 16) || misaligned(X, 16) || misaligned(dY, 16) || misaligned(dX, 16) || misaligned(grad_shard, 16))
    return OSDP_ERR_ALIGN;
  cudaStream_t cs = (cudaStream_t)compute_stream, ms = (cudaStream_t)comm_stream;
  const bool two = ms != cs;
  const ZdpWs w = zdp_ws(g, OSDP_BWD);
  const ZdpBuf gb = zdp_buf(g, g.e), rb = zdp_buf(g, 4);
  char* ws = (char*)workspace;
  const char* shard = (const char*)param_shard;
  ZdpEvents* ev = nullptr;
  OSDP_TRY(zdp_events(&ev));
  if (two) {
    OSDP_CUDA_TRY(cudaEventRecord(ev->entry, cs));
    OSDP_CUDA_TRY(cudaStreamWaitEvent(ms, ev->entry, 0));
  }
  ZdpJoin join{cs, ms, ev->tail, two};
  std::vector<osdp_zdp_step> steps;
  zdp_steps(g, OSDP_BWD, &steps);
  int used[2] = {0, 0}, scattered[2] = {0, 0};
  for (const osdp_zdp_step& stp : steps) {
    osdp_zdp_slice sl;
    zdp_slice(g, stp.slice, &sl);
    const int b = stp.buffer;
    if (stp.op == OSDP_ZDP_GATHER) {
      if (two && used[b] > 0) OSDP_CUDA_TRY(cudaStreamWaitEvent(ms, ev->freed[b], 0));
      char* G = ws + w.gbuf[b];
      OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.w1_off * g.e, G + gb.w1, (size_t)sl.w1_elems * g.e, ms));
      OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.b1_off * g.e, G + gb.b1, (size_t)sl.b1_elems * g.e, ms));
      OSDP_TRY(zdp_all_gather(comm, shard + (size_t)sl.w2_off * g.e, G + gb.w2, (size_t)sl.w2_elems * g.e, ms));
      if (two) OSDP_CUDA_TRY(cudaEventRecord(ev->gathered[b], ms));
    } else if (stp.op == OSDP_ZDP_COMPUTE) {
      if (two) {
        OSDP_CUDA_TRY(cudaStreamWaitEvent(cs, ev->gathered[b], 0));
        if (scattered[b] > 0) OSDP_CUDA_TRY(cudaStreamWaitEvent(cs, ev->scattered[b], 0));   // staging buffer b is free again
      }
      const char* G = ws + w.gbuf[b];
      char* R = ws + w.rbuf[b];
      const int fs = (int)(sl.hi - sl.lo);
      const FfnSliceW sw = {G + gb.w1, fs, G + gb.b1, G + gb.w2};
      const FfnSliceG sg = {(float*)(R + rb.w1), fs, (float*)(R + rb.b1), (float*)(R + rb.w2)};
      OSDP_TRY(ffn_slice_backward(g.dt, g.T, g.h, fs, X, dY, sw, sg, ws + w.zs, ws + w.hs, dX, (float*)(ws + w.acc),
                                  (float*)(ws + w.scratch1), (float*)(ws + w.scratch2),
                                  stp.slice == 0 ? (float*)(ws + w.db2s) : nullptr, g.k == 1, stp.slice == 0, cs));
      if (two) {
        OSDP_CUDA_TRY(cudaEventRecord(ev->freed[b], cs));
        OSDP_CUDA_TRY(cudaEventRecord(ev->grads[b], cs));
      }
      ++used[b];
    } else {   // reduce-scatter
      if (stp.slice == g.k) {   // db2: staged by the first slice's column sums
        if (two) OSDP_CUDA_TRY(cudaStreamWaitEvent(ms, ev->grads[0], 0));
        OSDP_TRY(zdp_reduce_scatter(comm, (const float*)(ws + w.db2s), grad_shard + sl.b1_off, (size_t)sl.b1_elems, ms));
        continue;
      }
      if (two) OSDP_CUDA_TRY(cudaStreamWaitEvent(ms, ev->grads[b], 0));
      const char* R = ws + w.rbuf[b];
      OSDP_TRY(zdp_reduce_scatter(comm, (const float*)(R + rb.w1), grad_shard + sl.w1_off, (size_t)sl.w1_elems, ms));
      OSDP_TRY(zdp_reduce_scatter(comm, (const float*)(R + rb.b1), grad_shard + sl.b1_off, (size_t)sl.b1_elems, ms));
      OSDP_TRY(zdp_reduce_scatter(comm, (const float*)(R + rb.w2), grad_shard + sl.w2_off, (size_t)sl.w2_elems, ms));
      if (two) OSDP_CUDA_TRY(cudaEventRecord(ev->scattered[b], ms));
      ++scattered[b];
    }
  }
  if (g.k > 1) {   // dX = storage(dXacc)
    trace_set_step(10);
    sm100::DeviceInfo dev;
    OSDP_TRY(sm100::current_device(&dev));
    OSDP_TRY(launch_acc_to_out(g.dt, (const float*)(ws + w.acc), nullptr, dX, g.T, (int)g.h, dev.sms, cs));
  }
  if (two) {   // join: the gradient shard is complete in compute-stream order
    OSDP_CUDA_TRY(cudaEventRecord(ev->tail, ms));
    OSDP_CUDA_TRY(cudaStreamWaitEvent(cs, ev->tail, 0));
  }
  join.armed = false;
  return OSDP_OK;
}

}  // extern "C"
