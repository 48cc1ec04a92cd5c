// osdp_api.cu — the C ABI of osdp-b200 (include/osdp.h) and the host-side slice scheduler (step A0).
//
// The scheduler follows PAPER.md:165: slices are processed one after another in order on the caller's
// stream, the per-slice buffers in the caller's workspace are reused serially, and results that span slices
// (dW1, dW2, db1, db2) are summed: "=" on slice 0, "+=" afterwards, in fixed slice order.
#include <mutex>
#include <string>
#include <vector>

#include "cast.cuh"
#include "common.cuh"
#include "gemm_f32.cuh"
#include "gemm_sm100.cuh"
#include "reduce.cuh"
#include "slice_sm100.cuh"

namespace osdp {

namespace {
thread_local std::string g_last_error;
thread_local int64_t g_launches = 0;
}  // namespace

void note_cuda_error(cudaError_t e, const char* where) {
  g_last_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e) + " at " + where;
}
void count_launch() { ++g_launches; }

namespace {
struct TraceState {
  bool on = false;
  int step = 0;
  std::vector<cudaEvent_t> pool;    // 2 events per recorded launch, reused across reads
  std::vector<int32_t> steps;       // step id per recorded launch
  bool failed = false;
  cudaEvent_t get(size_t i) {
    while (pool.size() <= i) {
      cudaEvent_t e = nullptr;
      if (cudaEventCreate(&e) != cudaSuccess) { failed = true; return nullptr; }
      pool.push_back(e);
    }
    return pool[i];
  }
};
thread_local TraceState g_trace;
}  // namespace

void trace_set_step(int step_id) { g_trace.step = step_id; }
void trace_before(cudaStream_t st) {
  if (!g_trace.on) return;
  cudaEvent_t e = g_trace.get(2 * g_trace.steps.size());
  if (e && cudaEventRecord(e, st) != cudaSuccess) g_trace.failed = true;
}
void trace_after(cudaStream_t st) {
  if (!g_trace.on) return;
  cudaEvent_t e = g_trace.get(2 * g_trace.steps.size() + 1);
  if (e && cudaEventRecord(e, st) != cudaSuccess) g_trace.failed = true;
  g_trace.steps.push_back(g_trace.step);
}

namespace sm100 {
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  });
  if (!fn) note_cuda_error(cudaErrorNotSupported, "cudaGetDriverEntryPoint(cuTensorMapEncodeTiled)");
  return fn;
}
std::mutex& launch_setup_mutex() {
  static std::mutex m;
  return m;
}
// Ordinal and SM count of the device current to the calling thread (cached per ordinal after the first query).
int current_device(DeviceInfo* out) {
  static std::atomic<int> sms_of[kMaxDevices];
  int dev = 0;
  OSDP_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return OSDP_ERR_ARG;
  int n = sms_of[dev].load(std::memory_order_acquire);
  if (n == 0) {
    OSDP_CUDA_TRY(cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
    if (n <= 0) n = 1;
    sms_of[dev].store(n, std::memory_order_release);
  }
  out->ordinal = dev;
  out->sms = n;
  return OSDP_OK;
}
}  // namespace sm100

namespace {

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline size_t elem_size(int dtype) { return dtype == OSDP_BF16 ? 2 : 4; }

int check_desc(const osdp_mlp_desc* d) {
  if (!d) return OSDP_ERR_NULL;
  if (d->dtype != OSDP_F32 && d->dtype != OSDP_BF16) return OSDP_ERR_DTYPE;
  const int64_t mult = 16 / (int64_t)elem_size(d->dtype);
  if (d->tokens < 1 || d->hidden < 1 || d->ffn < 1) return OSDP_ERR_SHAPE;
  if (d->hidden % mult || d->ffn % mult) return OSDP_ERR_SHAPE;
  if (d->tokens > (1ll << 30) || d->hidden > (1ll << 30) || d->ffn > (1ll << 30)) return OSDP_ERR_SHAPE;
  if (d->k < 1 || (int64_t)d->k > d->tokens) return OSDP_ERR_K;
  return OSDP_OK;
}

inline size_t slice_buf_bytes(const osdp_mlp_desc* d) {
  const int64_t ts = (d->tokens + d->k - 1) / d->k;
  return align_up((size_t)ts * (size_t)d->ffn * elem_size(d->dtype), 256);
}
// Column-sum scratch: db1 = one fp32 partial row per 32-row band of the slice's dZ_s (written by
// the A4 epilogue), db2 = kReduceRowChunks partial rows of dY.
inline size_t db1_scratch_bytes(int64_t slice_rows, int64_t cols) {
  return align_up((size_t)((slice_rows + kBandRows - 1) / kBandRows) * (size_t)cols * 4, 256);
}
inline size_t db2_scratch_bytes(int64_t h) { return align_up((size_t)kReduceRowChunks * (size_t)h * 4, 256); }
// Tile counter and per-tile flags of the one-kernel-per-slice path (slice_sm100.cuh): kSliceFlags0 + 2 words per 256 x 256
// tile of a slice's [rows x cols] GEMM, for each of the k slices.  They live at the END of the caller's workspace, which
// is exclusive to one call in flight by contract, so any number of calls on any number of streams, and captured graphs
// replayed side by side, have their own words (round 2 kept 16 static blocks handed out round-robin).  Pure host
// arithmetic, independent of the tuning knobs: the bytes are reserved whenever the path COULD be chosen (bf16, the
// call's words fit kSliceSyncWords = 128 KiB), else 0.
inline int64_t tiles_256(int64_t m, int64_t n) { return ((m + 255) / 256) * ((n + 255) / 256); }
inline int64_t slice_sync_words(int dtype, int64_t rows, int64_t cols, int64_t k) {
  if (dtype != OSDP_BF16) return 0;
  const int64_t per_slice = sm100::kSliceFlags0 + 2 * tiles_256(rows, cols);
  return per_slice * k > sm100::kSliceSyncWords ? 0 : per_slice * k;
}
inline size_t slice_sync_bytes(const osdp_mlp_desc* d) {
  return align_up((size_t)slice_sync_words(d->dtype, (d->tokens + d->k - 1) / d->k, d->ffn, d->k) * 4, 256);
}
inline size_t workspace_tensor_bytes(const osdp_mlp_desc* d, int pass) {   // everything but the sync words
  if (pass == OSDP_FWD) return slice_buf_bytes(d);
  const int64_t ts = (d->tokens + d->k - 1) / d->k;
  return 2 * slice_buf_bytes(d) + db1_scratch_bytes(ts, d->ffn) + db2_scratch_bytes(d->hidden);
}
size_t workspace_bytes(const osdp_mlp_desc* d, int pass) { return workspace_tensor_bytes(d, pass) + slice_sync_bytes(d); }

// ---- ffn-axis split: slice s owns ffn columns [ffn_lo(s), ffn_lo(s + 1)), whole 16-byte units
inline int64_t ffn_unit(const osdp_mlp_desc* d) { return 16 / (int64_t)elem_size(d->dtype); }
inline int64_t ffn_lo(const osdp_mlp_desc* d, int64_t s) {
  const int64_t u = ffn_unit(d), units = d->ffn / u;
  return (s * units / d->k) * u;
}
inline int64_t ffn_slice_max(const osdp_mlp_desc* d) {
  const int64_t u = ffn_unit(d), units = d->ffn / u;
  return ((units + d->k - 1) / d->k) * u;
}
int check_desc_ffn(const osdp_mlp_desc* d) {
  const int rc = check_desc(d);
  if (rc == OSDP_ERR_K) {   // check_desc bounds k by tokens; here the bound is the number of 16-byte ffn units
    if (d->k < 1) return OSDP_ERR_K;
  } else if (rc != OSDP_OK) {
    return rc;
  }
  if ((int64_t)d->k > d->ffn / ffn_unit(d)) return OSDP_ERR_K;
  return OSDP_OK;
}
inline size_t ffn_slice_buf_bytes(const osdp_mlp_desc* d) {
  return align_up((size_t)d->tokens * (size_t)ffn_slice_max(d) * elem_size(d->dtype), 256);
}
inline size_t ffn_acc_bytes(const osdp_mlp_desc* d) {   // fp32 accumulator of Y / dX across slices; not needed at k = 1
  return d->k == 1 ? 0 : align_up((size_t)d->tokens * (size_t)d->hidden * 4, 256);
}
inline size_t ffn_slice_sync_bytes(const osdp_mlp_desc* d) {   // slice-kernel words of the call (see slice_sync_words)
  return align_up((size_t)slice_sync_words(d->dtype, d->tokens, ffn_slice_max(d), d->k) * 4, 256);
}
inline size_t ffn_workspace_tensor_bytes(const osdp_mlp_desc* d, int pass) {   // everything but the sync words
  if (pass == OSDP_FWD) return ffn_slice_buf_bytes(d) + ffn_acc_bytes(d);
  return 2 * ffn_slice_buf_bytes(d) + ffn_acc_bytes(d) + db1_scratch_bytes(d->tokens, ffn_slice_max(d)) +
         db2_scratch_bytes(d->hidden);
}
size_t ffn_workspace_bytes(const osdp_mlp_desc* d, int pass) {
  return ffn_workspace_tensor_bytes(d, pass) + ffn_slice_sync_bytes(d);
}

inline bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; }

int check_arch() {
  int dev = 0, major = 0;
  OSDP_CUDA_TRY(cudaGetDevice(&dev));
  OSDP_CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  return major == 10 ? OSDP_OK : OSDP_ERR_ARCH;
}

// One GEMM of the path, dispatched on storage dtype.  For bf16 the operands go through TMA/tcgen05; for fp32
// through the FFMA kernel with explicit strides.
template <int A_MAJOR, int B_MAJOR, int EPI>
int gemm(int dtype, const void* A, int64_t lda, const void* B, int64_t ldb, const GemmShape& s, const EpiParams& ep,
         cudaStream_t st) {
  if (dtype == OSDP_BF16) return sm100::launch_gemm_bf16<A_MAJOR, B_MAJOR, EPI>(A, lda, B, ldb, s, ep, st);
  StridedOperands op;
  op.A = (const float*)A;
  op.a_sm = A_MAJOR == MAJOR_K ? lda : 1;
  op.a_sk = A_MAJOR == MAJOR_K ? 1 : lda;
  op.B = (const float*)B;
  op.b_sk = B_MAJOR == MAJOR_K ? 1 : ldb;
  op.b_sn = B_MAJOR == MAJOR_K ? ldb : 1;
  return launch_gemm_f32<EPI>(op, s, ep, st);
}

// out (+)= colsum(src [rows x cols]) in kReduceRowChunks equal row chunks (db2, and the Linear operator's db)
int colsum_rows(int dtype, const void* src, int cols, float* out, int rows, float* scratch, int beta, cudaStream_t st) {
  if (dtype == OSDP_BF16) return launch_colsum<__nv_bfloat16>((const __nv_bfloat16*)src, cols, cols, out, rows, 0, scratch, beta, st);
  return launch_colsum<float>((const float*)src, cols, cols, out, rows, 0, scratch, beta, st);
}
// db1 (+)= colsum(dZ_s [rows x cols]) from the 32-row band partials.  bf16: the A4 epilogue has already written them to
// `scratch` (one launch here); fp32: the FFMA GEMM has no such epilogue, a kernel makes the same partials first.
int db1_from_bands(int dtype, const void* dZs, int cols, float* out, int rows, float* scratch, int beta, cudaStream_t st) {
  if (dtype == OSDP_BF16)
    return launch_colsum_final(scratch, cols, (rows + kBandRows - 1) / kBandRows, out, 0, 0, nullptr, beta, st);
  return launch_colsum<float>((const float*)dZs, cols, cols, out, rows, kBandRows, scratch, beta, st);
}

#define OSDP_TRY(expr)            \
  do {                            \
    int _rc = (expr);             \
    if (_rc != OSDP_OK) return _rc; \
  } while (0)

// ---- helper streams: independent launches of one slice side by side ------------------------------------------
// Once dZ_s exists, dW2 (+)= H_s^T dY_s, dW1 (+)= X_s^T dZ_s, dX_s = dZ_s W1^T and the two column sums are independent
// (SURVEY.md section 7 "co-scheduling").  On small slices each of them fills a fraction of the machine for a few
// microseconds, most of it fixed cost, so they are enqueued side by side: the caller's stream forks into helper
// streams (event record + wait) and joins them again before the next slice reuses the slice buffers.  Seen from the
// caller the call still only adds work to `stream` in order (and stays CUDA-graph capturable: fork/join through events
// becomes parallel branches).  Streams and events belong to the calling host thread and the current device, are
// created on first use and never shared between host threads.
constexpr int kForkBranches = 3;
struct ForkCtx {
  cudaStream_t side[kForkBranches] = {};
  cudaEvent_t fork_ev = nullptr;
  cudaEvent_t join_ev[kForkBranches] = {};
  bool ready = false;
};
int fork_ctx(ForkCtx** out) {
  static thread_local ForkCtx ctx[sm100::kMaxDevices];
  sm100::DeviceInfo dev;
  const int rc = sm100::current_device(&dev);
  if (rc != OSDP_OK) return rc;
  ForkCtx& c = ctx[dev.ordinal];
  if (!c.ready) {
    for (int i = 0; i < kForkBranches; ++i) {
      OSDP_CUDA_TRY(cudaStreamCreateWithFlags(&c.side[i], cudaStreamNonBlocking));
      OSDP_CUDA_TRY(cudaEventCreateWithFlags(&c.join_ev[i], cudaEventDisableTiming));
    }
    OSDP_CUDA_TRY(cudaEventCreateWithFlags(&c.fork_ev, cudaEventDisableTiming));
    c.ready = true;
  }
  *out = &c;
  return OSDP_OK;
}
// Everything enqueued on `st` so far happens before whatever is enqueued on the side streams from now on.
int fork_from(ForkCtx* c, cudaStream_t st) {
  OSDP_CUDA_TRY(cudaEventRecord(c->fork_ev, st));
  for (int i = 0; i < kForkBranches; ++i) OSDP_CUDA_TRY(cudaStreamWaitEvent(c->side[i], c->fork_ev, 0));
  return OSDP_OK;
}
// Everything enqueued on the side streams so far happens before whatever is enqueued on `st` from now on.
int join_into(ForkCtx* c, cudaStream_t st) {
  for (int i = 0; i < kForkBranches; ++i) {
    OSDP_CUDA_TRY(cudaEventRecord(c->join_ev[i], c->side[i]));
    OSDP_CUDA_TRY(cudaStreamWaitEvent(st, c->join_ev[i], 0));
  }
  return OSDP_OK;
}


// ---- one persistent kernel per slice (slice_sm100.cuh) ----------------------------------------------------------
// Taken for bf16 when the slice is small in TOKENS: its [T_s x ffn] GEMMs (A1, A3, A4) have at most
// OSDP_TUNE_SLICE_KERNEL_MAX_TILES tiles of 256 x 256, i.e. about one wave, which is where a launch per GEMM is mostly
// fill and drain (measured: at 128 tiles C2 k = 4 +7 %, C5 layer k = 16 +1 %, C4 k = 32 +6 %; at 64 tiles +10-27 %; at 256
// tiles the launch-per-GEMM path with its 512 x 256 tiles wins; the dW GEMMs' tile count does not matter), and the call's
// flags fit the per-call block.  A2 / A7 (long contraction, few
// output tiles) take 128-column tiles when that still fits one wave of CTA pairs, so they spread over twice as many SMs.
struct SlicePlan {
  bool use = false;
  int bn_narrow = 256;   // tile width of A2 / A7
  int words_per_slice = 0, words = 0;
};
int slice_plan(const osdp_mlp_desc* d, int pass, SlicePlan* out) {
  *out = SlicePlan{};
  const int64_t max_tiles = sm100::tuning().slice_kernel_max_tiles.load();
  if (d->dtype != OSDP_BF16 || max_tiles <= 0) return OSDP_OK;
  sm100::DeviceInfo dev;
  OSDP_TRY(sm100::current_device(&dev));
  const int64_t ts = (d->tokens + d->k - 1) / d->k;
  (void)pass;
  const int64_t t_tf = tiles_256(ts, d->ffn), t_th = tiles_256(ts, d->hidden);
  if (t_tf > max_tiles) return OSDP_OK;
  out->bn_narrow = 2 * t_th <= dev.sms / 2 ? 128 : 256;
  const int64_t per_slice = sm100::kSliceFlags0 + 2 * t_tf;   // flags of the publishing phase (A1 / fused A3 + A4) only
  if (per_slice * d->k > sm100::kSliceSyncWords) return OSDP_OK;
  out->use = true;
  out->words_per_slice = (int)per_slice;
  out->words = (int)(per_slice * d->k);
  return OSDP_OK;
}

// The call's tile counter / flag words: `bytes_before` into the caller's workspace (exclusive to this call), zeroed on
// the call's stream before its first launch - the workspace holds whatever the caller left there.
int slice_sync_setup(const SlicePlan& sp, void* workspace, size_t bytes_before, int launches, cudaStream_t st,
                     unsigned int** sync, unsigned int* epoch0) {
  *sync = reinterpret_cast<unsigned int*>((char*)workspace + bytes_before);
  OSDP_CUDA_TRY(cudaMemsetAsync(*sync, 0, (size_t)sp.words * 4, st));
  *epoch0 = sm100::slice_epochs(launches);
  return OSDP_OK;
}

// The same for the ffn-axis split: a slice is ffn columns [lo, hi), its [T x fs] GEMMs (A1 / A3 + A4) decide.  Its own
// knob, off by default: measured C3 k = 64 +35 %, C5 layer shape k = 16 / 32 +31 / +37 %, but C2 k = 4 / 8 -17 / -15 % and C4
// k = 32 -10 % (the slice's dW GEMMs are few tiles with K = T, and they then run beside the dX tiles instead of alone).
int ffn_slice_plan(const osdp_mlp_desc* d, int64_t fs_max, SlicePlan* out) {
  *out = SlicePlan{};
  const int64_t max_tiles = sm100::tuning().slice_kernel_ffn_max_tiles.load();
  if (d->dtype != OSDP_BF16 || max_tiles <= 0) return OSDP_OK;
  sm100::DeviceInfo dev;
  OSDP_TRY(sm100::current_device(&dev));
  const int64_t t_tf = tiles_256(d->tokens, fs_max), t_th = tiles_256(d->tokens, d->hidden);
  if (t_tf > max_tiles) return OSDP_OK;
  out->bn_narrow = 2 * t_th <= dev.sms / 2 ? 128 : 256;
  const int64_t per_slice = sm100::kSliceFlags0 + 2 * t_tf;
  if (per_slice * d->k > sm100::kSliceSyncWords) return OSDP_OK;
  out->use = true;
  out->words_per_slice = (int)per_slice;
  out->words = (int)(per_slice * d->k);
  return OSDP_OK;
}
// One-kernel-per-slice launch context of an ffn-split call (sync == nullptr: one launch per GEMM)
struct FfnSliceKernel {
  unsigned int* sync = nullptr;   // this slice's flags
  unsigned int epoch = 0;
  int bn_narrow = 256;
};

// ---- one slice of the ffn-axis split.  The slice's weights are given by pointer + leading
// dimension, so the same code serves weights sliced in place (W1 + lo, ld = f) and gathered slice buffers (ZDP, ld = fs).
struct FfnSliceW {
  const void* W1s;   // W1[:, lo:hi]   [h x fs], leading dimension ldw1
  int64_t ldw1;
  const void* b1s;   // b1[lo:hi]
  const void* W2s;   // W2[lo:hi, :]   [fs x h], leading dimension h
};
struct FfnSliceG {
  float* dW1s;       // dW1[:, lo:hi]  [h x fs], leading dimension ldg1
  int64_t ldg1;
  float* db1s;       // db1[lo:hi]
  float* dW2s;       // dW2[lo:hi, :]  [fs x h], leading dimension h
};
// H_s = gelu(X W1s + b1s); Y (+)= H_s W2s.  single = the operator has one slice (Y written directly, + b2).
int ffn_slice_forward(int dt, int64_t T, int64_t h, int fs, const void* X, const FfnSliceW& w, const void* b2, void* Y,
                      void* Hs, float* Yacc, bool single, bool first, cudaStream_t st, const FfnSliceKernel* sk = nullptr) {
  if (sk && sk->sync) {   // A1 -> A2 in one launch (slice_sm100.cuh); Y (+)= goes through the fp32 reduce-add epilogue
    trace_set_step(21);
    sm100::SliceGemm g[2] = {};
    g[0] = {X, h, w.W1s, w.ldw1, MAJOR_K, MAJOR_MN, EPI_BIAS_GELU, GemmShape{(int)T, fs, (int)h},
            EpiParams{w.b1s, Hs, nullptr, nullptr, fs, 0}, sm100::DEP_NONE, 0, 256, 1, 0};
    if (single)
      g[1] = {Hs, fs, w.W2s, h, MAJOR_K, MAJOR_MN, EPI_BIAS, GemmShape{(int)T, (int)h, fs},
              EpiParams{b2, Y, nullptr, nullptr, h, 0}, sm100::DEP_ROW, 0, sk->bn_narrow, 0, 0};
    else
      g[1] = {Hs, fs, w.W2s, h, MAJOR_K, MAJOR_MN, EPI_ACCUM_F32, GemmShape{(int)T, (int)h, fs},
              EpiParams{nullptr, Yacc, nullptr, nullptr, h, first ? 0 : 1}, sm100::DEP_ROW, 0, 256, 0, 0};
    return sm100::launch_mlp_slice(g, 2, sk->sync, sk->epoch, nullptr, false, st);
  }
  trace_set_step(1);
  EpiParams e1 = {w.b1s, Hs, nullptr, nullptr, fs, 0};
  OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS_GELU>(dt, X, h, w.W1s, w.ldw1, GemmShape{(int)T, fs, (int)h}, e1, st)));
  // the paper's split: contraction axis sliced, partial products summed
  trace_set_step(2);
  if (single) {
    EpiParams e2 = {b2, Y, nullptr, nullptr, h, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS>(dt, Hs, fs, w.W2s, h, GemmShape{(int)T, (int)h, fs}, e2, st)));
  } else {
    EpiParams e2 = {nullptr, Yacc, nullptr, nullptr, h, first ? 0 : 1};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_ACCUM_F32>(dt, Hs, fs, w.W2s, h, GemmShape{(int)T, (int)h, fs}, e2, st)));
  }
  return OSDP_OK;
}
// Z_s, H_s recomputed; dZ_s; the slice's own parts of dW2, dW1, db1 (written once); dX (+)= dZ_s W1s^T.
// db2 != nullptr: also db2 = colsum(dY) (once per call, with the first slice).
int ffn_slice_backward(int dt, int64_t T, int64_t h, int fs, const void* X, const void* dY, const FfnSliceW& w,
                       const FfnSliceG& g, void* Zs, void* Hs, void* dX, float* dXacc, float* scratch1, float* scratch2,
                       float* db2, bool single, bool first, cudaStream_t st, const FfnSliceKernel* sk = nullptr) {
  if (sk && sk->sync) {   // (A3 + A4) -> A7 | A5 | A6 (+ db1) in one launch; the slice's dW / db1 parts are written once
    if (db2) {
      trace_set_step(8);
      OSDP_TRY(colsum_rows(dt, dY, (int)h, db2, (int)T, scratch2, 0, st));
    }
    trace_set_step(22);
    sm100::SliceGemm ph[4] = {};
    ph[0] = {X, h, w.W1s, w.ldw1, MAJOR_K, MAJOR_MN, sm100::kEpiFusedA34, GemmShape{(int)T, fs, (int)h},
            EpiParams{w.b1s, Zs, Hs, nullptr, fs, 0, scratch1, fs}, sm100::DEP_NONE, 0, 256, 1, 0,
            dY, h, w.W2s, h, MAJOR_K, MAJOR_K, (int)h};
    // list order = claim order: everything after the fused tiles is ready at the same time, so the phase with the
    // longest contraction (fewest, longest tiles) goes first: here usually the dW GEMMs (K = T), dX (K = fs) fills in
    const int ix = T > fs ? 3 : 1, i5 = T > fs ? 1 : 2, i6 = T > fs ? 2 : 3;
    if (single)
      ph[ix] = {Zs, fs, w.W1s, w.ldw1, MAJOR_K, MAJOR_K, EPI_PLAIN, GemmShape{(int)T, (int)h, fs},
                EpiParams{nullptr, dX, nullptr, nullptr, h, 0}, sm100::DEP_ROW, 0, sk->bn_narrow, 0, 0};
    else
      ph[ix] = {Zs, fs, w.W1s, w.ldw1, MAJOR_K, MAJOR_K, EPI_ACCUM_F32, GemmShape{(int)T, (int)h, fs},
                EpiParams{nullptr, dXacc, nullptr, nullptr, h, first ? 0 : 1}, sm100::DEP_ROW, 0, 256, 0, 0};
    ph[i5] = {Hs, fs, dY, h, MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32, GemmShape{fs, (int)h, (int)T},
              EpiParams{nullptr, g.dW2s, nullptr, nullptr, h, 0}, sm100::DEP_COL_AS_M, 0, 256, 0, 0};
    ph[i6] = {X, h, Zs, fs, MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32, GemmShape{(int)h, fs, (int)T},
              EpiParams{nullptr, g.dW1s, nullptr, nullptr, g.ldg1, 0}, sm100::DEP_COL_AS_N, 0, 256, 0, 1};
    const sm100::SliceDb1 dj = {scratch1, fs, g.db1s, (int)((T + kBandRows - 1) / kBandRows), 0};
    return sm100::launch_mlp_slice(ph, 4, sk->sync, sk->epoch, &dj, false, st);
  }
  // dW2, dW1, dX (+)= and the column sums only need dZ_s: side by side on small slices (helper streams above)
  const int64_t fork_max = sm100::tuning().fork_max_tiles.load();
  const bool fork = fork_max > 0 && tiles_256(fs, h) <= fork_max && tiles_256(T, h) <= fork_max;
  ForkCtx* fc = nullptr;
  if (fork) OSDP_TRY(fork_ctx(&fc));
  trace_set_step(3);
  EpiParams e3 = {w.b1s, Zs, Hs, nullptr, fs, 0};
  OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS_GELU_DUAL>(dt, X, h, w.W1s, w.ldw1, GemmShape{(int)T, fs, (int)h}, e3, st)));
  trace_set_step(4);   // the epilogue also leaves the 32-row band sums of dZ_s in scratch1 (db1)
  EpiParams e4 = {nullptr, Zs, nullptr, Zs, fs, 0, scratch1, fs};
  OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_DGELU>(dt, dY, h, w.W2s, h, GemmShape{(int)T, fs, (int)h}, e4, st)));
  if (fork) OSDP_TRY(fork_from(fc, st));
  cudaStream_t s1 = fork ? fc->side[0] : st, s2 = fork ? fc->side[1] : st, s3 = fork ? fc->side[2] : st;
  trace_set_step(5);   // rows of dW2 belong to exactly one slice: written once, no accumulation
  EpiParams e5 = {nullptr, g.dW2s, nullptr, nullptr, h, 0};
  OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, Hs, fs, dY, h, GemmShape{fs, (int)h, (int)T}, e5, st)));
  trace_set_step(8);
  OSDP_TRY(db1_from_bands(dt, Zs, fs, g.db1s, (int)T, scratch1, 0, s3));
  if (db2) OSDP_TRY(colsum_rows(dt, dY, (int)h, db2, (int)T, scratch2, 0, s3));
  trace_set_step(6);   // columns of dW1 belong to exactly one slice
  EpiParams e6 = {nullptr, g.dW1s, nullptr, nullptr, g.ldg1, 0};
  OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, X, h, Zs, fs, GemmShape{(int)h, fs, (int)T}, e6, s1)));
  trace_set_step(7);   // the only result that spans slices
  if (single) {
    EpiParams e7 = {nullptr, dX, nullptr, nullptr, h, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_PLAIN>(dt, Zs, fs, w.W1s, w.ldw1, GemmShape{(int)T, (int)h, fs}, e7, s2)));
  } else {
    EpiParams e7 = {nullptr, dXacc, nullptr, nullptr, h, first ? 0 : 1};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_ACCUM_F32>(dt, Zs, fs, w.W1s, w.ldw1, GemmShape{(int)T, (int)h, fs}, e7, s2)));
  }
  if (fork) OSDP_TRY(join_into(fc, st));   // the next slice overwrites Z_s / H_s
  return OSDP_OK;
}

}  // namespace
}  // namespace osdp

using namespace osdp;

extern "C" {

const char* osdp_status_string(int status) {
  switch (status) {
    case OSDP_OK: return "ok";
    case OSDP_ERR_NULL: return "null pointer";
    case OSDP_ERR_SHAPE: return "bad shape";
    case OSDP_ERR_K: return "bad split count k";
    case OSDP_ERR_DTYPE: return "unsupported dtype";
    case OSDP_ERR_WORKSPACE: return "workspace too small or misaligned";
    case OSDP_ERR_ALIGN: return "tensor pointer not 16-byte aligned";
    case OSDP_ERR_ARCH: return "device is not sm_100";
    case OSDP_ERR_CUDA: return "CUDA error";
    case OSDP_ERR_INFEASIBLE: return "no plan fits the memory limit";
    case OSDP_ERR_ARG: return "invalid argument";
    case OSDP_ERR_SEARCH_LIMIT: return "planner node budget exhausted";
    case OSDP_ERR_COMM: return "a caller-supplied collective failed";
    case OSDP_ERR_STATIC_LIMIT: return "more columns than the static scratch of osdp_bias_grad_static holds";
    default: return "unknown status";
  }
}

const char* osdp_last_cuda_error(void) { return g_last_error.c_str(); }
const char* osdp_version(void) { return "osdp-b200 0.1.0 (sm_100a)"; }
int64_t osdp_last_launch_count(void) { return g_launches; }

int osdp_set_tuning(int key, int64_t value) {
  sm100::Tuning& t = sm100::tuning();
  switch (key) {
    case OSDP_TUNE_MT2_MIN_K:
      if (value < 1) return OSDP_ERR_ARG;
      t.mt2_min_k = value;
      return OSDP_OK;
    case OSDP_TUNE_MT2_MIN_TILES:
      if (value < 0) return OSDP_ERR_ARG;
      t.mt2_min_tiles = value;
      return OSDP_OK;
    case OSDP_TUNE_WAVE_SYNC:
      if (value < 0 || value > (1 << 20)) return OSDP_ERR_ARG;
      t.wave_sync = value;
      return OSDP_OK;
    case OSDP_TUNE_BAND_MIB:
      if (value < 0 || value > 1024) return OSDP_ERR_ARG;
      t.band_mib = value;
      return OSDP_OK;
    case OSDP_TUNE_CLUSTER_MIN_TILES:
      if (value < 0) return OSDP_ERR_ARG;
      t.cluster_min_tiles = value;
      return OSDP_OK;
    case OSDP_TUNE_MT2_MIN_K_ACC:
      if (value < 1) return OSDP_ERR_ARG;
      t.mt2_min_k_acc = value;
      return OSDP_OK;
    case OSDP_TUNE_FORK_MAX_TILES:
      if (value < 0) return OSDP_ERR_ARG;
      t.fork_max_tiles = value;
      return OSDP_OK;
    case OSDP_TUNE_SLICE_KERNEL_MAX_TILES:
      if (value < 0) return OSDP_ERR_ARG;
      t.slice_kernel_max_tiles = value;
      return OSDP_OK;
    case OSDP_TUNE_SLICE_KERNEL_FFN_MAX_TILES:
      if (value < 0) return OSDP_ERR_ARG;
      t.slice_kernel_ffn_max_tiles = value;
      return OSDP_OK;
    case OSDP_TUNE_BALANCE_N:
      if (value < 0 || value > 1) return OSDP_ERR_ARG;
      t.balance_n = value;
      return OSDP_OK;
    default: return OSDP_ERR_ARG;
  }
}

int64_t osdp_get_tuning(int key) {
  sm100::Tuning& t = sm100::tuning();
  switch (key) {
    case OSDP_TUNE_MT2_MIN_K: return t.mt2_min_k;
    case OSDP_TUNE_MT2_MIN_TILES: return t.mt2_min_tiles;
    case OSDP_TUNE_WAVE_SYNC: return t.wave_sync;
    case OSDP_TUNE_BAND_MIB: return t.band_mib;
    case OSDP_TUNE_CLUSTER_MIN_TILES: return t.cluster_min_tiles;
    case OSDP_TUNE_MT2_MIN_K_ACC: return t.mt2_min_k_acc;
    case OSDP_TUNE_FORK_MAX_TILES: return t.fork_max_tiles;
    case OSDP_TUNE_SLICE_KERNEL_MAX_TILES: return t.slice_kernel_max_tiles;
    case OSDP_TUNE_SLICE_KERNEL_FFN_MAX_TILES: return t.slice_kernel_ffn_max_tiles;
    case OSDP_TUNE_BALANCE_N: return t.balance_n;
    default: return -1;
  }
}

int osdp_trace_enable(int on) {
  g_trace.on = on != 0;
  if (!g_trace.on) g_trace.steps.clear();
  return OSDP_OK;
}

int64_t osdp_trace_read(int64_t max_entries, int32_t* step_ids, float* ms) {
  const int64_t n = (int64_t)g_trace.steps.size();
  bool bad = g_trace.failed;
  for (int64_t i = 0; i < n && !bad; ++i) {
    float t = 0.f;
    if (cudaEventSynchronize(g_trace.pool[2 * i + 1]) != cudaSuccess ||
        cudaEventElapsedTime(&t, g_trace.pool[2 * i], g_trace.pool[2 * i + 1]) != cudaSuccess) {
      bad = true;
      break;
    }
    if (i < max_entries) {
      if (step_ids) step_ids[i] = g_trace.steps[i];
      if (ms) ms[i] = t;
    }
  }
  g_trace.steps.clear();
  g_trace.failed = false;
  return bad ? -1 : n;
}

const char* osdp_step_name(int step_id) {
  switch (step_id) {
    case 1: return "A1 fwd GEMM1 + bias + GeLU";
    case 2: return "A2 fwd GEMM2 + bias";
    case 3: return "A3 bwd recompute GEMM1 (Z, H)";
    case 4: return "A4 bwd dH GEMM + GeLU'";
    case 5: return "A5 dW2 += H^T dY";
    case 6: return "A6 dW1 += X^T dZ";
    case 7: return "A7 dX = dZ W1^T";
    case 8: return "A8 db2 and db1 column sums";
    case 10: return "fp32 accumulator -> output (ffn / contraction-axis split)";
    case 11: return "Linear fwd Y = X W + b";
    case 12: return "Linear bwd dX = dY W^T";
    case 13: return "Linear bwd dW += X^T dY";
    case 21: return "slice kernel fwd (A1 -> A2 in one launch)";
    case 22: return "slice kernel bwd ((A3 + A4 fused) -> A7 | A5 | A6 + db1 in one launch)";
    default: return "unknown";
  }
}

size_t osdp_split_mlp_workspace_bytes(const osdp_mlp_desc* desc, int pass) {
  if (check_desc(desc) != OSDP_OK || (pass != OSDP_FWD && pass != OSDP_BWD)) return 0;
  return workspace_bytes(desc, pass);
}

int osdp_mlp_op_cost(const osdp_mlp_desc* desc, int pass, osdp_op_cost* out) {
  if (!out) return OSDP_ERR_NULL;
  OSDP_TRY(check_desc(desc));
  if (pass != OSDP_FWD && pass != OSDP_BWD) return OSDP_ERR_ARG;
  const uint64_t T = desc->tokens, h = desc->hidden, f = desc->ffn, e = elem_size(desc->dtype);
  osdp_op_cost c = {};
  c.S = (double)((2 * h * f + f + h) * e);
  // Model states (what ZDP shards) are the parameters and, in the backward, their fp32 gradients; the
  // T x h tensors are activations of this call's token batch (one unit of batch = desc->tokens tokens).
  if (pass == OSDP_FWD) {
    c.model_bytes = (2 * h * f + f + h) * e;                          // W1, W2, b1, b2
    c.act_bytes = 2 * T * h * e;                                      // X, Y
    c.extra_transient = T * f * e;                                    // H
    c.extra_fixed = slice_sync_bytes(desc);                           // tile counter / flags of the one-kernel-per-slice path
  } else {
    c.model_bytes = (2 * h * f + f + h) * e + (2 * h * f + f + h) * 4;   // W, b; fp32 dW, db
    c.act_bytes = 3 * T * h * e;                                      // X, dY, dX
    c.extra_transient = 2 * T * f * e + (T * f * 4) / kBandRows;      // Z/dZ, H and the db1 band partials: all per slice
    c.extra_fixed = db2_scratch_bytes(h) + slice_sync_bytes(desc);
  }
  *out = c;
  return OSDP_OK;
}

int osdp_split_mlp_forward(const osdp_mlp_desc* desc, const void* X, const void* W1, const void* b1, const void* W2,
                           const void* b2, void* Y, void* workspace, size_t workspace_bytes_given, void* stream) {
  g_launches = 0;
  OSDP_TRY(check_desc(desc));
  if (!X || !W1 || !b1 || !W2 || !b2 || !Y || !workspace) return OSDP_ERR_NULL;
  if (misaligned(X, 16) || misaligned(W1, 16) || misaligned(b1, 16) || misaligned(W2, 16) || misaligned(b2, 16) ||
      misaligned(Y, 16))
    return OSDP_ERR_ALIGN;
  if (misaligned(workspace, 256) || workspace_bytes_given < workspace_bytes(desc, OSDP_FWD)) return OSDP_ERR_WORKSPACE;
  if (desc->dtype == OSDP_BF16) OSDP_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t T = desc->tokens, h = desc->hidden, f = desc->ffn;
  const size_t e = elem_size(desc->dtype);
  const int dt = desc->dtype;
  void* Hs = workspace;

  SlicePlan sp;
  OSDP_TRY(slice_plan(desc, OSDP_FWD, &sp));
  unsigned int* sync = nullptr;
  unsigned int epoch0 = 0;
  // A workspace with room for two H_s buffers (the backward's is: callers that train pass the same workspace to both
  // passes) lets consecutive slices alternate buffers, and slice s then need not wait for slice s - 1 at all (see
  // late_wait in slice_sm100.cuh); with the forward's own minimum the slices run one after another as the paper says.
  const bool two_bufs = workspace_bytes_given >= 2 * slice_buf_bytes(desc) + slice_sync_bytes(desc);
  if (sp.use)
    OSDP_TRY(slice_sync_setup(sp, workspace, (two_bufs ? 2 : 1) * slice_buf_bytes(desc), desc->k, st, &sync, &epoch0));
  bool first_launch = true;

  for (int s = 0; s < desc->k; ++s) {
    const int64_t lo = (int64_t)s * T / desc->k, hi = (int64_t)(s + 1) * T / desc->k;
    const int Ts = (int)(hi - lo);
    if (Ts == 0) continue;
    const char* Xs = (const char*)X + (size_t)lo * h * e;
    char* Ys = (char*)Y + (size_t)lo * h * e;
    if (sp.use) {   // A1 -> A2 in one launch: an A2 tile starts when its 256 rows of H_s are complete
      void* Hb = two_bufs ? (char*)workspace + (size_t)(s & 1) * slice_buf_bytes(desc) : Hs;
      trace_set_step(21);
      sm100::SliceGemm g[2] = {};
      g[0] = {Xs, h, W1, f, MAJOR_K, MAJOR_MN, EPI_BIAS_GELU, GemmShape{Ts, (int)f, (int)h},
              EpiParams{b1, Hb, nullptr, nullptr, f, 0}, sm100::DEP_NONE, 0, 256, 1, 0};
      g[1] = {Hb, f, W2, h, MAJOR_K, MAJOR_MN, EPI_BIAS, GemmShape{Ts, (int)h, (int)f},
              EpiParams{b2, Ys, nullptr, nullptr, h, 0}, sm100::DEP_ROW, 0, sp.bn_narrow, 0, 0};
      OSDP_TRY(sm100::launch_mlp_slice(g, 2, sync + (size_t)s * sp.words_per_slice, epoch0 + (unsigned int)s, nullptr,
                                       two_bufs && !first_launch, st));
      first_launch = false;
      continue;
    }
    // A1: H_s = gelu(X_s W1 + b1)
    trace_set_step(1);
    EpiParams e1 = {b1, Hs, nullptr, nullptr, f, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS_GELU>(dt, Xs, h, W1, f, GemmShape{Ts, (int)f, (int)h}, e1, st)));
    // A2: Y_s = H_s W2 + b2
    trace_set_step(2);
    EpiParams e2 = {b2, Ys, nullptr, nullptr, h, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS>(dt, Hs, f, W2, h, GemmShape{Ts, (int)h, (int)f}, e2, st)));
  }
  return OSDP_OK;
}

int osdp_split_mlp_backward(const osdp_mlp_desc* desc, const void* X, const void* W1, const void* b1, const void* W2,
                            const void* b2, const void* dY, void* dX, float* dW1, float* db1, float* dW2, float* db2,
                            void* workspace, size_t workspace_bytes_given, void* stream) {
  (void)b2;
  g_launches = 0;
  OSDP_TRY(check_desc(desc));
  if (!X || !W1 || !b1 || !W2 || !dY || !dX || !dW1 || !db1 || !dW2 || !db2 || !workspace) return OSDP_ERR_NULL;
  if (misaligned(X, 16) || misaligned(W1, 16) || misaligned(b1, 16) || misaligned(W2, 16) || misaligned(dY, 16) ||
      misaligned(dX, 16) || misaligned(dW1, 16) || misaligned(db1, 16) || misaligned(dW2, 16) || misaligned(db2, 16))
    return OSDP_ERR_ALIGN;
  if (misaligned(workspace, 256) || workspace_bytes_given < workspace_bytes(desc, OSDP_BWD)) return OSDP_ERR_WORKSPACE;
  if (desc->dtype == OSDP_BF16) OSDP_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t T = desc->tokens, h = desc->hidden, f = desc->ffn;
  const size_t e = elem_size(desc->dtype);
  const int dt = desc->dtype;
  const size_t buf = slice_buf_bytes(desc);
  void* Zs = workspace;                                  // Z_s, then dZ_s in place
  void* Hs = (char*)workspace + buf;                     // H_s
  const int64_t ts_max = (T + desc->k - 1) / desc->k;
  float* scratch1 = (float*)((char*)workspace + 2 * buf);                                   // db1: band partials of dZ_s
  float* scratch2 = (float*)((char*)workspace + 2 * buf + db1_scratch_bytes(ts_max, f));    // db2: chunk partials of dY

  // db2 = colsum(dY): dY is whole in memory, so one fixed-order reduction per call (not per slice; bit-identical for every k)
  trace_set_step(8);
  OSDP_TRY(colsum_rows(dt, dY, (int)h, db2, (int)T, scratch2, 0, st));

  // Small slices: the three GEMMs and the column sums that only need dZ_s run side by side (helper streams above).
  const int64_t fork_max = sm100::tuning().fork_max_tiles.load();
  const bool fork = fork_max > 0 && tiles_256(f, h) <= fork_max && tiles_256(ts_max, h) <= fork_max;
  ForkCtx* fc = nullptr;
  SlicePlan sp;
  OSDP_TRY(slice_plan(desc, OSDP_BWD, &sp));
  unsigned int* sync = nullptr;
  unsigned int epoch0 = 0;
  if (sp.use) OSDP_TRY(slice_sync_setup(sp, workspace, workspace_tensor_bytes(desc, OSDP_BWD), desc->k, st, &sync, &epoch0));
  if (fork && !sp.use) OSDP_TRY(fork_ctx(&fc));

  int first = 1;
  for (int s = 0; s < desc->k; ++s) {
    const int64_t lo = (int64_t)s * T / desc->k, hi = (int64_t)(s + 1) * T / desc->k;
    const int Ts = (int)(hi - lo);
    if (Ts == 0) continue;
    const int beta = first ? 0 : 1;
    first = 0;
    const char* Xs = (const char*)X + (size_t)lo * h * e;
    const char* dYs = (const char*)dY + (size_t)lo * h * e;
    char* dXs = (char*)dX + (size_t)lo * h * e;
    if (sp.use) {
      // (A3 + A4) -> A5 | A7 | A6 (+ db1) in one launch.  A3 and A4 share their output tile grid, so one tile runs both
      // contractions into the two TMEM accumulators and one epilogue makes H_s and dZ_s (Z_s never goes to memory).
      // List order = claim order; everything after the fused tiles becomes ready at about the same time, so the
      // long-contraction dX tiles (few tiles, four times the k-blocks of the others) go first and the dW tiles fill in.
      trace_set_step(22);
      sm100::SliceGemm g[4] = {};
      g[0] = {Xs, h, W1, f, MAJOR_K, MAJOR_MN, sm100::kEpiFusedA34, GemmShape{Ts, (int)f, (int)h},
              EpiParams{b1, Zs, Hs, nullptr, f, 0, scratch1, f}, sm100::DEP_NONE, 0, 256, 1, 0,
              dYs, h, W2, h, MAJOR_K, MAJOR_K, (int)h};
      g[1] = {Zs, f, W1, f, MAJOR_K, MAJOR_K, EPI_PLAIN, GemmShape{Ts, (int)h, (int)f},
              EpiParams{nullptr, dXs, nullptr, nullptr, h, 0}, sm100::DEP_ROW, 0, sp.bn_narrow, 0, 0};
      g[2] = {Hs, f, dYs, h, MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32, GemmShape{(int)f, (int)h, Ts},
              EpiParams{nullptr, dW2, nullptr, nullptr, h, beta}, sm100::DEP_COL_AS_M, 0, 256, 0, 0};
      g[3] = {Xs, h, Zs, f, MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32, GemmShape{(int)h, (int)f, Ts},
              EpiParams{nullptr, dW1, nullptr, nullptr, f, beta}, sm100::DEP_COL_AS_N, 0, 256, 0, 1};
      const sm100::SliceDb1 dj = {scratch1, f, db1, (Ts + kBandRows - 1) / kBandRows, beta};
      OSDP_TRY(sm100::launch_mlp_slice(g, 4, sync + (size_t)s * sp.words_per_slice, epoch0 + (unsigned int)s, &dj, false, st));
      continue;
    }
    // A3: Z_s = X_s W1 + b1, H_s = gelu(Z_s)
    trace_set_step(3);
    EpiParams e3 = {b1, Zs, Hs, nullptr, f, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS_GELU_DUAL>(dt, Xs, h, W1, f, GemmShape{Ts, (int)f, (int)h}, e3, st)));
    // A4: dZ_s = (dY_s W2^T) (.) gelu'(Z_s), in place over Z_s; the epilogue also leaves the 32-row band sums (db1)
    trace_set_step(4);
    EpiParams e4 = {nullptr, Zs, nullptr, Zs, f, 0, scratch1, f};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_DGELU>(dt, dYs, h, W2, h, GemmShape{Ts, (int)f, (int)h}, e4, st)));
    if (fork) OSDP_TRY(fork_from(fc, st));
    // A5: dW2 (+)= H_s^T dY_s
    trace_set_step(5);
    EpiParams e5 = {nullptr, dW2, nullptr, nullptr, h, beta};
    OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, Hs, f, dYs, h, GemmShape{(int)f, (int)h, Ts}, e5, st)));
    // A8: db1 (+)= colsum(dZ_s), fixed-order sum of the band partials
    trace_set_step(8);
    OSDP_TRY(db1_from_bands(dt, Zs, (int)f, db1, Ts, scratch1, beta, fork ? fc->side[2] : st));
    // A6: dW1 (+)= X_s^T dZ_s
    trace_set_step(6);
    EpiParams e6 = {nullptr, dW1, nullptr, nullptr, f, beta};
    OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, Xs, h, Zs, f, GemmShape{(int)h, (int)f, Ts}, e6,
                                                      fork ? fc->side[0] : st)));
    // A7: dX_s = dZ_s W1^T
    trace_set_step(7);
    EpiParams e7 = {nullptr, dXs, nullptr, nullptr, h, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_PLAIN>(dt, Zs, f, W1, f, GemmShape{Ts, (int)h, (int)f}, e7,
                                                fork ? fc->side[1] : st)));
    if (fork) OSDP_TRY(join_into(fc, st));   // the next slice overwrites Z_s / H_s
  }
  return OSDP_OK;
}

// ============================================================================================ ffn-axis split
size_t osdp_ffn_split_mlp_workspace_bytes(const osdp_mlp_desc* desc, int pass) {
  if (check_desc_ffn(desc) != OSDP_OK || (pass != OSDP_FWD && pass != OSDP_BWD)) return 0;
  return ffn_workspace_bytes(desc, pass);
}

int osdp_ffn_split_mlp_op_cost(const osdp_mlp_desc* desc, int pass, osdp_op_cost* out) {
  if (!out) return OSDP_ERR_NULL;
  OSDP_TRY(check_desc_ffn(desc));
  if (pass != OSDP_FWD && pass != OSDP_BWD) return OSDP_ERR_ARG;
  const uint64_t T = desc->tokens, h = desc->hidden, f = desc->ffn, e = elem_size(desc->dtype);
  osdp_op_cost c = {};
  c.S = (double)((2 * h * f + f + h) * e);
  const uint64_t acc = align_up((size_t)T * h * 4, 256);   // cross-slice fp32 accumulator (any k > 1)
  if (pass == OSDP_FWD) {
    c.model_bytes = (2 * h * f + f + h) * e;
    c.act_bytes = 2 * T * h * e;
    c.extra_transient = T * f * e;
    c.extra_fixed = acc + ffn_slice_sync_bytes(desc);
  } else {
    c.model_bytes = (2 * h * f + f + h) * e + (2 * h * f + f + h) * 4;
    c.act_bytes = 3 * T * h * e;
    c.extra_transient = 2 * T * f * e + db1_scratch_bytes(T, f);     // db1 band partials of one slice: ceil(T / 32) x f / k floats
    c.extra_fixed = acc + db2_scratch_bytes(h) + ffn_slice_sync_bytes(desc);
  }
  *out = c;
  return OSDP_OK;
}

int osdp_ffn_split_mlp_forward(const osdp_mlp_desc* desc, const void* X, const void* W1, const void* b1, const void* W2,
                               const void* b2, void* Y, void* workspace, size_t workspace_bytes_given, void* stream) {
  g_launches = 0;
  OSDP_TRY(check_desc_ffn(desc));
  if (!X || !W1 || !b1 || !W2 || !b2 || !Y || !workspace) return OSDP_ERR_NULL;
  if (misaligned(X, 16) || misaligned(W1, 16) || misaligned(b1, 16) || misaligned(W2, 16) || misaligned(b2, 16) ||
      misaligned(Y, 16))
    return OSDP_ERR_ALIGN;
  if (misaligned(workspace, 256) || workspace_bytes_given < ffn_workspace_bytes(desc, OSDP_FWD)) return OSDP_ERR_WORKSPACE;
  if (desc->dtype == OSDP_BF16) OSDP_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t T = desc->tokens, h = desc->hidden;
  const size_t e = elem_size(desc->dtype);
  const int dt = desc->dtype, k = desc->k;
  void* Hs = workspace;
  float* Yacc = (float*)((char*)workspace + ffn_slice_buf_bytes(desc));
  SlicePlan sp;
  OSDP_TRY(ffn_slice_plan(desc, ffn_slice_max(desc), &sp));
  unsigned int* sync = nullptr;
  unsigned int epoch0 = 0;
  if (sp.use) OSDP_TRY(slice_sync_setup(sp, workspace, ffn_workspace_tensor_bytes(desc, OSDP_FWD), k, st, &sync, &epoch0));

  for (int s = 0; s < k; ++s) {
    const int64_t lo = ffn_lo(desc, s), hi = ffn_lo(desc, s + 1);
    const int fs = (int)(hi - lo);
    if (fs == 0) continue;   // cannot happen for k <= units; kept for symmetry with the token split
    const FfnSliceW w = {(const char*)W1 + (size_t)lo * e, desc->ffn, (const char*)b1 + (size_t)lo * e,
                         (const char*)W2 + (size_t)lo * h * e};
    FfnSliceKernel sk;
    if (sp.use) sk = FfnSliceKernel{sync + (size_t)s * sp.words_per_slice, epoch0 + (unsigned int)s, sp.bn_narrow};
    OSDP_TRY(ffn_slice_forward(dt, T, h, fs, X, w, b2, Y, Hs, Yacc, k == 1, s == 0, st, &sk));
  }
  if (k > 1) {   // Y = storage(Yacc + b2)
    trace_set_step(10);
    sm100::DeviceInfo dev;
    OSDP_TRY(sm100::current_device(&dev));
    OSDP_TRY(launch_acc_to_out(dt, Yacc, b2, Y, T, (int)h, dev.sms, st));
  }
  return OSDP_OK;
}

int osdp_ffn_split_mlp_backward(const osdp_mlp_desc* desc, const void* X, const void* W1, const void* b1, const void* W2,
                                const void* b2, const void* dY, void* dX, float* dW1, float* db1, float* dW2, float* db2,
                                void* workspace, size_t workspace_bytes_given, void* stream) {
  (void)b2;
  g_launches = 0;
  OSDP_TRY(check_desc_ffn(desc));
  if (!X || !W1 || !b1 || !W2 || !dY || !dX || !dW1 || !db1 || !dW2 || !db2 || !workspace) return OSDP_ERR_NULL;
  if (misaligned(X, 16) || misaligned(W1, 16) || misaligned(b1, 16) || misaligned(W2, 16) || misaligned(dY, 16) ||
      misaligned(dX, 16) || misaligned(dW1, 16) || misaligned(db1, 16) || misaligned(dW2, 16) || misaligned(db2, 16))
    return OSDP_ERR_ALIGN;
  if (misaligned(workspace, 256) || workspace_bytes_given < ffn_workspace_bytes(desc, OSDP_BWD)) return OSDP_ERR_WORKSPACE;
  if (desc->dtype == OSDP_BF16) OSDP_TRY(check_arch());
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t T = desc->tokens, h = desc->hidden, f = desc->ffn;
  const size_t e = elem_size(desc->dtype);
  const int dt = desc->dtype, k = desc->k;
  const size_t buf = ffn_slice_buf_bytes(desc);
  void* Zs = workspace;                                  // Z_s, then dZ_s in place       [T x fs]
  void* Hs = (char*)workspace + buf;                     // H_s                           [T x fs]
  float* dXacc = (float*)((char*)workspace + 2 * buf);   // fp32 accumulator of dX        [T x h]   (k > 1)
  float* scratch1 = (float*)((char*)workspace + 2 * buf + ffn_acc_bytes(desc));                      // db1 band partials
  float* scratch2 = (float*)((char*)scratch1 + db1_scratch_bytes(T, ffn_slice_max(desc)));           // db2 chunk partials
  SlicePlan sp;
  OSDP_TRY(ffn_slice_plan(desc, ffn_slice_max(desc), &sp));
  unsigned int* sync = nullptr;
  unsigned int epoch0 = 0;
  if (sp.use) OSDP_TRY(slice_sync_setup(sp, workspace, ffn_workspace_tensor_bytes(desc, OSDP_BWD), k, st, &sync, &epoch0));

  for (int s = 0; s < k; ++s) {
    const int64_t lo = ffn_lo(desc, s), hi = ffn_lo(desc, s + 1);
    const int fs = (int)(hi - lo);
    if (fs == 0) continue;
    const FfnSliceW w = {(const char*)W1 + (size_t)lo * e, f, (const char*)b1 + (size_t)lo * e,
                         (const char*)W2 + (size_t)lo * h * e};
    const FfnSliceG g = {dW1 + lo, f, db1 + lo, dW2 + (size_t)lo * h};
    FfnSliceKernel sk;
    if (sp.use) sk = FfnSliceKernel{sync + (size_t)s * sp.words_per_slice, epoch0 + (unsigned int)s, sp.bn_narrow};
    OSDP_TRY(ffn_slice_backward(dt, T, h, fs, X, dY, w, g, Zs, Hs, dX, dXacc, scratch1, scratch2, s == 0 ? db2 : nullptr,
                                k == 1, s == 0, st, &sk));
  }
  if (k > 1) {   // dX = storage(dXacc)
    trace_set_step(10);
    sm100::DeviceInfo dev;
    OSDP_TRY(sm100::current_device(&dev));
    OSDP_TRY(launch_acc_to_out(dt, dXacc, nullptr, dX, T, (int)h, dev.sms, st));
  }
  return OSDP_OK;
}

}  // extern "C"

#include "linear_api.inl"
#include "zdp_api.inl"
