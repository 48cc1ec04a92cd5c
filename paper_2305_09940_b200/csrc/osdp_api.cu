// osdp_api.cu — the C ABI of osdp-b200 (include/osdp.h) and the host-side slice scheduler (step A0).
//
// The scheduler follows PAPER.md:165: slices are processed one after another in order on the caller's
// stream, the per-slice buffers in the caller's workspace are reused serially, and results that span slices
// (dW1, dW2, db1, db2) are summed: "=" on slice 0, "+=" afterwards, in fixed slice order.
#include <mutex>
#include <string>

#include "common.cuh"
#include "gemm_f32.cuh"
#include "gemm_sm100.cuh"
#include "reduce.cuh"

namespace osdp {

namespace {
thread_local std::string g_last_error;
thread_local int64_t g_launches = 0;
}  // namespace

void note_cuda_error(cudaError_t e, const char* where) {
  g_last_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e) + " at " + where;
}
void count_launch() { ++g_launches; }

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
int num_sms() {
  static int n = 0;
  if (n == 0) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    if (n <= 0) n = 1;
  }
  return n;
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
inline size_t reduce_scratch_bytes(const osdp_mlp_desc* d) {
  const int64_t c = d->hidden > d->ffn ? d->hidden : d->ffn;
  return align_up((size_t)kReduceRowChunks * (size_t)c * 4, 256);
}
size_t workspace_bytes(const osdp_mlp_desc* d, int pass) {
  if (pass == OSDP_FWD) return slice_buf_bytes(d);
  return 2 * slice_buf_bytes(d) + reduce_scratch_bytes(d);
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

int colsum(int dtype, const void* src, int rows, int cols, int64_t ld, float* scratch, float* out, int beta,
           cudaStream_t st) {
  if (dtype == OSDP_BF16) return launch_colsum<__nv_bfloat16>((const __nv_bfloat16*)src, rows, cols, ld, scratch, out, beta, st);
  return launch_colsum<float>((const float*)src, rows, cols, ld, scratch, out, beta, st);
}

#define OSDP_TRY(expr)            \
  do {                            \
    int _rc = (expr);             \
    if (_rc != OSDP_OK) return _rc; \
  } while (0)

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
    default: return "unknown status";
  }
}

const char* osdp_last_cuda_error(void) { return g_last_error.c_str(); }
const char* osdp_version(void) { return "osdp-b200 0.1.0 (sm_100a)"; }
int64_t osdp_last_launch_count(void) { return g_launches; }

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
  if (pass == OSDP_FWD) {
    c.model_bytes = (2 * T * h + 2 * h * f + f + h) * e;             // X, Y, W1, W2, b1, b2
    c.extra_transient = T * f * e;                                    // H
    c.extra_fixed = 0;
  } else {
    c.model_bytes = (3 * T * h + 2 * h * f + f + h) * e + (2 * h * f + f + h) * 4;   // X, dY, dX, W, b; fp32 grads
    c.extra_transient = 2 * T * f * e;                                // Z/dZ and H
    c.extra_fixed = reduce_scratch_bytes(desc);
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

  for (int s = 0; s < desc->k; ++s) {
    const int64_t lo = (int64_t)s * T / desc->k, hi = (int64_t)(s + 1) * T / desc->k;
    const int Ts = (int)(hi - lo);
    if (Ts == 0) continue;
    const char* Xs = (const char*)X + (size_t)lo * h * e;
    char* Ys = (char*)Y + (size_t)lo * h * e;
    // A1: H_s = gelu(X_s W1 + b1)
    EpiParams e1 = {b1, Hs, nullptr, nullptr, f, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS_GELU>(dt, Xs, h, W1, f, GemmShape{Ts, (int)f, (int)h}, e1, st)));
    // A2: Y_s = H_s W2 + b2
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
  float* scratch = (float*)((char*)workspace + 2 * buf);   // column-sum partials

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
    // A3: Z_s = X_s W1 + b1, H_s = gelu(Z_s)
    EpiParams e3 = {b1, Zs, Hs, nullptr, f, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_MN, EPI_BIAS_GELU_DUAL>(dt, Xs, h, W1, f, GemmShape{Ts, (int)f, (int)h}, e3, st)));
    // A4: dZ_s = (dY_s W2^T) (.) gelu'(Z_s), in place over Z_s
    EpiParams e4 = {nullptr, Zs, nullptr, Zs, f, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_DGELU>(dt, dYs, h, W2, h, GemmShape{Ts, (int)f, (int)h}, e4, st)));
    // A5: dW2 (+)= H_s^T dY_s
    EpiParams e5 = {nullptr, dW2, nullptr, nullptr, h, beta};
    OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, Hs, f, dYs, h, GemmShape{(int)f, (int)h, Ts}, e5, st)));
    // A8: db2 (+)= colsum(dY_s);  db1 (+)= colsum(dZ_s)
    OSDP_TRY(colsum(dt, dYs, Ts, (int)h, h, scratch, db2, beta, st));
    OSDP_TRY(colsum(dt, Zs, Ts, (int)f, f, scratch, db1, beta, st));
    // A6: dW1 (+)= X_s^T dZ_s
    EpiParams e6 = {nullptr, dW1, nullptr, nullptr, f, beta};
    OSDP_TRY((gemm<MAJOR_MN, MAJOR_MN, EPI_ACCUM_F32>(dt, Xs, h, Zs, f, GemmShape{(int)h, (int)f, Ts}, e6, st)));
    // A7: dX_s = dZ_s W1^T
    EpiParams e7 = {nullptr, dXs, nullptr, nullptr, h, 0};
    OSDP_TRY((gemm<MAJOR_K, MAJOR_K, EPI_PLAIN>(dt, Zs, f, W1, f, GemmShape{Ts, (int)h, (int)f}, e7, st)));
  }
  return OSDP_OK;
}

}  // extern "C"
