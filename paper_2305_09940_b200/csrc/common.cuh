// common.cuh — shared host/device declarations of the osdp-b200 kernels.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/osdp.h"

namespace osdp {

// ---- GEMM problem as the slice scheduler states it -------------------------------------------------------
// C[M x N] = A[M x K] * B[K x N] with fp32 accumulation, then an epilogue.
// "K-major" = the contraction index is contiguous in memory; "MN-major" = the M (for A) / N (for B) index is.
//   A K-major : stored [M x K] row-major, leading dimension lda   (X_s, H_s, dY_s, dZ_s as left operands)
//   A MN-major: stored [K x M] row-major, leading dimension lda   (H_s^T, X_s^T for the dW GEMMs)
//   B K-major : stored [N x K] row-major, leading dimension ldb   (W2^T, W1^T given as W2, W1)
//   B MN-major: stored [K x N] row-major, leading dimension ldb   (W1, W2, dY_s, dZ_s as right operands)
enum Major : int { MAJOR_K = 0, MAJOR_MN = 1 };

// Epilogues (DESIGN.md steps):
enum Epi : int {
  EPI_BIAS_GELU = 0,       // A1: out0 = gelu(acc + bias)                       (storage dtype)
  EPI_BIAS = 1,            // A2: out0 = acc + bias                             (storage dtype)
  EPI_BIAS_GELU_DUAL = 2,  // A3: out0 = acc + bias (Z_s), out1 = gelu(out0-before-rounding) (H_s)
  EPI_DGELU = 3,           // A4: out0 = acc * gelu'(aux)   (aux = stored Z_s; out0 may alias aux)
  EPI_ACCUM_F32 = 4,       // A5/A6: out0(fp32) = (beta ? out0 : 0) + acc
  EPI_PLAIN = 5            // A7: out0 = acc                                    (storage dtype)
};

struct EpiParams {
  const void* bias;   // [N] storage dtype (BIAS* epilogues)
  void* out0;         // primary output, leading dimension ldo
  void* out1;         // EPI_BIAS_GELU_DUAL: H_s
  const void* aux;    // EPI_DGELU: Z_s
  int64_t ldo;        // leading dimension (elements) of out0/out1/aux
  int beta;           // EPI_ACCUM_F32: 0 = overwrite (first slice), 1 = accumulate
  // EPI_DGELU (A4): the epilogue also leaves the column sums of every 32-row band of dZ_s here,
  // colsum[(row / 32) * ld_colsum + col], for the fixed-order db1 reduction (reduce.cuh); nullptr = not wanted
  float* colsum = nullptr;
  int64_t ld_colsum = 0;
};

struct GemmShape {
  int M, N, K;
};

// tanh-GeLU constants (reading S2).
__host__ __device__ constexpr float kGeluC() { return 0.7978845608028654f; }
__host__ __device__ constexpr float kGeluA() { return 0.044715f; }

// ---- host-side error bookkeeping (osdp_api.cu) -------------------------------------------------------------
void note_cuda_error(cudaError_t e, const char* where);
void count_launch();
// Per-launch event trace (osdp_trace_*): launch wrappers bracket every kernel with LaunchTrace.
void trace_set_step(int step_id);
void trace_before(cudaStream_t st);
void trace_after(cudaStream_t st);
struct LaunchTrace {
  cudaStream_t st;
  explicit LaunchTrace(cudaStream_t s) : st(s) { trace_before(st); }
  ~LaunchTrace() { trace_after(st); count_launch(); }
};

#define OSDP_CUDA_TRY(expr)                                   \
  do {                                                        \
    cudaError_t _e = (expr);                                  \
    if (_e != cudaSuccess) {                                  \
      ::osdp::note_cuda_error(_e, #expr);                     \
      return OSDP_ERR_CUDA;                                   \
    }                                                         \
  } while (0)

}  // namespace osdp
