// reduce.cuh — A8 / db1: column sums of a [rows x cols] tensor into an fp32 vector.
//
// Deterministic: fixed two-stage reduction order, no float atomics (SURVEY.md §7 "Deterministic accumulation").
// Stage 1 leaves partial sums of row chunks in a scratch [chunks x cols]:
//   db1 (bf16): the A4 GEMM's epilogue writes the sums of every 32-row band of dZ_s itself (gemm_sm100.cuh), so dZ_s is
//               never read again;
//   db1 (fp32) and db2: colsum_partial_kernel, HBM-bound (reads the tensor once): grid (column blocks x chunks); every
//               warp owns whole rows (lanes across 16-byte column vectors: coalesced), rows ascending, then the 8 warps
//               of the CTA are summed in warp order through shared memory.
// Stage 2 (colsum_final_kernel): one thread per column sums the partials in chunk order and adds to (beta = 1) or
// overwrites (beta = 0) the output.
#pragma once
#include "common.cuh"

namespace osdp {

constexpr int kReduceRowChunks = 32;   // db2: chunks of the whole call's rows (scratch 32 x h floats)
constexpr int kBandRows = 32;          // db1: one partial row per 32-row band of the slice (scratch ceil(T_s / 32) x f floats)
constexpr int kReduceThreads = 256;

template <typename T> struct VecOf;
template <> struct VecOf<float> {
  static constexpr int N = 4;
  __device__ static void load(const float* p, float (&v)[4]) {
    const float4 x = *reinterpret_cast<const float4*>(p);
    v[0] = x.x; v[1] = x.y; v[2] = x.z; v[3] = x.w;
  }
};
template <> struct VecOf<__nv_bfloat16> {
  static constexpr int N = 8;
  __device__ static void load(const __nv_bfloat16* p, float (&v)[8]) {
    const uint4 x = *reinterpret_cast<const uint4*>(p);
    const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      v[2 * i] = __uint_as_float(w[i] << 16);
      v[2 * i + 1] = __uint_as_float(w[i] & 0xFFFF0000u);
    }
  }
};

// One column-sum job: src [rows x cols] (leading dimension ld) -> out [cols]; partials live at scratch + offset.
struct ColsumJob {
  const void* src;
  int cols;
  int64_t ld;
  float* out;
  int64_t scratch_off;   // floats; the job owns chunks x cols floats from there
  int col_blocks;        // CTAs along the columns (stage 1) / along the columns in 256s (stage 2)
  int chunks;            // partial rows of this job (stage 2)
};

// Stage 1 for TWO tensors with the same row count in one launch (db2 from dY_s and db1 from dZ_s): blockIdx.x
// first walks the column blocks of job 0, then those of job 1.
template <typename T>
__global__ void __launch_bounds__(kReduceThreads) colsum_partial_kernel(const ColsumJob j0, const ColsumJob j1, int rows,
                                                                        float* __restrict__ scratch, int rows_per_chunk) {
  constexpr int V = VecOf<T>::N;
  constexpr int kWarps = kReduceThreads / 32;
  __shared__ float red[kWarps][32 * V];
  const bool second = (int)blockIdx.x >= j0.col_blocks;
  const ColsumJob& job = second ? j1 : j0;
  const int bx = second ? (int)blockIdx.x - j0.col_blocks : (int)blockIdx.x;
  const T* __restrict__ src = reinterpret_cast<const T*>(job.src);
  float* __restrict__ partial = scratch + job.scratch_off;
  const int cols = job.cols;
  const int lane = threadIdx.x % 32, warp = threadIdx.x / 32;
  const int c = (bx * 32 + lane) * V;
  const int r_begin = blockIdx.y * rows_per_chunk;
  const int r_end = min(rows, r_begin + rows_per_chunk);
  float acc[V];
#pragma unroll
  for (int i = 0; i < V; ++i) acc[i] = 0.0f;
  if (c < cols) {
    for (int r = r_begin + warp; r < r_end; r += kWarps) {
      float v[V];
      VecOf<T>::load(src + (int64_t)r * job.ld + c, v);
#pragma unroll
      for (int i = 0; i < V; ++i) acc[i] += v[i];
    }
  }
#pragma unroll
  for (int i = 0; i < V; ++i) red[warp][lane * V + i] = acc[i];
  __syncthreads();
  for (int j = threadIdx.x; j < 32 * V; j += kReduceThreads) {
    float s = 0.0f;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) s += red[w][j];
    const int col = bx * 32 * V + j;
    if (col < cols) partial[(int64_t)blockIdx.y * cols + col] = s;
  }
}

__global__ void colsum_final_kernel(const ColsumJob j0, const ColsumJob j1, const float* __restrict__ scratch, int beta) {
  const bool second = (int)blockIdx.x >= j0.col_blocks;
  const ColsumJob& job = second ? j1 : j0;
  const int bx = second ? (int)blockIdx.x - j0.col_blocks : (int)blockIdx.x;
  const int col = bx * blockDim.x + threadIdx.x;
  if (col >= job.cols) return;
  const float* __restrict__ partial = scratch + job.scratch_off;
  float s = 0.0f;
#pragma unroll 8
  for (int r = 0; r < job.chunks; ++r) s += partial[(int64_t)r * job.cols + col];
  job.out[col] = beta ? job.out[col] + s : s;
}

// Stage 2 alone: out_a (+)= sum of chunks_a partial rows at scratch, out_b likewise at scratch + chunks_a * cols_a
// (either job may be empty: cols = 0).
inline int launch_colsum_final(float* scratch, int cols_a, int chunks_a, float* out_a, int cols_b, int chunks_b, float* out_b,
                               int beta, cudaStream_t st) {
  ColsumJob j0{nullptr, cols_a, 0, out_a, 0, (cols_a + 255) / 256, chunks_a};
  ColsumJob j1{nullptr, cols_b, 0, out_b, (int64_t)chunks_a * cols_a, (cols_b + 255) / 256, chunks_b};
  if (j0.col_blocks + j1.col_blocks == 0) return OSDP_OK;
  {
    LaunchTrace tr(st);
    colsum_final_kernel<<<j0.col_blocks + j1.col_blocks, 256, 0, st>>>(j0, j1, scratch, beta);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

// out (+)= colsum(A [rows x cols]) in two launches; rows_per_chunk rows per partial (0 = kReduceRowChunks equal chunks).
// scratch: chunks x cols floats.
template <typename T>
inline int launch_colsum(const T* A, int cols, int64_t lda, float* out, int rows, int rows_per_chunk, float* scratch, int beta,
                         cudaStream_t st) {
  constexpr int V = VecOf<T>::N;
  if (cols == 0 || rows == 0) return OSDP_OK;
  if (rows_per_chunk <= 0) rows_per_chunk = (rows + kReduceRowChunks - 1) / kReduceRowChunks;
  int chunks = (rows + rows_per_chunk - 1) / rows_per_chunk;
  if (chunks > 65535) {   // grid.y limit: coarser chunks (the scratch sized for the finer ones still fits)
    rows_per_chunk = (rows + 65534) / 65535;
    chunks = (rows + rows_per_chunk - 1) / rows_per_chunk;
  }
  ColsumJob j0{A, cols, lda, out, 0, (cols + 32 * V - 1) / (32 * V), chunks};
  ColsumJob j1{nullptr, 0, 0, nullptr, 0, 0, 0};
  {
    LaunchTrace tr(st);
    colsum_partial_kernel<T><<<dim3(j0.col_blocks, chunks), kReduceThreads, 0, st>>>(j0, j1, rows, scratch, rows_per_chunk);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return launch_colsum_final(scratch, cols, chunks, out, 0, 0, nullptr, beta, st);
}

}  // namespace osdp
