// reduce.cuh — A8 / db1: column sums of a [rows x cols] slice tensor into an fp32 vector.
//
// HBM-bound (reads the slice once).  Deterministic: fixed two-stage reduction order, no float atomics
// (SURVEY.md §7 "Deterministic accumulation").  db2 (from dY_s) and db1 (from dZ_s) share the two launches.
// Stage 1: grid (column blocks of both tensors x kReduceRowChunks); every warp
// owns whole rows (lanes across 16-byte column vectors: coalesced), rows ascending, then the 8 warps of the
// CTA are summed in warp order through shared memory.  Stage 2: one thread per column sums the
// kReduceRowChunks partials in chunk order and adds to (beta = 1) or overwrites (beta = 0) the output.
#pragma once
#include "common.cuh"

namespace osdp {

constexpr int kReduceRowChunks = 32;   // scratch = kReduceRowChunks x (h + f) floats (osdp.h, A10)
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
  int64_t scratch_off;   // floats; the job owns kReduceRowChunks x cols floats from there
  int col_blocks;        // CTAs along the columns (stage 1) / along the columns in 256s (stage 2)
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
  for (int r = 0; r < kReduceRowChunks; ++r) s += partial[(int64_t)r * job.cols + col];
  job.out[col] = beta ? job.out[col] + s : s;
}

// db2 (+)= colsum(A [rows x cols_a]) and db1 (+)= colsum(B [rows x cols_b]) in two launches.
// scratch: kReduceRowChunks x (cols_a + cols_b) floats.
template <typename T>
inline int launch_colsum2(const T* A, int cols_a, int64_t lda, float* out_a, const T* B, int cols_b, int64_t ldb,
                          float* out_b, int rows, float* scratch, int beta, cudaStream_t st) {
  constexpr int V = VecOf<T>::N;
  const int rows_per_chunk = (rows + kReduceRowChunks - 1) / kReduceRowChunks;
  ColsumJob j0{A, cols_a, lda, out_a, 0, (cols_a + 32 * V - 1) / (32 * V)};
  ColsumJob j1{B, cols_b, ldb, out_b, (int64_t)kReduceRowChunks * cols_a, (cols_b + 32 * V - 1) / (32 * V)};
  {
    LaunchTrace tr(st);
    colsum_partial_kernel<T><<<dim3(j0.col_blocks + j1.col_blocks, kReduceRowChunks), kReduceThreads, 0, st>>>(
        j0, j1, rows, scratch, rows_per_chunk);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  j0.col_blocks = (cols_a + 255) / 256;
  j1.col_blocks = (cols_b + 255) / 256;
  {
    LaunchTrace tr(st);
    colsum_final_kernel<<<j0.col_blocks + j1.col_blocks, 256, 0, st>>>(j0, j1, scratch, beta);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace osdp
