// reduce.cuh — A8 / db1: column sums of a [rows x cols] slice tensor into an fp32 vector.
//
// HBM-bound (reads the slice once).  Deterministic: fixed two-stage reduction order, no float atomics
// (SURVEY.md §7 "Deterministic accumulation").  Stage 1: grid (column blocks x kReduceRowChunks); every warp
// owns whole rows (lanes across 16-byte column vectors: coalesced), rows ascending, then the 8 warps of the
// CTA are summed in warp order through shared memory.  Stage 2: one thread per column sums the
// kReduceRowChunks partials in chunk order and adds to (beta = 1) or overwrites (beta = 0) the output.
#pragma once
#include "common.cuh"

namespace osdp {

constexpr int kReduceRowChunks = 32;   // scratch = kReduceRowChunks x max(h, f) floats (osdp.h, A10)
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

template <typename T>
__global__ void __launch_bounds__(kReduceThreads) colsum_partial_kernel(const T* __restrict__ src, int rows, int cols,
                                                                        int64_t ld, float* __restrict__ partial,
                                                                        int rows_per_chunk) {
  constexpr int V = VecOf<T>::N;
  constexpr int kWarps = kReduceThreads / 32;
  __shared__ float red[kWarps][32 * V];
  const int lane = threadIdx.x % 32, warp = threadIdx.x / 32;
  const int c = (blockIdx.x * 32 + lane) * V;
  const int r_begin = blockIdx.y * rows_per_chunk;
  const int r_end = min(rows, r_begin + rows_per_chunk);
  float acc[V];
#pragma unroll
  for (int i = 0; i < V; ++i) acc[i] = 0.0f;
  if (c < cols) {
    for (int r = r_begin + warp; r < r_end; r += kWarps) {
      float v[V];
      VecOf<T>::load(src + (int64_t)r * ld + c, v);
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
    const int col = blockIdx.x * 32 * V + j;
    if (col < cols) partial[(int64_t)blockIdx.y * cols + col] = s;
  }
}

__global__ void colsum_final_kernel(const float* __restrict__ partial, int cols, float* __restrict__ out, int beta) {
  const int col = blockIdx.x * blockDim.x + threadIdx.x;
  if (col >= cols) return;
  float s = 0.0f;
#pragma unroll 8
  for (int r = 0; r < kReduceRowChunks; ++r) s += partial[(int64_t)r * cols + col];
  out[col] = beta ? out[col] + s : s;
}

template <typename T>
inline int launch_colsum(const T* src, int rows, int cols, int64_t ld, float* scratch, float* out, int beta,
                         cudaStream_t st) {
  constexpr int V = VecOf<T>::N;
  const int rows_per_chunk = (rows + kReduceRowChunks - 1) / kReduceRowChunks;
  dim3 grid((cols + 32 * V - 1) / (32 * V), kReduceRowChunks);
  {
    LaunchTrace tr(st);
    colsum_partial_kernel<T><<<grid, kReduceThreads, 0, st>>>(src, rows, cols, ld, scratch, rows_per_chunk);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  {
    LaunchTrace tr(st);
    colsum_final_kernel<<<(cols + 255) / 256, 256, 0, st>>>(scratch, cols, out, beta);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace osdp
