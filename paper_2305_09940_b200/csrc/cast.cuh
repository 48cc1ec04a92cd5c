// cast.cuh — last step of the ffn-axis split: the fp32 cross-slice accumulator of Y or dX
// becomes the storage-dtype output, plus the output bias for Y.  out[r, c] = T(acc[r, c] + bias[c]).
//
// HBM-bound: reads rows x cols fp32 once, writes rows x cols T once.  Each thread converts 8 consecutive columns
// (two 16-byte loads, one 16-byte store for bf16 / two for fp32); cols is a multiple of 8 (bf16) or 4 (fp32).
#pragma once
#include "common.cuh"

namespace osdp {

constexpr int kCastThreads = 256;

template <typename T, int V>
__global__ void __launch_bounds__(kCastThreads) acc_to_out_kernel(const float* __restrict__ acc, const T* __restrict__ bias,
                                                                  T* __restrict__ out, int64_t rows, int cols) {
  const int vec_per_row = cols / V;
  const int64_t total = rows * (int64_t)vec_per_row;
  for (int64_t i = (int64_t)blockIdx.x * kCastThreads + threadIdx.x; i < total; i += (int64_t)gridDim.x * kCastThreads) {
    const int c = (int)(i % vec_per_row) * V;
    const int64_t off = (i / vec_per_row) * (int64_t)cols + c;
    float v[V];
#pragma unroll
    for (int j = 0; j < V; j += 4) {
      const float4 x = *reinterpret_cast<const float4*>(acc + off + j);
      v[j] = x.x; v[j + 1] = x.y; v[j + 2] = x.z; v[j + 3] = x.w;
    }
    if (bias != nullptr) {
#pragma unroll
      for (int j = 0; j < V; ++j) v[j] += (float)bias[c + j];
    }
    if constexpr (sizeof(T) == 2) {
      uint4 o;
      uint32_t* w = reinterpret_cast<uint32_t*>(&o);
#pragma unroll
      for (int j = 0; j < V; j += 2) {
        const __nv_bfloat162 p = __floats2bfloat162_rn(v[j], v[j + 1]);
        w[j / 2] = *reinterpret_cast<const uint32_t*>(&p);
      }
      *reinterpret_cast<uint4*>(out + off) = o;
    } else {
      *reinterpret_cast<float4*>(out + off) = make_float4(v[0], v[1], v[2], v[3]);
    }
  }
}

// dtype-dispatched launch; grid = enough CTAs to fill the machine several times over, grid-stride inside.
inline int launch_acc_to_out(int dtype, const float* acc, const void* bias, void* out, int64_t rows, int cols, int sms,
                             cudaStream_t st) {
  const int64_t vecs = rows * (int64_t)(cols / (dtype == OSDP_BF16 ? 8 : 4));
  int64_t blocks = (vecs + kCastThreads - 1) / kCastThreads;
  const int64_t cap = (int64_t)sms * 16;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  {
    LaunchTrace tr(st);
    if (dtype == OSDP_BF16)
      acc_to_out_kernel<__nv_bfloat16, 8><<<(unsigned)blocks, kCastThreads, 0, st>>>(
          acc, (const __nv_bfloat16*)bias, (__nv_bfloat16*)out, rows, cols);
    else
      acc_to_out_kernel<float, 4><<<(unsigned)blocks, kCastThreads, 0, st>>>(acc, (const float*)bias, (float*)out, rows, cols);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace osdp
