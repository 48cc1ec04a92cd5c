// gemm_f32.cuh — fp32 path (config C1): plain FFMA tiled GEMM with the same fused epilogues.
//
// Why not tensor cores here: tcgen05 kind::tf32 keeps a 10-bit mantissa and cannot meet the fp32 config's
// 1e-4 relative bound with 1e-5 split-invariance (SURVEY.md §7 "fp32 config accuracy"); the fp32 config is
// 1.9 GFLOP, so exact-fp32 FFMA is the right tool.  Every output element is accumulated over k in ascending
// order by ONE thread, so Y/dX rows are bit-identical for every split count k.
#pragma once
#include "common.cuh"
#include "epilogue_math.cuh"

namespace osdp {

constexpr int F32_BM = 64, F32_BN = 64, F32_BK = 16, F32_THREADS = 256;

struct StridedOperands {
  const float* A; int64_t a_sm, a_sk;   // A(m,k) = A[m*a_sm + k*a_sk]
  const float* B; int64_t b_sk, b_sn;   // B(k,n) = B[k*b_sk + n*b_sn]
};

template <int EPI>
__device__ __forceinline__ void f32_epilogue_store(float acc, int m, int n, const EpiParams& ep) {
  const int64_t o = (int64_t)m * ep.ldo + n;
  if constexpr (EPI == EPI_BIAS_GELU) {
    ((float*)ep.out0)[o] = gelu_fwd<true>(acc + ((const float*)ep.bias)[n]);
  } else if constexpr (EPI == EPI_BIAS) {
    ((float*)ep.out0)[o] = acc + ((const float*)ep.bias)[n];
  } else if constexpr (EPI == EPI_BIAS_GELU_DUAL) {
    const float z = acc + ((const float*)ep.bias)[n];
    ((float*)ep.out0)[o] = z;
    ((float*)ep.out1)[o] = gelu_fwd<true>(z);
  } else if constexpr (EPI == EPI_DGELU) {
    const float z = ((const float*)ep.aux)[o];
    ((float*)ep.out0)[o] = acc * gelu_bwd<true>(z);
  } else if constexpr (EPI == EPI_ACCUM_F32) {
    float* p = (float*)ep.out0 + o;
    *p = ep.beta ? (*p + acc) : acc;
  } else {
    ((float*)ep.out0)[o] = acc;
  }
}

template <int EPI>
__global__ void __launch_bounds__(F32_THREADS) gemm_f32_kernel(StridedOperands op, GemmShape s, EpiParams ep) {
  __shared__ float As[F32_BK][F32_BM + 4];
  __shared__ float Bs[F32_BK][F32_BN + 4];
  const int tid = threadIdx.x;
  const int m0 = blockIdx.y * F32_BM, n0 = blockIdx.x * F32_BN;
  const int ty = tid / 16, tx = tid % 16;
  float acc[4][4] = {};
  const bool a_kcontig = (op.a_sk == 1), b_ncontig = (op.b_sn == 1);

  for (int k0 = 0; k0 < s.K; k0 += F32_BK) {
#pragma unroll
    for (int i = 0; i < (F32_BM * F32_BK) / F32_THREADS; ++i) {
      const int e = tid + i * F32_THREADS;
      const int m = a_kcontig ? e / F32_BK : e % F32_BM;
      const int k = a_kcontig ? e % F32_BK : e / F32_BM;
      const int gm = m0 + m, gk = k0 + k;
      As[k][m] = (gm < s.M && gk < s.K) ? op.A[(int64_t)gm * op.a_sm + (int64_t)gk * op.a_sk] : 0.0f;
    }
#pragma unroll
    for (int i = 0; i < (F32_BN * F32_BK) / F32_THREADS; ++i) {
      const int e = tid + i * F32_THREADS;
      const int n = b_ncontig ? e % F32_BN : e / F32_BK;
      const int k = b_ncontig ? e / F32_BN : e % F32_BK;
      const int gn = n0 + n, gk = k0 + k;
      Bs[k][n] = (gn < s.N && gk < s.K) ? op.B[(int64_t)gk * op.b_sk + (int64_t)gn * op.b_sn] : 0.0f;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < F32_BK; ++k) {
      float a[4], b[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[k][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) b[j] = Bs[k][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int m = m0 + ty * 4 + i, n = n0 + tx * 4 + j;
      if (m < s.M && n < s.N) f32_epilogue_store<EPI>(acc[i][j], m, n, ep);
    }
}

template <int EPI>
inline int launch_gemm_f32(const StridedOperands& op, const GemmShape& s, const EpiParams& ep, cudaStream_t st) {
  dim3 grid((s.N + F32_BN - 1) / F32_BN, (s.M + F32_BM - 1) / F32_BM);
  {
    LaunchTrace tr(st);
    gemm_f32_kernel<EPI><<<grid, F32_THREADS, 0, st>>>(op, s, ep);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace osdp
