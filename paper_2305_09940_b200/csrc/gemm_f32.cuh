// gemm_f32.cuh — fp32 path (config C1): exact-fp32 FFMA GEMM with the same fused epilogues.
//
// Why not tensor cores here: tcgen05 kind::tf32 keeps a 10-bit mantissa and cannot meet the fp32 config's
// 1e-4 relative bound with 1e-5 split-invariance (SURVEY.md §7 "fp32 config accuracy"); the fp32 config is
// 1.9 GFLOP, so exact-fp32 FFMA is the right tool.  The shapes are tiny (T_s = 128 rows per slice at C1), so the
// kernel is built for latency, not for bandwidth:
//   * 64 x 64 x 16 tiles, 256 threads, 4 x 4 outputs per thread, operands fetched with 16-byte loads along
//     whichever axis is contiguous in memory (both majornesses of both operands), two shared-memory stages with the
//     next tile's global loads in flight during the FFMAs (one __syncthreads per k-step);
//   * split-K inside a thread-block cluster: GEMMs with a long contraction (A2 / A7 at C1: 128 x 256 x 1024 = 8 output
//     tiles of 64 k-steps) run as clusters of up to 8 CTAs, each CTA takes a contiguous K range and CTA 0 adds the
//     partial tiles in rank order through distributed shared memory, then runs the epilogue.
// Determinism: the split count depends on K only (never on the slice's rows or columns), every partial is accumulated
// in ascending k and the partials are added in rank order, so results are bit-reproducible and Y / dX rows are
// bit-identical for every token split count k.
#pragma once
#include <cooperative_groups.h>

#include "common.cuh"
#include "epilogue_math.cuh"

namespace osdp {

constexpr int F32_BM = 64, F32_BN = 64, F32_BK = 16, F32_THREADS = 256, F32_PAD = 4, F32_MAX_SPLIT = 8;

struct StridedOperands {
  const float* A; int64_t a_sm, a_sk;   // A(m,k) = A[m*a_sm + k*a_sk]
  const float* B; int64_t b_sk, b_sn;   // B(k,n) = B[k*b_sk + n*b_sn]
};

// out[m, n .. n+3] for one thread's four consecutive columns (n + 3 < N is guaranteed by the caller; N % 4 == 0).
template <int EPI>
__device__ __forceinline__ void f32_epilogue_store4(const float (&acc)[4], int m, int n, const EpiParams& ep) {
  const int64_t o = (int64_t)m * ep.ldo + n;
  float4 r;
  float* v = reinterpret_cast<float*>(&r);
  if constexpr (EPI == EPI_BIAS_GELU || EPI == EPI_BIAS || EPI == EPI_BIAS_GELU_DUAL) {
    const float4 b = *reinterpret_cast<const float4*>((const float*)ep.bias + n);
    const float bb[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) v[j] = acc[j] + bb[j];
    if constexpr (EPI == EPI_BIAS_GELU_DUAL) *reinterpret_cast<float4*>((float*)ep.out0 + o) = r;
    if constexpr (EPI != EPI_BIAS) {
#pragma unroll
      for (int j = 0; j < 4; ++j) v[j] = gelu_fwd<true>(v[j]);
    }
    *reinterpret_cast<float4*>((float*)(EPI == EPI_BIAS_GELU_DUAL ? ep.out1 : ep.out0) + o) = r;
  } else if constexpr (EPI == EPI_DGELU) {
    const float4 z = *reinterpret_cast<const float4*>((const float*)ep.aux + o);
    const float zz[4] = {z.x, z.y, z.z, z.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) v[j] = acc[j] * gelu_bwd<true>(zz[j]);
    *reinterpret_cast<float4*>((float*)ep.out0 + o) = r;
  } else if constexpr (EPI == EPI_ACCUM_F32) {
    float4* p = reinterpret_cast<float4*>((float*)ep.out0 + o);
    if (ep.beta) {
      const float4 old = *p;
      r = make_float4(old.x + acc[0], old.y + acc[1], old.z + acc[2], old.w + acc[3]);
    } else {
      r = make_float4(acc[0], acc[1], acc[2], acc[3]);
    }
    *p = r;
  } else {
    *reinterpret_cast<float4*>((float*)ep.out0 + o) = make_float4(acc[0], acc[1], acc[2], acc[3]);
  }
}

template <int EPI>
__global__ void __launch_bounds__(F32_THREADS) gemm_f32_kernel(StridedOperands op, GemmShape s, EpiParams ep, int tiles_n,
                                                               int k_per_split) {
  namespace cg = cooperative_groups;
  constexpr int LDS = F32_BM + F32_PAD;                       // 68 floats: rows stay 16-byte aligned
  __shared__ __align__(16) float smem[2 * 2 * F32_BK * LDS];  // As[2][BK][LDS] | Bs[2][BK][LDS]; reused for the split-K partial
  float(*As)[F32_BK][LDS] = reinterpret_cast<float(*)[F32_BK][LDS]>(smem);
  float(*Bs)[F32_BK][LDS] = reinterpret_cast<float(*)[F32_BK][LDS]>(smem + 2 * F32_BK * LDS);
  static_assert(2 * 2 * F32_BK * LDS >= F32_BM * F32_BN, "split-K partial tile fits the operand stages");

  cg::cluster_group cluster = cg::this_cluster();
  const unsigned split = cluster.num_blocks(), rank = cluster.block_rank();
  const int tid = threadIdx.x;
  const int tile = blockIdx.x / split;
  const int m0 = (tile / tiles_n) * F32_BM, n0 = (tile % tiles_n) * F32_BN;
  const int k_begin = (int)rank * k_per_split, k_end = min(s.K, k_begin + k_per_split);
  const int ty = tid / 16, tx = tid % 16;
  const bool a_kmajor = (op.a_sk == 1), b_nmajor = (op.b_sn == 1);

  // One 16-byte load per operand per thread per k-step, along the contiguous axis.
  //   k-contiguous operand ([rows x K]): thread -> row tid / 4, k offset (tid % 4) * 4   (K % 4 == 0)
  //   mn-contiguous operand ([K x cols]): thread -> k row tid / 16, column (tid % 16) * 4 (cols % 4 == 0)
  const int a_r = a_kmajor ? tid / 4 : tid / 16, a_c = a_kmajor ? (tid % 4) * 4 : (tid % 16) * 4;
  const int b_r = b_nmajor ? tid / 16 : tid / 4, b_c = b_nmajor ? (tid % 16) * 4 : (tid % 4) * 4;
  float4 ra, rb;
  auto fetch = [&](int k0) {
    ra = rb = make_float4(0.f, 0.f, 0.f, 0.f);
    if (a_kmajor) {
      if (m0 + a_r < s.M && k0 + a_c < k_end) ra = *reinterpret_cast<const float4*>(op.A + (int64_t)(m0 + a_r) * op.a_sm + k0 + a_c);
    } else {
      if (k0 + a_r < k_end && m0 + a_c < s.M) ra = *reinterpret_cast<const float4*>(op.A + (int64_t)(k0 + a_r) * op.a_sk + m0 + a_c);
    }
    if (b_nmajor) {
      if (k0 + b_r < k_end && n0 + b_c < s.N) rb = *reinterpret_cast<const float4*>(op.B + (int64_t)(k0 + b_r) * op.b_sk + n0 + b_c);
    } else {
      if (n0 + b_r < s.N && k0 + b_c < k_end) rb = *reinterpret_cast<const float4*>(op.B + (int64_t)(n0 + b_r) * op.b_sn + k0 + b_c);
    }
  };
  auto stage = [&](int buf) {
    if (a_kmajor) {
      As[buf][a_c + 0][a_r] = ra.x; As[buf][a_c + 1][a_r] = ra.y; As[buf][a_c + 2][a_r] = ra.z; As[buf][a_c + 3][a_r] = ra.w;
    } else {
      *reinterpret_cast<float4*>(&As[buf][a_r][a_c]) = ra;
    }
    if (b_nmajor) {
      *reinterpret_cast<float4*>(&Bs[buf][b_r][b_c]) = rb;
    } else {
      Bs[buf][b_c + 0][b_r] = rb.x; Bs[buf][b_c + 1][b_r] = rb.y; Bs[buf][b_c + 2][b_r] = rb.z; Bs[buf][b_c + 3][b_r] = rb.w;
    }
  };

  // Programmatic dependent launch: the index arithmetic above overlapped the tail of the previous kernel of the stream;
  // from here on this kernel reads what that kernel wrote.  These launches are a few microseconds each and several CTAs
  // fit an SM, so the next kernel's CTAs are resident and waiting here when the previous grid completes.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  float acc[4][4] = {};
  int buf = 0;
  if (k_begin < k_end) {
    fetch(k_begin);
    stage(0);
  }
  __syncthreads();
  for (int k0 = k_begin; k0 < k_end; k0 += F32_BK) {
    const bool more = k0 + F32_BK < k_end;
    if (more) fetch(k0 + F32_BK);          // in flight during the FFMAs below
#pragma unroll
    for (int k = 0; k < F32_BK; ++k) {
      const float4 a4 = *reinterpret_cast<const float4*>(&As[buf][k][ty * 4]);
      const float4 b4 = *reinterpret_cast<const float4*>(&Bs[buf][k][tx * 4]);
      const float a[4] = {a4.x, a4.y, a4.z, a4.w}, b[4] = {b4.x, b4.y, b4.z, b4.w};
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fmaf(a[i], b[j], acc[i][j]);
    }
    if (more) stage(buf ^ 1);
    __syncthreads();
    buf ^= 1;
  }

  if (split > 1) {   // add the partial tiles of the cluster in rank order (distributed shared memory)
    float* part = smem;                                   // [BM][BN]; every thread is past the last read of As / Bs
    if (rank != 0) {
#pragma unroll
      for (int i = 0; i < 4; ++i)
        *reinterpret_cast<float4*>(part + (ty * 4 + i) * F32_BN + tx * 4) = make_float4(acc[i][0], acc[i][1], acc[i][2], acc[i][3]);
    }
    cluster.sync();
    if (rank == 0) {
      for (unsigned r = 1; r < split; ++r) {
        const float* remote = cluster.map_shared_rank(part, r);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const float4 p = *reinterpret_cast<const float4*>(remote + (ty * 4 + i) * F32_BN + tx * 4);
          acc[i][0] += p.x; acc[i][1] += p.y; acc[i][2] += p.z; acc[i][3] += p.w;
        }
      }
    }
    cluster.sync();                                       // nobody leaves while its partial may still be read
    if (rank != 0) return;
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i, n = n0 + tx * 4;
    if (m < s.M && n < s.N) f32_epilogue_store4<EPI>(acc[i], m, n, ep);
  }
}

// Split count of the contraction: a function of K ONLY (see the header note on determinism: every output element of
// every GEMM with this contraction length is summed in the same order, whatever the slice rows / slice columns are, so
// token slices leave Y / dX rows and ffn slices leave dW1 / dW2 / db1 bit-identical).  >= 8 k-steps per CTA.
inline int f32_split_k(const GemmShape& s) {
  const int iters = (s.K + F32_BK - 1) / F32_BK;
  int split = 1;
  while (split < F32_MAX_SPLIT && iters / (2 * split) >= 8) split *= 2;
  return split;
}

template <int EPI>
inline int launch_gemm_f32(const StridedOperands& op, const GemmShape& s, const EpiParams& ep, cudaStream_t st) {
  // 16-byte loads: the contiguous extent of every operand and of the output is a multiple of 4 floats
  const bool a_kmajor = op.a_sk == 1, b_nmajor = op.b_sn == 1;
  if ((a_kmajor ? s.K : s.M) % 4 || (b_nmajor ? s.N : s.K) % 4 || s.N % 4 || ep.ldo % 4) return OSDP_ERR_SHAPE;
  const int64_t tiles_m = (s.M + F32_BM - 1) / F32_BM, tiles_n = (s.N + F32_BN - 1) / F32_BN;
  const int split = f32_split_k(s);
  const int iters = (s.K + F32_BK - 1) / F32_BK;
  const int k_per_split = ((iters + split - 1) / split) * F32_BK;
  if (tiles_m * tiles_n * split > 0x7FFFFFFFll) return OSDP_ERR_SHAPE;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(tiles_m * tiles_n * split));
  cfg.blockDim = dim3(F32_THREADS);
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)split;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol in the kernel
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  cudaError_t err;
  {
    LaunchTrace tr(st);
    err = cudaLaunchKernelEx(&cfg, gemm_f32_kernel<EPI>, op, s, ep, (int)tiles_n, k_per_split);
  }
  OSDP_CUDA_TRY(err);
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace osdp
