// gemm_sm100.cuh — the bf16 slice GEMM of osdp-b200, hand-written for sm_100a.
//
//   C[M x N] = A[M x K] * B[K x N]   (bf16 x bf16 -> fp32 in TMEM), then a fused epilogue (common.cuh Epi).
//
// Structure (one persistent CTA per SM, 256 threads, warp-specialised):
//   warp 0      TMA producer: cp.async.bulk.tensor (128B-swizzled boxes) into a kStages-deep smem ring
//   warp 1      MMA issuer: one lane issues tcgen05.mma.cta_group::1.kind::f16 (128 x 256 x 16) from smem
//               descriptors into one of two 256-column TMEM accumulator stages; tcgen05.commit frees
//               smem slots and publishes finished accumulators
//   warp 2      TMEM allocator (512 columns) / deallocator
//   warps 4..7  epilogue: tcgen05.ld (32 lanes x 32 columns per warp), bias / GeLU / GeLU' / fp32
//               accumulate, 16-byte global stores; overlaps the next tile's main loop through the second
//               accumulator stage
// Three mbarrier pipelines: smem full/empty (TMA <-> MMA), TMEM full/empty (MMA <-> epilogue).
//
// Operand majorness: both K-major and MN-major operands are supported directly by
// the UMMA shared-memory descriptors, so the dW GEMMs (A = H_s^T, X_s^T; B = dY_s, dZ_s) need no transposes.
//   K-major tile  [rows x 64 k]      : one TMA box {64, rows};   smem rows of 128 B, 8-row swizzle atoms,
//                                      descriptor SBO = 1024 B, k-step of 16 elements = +32 B
//   MN-major tile [64 k x mn]        : mn/64 TMA boxes {64, 64}; each box 64 k-rows of 128 B (8 KiB),
//                                      descriptor LBO = 8192 B (next 64 mn), SBO = 1024 B (next 8 k), k-step = +2048 B
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "epilogue_math.cuh"

namespace osdp {
namespace sm100 {

constexpr int BLOCK_M = 128;
constexpr int BLOCK_N = 256;
constexpr int BLOCK_K = 64;
constexpr int UMMA_K = 16;
constexpr int kStages = 4;
constexpr int kAccStages = 2;
constexpr int kTmemCols = 512;
constexpr int kThreads = 256;
constexpr int kEpiWarp0 = 4;
constexpr int kNumEpiWarps = 4;
constexpr uint32_t kAStageBytes = BLOCK_M * BLOCK_K * 2;   // 16 KiB
constexpr uint32_t kBStageBytes = BLOCK_N * BLOCK_K * 2;   // 32 KiB
constexpr uint32_t kStageBytes = kAStageBytes + kBStageBytes;
constexpr uint32_t kSmemTiles = kStages * kStageBytes;     // 192 KiB
constexpr uint32_t kSmemBytes = kSmemTiles + 1024 /*align slack*/ + 256 /*barriers*/;
constexpr int kGroupM = 16;   // tile rasterisation: bands of 16 m-tiles, n walks across the band

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok;
}
__device__ __forceinline__ uint64_t global_timer_ns() {
  uint64_t t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
// Wait for the phase with the given parity to complete.  A pipeline bug must not hang the GPU: after ~20 s
// without progress the kernel traps (the launch then reports an error instead of wedging the device).
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  if (mbar_try_wait(bar, parity)) return;
  uint64_t t0 = 0;
  uint32_t spins = 0;
  while (!mbar_try_wait(bar, parity)) {
    if ((++spins & 0xFFFu) == 0) {
      const uint64_t now = global_timer_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > 20ull * 1000 * 1000 * 1000) __trap();
    }
  }
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c_inner, int c_outer) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c_inner), "r"(c_outer)
      : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"((uint64_t)map) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// D[tmem] (+)= A[smem desc] * B[smem desc]; accumulate = 0 overwrites D.
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// Arrive on an mbarrier when all tcgen05.mma issued so far by this thread have completed
// (implies tcgen05.fence::before_thread_sync).
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// 32 lanes x 32 consecutive fp32 columns: thread i of the warp gets row (lane base + i), v[j] = column j.
__device__ __forceinline__ void tmem_ld_32x32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
        "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
        "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
        "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// ------------------------------------------------------------------------------------------------ descriptors
// Shared-memory matrix descriptor (sm_100 format): start address >> 4 in bits [0,14), leading byte offset >> 4
// in [16,30), stride byte offset >> 4 in [32,46), descriptor version 1 in [46,48), layout type in [61,64)
// (2 = 128-byte swizzle).
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = (uint64_t)((saddr & 0x3FFFFu) >> 4);
  d |= (uint64_t)(lbo_bytes >> 4) << 16;
  d |= (uint64_t)(sbo_bytes >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
template <int MAJOR>
__device__ __forceinline__ uint64_t operand_desc(uint32_t tile_addr, int k16) {
  if constexpr (MAJOR == MAJOR_K) return make_smem_desc(tile_addr + k16 * (UMMA_K * 2), 0, 1024);
  else                            return make_smem_desc(tile_addr + k16 * (UMMA_K * 128), BLOCK_K * 128, 1024);
}
// Instruction descriptor for kind::f16: D = fp32 (bit 4), A = B = bf16 (bits 7, 10), A/B major (bits 15, 16;
// 1 = MN-major), N >> 3 in [17,23), M >> 4 in [24,29).
template <int A_MAJOR, int B_MAJOR>
__host__ __device__ constexpr uint32_t make_idesc() {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)A_MAJOR << 15) | ((uint32_t)B_MAJOR << 16) |
         ((uint32_t)(BLOCK_N >> 3) << 17) | ((uint32_t)(BLOCK_M >> 4) << 24);
}

// --------------------------------------------------------------------------------------------------- epilogue
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  const __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&p);
}
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

// One thread's 32 consecutive columns [n, n+32) of row `row` (valid when row_ok); groups of 8 columns are
// written only while n + 8 g < N (N is a multiple of 8).
template <int EPI>
__device__ __forceinline__ void epilogue_chunk(const uint32_t (&acc)[32], int64_t row, bool row_ok, int n, int N,
                                               const EpiParams& ep) {
#pragma unroll
  for (int g = 0; g < 4; ++g) {
    const int ng = n + 8 * g;
    if (ng >= N) break;   // warp-uniform
    float v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __uint_as_float(acc[8 * g + j]);

    if constexpr (EPI == EPI_BIAS_GELU || EPI == EPI_BIAS || EPI == EPI_BIAS_GELU_DUAL) {
      const uint4 b = __ldg(reinterpret_cast<const uint4*>((const __nv_bfloat16*)ep.bias + ng));
      const uint32_t bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        v[2 * j] += bf16_lo(bw[j]);
        v[2 * j + 1] += bf16_hi(bw[j]);
      }
    }
    if constexpr (EPI == EPI_ACCUM_F32) {
      if (row_ok) {
        float4* p = reinterpret_cast<float4*>((float*)ep.out0 + row * ep.ldo + ng);
        float4 lo = make_float4(v[0], v[1], v[2], v[3]), hi = make_float4(v[4], v[5], v[6], v[7]);
        if (ep.beta) {
          const float4 a = p[0], c = p[1];
          lo.x += a.x; lo.y += a.y; lo.z += a.z; lo.w += a.w;
          hi.x += c.x; hi.y += c.y; hi.z += c.z; hi.w += c.w;
        }
        p[0] = lo;
        p[1] = hi;
      }
    } else if constexpr (EPI == EPI_DGELU) {
      if (row_ok) {
        const int64_t o = row * ep.ldo + ng;
        const uint4 z = *reinterpret_cast<const uint4*>((const __nv_bfloat16*)ep.aux + o);
        const uint32_t zw[4] = {z.x, z.y, z.z, z.w};
        uint32_t w[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
          w[j] = pack_bf16x2(v[2 * j] * gelu_bwd<false>(bf16_lo(zw[j])), v[2 * j + 1] * gelu_bwd<false>(bf16_hi(zw[j])));
        *reinterpret_cast<uint4*>((__nv_bfloat16*)ep.out0 + o) = make_uint4(w[0], w[1], w[2], w[3]);
      }
    } else {
      if (row_ok) {
        const int64_t o = row * ep.ldo + ng;
        uint32_t w[4];
        if constexpr (EPI == EPI_BIAS_GELU_DUAL) {
#pragma unroll
          for (int j = 0; j < 4; ++j) w[j] = pack_bf16x2(v[2 * j], v[2 * j + 1]);
          *reinterpret_cast<uint4*>((__nv_bfloat16*)ep.out0 + o) = make_uint4(w[0], w[1], w[2], w[3]);
        }
        if constexpr (EPI == EPI_BIAS_GELU || EPI == EPI_BIAS_GELU_DUAL) {
#pragma unroll
          for (int j = 0; j < 8; ++j) v[j] = gelu_fwd<false>(v[j]);
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) w[j] = pack_bf16x2(v[2 * j], v[2 * j + 1]);
        __nv_bfloat16* dst = (EPI == EPI_BIAS_GELU_DUAL) ? (__nv_bfloat16*)ep.out1 : (__nv_bfloat16*)ep.out0;
        *reinterpret_cast<uint4*>(dst + o) = make_uint4(w[0], w[1], w[2], w[3]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------- the kernel
struct TileCoord {
  int m_blk, n_blk;
};
__device__ __forceinline__ TileCoord tile_coord(int t, int num_m, int num_n) {
  const int per_group = kGroupM * num_n;
  const int g = t / per_group;
  const int first_m = g * kGroupM;
  const int gsize = min(kGroupM, num_m - first_m);
  const int local = t - g * per_group;
  return {first_m + local % gsize, local / gsize};
}

template <int A_MAJOR, int B_MAJOR, int EPI>
__global__ void __launch_bounds__(kThreads, 1)
gemm_bf16_sm100_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b,
                       const GemmShape shape, const EpiParams ep) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // 128B swizzle atoms need 1024 B alignment
  const uint32_t smem_a = smem_base;
  const uint32_t smem_b = smem_base + kStages * kAStageBytes;
  const uint32_t bars = smem_base + kSmemTiles;
  const uint32_t full_bar = bars;                                  // [kStages]
  const uint32_t empty_bar = bars + 8 * kStages;                   // [kStages]
  const uint32_t tfull_bar = bars + 16 * kStages;                  // [kAccStages]
  const uint32_t tempty_bar = bars + 16 * kStages + 8 * kAccStages;   // [kAccStages]
  const uint32_t tmem_slot = bars + 16 * kStages + 16 * kAccStages;   // uint32
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const int num_m = (shape.M + BLOCK_M - 1) / BLOCK_M, num_n = (shape.N + BLOCK_N - 1) / BLOCK_N;
  const int num_tiles = num_m * num_n;
  const int num_kb = (shape.K + BLOCK_K - 1) / BLOCK_K;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmap_a);
    tma_prefetch_desc(&tmap_b);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kStages; ++i) {
      mbar_init(full_bar + 8 * i, 1);
      mbar_init(empty_bar + 8 * i, 1);
    }
    for (int i = 0; i < kAccStages; ++i) {
      mbar_init(tfull_bar + 8 * i, 1);
      mbar_init(tempty_bar + 8 * i, kNumEpiWarps);
    }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(tmem_slot, kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  if (warp == 0) {
    // ================================================================== TMA producer
    int stage = 0;
    uint32_t phase = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x) {
      const TileCoord tc = tile_coord(t, num_m, num_n);
      const int m0 = tc.m_blk * BLOCK_M, n0 = tc.n_blk * BLOCK_N;
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(empty_bar + 8 * stage, phase ^ 1);
        if (lane == 0) {
          const uint32_t fb = full_bar + 8 * stage;
          const uint32_t sa = smem_a + stage * kAStageBytes, sb = smem_b + stage * kBStageBytes;
          const int k0 = kb * BLOCK_K;
          mbar_expect_tx(fb, kStageBytes);
          if constexpr (A_MAJOR == MAJOR_K) {
            tma_load_2d(sa, &tmap_a, fb, k0, m0);
          } else {
#pragma unroll
            for (int c = 0; c < BLOCK_M / 64; ++c) tma_load_2d(sa + c * (BLOCK_K * 128), &tmap_a, fb, m0 + 64 * c, k0);
          }
          if constexpr (B_MAJOR == MAJOR_K) {
            tma_load_2d(sb, &tmap_b, fb, k0, n0);
          } else {
#pragma unroll
            for (int c = 0; c < BLOCK_N / 64; ++c) tma_load_2d(sb + c * (BLOCK_K * 128), &tmap_b, fb, n0 + 64 * c, k0);
          }
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp == 1) {
    // ================================================================== MMA issuer
    constexpr uint32_t idesc = make_idesc<A_MAJOR, B_MAJOR>();
    int stage = 0;
    uint32_t phase = 0;
    int it = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x, ++it) {
      const int as = it & 1;
      const uint32_t aphase = (it >> 1) & 1;
      mbar_wait(tempty_bar + 8 * as, aphase ^ 1);   // epilogue has drained this accumulator stage
      tc_fence_after();
      const uint32_t tmem_d = tmem_base + as * BLOCK_N;
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(full_bar + 8 * stage, phase);      // TMA bytes have landed
        tc_fence_after();
        if (lane == 0) {
          const uint32_t sa = smem_a + stage * kAStageBytes, sb = smem_b + stage * kBStageBytes;
#pragma unroll
          for (int k = 0; k < BLOCK_K / UMMA_K; ++k)
            umma_bf16(tmem_d, operand_desc<A_MAJOR>(sa, k), operand_desc<B_MAJOR>(sb, k), idesc, (kb | k) != 0);
          umma_commit(empty_bar + 8 * stage);        // smem slot free once these MMAs have read it
          if (kb == num_kb - 1) umma_commit(tfull_bar + 8 * as);   // accumulator complete
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp >= kEpiWarp0) {
    // ================================================================== epilogue
    const int q = warp % 4;   // TMEM lane quarter this warp may access
    int it = 0;
    for (int t = blockIdx.x; t < num_tiles; t += gridDim.x, ++it) {
      const TileCoord tc = tile_coord(t, num_m, num_n);
      const int as = it & 1;
      const uint32_t aphase = (it >> 1) & 1;
      const int64_t row = (int64_t)tc.m_blk * BLOCK_M + q * 32 + lane;
      const bool row_ok = row < shape.M;
      const int n0 = tc.n_blk * BLOCK_N;
      mbar_wait(tfull_bar + 8 * as, aphase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BLOCK_N;
#pragma unroll 1
      for (int c = 0; c < BLOCK_N / 32; ++c) {
        if (n0 + c * 32 >= shape.N) break;   // warp-uniform
        uint32_t acc[32];
        tmem_ld_32x32(taddr + c * 32, acc);
        tmem_ld_wait();
        epilogue_chunk<EPI>(acc, row, row_ok, n0 + c * 32, shape.N, ep);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(tempty_bar + 8 * as);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, kTmemCols);
  }
}

// ------------------------------------------------------------------------------------------------------ host
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn();   // osdp_api.cu: resolved through cudaGetDriverEntryPoint (no libcuda link)
int num_sms();                     // osdp_api.cu

// bf16 matrix stored row-major [outer x inner] with `ld` elements between rows; 128B-swizzled box.
inline int make_tmap(CUtensorMap* map, const void* ptr, int64_t inner, int64_t outer, int64_t ld, int box_inner,
                     int box_outer) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return OSDP_ERR_CUDA;
  const cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * 2};
  const cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    note_cuda_error(cudaErrorInvalidValue, "cuTensorMapEncodeTiled");
    return OSDP_ERR_CUDA;
  }
  return OSDP_OK;
}

// A, B: bf16 device pointers stored as common.cuh describes for the given majorness.
template <int A_MAJOR, int B_MAJOR, int EPI>
inline int launch_gemm_bf16(const void* A, int64_t lda, const void* B, int64_t ldb, const GemmShape& s,
                            const EpiParams& ep, cudaStream_t st) {
  CUtensorMap ta, tb;
  int rc;
  if (A_MAJOR == MAJOR_K) rc = make_tmap(&ta, A, s.K, s.M, lda, BLOCK_K, BLOCK_M);
  else                    rc = make_tmap(&ta, A, s.M, s.K, lda, 64, BLOCK_K);
  if (rc != OSDP_OK) return rc;
  if (B_MAJOR == MAJOR_K) rc = make_tmap(&tb, B, s.K, s.N, ldb, BLOCK_K, BLOCK_N);
  else                    rc = make_tmap(&tb, B, s.N, s.K, ldb, 64, BLOCK_K);
  if (rc != OSDP_OK) return rc;

  auto kernel = gemm_bf16_sm100_kernel<A_MAJOR, B_MAJOR, EPI>;
  static bool attr_set = false;   // one process per GPU: the attribute is per function per device
  if (!attr_set) {
    OSDP_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes));
    attr_set = true;
  }
  const int num_m = (s.M + BLOCK_M - 1) / BLOCK_M, num_n = (s.N + BLOCK_N - 1) / BLOCK_N;
  const int tiles = num_m * num_n;
  const int sms = num_sms();
  const int grid = tiles < sms ? tiles : sms;
  {
    LaunchTrace tr(st);
    kernel<<<grid, kThreads, kSmemBytes, st>>>(ta, tb, s, ep);
  }
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace sm100
}  // namespace osdp
