// slice_sm100.cuh — one persistent kernel per SLICE of the token-split MLP (small slices).
//
// A slice of the operator-split MLP (slices "executed sequentially") is a short chain of GEMMs:
// forward A1 -> A2, backward (A3, A4) -> {A7, A5, A6}.  When a slice is small each GEMM is a fraction of a wave and a
// few microseconds of tensor time, and one launch per GEMM spends more time filling and draining the machine than
// computing.  This kernel runs ALL GEMMs of one slice in ONE launch: the tiles of every GEMM
// ("phase") form one list, CTA pairs claim tiles from it in order through a global counter, and a tile that reads
// another phase's output waits for exactly the producer tiles it needs (per-tile flags in global memory), so the
// machine drains once per slice and independent GEMMs (A7 | A5 | A6) fill each other's partial waves.
//
//   * Tile pipeline, warp roles, shared-memory ring, TMEM double buffering, epilogue math: those of the MT = 1
//     configuration of gemm_sm100.cuh (256 x 256 pair tiles, tcgen05.mma.cta_group::2, TMA loads / stores), with
//     operand majorness, epilogue kind and tile width (256 or 128 columns) read per phase at run time.
//   * A3 and A4 share their output tile grid and are ONE phase: a tile runs X_s W1 into TMEM accumulator 0 and
//     dY_s W2^T into accumulator 1, and one epilogue makes H_s and dZ_s from the same z (kEpiFusedA34 below).
//   * Tile claiming on demand (warp 3 of each pair's leader CTA: atomicAdd on the launch's tile counter when the
//     producer nears the end of its current tile; the index reaches both CTAs of the pair through a small shared-memory
//     queue): a tile only ever waits for tiles with a SMALLER list index, and those were claimed by pairs that are
//     already running.  So the kernel cannot deadlock however few of its CTAs are resident (two such launches on two
//     streams each holding SMs the other wants are fine), which a static tile-to-pair assignment could not promise,
//     and a pair inside a long tile does not sit on tiles the idle pairs could take.
//   * Publication: every epilogue warp waits for its TMA stores of the tile to complete (cp.async.bulk.wait_group 0)
//     and fences the async proxy, the 8 epilogue warps of the CTA meet at a named barrier, and one thread stores the
//     launch's EPOCH (release, gpu scope) into the tile's flag of this CTA; a tile is complete when both CTAs' flags
//     hold the epoch.  Consumers poll with ld.acquire.gpu, then fence.proxy.async before their TMA loads.  Flags and
//     the tile counter live at the end of the CALLER'S WORKSPACE (osdp_api.cu: slice_sync_words), which one call in
//     flight owns exclusively, so concurrent calls and concurrently replayed graphs never share them; the call zeroes
//     its words on its stream before the first launch (a memset node when captured).  The last pair to draw a
//     sentinel still puts the tile counter back to zero and the last CTA to leave clears the flags; the per-launch
//     epoch keeps the slices of one call apart.
//   * Forward slices pipeline: with room for two H_s buffers in the caller's workspace, slice s does not wait for
//     slice s - 1 (late_wait below), so its A1 tiles run beside the few long A2 tiles of the slice before.
//   * db1: the A6 tiles of the first tile row also add up the 32-row band sums that the fused epilogue left in the
//     scratch (bands in ascending order, one thread per column: the arithmetic of colsum_final_kernel).
//   * No remote mbarrier arrive is left unconsumed at exit, and the teardown is a release / acquire cluster barrier: a
//     remote arrive still in flight when the peer CTA has exited lands in the NEXT kernel's CTA on that SM (found the
//     hard way: a queue slot refilled before its slowest reader had read it).
// Results are bit-identical to the launch-per-GEMM path: same tile shape per output element, same ascending-k
// accumulation, same epilogue arithmetic, same db1 order (tests/test_gpu_slice_kernel.py).
#pragma once
#include <type_traits>

#include "gemm_sm100.cuh"

namespace osdp {
namespace sm100 {

constexpr int kSliceMaxPhases = 5;
constexpr int kSliceQueue = 4;              // tile indices a pair may hold ahead of its epilogue
constexpr int kSliceSyncWords = 32768;      // most words a call may take from the workspace: k x (kSliceFlags0 + 2 x publishing tiles of a slice)
constexpr unsigned int kPublishersPerTile = 2 * kNumEpiWarps;   // arrivals that hand a TMEM stage back
constexpr int kSliceFlags0 = 4;             // first flag word of a launch's part of the array
// A3 and A4 of the backward in one tile (they have the same output tile grid): accumulator 0 = X_s W1, accumulator 1 =
// dY_s W2^T; the epilogue forms z = acc0 + b1 once, stores H_s = gelu(z) (out1) and dZ_s = acc1 * gelu'(bf16(z)) (out0)
// and the 32-row band sums of dZ_s: the arithmetic of EPI_BIAS_GELU_DUAL followed by EPI_DGELU, without Z_s ever going
// to memory and without a tile-to-tile dependency.
constexpr int kEpiFusedA34 = 6;

// What a tile waits for before its first operand load (tiles of phase dep_phase, which precedes it in the list):
enum SliceDep : int {
  DEP_NONE = 0,
  DEP_ROW = 1,        // every tile of the same tile ROW (A operand = the producer's output rows: A2 <- A1, A7 <- A4)
  DEP_COL_AS_M = 2,   // every tile of producer COLUMN band = this tile's row band (A5: rows of dW2 are columns of H_s)
  DEP_COL_AS_N = 3    // every tile of producer COLUMN band = this tile's column band (A6: columns of dW1 are columns of dZ_s)
};

struct SlicePhase {
  int M, N, K;
  int a_major, b_major, epi;
  int bn;              // tile columns = UMMA N: 256, or 128 for long-K phases with few tiles (A2 / A7)
  int num_m, num_n;    // tile grid; tiles walk n fastest inside a tile row
  int tile_begin;      // list index of this phase's first tile
  int dep_kind, dep_phase;
  int publish;         // a later phase waits for this phase's tiles
  int db1;             // A6: tiles of tile row 0 also reduce the db1 band partials of their columns
  // Fused phase (epi == kEpiFusedA34): a tile runs TWO contractions into the two TMEM accumulator stages, first
  // A x B (K), then A2 x B2 (K2), and one epilogue combines them.  A2 / B2's tensor maps sit in phase slot `aux`.
  int fused, a2_major, b2_major, K2, aux;
  EpiParams ep;
};
struct SliceParams {
  int num_phases, total_tiles;
  int flag_tiles;      // tiles that have flags: list indices below this (the publishing phases come first in the list)
  unsigned int* sync;  // [0]: next list index to claim; [1]: pairs that have drawn their sentinel; [2]: CTAs that have left;
                       // [kSliceFlags0 + 2 t + r]: epoch once CTA r of the owning pair has published tile t
  unsigned int epoch;  // this launch's flag value (never 0; no two launches that can see the same flags share one)
  int late_wait;       // 1: this launch does not depend on the previous kernel of the stream (see the kernel)
  // db1 (+)= sum over bands of band[r * ld_band + c] (the A4 epilogue's 32-row band sums of dZ_s)
  const float* band;
  int64_t ld_band;
  float* db1;
  int bands, db1_beta;
  SlicePhase ph[kSliceMaxPhases];
};
struct SliceMaps {
  CUtensorMap m[kSliceMaxPhases][4];   // A, B, out0, out1 of each phase
};

// ------------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t mbar_try_wait_cluster(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
      "selp.u32 %0, 1, 0, p;\n"
      "}\n"
      : "=r"(ok)
      : "r"(bar), "r"(parity)
      : "memory");
  return ok;
}
// Wait (acquire at cluster scope: the data guarded by the barrier was written by the peer CTA).
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  if (mbar_try_wait_cluster(bar, parity)) return;
  uint64_t t0 = 0;
  uint32_t spins = 0;
  while (!mbar_try_wait_cluster(bar, parity)) {
    if ((++spins & 0xFFFu) == 0) {
      const uint64_t now = global_timer_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > 20ull * 1000 * 1000 * 1000) __trap();
    }
  }
}
__device__ __forceinline__ void mbar_arrive_release_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void st_shared_cluster_u32(uint32_t cluster_addr, uint32_t v) {
  asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(cluster_addr), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_shared_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned int* p, unsigned int x) {
  asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(x) : "memory");
}
__device__ __forceinline__ void epilogue_warps_sync() { asm volatile("bar.sync 1, 256;" ::: "memory"); }   // warps 4-11
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }

// The flag holds this launch's epoch.  A scheduling bug must not wedge the GPU: trap after ~20 s.
__device__ __forceinline__ void flag_wait(const unsigned int* f, unsigned int epoch) {
  if (ld_acquire_gpu(f) == epoch) return;
  uint64_t t0 = 0;
  uint32_t spins = 0;
  while (ld_acquire_gpu(f) != epoch) {
    __nanosleep(32);
    if ((++spins & 0x3FFu) == 0) {
      const uint64_t now = global_timer_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > 20ull * 1000 * 1000 * 1000) __trap();
    }
  }
}


__device__ __forceinline__ uint32_t make_idesc_rt(int a_major, int b_major, int bn) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_major << 15) | ((uint32_t)b_major << 16) |
         ((uint32_t)(bn >> 3) << 17) | ((uint32_t)(UMMA_M >> 4) << 24);
}
__device__ __forceinline__ uint64_t operand_desc_rt(int major, uint32_t tile_addr, int k16) {
  return major == MAJOR_K ? make_smem_desc(tile_addr + k16 * (UMMA_K * 2), 0, 1024)
                          : make_smem_desc(tile_addr + k16 * (UMMA_K * 128), BLOCK_K * 128, 1024);
}

struct SliceTile {
  int phase, m_blk, n_blk;
};
__device__ __forceinline__ SliceTile slice_tile(const SliceParams& P, int t) {
  int p = 0;
  while (p + 1 < P.num_phases && t >= P.ph[p + 1].tile_begin) ++p;
  const int local = t - P.ph[p].tile_begin;
  const int nn = P.ph[p].num_n;
  return {p, local / nn, local % nn};
}

// ------------------------------------------------------------------------------------------------- the kernel
__global__ void __launch_bounds__(kThreads, 1)
mlp_slice_kernel(const __grid_constant__ SliceMaps maps, const __grid_constant__ SliceParams P) {
  using Cfg = TileCfg<1, 1>;
  constexpr int kStages = Cfg::kStages;
  constexpr int kAccStages = 2;
  constexpr uint32_t kAStageBytes = Cfg::kAStageBytes;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t smem_a = smem_base;
  const uint32_t smem_b = smem_base + kStages * kAStageBytes;
  const uint32_t smem_store = smem_base + Cfg::kSmemTiles;
  const uint32_t bars = smem_store + Cfg::kSmemStore;
  const uint32_t full_bar = bars;                               // [kStages]    (pair leader)
  const uint32_t empty_bar = full_bar + 8 * kStages;            // [kStages]    (each CTA)
  const uint32_t tfull_bar = empty_bar + 8 * kStages;           // [kAccStages] (each CTA)
  const uint32_t tempty_bar = tfull_bar + 8 * kAccStages;       // [kAccStages] (pair leader)
  const uint32_t qfull_bar = tempty_bar + 8 * kAccStages;       // [kSliceQueue] (each CTA): slot holds a tile index
  const uint32_t qempty_bar = qfull_bar + 8 * kSliceQueue;      // [kSliceQueue] (pair leader): every reader has read it
  const uint32_t tile_q = qempty_bar + 8 * kSliceQueue;         // [kSliceQueue] uint32
  const uint32_t req_bar = tile_q + 4 * kSliceQueue;            // (pair leader): the producer wants its next tile
  const uint32_t tmem_slot = req_bar + 8;
  static_assert(16 * kStages + 16 * kAccStages + 20 * kSliceQueue + 8 + 4 <= 256, "barrier area");
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t rank = cluster_ctarank() & 1u;   // cluster = one pair
  const bool leader = rank == 0;
  // readers of a queue slot: producer warp + 8 epilogue warps in each CTA, and the leader's MMA warp
  constexpr uint32_t kQueueReaders = 2 * (1 + kNumEpiWarps) + 1;

  if (warp == 0 && lane == 0) {
    for (int p = 0; p < P.num_phases; ++p) {
      tma_prefetch_desc(&maps.m[p][0]);
      tma_prefetch_desc(&maps.m[p][1]);
      tma_prefetch_desc(&maps.m[p][2]);
      if (P.ph[p].epi == EPI_BIAS_GELU_DUAL || P.ph[p].fused) tma_prefetch_desc(&maps.m[p][3]);
      if (P.ph[p].fused) {
        tma_prefetch_desc(&maps.m[P.ph[p].aux][0]);
        tma_prefetch_desc(&maps.m[P.ph[p].aux][1]);
      }
    }
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kStages; ++i) {
      mbar_init(full_bar + 8 * i, 1);
      mbar_init(empty_bar + 8 * i, 1);
    }
    for (int i = 0; i < kAccStages; ++i) {
      mbar_init(tfull_bar + 8 * i, 1);
      mbar_init(tempty_bar + 8 * i, kPublishersPerTile);
    }
    for (int i = 0; i < kSliceQueue; ++i) {
      mbar_init(qfull_bar + 8 * i, 1);
      mbar_init(qempty_bar + 8 * i, kQueueReaders);
    }
    mbar_init(req_bar, 1);
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(tmem_slot, kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  cluster_sync();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  // Programmatic dependent launch.  Normally every thread waits for the previous kernel of the stream to complete
  // before it touches memory, and then lets the next kernel start its set-up.  late_wait (forward slices s > 0 when the
  // caller's workspace holds two H_s buffers): nothing this launch reads or writes is touched by the previous kernel
  // (slice s - 1 uses the other buffer, other rows of Y), and the kernel before that (slice s - 2, the last user of this
  // launch's buffer) had completed before the previous kernel let this one start.  So only one thread per CTA waits, off
  // the critical path, and only then lets the NEXT kernel (slice s + 1, which reuses slice s - 1's buffer) start: the
  // A1 tiles of this slice run beside the long-contraction A2 tiles of the previous one, which occupy few SMs.
  if (!P.late_wait) {
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  } else if (warp == 2) {
    if (lane == 0) {
      asm volatile("griddepcontrol.wait;" ::: "memory");
      asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    }
    __syncwarp();
  }

  unsigned int* const flags = P.sync + kSliceFlags0;   // two words per tile (one per CTA of the owning pair)
  const unsigned int epoch = P.epoch;
  const uint32_t qempty_leader = mapa(qempty_bar, 0);
  // Next list index of this pair (every reader warp calls this once per tile, in the same order).
  auto next_tile = [&](int it) -> int {
    const int slot = it % kSliceQueue;
    mbar_wait_cluster(qfull_bar + 8 * slot, (uint32_t)(it / kSliceQueue) & 1u);
    const int t = (int)ld_shared_u32(tile_q + 4 * slot);
    __syncwarp();
    // The sentinel's slot is never refilled, so nobody waits for it to be handed back: a remote arrive that nobody
    // consumes could still be in flight when the leader CTA has exited and land in the barriers of the NEXT kernel's CTA
    // on that SM (seen as a spurious arrival: a slot refilled before its slowest reader had read it).
    if (lane == 0 && t < P.total_tiles) mbar_arrive_cluster(qempty_leader + 8 * slot);
    return t;
  };
  // All producer tiles this tile reads have been published (whole warp; lanes share the polling).
  auto wait_deps = [&](const SlicePhase& S, const SliceTile& tl) {
    const SlicePhase& D = P.ph[S.dep_phase];
    const unsigned int* df = flags + 2 * D.tile_begin;
    if (S.dep_kind == DEP_ROW) {
      for (int i = lane; i < 2 * D.num_n; i += 32) flag_wait(df + 2 * (tl.m_blk * D.num_n) + i, epoch);
    } else {
      const int col = S.dep_kind == DEP_COL_AS_M ? tl.m_blk : tl.n_blk;
      for (int i = lane; i < 2 * D.num_m; i += 32) flag_wait(df + 2 * ((i >> 1) * D.num_n + col) + (i & 1), epoch);
    }
    __syncwarp();
  };

  if (warp == 3) {
    // ================================================================== tile scheduler (pair leader)
    // The whole warp stays in the loop (lane 0 works): the cluster barrier at the end of the kernel is .aligned.
    if (leader) {
      const uint32_t qfull_own = mapa(qfull_bar, 0), qfull_peer = mapa(qfull_bar, 1);
      const uint32_t tq_peer = mapa(tile_q, 1);
      for (int it = 0;; ++it) {
        const int slot = it % kSliceQueue;
        // Claim on demand: tile it + 1 is drawn when the producer is close to the end of tile it's loads (the claim's
        // latency hides behind the shared-memory ring), not as far ahead as the queue has room: tiles claimed early are
        // tiles other pairs cannot take, and a pair in a long tile would sit on work the idle ones should do.
        if (it > 0) mbar_wait(req_bar, (uint32_t)(it - 1) & 1u);
        mbar_wait(qempty_bar + 8 * slot, ((uint32_t)(it / kSliceQueue) & 1u) ^ 1u);
        unsigned int t = 0;
        if (lane == 0) {
          t = atomicAdd(P.sync, 1u);
          asm volatile("st.shared.u32 [%0], %1;" ::"r"(tile_q + 4 * slot), "r"(t) : "memory");
          st_shared_cluster_u32(tq_peer + 4 * slot, t);
          mbar_arrive_release_cluster(qfull_own + 8 * slot);
          mbar_arrive_release_cluster(qfull_peer + 8 * slot);
        }
        t = __shfl_sync(0xFFFFFFFFu, t, 0);
        if (t >= (unsigned int)P.total_tiles) break;   // the sentinel: every reader leaves its loop
      }
      // Every pair of the grid draws exactly one sentinel, and that is its last access to the tile counter: the last
      // pair to get here leaves both counters at zero for the next launch that uses this part of the array.
      if (lane == 0 && atomicAdd(P.sync + 1, 1u) == gridDim.x / 2 - 1) {
        P.sync[0] = 0u;
        P.sync[1] = 0u;
      }
      __syncwarp();
    }
  } else if (warp == 0) {
    // ================================================================== TMA producer (both CTAs)
    constexpr uint64_t pol = kEvictNormal;
    int stage = 0;
    uint32_t phase = 0;
    for (int it = 0;; ++it) {
      const int t = next_tile(it);
      if (t >= P.total_tiles) break;
      const SliceTile tl = slice_tile(P, t);
      const SlicePhase& S = P.ph[tl.phase];
      const CUtensorMap* map_a = &maps.m[tl.phase][0];
      const CUtensorMap* map_b = &maps.m[tl.phase][1];
      if (S.dep_kind != DEP_NONE) {
        wait_deps(S, tl);
        fence_proxy_async_global();   // what the producers' TMA stores wrote -> visible to this thread's TMA loads
      }
      const int half_n = S.bn / 2;
      const int m0 = tl.m_blk * UMMA_M + (int)rank * BLOCK_M;
      const int n0 = tl.n_blk * S.bn + (int)rank * half_n;
      const uint32_t tx_bytes = 2u * (kAStageBytes + (uint32_t)half_n * (BLOCK_K * 2));
      const int nseg = S.fused ? 2 : 1;
      for (int seg = 0; seg < nseg; ++seg) {
      const int a_major = seg ? S.a2_major : S.a_major, b_major = seg ? S.b2_major : S.b_major;
      if (seg) {
        map_a = &maps.m[S.aux][0];
        map_b = &maps.m[S.aux][1];
      }
      const int num_kb = ((seg ? S.K2 : S.K) + BLOCK_K - 1) / BLOCK_K;
      // when to ask for the next tile: a ring's worth of k-blocks before the end of this tile's loads
      const int req_kb = seg + 1 < nseg ? -1 : (num_kb > kStages + 2 ? num_kb - (kStages + 2) : 0);
      for (int kb = 0; kb < num_kb; ++kb) {
        if (kb == req_kb && leader && lane == 0) mbar_arrive(req_bar);
        mbar_wait(empty_bar + 8 * stage, phase ^ 1);
        if (lane == 0) {
          const uint32_t fb_local = full_bar + 8 * stage;
          const uint32_t fb = mapa(fb_local, 0);
          const uint32_t sa = smem_a + stage * kAStageBytes, sb = smem_b + stage * kBStageBytes;
          const int k0 = kb * BLOCK_K;
          if (leader) mbar_expect_tx(fb_local, tx_bytes);
          if (a_major == MAJOR_K) {
            tma_load_2d(sa, map_a, fb, k0, m0, pol);
          } else {
#pragma unroll
            for (int c = 0; c < BLOCK_M / 64; ++c) tma_load_2d(sa + c * (BLOCK_K * 128), map_a, fb, m0 + 64 * c, k0, pol);
          }
          if (b_major == MAJOR_K) {
            tma_load_2d(sb, map_b, fb, k0, n0, pol);
          } else {
            for (int c = 0; c < half_n / 64; ++c) tma_load_2d(sb + c * (BLOCK_K * 128), map_b, fb, n0 + 64 * c, k0, pol);
          }
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
      }   // seg
    }
  } else if (warp == 1) {
    // ================================================================== MMA issuer (pair leader)
    if (leader) {
      int stage = 0;
      uint32_t phase = 0;
      uint32_t acc = 0;   // accumulator stages handed out so far (a fused tile takes two)
      for (int it = 0;; ++it) {
        const int t = next_tile(it);
        if (t >= P.total_tiles) break;
        const SliceTile tl = slice_tile(P, t);
        const SlicePhase& S = P.ph[tl.phase];
        const int nseg = S.fused ? 2 : 1;
        for (int seg = 0; seg < nseg; ++seg, ++acc) {
        const int a_major = seg ? S.a2_major : S.a_major, b_major = seg ? S.b2_major : S.b_major;
        const uint32_t idesc = make_idesc_rt(a_major, b_major, S.bn);
        const int num_kb = ((seg ? S.K2 : S.K) + BLOCK_K - 1) / BLOCK_K;
        const int as = (int)(acc % kAccStages);
        mbar_wait(tempty_bar + 8 * as, ((acc / kAccStages) & 1u) ^ 1u);
        tc_fence_after();
        const uint32_t tmem_d = tmem_base + as * BLOCK_N;
        for (int kb = 0; kb < num_kb; ++kb) {
          mbar_wait(full_bar + 8 * stage, phase);
          tc_fence_after();
          if (lane == 0) {
            const uint32_t sa = smem_a + stage * kAStageBytes, sb = smem_b + stage * kBStageBytes;
#pragma unroll
            for (int k = 0; k < BLOCK_K / UMMA_K; ++k)
              umma_bf16(tmem_d, operand_desc_rt(a_major, sa, k), operand_desc_rt(b_major, sb, k), idesc, (kb | k) != 0);
            umma_commit(empty_bar + 8 * stage, (uint16_t)3);
            if (kb == num_kb - 1) umma_commit(tfull_bar + 8 * as, (uint16_t)3);
          }
          __syncwarp();
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        }   // seg
      }
    }
  } else if (warp >= kEpiWarp0) {
    // ================================================================== epilogue (both CTAs, own rows)
    const int q = warp % 4;
    const int cg = (warp - kEpiWarp0) / 4;
    StorePipe<1> pipe{smem_store + (uint32_t)(warp - kEpiWarp0) * kStoreBufBytes, lane};
    const uint32_t tempty_leader = mapa(tempty_bar, 0);
    uint32_t acc_used = 0;   // accumulator stages consumed so far (mirrors the MMA warp's count)
    for (int it = 0;; ++it) {
      const int t = next_tile(it);
      if (t >= P.total_tiles) break;
      const SliceTile tl = slice_tile(P, t);
      const SlicePhase& S = P.ph[tl.phase];
      const CUtensorMap* map0 = &maps.m[tl.phase][2];
      const CUtensorMap* map1 = &maps.m[tl.phase][3];
      const EpiParams& ep = S.ep;
      const int as = (int)(acc_used % kAccStages);
      const uint32_t aphase = (acc_used / kAccStages) & 1u;
      acc_used += S.fused ? 2u : 1u;
      const int M = S.M, N = S.N;
      const int n0 = tl.n_blk * S.bn;
      const int n_end = min(n0 + S.bn, N);
      const int row0 = tl.m_blk * UMMA_M + (int)rank * BLOCK_M + q * 32;   // this warp's 32-row band
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BLOCK_N;

      // ---- one contraction per tile: bias + GeLU (A1), bias (A2), plain (A7), fp32 store / reduce-add (A5, A6)
      auto run = [&](auto tag) {
        constexpr int EPI = decltype(tag)::value;
        using Tr = EpiTraits<EPI>;
        constexpr int kChunk = Tr::kChunkCols;
        constexpr bool kHasBias = (EPI == EPI_BIAS_GELU || EPI == EPI_BIAS);
        uint32_t bias_reg[2] = {0u, 0u};
        if constexpr (kHasBias) {
          const __nv_bfloat16* bias = reinterpret_cast<const __nv_bfloat16*>(ep.bias);
#pragma unroll
          for (int ci = 0; ci < 2; ++ci) {
            const int c = n0 + (cg + 2 * ci) * 64 + 2 * lane;
            bias_reg[ci] = c < N ? __ldg(reinterpret_cast<const uint32_t*>(bias + c)) : 0u;
          }
        }
        auto load8 = [&](const uint32_t* a, uint32_t bias_cur, int j, float (&v)[8]) {
#pragma unroll
          for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(a[i]);
          if constexpr (kHasBias) {
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              const uint32_t bw = __shfl_sync(0xFFFFFFFFu, bias_cur, 4 * j + i);
              v[2 * i] += bf16_lo(bw);
              v[2 * i + 1] += bf16_hi(bw);
            }
          }
        };
        auto pack8 = [](const float (&v)[8]) {
          return make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]), pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
        };
        if constexpr (Tr::kF32Out) {   // short slices: ask L2 for the old dW tile while the main loop runs (gemm_sm100.cuh)
          if (ep.beta != 0 && S.K <= kPrefetchMaxK && lane == 0 && row0 < M) {
            for (int n = n0 + cg * kChunk; n < n_end; n += 2 * kChunk) tma_prefetch_l2_2d(map0, n, row0);
          }
        }
        mbar_wait(tfull_bar + 8 * as, aphase);
        tc_fence_after();
        bool released = false;
        if (row0 < M) {
#pragma unroll 1
          for (int n = n0 + cg * kChunk; n < n_end; n += 2 * kChunk) {
            uint32_t acc[kChunk];
#pragma unroll
            for (int i = 0; i < kChunk / 32; ++i)
              tmem_ld_32x32(taddr + (n - n0) + 32 * i, *reinterpret_cast<uint32_t(*)[32]>(&acc[32 * i]));
            tmem_ld_wait();
            if (n + 2 * kChunk >= n_end) {   // this warp's last read of the accumulator stage
              tc_fence_before();
              __syncwarp();
              if (lane == 0) mbar_arrive_cluster(tempty_leader + 8 * as);
              released = true;
            }
            [[maybe_unused]] const uint32_t bias_cur = (n - n0) >= 2 * kChunk ? bias_reg[1] : bias_reg[0];
            pipe.begin();
            if constexpr (Tr::kF32Out) {
#pragma unroll
              for (int j = 0; j < 8; ++j) pipe.put(j, make_uint4(acc[4 * j], acc[4 * j + 1], acc[4 * j + 2], acc[4 * j + 3]));
              pipe.commit(map0, n, row0, ep.beta != 0);
            } else {
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                float v[8];
                load8(&acc[8 * j], bias_cur, j, v);
                if constexpr (EPI == EPI_BIAS_GELU) {
#pragma unroll
                  for (int i = 0; i < 8; ++i) v[i] = gelu_fwd<false>(v[i]);
                }
                pipe.put(j, pack8(v));
              }
              pipe.commit(map0, n, row0, false);
            }
          }
        }
        if (!released) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) mbar_arrive_cluster(tempty_leader + 8 * as);
        }
      };

      // ---- fused A3 + A4 tile: accumulator 0 in stage `as`, accumulator 1 in the other stage
      auto run_fused = [&]() {
        const int as1 = as ^ 1;
        const uint32_t aphase1 = ((acc_used - 1u) / kAccStages) & 1u;
        const uint32_t taddr1 = tmem_base + ((uint32_t)(q * 32) << 16) + as1 * BLOCK_N;
        const __nv_bfloat16* bias = reinterpret_cast<const __nv_bfloat16*>(ep.bias);
        uint32_t bias_reg[2];
#pragma unroll
        for (int ci = 0; ci < 2; ++ci) {
          const int c = n0 + (cg + 2 * ci) * 64 + 2 * lane;
          bias_reg[ci] = c < N ? __ldg(reinterpret_cast<const uint32_t*>(bias + c)) : 0u;
        }
        // z (fp32) = accumulator 0 + b1 for 8 consecutive columns; j = index of the 8-column group inside the chunk
        auto z8 = [&](const uint32_t* a, uint32_t bias_cur, int j, float (&v)[8]) {
#pragma unroll
          for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(a[i]);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            const uint32_t bw = __shfl_sync(0xFFFFFFFFu, bias_cur, 4 * j + i);
            v[2 * i] += bf16_lo(bw);
            v[2 * i + 1] += bf16_hi(bw);
          }
        };
        auto pack8 = [](const float (&v)[8]) {
          return make_uint4(pack_bf16x2(v[0], v[1]), pack_bf16x2(v[2], v[3]), pack_bf16x2(v[4], v[5]), pack_bf16x2(v[6], v[7]));
        };
        // pass 1 (needs only X_s W1, which finishes first): H_s = gelu(z)
        mbar_wait(tfull_bar + 8 * as, aphase);
        tc_fence_after();
        if (row0 < M) {
#pragma unroll 1
          for (int n = n0 + cg * 64; n < n_end; n += 128) {
            uint32_t a0[64];
            tmem_ld_32x32(taddr + (n - n0), *reinterpret_cast<uint32_t(*)[32]>(&a0[0]));
            tmem_ld_32x32(taddr + (n - n0) + 32, *reinterpret_cast<uint32_t(*)[32]>(&a0[32]));
            tmem_ld_wait();
            const uint32_t bias_cur = (n - n0) >= 128 ? bias_reg[1] : bias_reg[0];
            pipe.begin();
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              float v[8];
              z8(&a0[8 * j], bias_cur, j, v);
#pragma unroll
              for (int i = 0; i < 8; ++i) v[i] = gelu_fwd<false>(v[i]);
              pipe.put(j, pack8(v));
            }
            pipe.commit(map1, n, row0, false);
          }
        }
        // pass 2: dZ_s = (dY_s W2^T) * gelu'(Z_s), Z_s = z rounded to bf16 exactly as EPI_BIAS_GELU_DUAL would store it
        mbar_wait(tfull_bar + 8 * as1, aphase1);
        tc_fence_after();
        bool released = false;
        if (row0 < M) {
#pragma unroll 1
          for (int n = n0 + cg * 64; n < n_end; n += 128) {
            const uint32_t bias_cur = (n - n0) >= 128 ? bias_reg[1] : bias_reg[0];
            pipe.begin();
#pragma unroll
            for (int half = 0; half < 2; ++half) {
              uint32_t a0[32], a1[32];
              tmem_ld_32x32(taddr + (n - n0) + 32 * half, a0);
              tmem_ld_32x32(taddr1 + (n - n0) + 32 * half, a1);
              tmem_ld_wait();
              if (half == 1 && n + 128 >= n_end) {   // this warp's last read of both accumulator stages
                tc_fence_before();
                __syncwarp();
                if (lane == 0) {
                  mbar_arrive_cluster(tempty_leader + 8 * as);
                  mbar_arrive_cluster(tempty_leader + 8 * as1);
                }
                released = true;
              }
#pragma unroll
              for (int jj = 0; jj < 4; ++jj) {
                const int j = 4 * half + jj;
                float z[8], d[8];
                z8(&a0[8 * jj], bias_cur, j, z);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  const uint32_t zw = pack_bf16x2(z[2 * i], z[2 * i + 1]);
                  d[2 * i] = __uint_as_float(a1[8 * jj + 2 * i]) * gelu_bwd<false>(bf16_lo(zw));
                  d[2 * i + 1] = __uint_as_float(a1[8 * jj + 2 * i + 1]) * gelu_bwd<false>(bf16_hi(zw));
                }
                pipe.put(j, pack8(d));
              }
            }
            pipe.commit(map0, n, row0, false);
            if (ep.colsum != nullptr) {   // db1 band sums from the staged bf16 values (step A4)
              const uint32_t src = pipe.committed_buf() + ((lane & 3) << 2);
              float s0 = 0.0f, s1 = 0.0f;
#pragma unroll
              for (int r = 0; r < 32; ++r) {
                uint32_t w;
                asm volatile("ld.shared.b32 %0, [%1];" : "=r"(w) : "r"(src + r * 128 + ((((uint32_t)lane >> 2) ^ (r & 7)) << 4)));
                s0 += bf16_lo(w);
                s1 += bf16_hi(w);
              }
              const int c = n + 2 * lane;
              if (c < N) *reinterpret_cast<float2*>(ep.colsum + (int64_t)(row0 >> 5) * ep.ld_colsum + c) = make_float2(s0, s1);
            }
          }
        }
        if (!released) {
          tc_fence_before();
          __syncwarp();
          if (lane == 0) {
            mbar_arrive_cluster(tempty_leader + 8 * as);
            mbar_arrive_cluster(tempty_leader + 8 * as1);
          }
        }
      };
      switch (S.epi) {
        case kEpiFusedA34: run_fused(); break;
        case EPI_BIAS_GELU: run(std::integral_constant<int, EPI_BIAS_GELU>{}); break;
        case EPI_BIAS: run(std::integral_constant<int, EPI_BIAS>{}); break;
        case EPI_ACCUM_F32: run(std::integral_constant<int, EPI_ACCUM_F32>{}); break;
        default: run(std::integral_constant<int, EPI_PLAIN>{}); break;
      }
      if (S.publish) {   // this CTA's part of the tile is in global memory: let the consumers go
        if (lane == 0) {
          bulk_wait<0>();
          fence_proxy_async_global();
        }
        __syncwarp();
        epilogue_warps_sync();   // all 8 epilogue warps: TMA stores complete, band-sum stores (A4) issued
        if (warp == kEpiWarp0 && lane == 0) st_release_gpu(flags + 2 * t + (int)rank, epoch);
      }
      if (S.db1 && tl.m_blk == 0 && rank == 0) {
        // db1 (+)= colsum(dZ_s) for this tile's columns: the A4 tiles of this column band are complete (the producer
        // warp waited for them; this warp acquires them itself before reading the band sums), bands in ascending order.
        const SlicePhase& D = P.ph[S.dep_phase];
        for (int i = lane; i < 2 * D.num_m; i += 32)
          flag_wait(flags + 2 * (D.tile_begin + (i >> 1) * D.num_n + tl.n_blk) + (i & 1), epoch);
        __syncwarp();
        const int c = n0 + (warp - kEpiWarp0) * 32 + lane;
        if (c < n_end) {
          float s = 0.0f;
#pragma unroll 8
          for (int r = 0; r < P.bands; ++r) s += __ldcg(P.band + (int64_t)r * P.ld_band + c);
          P.db1[c] = P.db1_beta ? P.db1[c] + s : s;
        }
      }
    }
    if (lane == 0) bulk_wait<0>();
    __syncwarp();
  }

  // Release / acquire (not the relaxed rendezvous of gemm_sm100.cuh): the epilogue warps' last remote arrivals on the
  // leader's TMEM-empty barriers have nobody waiting for them, and they must have landed before the leader may exit.
  tc_fence_before();
  cluster_sync();
  if (warp == 2) {
    tc_fence_after();
    tmem_dealloc(tmem_base, kTmemCols);
    // The last CTA of the grid to get here (every role of every CTA has finished: nobody polls a flag any more) clears
    // the launch's flags, so the same launch can be replayed from a CUDA graph (same epoch) or its part of the array be
    // handed to a later launch.
    unsigned int last = 0;
    if (lane == 0) last = atomicAdd(P.sync + 2, 1u) == gridDim.x - 1 ? 1u : 0u;
    if (__shfl_sync(0xFFFFFFFFu, last, 0)) {
      for (int i = lane; i < 2 * P.flag_tiles; i += 32) flags[i] = 0u;
      if (lane == 0) P.sync[2] = 0u;
    }
  }
}

// ------------------------------------------------------------------------------------------------------ host
struct SliceGemm {   // one phase as the scheduler states it (operands as in launch_gemm_bf16)
  const void* A;
  int64_t lda;
  const void* B;
  int64_t ldb;
  int a_major, b_major, epi;
  GemmShape s;
  EpiParams ep;
  int dep_kind, dep_phase;
  int bn;        // 256 or 128
  int publish;
  int db1;
  // fused phase (epi == kEpiFusedA34): the second contraction A2 [M x K2] x B2 [K2 x N]
  const void* A2 = nullptr;
  int64_t lda2 = 0;
  const void* B2 = nullptr;
  int64_t ldb2 = 0;
  int a2_major = 0, b2_major = 0, K2 = 0;
};
struct SliceDb1 {
  const float* band;
  int64_t ld_band;
  float* db1;
  int bands, beta;
};

inline int slice_tiles(const GemmShape& s, int bn) { return ((s.M + UMMA_M - 1) / UMMA_M) * ((s.N + bn - 1) / bn); }

// Epoch of a call's first launch (launch s uses epoch + s): consecutive, never 0, never wrapping inside a call.
inline unsigned int slice_epochs(int launches) {
  static std::atomic<uint64_t> epoch_seq{0};
  return (unsigned int)(epoch_seq.fetch_add((uint64_t)launches) % 0xF0000000ull) + 1u;
}

inline int launch_mlp_slice(const SliceGemm* g, int n, unsigned int* sync, unsigned int epoch, const SliceDb1* db1,
                            bool late_wait, cudaStream_t st) {
  using Cfg = TileCfg<1, 1>;
  if (n < 1 || n > kSliceMaxPhases) return OSDP_ERR_ARG;
  SliceMaps maps;
  SliceParams P = {};
  P.num_phases = n;
  P.sync = sync;
  P.epoch = epoch;
  P.late_wait = late_wait ? 1 : 0;
  if (db1) {
    P.band = db1->band;
    P.ld_band = db1->ld_band;
    P.db1 = db1->db1;
    P.bands = db1->bands;
    P.db1_beta = db1->beta;
  }
  int tiles = 0;
  for (int p = 0; p < n; ++p) {
    const SliceGemm& G = g[p];
    SlicePhase& S = P.ph[p];
    S.M = G.s.M; S.N = G.s.N; S.K = G.s.K;
    S.a_major = G.a_major; S.b_major = G.b_major; S.epi = G.epi;
    S.bn = G.bn;
    S.num_m = (G.s.M + UMMA_M - 1) / UMMA_M;
    S.num_n = (G.s.N + G.bn - 1) / G.bn;
    S.tile_begin = tiles;
    S.dep_kind = G.dep_kind; S.dep_phase = G.dep_phase;
    S.publish = G.publish; S.db1 = G.db1;
    S.fused = G.epi == kEpiFusedA34 ? 1 : 0;
    S.ep = G.ep;
    tiles += S.num_m * S.num_n;
    if (G.publish) {
      if (P.flag_tiles != S.tile_begin) return OSDP_ERR_ARG;   // publishing phases must lead the list
      P.flag_tiles = tiles;
    }
    int rc;
    if (G.a_major == MAJOR_K) rc = make_tmap(&maps.m[p][0], G.A, G.s.K, G.s.M, G.lda, BLOCK_K, BLOCK_M);
    else                      rc = make_tmap(&maps.m[p][0], G.A, G.s.M, G.s.K, G.lda, 64, BLOCK_K);
    if (rc != OSDP_OK) return rc;
    if (G.b_major == MAJOR_K) rc = make_tmap(&maps.m[p][1], G.B, G.s.K, G.s.N, G.ldb, BLOCK_K, G.bn / 2);
    else                      rc = make_tmap(&maps.m[p][1], G.B, G.s.N, G.s.K, G.ldb, 64, BLOCK_K);
    if (rc != OSDP_OK) return rc;
    const bool f32out = G.epi == EPI_ACCUM_F32;
    rc = make_tmap(&maps.m[p][2], G.ep.out0, G.s.N, G.s.M, G.ep.ldo, f32out ? 32 : 64, 32, f32out);
    if (rc != OSDP_OK) return rc;
    maps.m[p][3] = maps.m[p][2];
    if (S.fused) {   // the second contraction's operand maps go to the first phase slot this launch does not use
      if (n >= kSliceMaxPhases || G.bn != BLOCK_N) return OSDP_ERR_ARG;
      S.a2_major = G.a2_major; S.b2_major = G.b2_major; S.K2 = G.K2; S.aux = n;
      if (G.a2_major == MAJOR_K) rc = make_tmap(&maps.m[n][0], G.A2, G.K2, G.s.M, G.lda2, BLOCK_K, BLOCK_M);
      else                       rc = make_tmap(&maps.m[n][0], G.A2, G.s.M, G.K2, G.lda2, 64, BLOCK_K);
      if (rc != OSDP_OK) return rc;
      if (G.b2_major == MAJOR_K) rc = make_tmap(&maps.m[n][1], G.B2, G.K2, G.s.N, G.ldb2, BLOCK_K, G.bn / 2);
      else                       rc = make_tmap(&maps.m[n][1], G.B2, G.s.N, G.K2, G.ldb2, 64, BLOCK_K);
      if (rc != OSDP_OK) return rc;
    }
    if (G.epi == EPI_BIAS_GELU_DUAL || S.fused) {
      rc = make_tmap(&maps.m[p][3], G.ep.out1, G.s.N, G.s.M, G.ep.ldo, 64, 32, false);
      if (rc != OSDP_OK) return rc;
    }
  }
  for (int p = n; p < kSliceMaxPhases; ++p)
    for (int i = (p == n && P.ph[0].fused ? 2 : 0); i < 4; ++i) maps.m[p][i] = maps.m[0][i];
  P.total_tiles = tiles;

  DeviceInfo dev;
  int rc = current_device(&dev);
  if (rc != OSDP_OK) return rc;
  static std::atomic<int> ready_of[kMaxDevices];
  if (ready_of[dev.ordinal].load(std::memory_order_acquire) == 0) {
    std::lock_guard<std::mutex> lock(launch_setup_mutex());
    OSDP_CUDA_TRY(cudaFuncSetAttribute(mlp_slice_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::kSmemBytes));
    ready_of[dev.ordinal].store(1, std::memory_order_release);
  }
  const int pairs = dev.sms / 2;
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(kThreads);
  cfg.gridDim = dim3(2 * (tiles < pairs ? tiles : pairs));
  cfg.dynamicSmemBytes = Cfg::kSmemBytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  cudaError_t err;
  {
    LaunchTrace tr(st);
    err = cudaLaunchKernelEx(&cfg, mlp_slice_kernel, maps, P);
  }
  OSDP_CUDA_TRY(err);
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

}  // namespace sm100
}  // namespace osdp
