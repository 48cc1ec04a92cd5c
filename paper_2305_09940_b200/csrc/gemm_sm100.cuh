// gemm_sm100.cuh — the bf16 slice GEMM of osdp-b200, hand-written for sm_100a.
//
//   C[M x N] = A[M x K] * B[K x N]   (bf16 x bf16 -> fp32 in TMEM), then a fused epilogue (common.cuh Epi).
//
// Structure: persistent CTA PAIRS (cluster of 2 = one TPC, one CTA per SM, 384 threads each, warp-specialised).
// Every MMA is tcgen05.mma.cta_group::2 (UMMA 256 x 256 x 16): CTA r of the pair supplies 128 A-rows (its TMEM
// lanes) and ONE HALF (128 columns) of the B tile, so every B byte is fetched from L2 and written to shared memory
// once per pair.  A CTA owns MT such row halves: MT = 1 -> 256 x 256 pair tiles, two TMEM accumulator stages
// (epilogue overlapped); MT = 2 -> 512 x 256 pair tiles, one stage, 25 % less operand traffic (TileCfg below).
//   warp 0      TMA producer (both CTAs): cp.async.bulk.tensor.cta_group::2 (128B-swizzled boxes) into a
//               kStages-deep smem ring; both CTAs' loads complete_tx on the LEADER's full barrier; lines up with
//               the other pairs at tile boundaries (wave sync, MT = 2)
//   warp 1      MMA issuer (leader CTA only): one lane issues the UMMAs from smem descriptors into TMEM;
//               tcgen05.commit (multicast to both CTAs) frees the smem slots and publishes finished accumulators
//   warp 2      TMEM allocator (512 columns, cta_group::2) / deallocator
//   warps 4..11 epilogue, two per TMEM lane quarter on alternate column chunks: tcgen05.ld (32 lanes x 32 columns),
//               bias / GeLU / GeLU' in fp32, then the warp's 32 rows x 128 B output segment goes to a 128B-swizzled
//               smem staging buffer and out through TMA (cp.async.bulk.tensor store; cp.reduce.async.bulk.tensor
//               .add for fp32 cross-slice accumulation)
// Three mbarrier pipelines: smem full/empty (TMA <-> MMA), TMEM full/empty (MMA <-> epilogue).  Launched with
// programmatic stream serialization: the set-up overlaps the previous kernel's tail (griddepcontrol).
// Optionally CM x CN pairs form one cluster and TMA-multicast the operand tiles they share (off by default).
//
// Operand majorness: both K-major and MN-major operands are supported directly by
// the UMMA shared-memory descriptors, so the dW GEMMs (A = H_s^T, X_s^T; B = dY_s, dZ_s) need no transposes.
//   K-major tile  [rows x 64 k]      : one TMA box {64, rows};   smem rows of 128 B, 8-row swizzle atoms,
//                                      descriptor SBO = 1024 B, k-step of 16 elements = +32 B
//   MN-major tile [64 k x mn]        : mn/64 TMA boxes {64, 64}; each box 64 k-rows of 128 B (8 KiB),
//                                      descriptor LBO = 8192 B (next 64 mn), SBO = 1024 B (next 8 k), k-step = +2048 B
#pragma once
#include <cuda.h>

#include <atomic>
#include <cmath>
#include <mutex>

#include "common.cuh"
#include "epilogue_math.cuh"

namespace osdp {
namespace sm100 {

constexpr int BLOCK_M = 128;       // rows per UMMA per CTA (TMEM lanes)
constexpr int UMMA_M = 2 * BLOCK_M;   // UMMA M of a CTA pair (cta_group::2)
constexpr int BLOCK_N = 256;       // columns per pair tile = UMMA N
constexpr int HALF_N = BLOCK_N / 2;   // B columns staged by each CTA
constexpr int BLOCK_K = 64;
constexpr int UMMA_K = 16;
// Kernel selection knobs (osdp_set_tuning): defaults are the measured best on C3/C4.
struct Tuning {
  std::atomic<int64_t> mt2_min_k{4096};     // MT = 2 from this contraction length on (bf16-output epilogues)
  std::atomic<int64_t> mt2_min_k_acc{4096}; // the same for the fp32-accumulate epilogue (dW GEMMs: K = slice rows)
  std::atomic<int64_t> mt2_min_tiles{0};    // 0: MT = 2 when it idles at most ~10 % more MMA slots than MT = 1; > 0: plain threshold
  std::atomic<int64_t> wave_sync{1};        // line the producers up at tile boundaries (MT = 2 launches)
  std::atomic<int64_t> band_mib{0};         // 0: square-wave raster bands; > 0: band = tile rows whose A rows fit this many MiB of L2
  std::atomic<int64_t> cluster_min_tiles{0};   // > 0: multicast clusters for launches of at least this many pair tiles
  std::atomic<int64_t> fork_max_tiles{256};    // backward: A5 | A6 | A7 | column sums run concurrently when each GEMM has at most this many 256 x 256 tiles
  std::atomic<int64_t> balance_n{1};           // dX GEMM: narrower tiles (UMMA N < 256) when that fills the last wave; 0 = always 256 columns
  std::atomic<int64_t> slice_kernel_ffn_max_tiles{0};   // the same for the ffn-axis split ([T x f_s] GEMMs); off by default: wins and losses are mixed
  std::atomic<int64_t> slice_kernel_max_tiles{128}; // token split: one persistent kernel per slice (slice_sm100.cuh) when the slice's [T_s x ffn] GEMMs have at most this many 256 x 256 tiles; 0 = never
};
inline Tuning& tuning() {
  static Tuning t;
  return t;
}
constexpr int kPrefetchMaxK = 1024;   // fp32 accumulate launches with K up to this prefetch the old output tile into L2
constexpr int kTmemCols = 512;
constexpr int kThreads = 384;      // warps 0-3: TMA, MMA, TMEM alloc, (idle); warps 4-11: epilogue
constexpr int kEpiWarp0 = 4;
constexpr int kNumEpiWarps = 8;    // two per TMEM lane quarter (warp % 4), taking alternate column chunks
constexpr uint32_t kBStageBytes = HALF_N * BLOCK_K * 2;    // 16 KiB (this CTA's half of the B tile)
constexpr uint32_t kStoreBufBytes = 32 * 128;              // one warp's 32 rows x 128 B output segment

// Two tile shapes share the kernel.  MT = M-halves (UMMAs of 128 rows) per CTA:
//   MT = 1: CTA 128 x 256, pair 256 x 256; TMEM holds TWO accumulator stages, so the epilogue of tile i overlaps
//           the main loop of tile i + 1; 6 smem stages of 32 KiB; 64 KiB of operands per 8.4 MFLOP k-block.
//   MT = 2: CTA 256 x 256, pair 512 x 256; the accumulator fills all 512 TMEM columns (one stage, epilogue
//           exposed); 4 smem stages of 48 KiB; 96 KiB of operands per 16.8 MFLOP k-block, i.e. 25 % less
//           L2 -> SM -> smem traffic per flop.  Large GEMMs run power-limited, where that traffic is what
//           decides the clock, so long-K GEMMs take MT = 2.
template <int MT, int NBUF>
struct TileCfg {
  static constexpr int kCtaM = MT * BLOCK_M;       // rows per CTA
  static constexpr int kPairM = 2 * kCtaM;         // rows per pair tile
  // NBUF = output staging buffers per epilogue warp.  The fp32 epilogue (EPI_ACCUM_F32) moves twice the bytes of the
  // bf16 ones and a warp with ONE buffer waits, chunk after chunk, until TMA has read the previous chunk out
  // (~15 k cycles to drain a 512 x 256 fp32 tile, exposed at MT = 2); with two buffers the wait disappears.  The second
  // buffer is paid for with one ring stage.
  static constexpr int kStoreBufs = NBUF;
  static constexpr uint32_t kSmemStore = kNumEpiWarps * NBUF * kStoreBufBytes;   // 32 / 64 KiB
  static constexpr int kStages = (MT == 1 ? 6 : 4) - (NBUF - 1);
  static constexpr int kAccStages = 2 / MT;
  static constexpr uint32_t kAStageBytes = kCtaM * BLOCK_K * 2;          // 16 / 32 KiB
  static constexpr uint32_t kStageBytes = kAStageBytes + kBStageBytes;   // per CTA; the leader's barrier expects 2x
  static constexpr uint32_t kSmemTiles = kStages * kStageBytes;
  static constexpr uint32_t kSmemBytes = kSmemTiles + kSmemStore + 1024 /*align slack*/ + 256 /*barriers*/;
  static_assert(kSmemBytes <= 227 * 1024, "shared memory per CTA");
};

// L2 cache-hint descriptor of the operand loads: evict_normal (what createpolicy.fractional.L2::evict_normal produces).
// evict_first on the streamed operand / evict_last on the band's rows were measured and doubled the DRAM reads
// (DESIGN.md section 7), so every load uses the default policy.
constexpr uint64_t kEvictNormal = 0x1000000000000000ull;

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
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
// shared::cluster address of the same smem offset in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
// Arrive on an mbarrier of another CTA of the cluster (shared::cluster address).  Default semantics (release at CTA
// scope): the barriers signalled this way hand over TMEM, whose ordering comes from tcgen05.wait::ld and the
// tcgen05 fences on both sides, not from generic-memory visibility; a cluster-scope release was measured to hold
// the arrival back by ~1.2 us (profiles/r01c_power_probes.md section 8).
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// Rendezvous only (no memory is handed over): the teardown, where a CTA just must not exit while a peer can still
// signal its barriers, write its smem or run UMMAs on its TMEM.
__device__ __forceinline__ void cluster_sync_relaxed() {
  asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.aligned;" ::: "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

// dst: this CTA's smem; bar: shared::cluster address of the mbarrier that receives complete_tx (the leader's).
// policy: an L2 cache-hint descriptor (kEvictNormal below).
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c_inner, int c_outer,
                                            uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint "
      "[%0], [%1, {%3, %4}], [%2], %5;"
      ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c_inner), "r"(c_outer), "l"(policy)
      : "memory");
}
// Same, delivered to the same smem offset of every CTA in `mask` (cluster ranks); each destination's bytes are
// signalled on the barrier at `bar`'s offset in the leader of that destination's pair.
__device__ __forceinline__ void tma_load_2d_mc(uint32_t dst, const CUtensorMap* map, uint32_t bar, int c_inner, int c_outer,
                                               uint16_t mask, uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint "
      "[%0], [%1, {%3, %4}], [%2], %5, %6;"
      ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c_inner), "r"(c_outer), "h"(mask), "l"(policy)
      : "memory");
}
// smem -> global tile store / fp32 reduce-add (bulk async-group completion).
__device__ __forceinline__ void tma_store_2d(const CUtensorMap* map, uint32_t src, int c_inner, int c_outer) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"((uint64_t)map), "r"(src), "r"(c_inner), "r"(c_outer)
               : "memory");
}
__device__ __forceinline__ void tma_reduce_add_2d(const CUtensorMap* map, uint32_t src, int c_inner, int c_outer) {
  asm volatile("cp.reduce.async.bulk.tensor.2d.global.shared::cta.add.bulk_group [%0, {%2, %3}], [%1];"
               ::"l"((uint64_t)map), "r"(src), "r"(c_inner), "r"(c_outer)
               : "memory");
}
// Bring the box at these coordinates into L2 (no shared-memory destination, nothing to wait for).
__device__ __forceinline__ void tma_prefetch_l2_2d(const CUtensorMap* map, int c_inner, int c_outer) {
  asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];"
               ::"l"((uint64_t)map), "r"(c_inner), "r"(c_outer)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void st_shared_v4(uint32_t addr, const uint4& v) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void tma_prefetch_desc(const CUtensorMap* map) {
  asm volatile("prefetch.tensormap [%0];" ::"l"((uint64_t)map) : "memory");
}

__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_relinquish() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// D[tmem] (+)= A[smem desc] * B[smem desc]; accumulate = 0 overwrites D.
__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// Arrive on the mbarrier at this smem offset in every CTA of `mask` (cluster ranks) when all tcgen05.mma issued so
// far by this thread have completed (implies tcgen05.fence::before_thread_sync).
__device__ __forceinline__ void umma_commit(uint32_t bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"(mask)
               : "memory");
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
         ((uint32_t)(BLOCK_N >> 3) << 17) | ((uint32_t)(UMMA_M >> 4) << 24);
}

// --------------------------------------------------------------------------------------------------- epilogue
__device__ __forceinline__ uint32_t pack_bf16x2(float lo, float hi) {
  const __nv_bfloat162 p = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&p);
}
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }

// Output columns per 128-byte row segment (one staged TMA store): 64 bf16 or 32 fp32.
template <int EPI>
struct EpiTraits {
  static constexpr bool kF32Out = (EPI == EPI_ACCUM_F32);
  static constexpr int kChunkCols = kF32Out ? 32 : 64;
  // Staging buffers per epilogue warp (TileCfg).  Two buffers (and one ring stage fewer) remove the wait for the
  // previous TMA store in the exposed MT = 2 epilogue; measured twice (bf16 and fp32 outputs, C4 k = 1 / 4 / 16): no
  // gain at the power cap and -2 % at k = 16 from the lost stage, so one buffer it is.
  static constexpr int kStoreBufs = 1;
};

// Per-warp output staging: NBUF buffers of 32 rows x 128 B (128B swizzle: 16-byte chunk j of row r sits at chunk
// j ^ (r & 7), which is also what makes the 16-byte st.shared of 8 consecutive rows conflict-free).  A warp fills
// it, hands it to TMA and meanwhile loads and computes its next chunk; the second warp of the same lane quarter
// covers the remaining latency.
template <int NBUF>
struct StorePipe {
  uint32_t base;    // smem address of this warp's NBUF buffers
  int lane;
  int cur = 0;      // buffer the next chunk goes to
  __device__ __forceinline__ uint32_t buf() const { return base + (uint32_t)cur * kStoreBufBytes; }
  // the buffer the last commit() handed to TMA (still intact until the next begin() on it)
  __device__ __forceinline__ uint32_t committed_buf() const {
    return base + (uint32_t)(NBUF > 1 ? (cur == 0 ? NBUF - 1 : cur - 1) : 0) * kStoreBufBytes;
  }
  __device__ __forceinline__ void begin() const {
    if (lane == 0) bulk_wait_read<NBUF - 1>();   // the store that last used this buffer has read it out
    __syncwarp();
  }
  __device__ __forceinline__ void put(int j, const uint4& v) const {
    st_shared_v4(buf() + lane * 128 + ((j ^ (lane & 7)) << 4), v);
  }
  __device__ __forceinline__ void commit(const CUtensorMap* map, int c_inner, int c_outer, bool reduce_add) {
    fence_proxy_async_smem();   // generic-proxy writes -> visible to the async proxy (TMA)
    __syncwarp();
    if (lane == 0) {
      if (reduce_add) tma_reduce_add_2d(map, buf(), c_inner, c_outer);
      else            tma_store_2d(map, buf(), c_inner, c_outer);
      bulk_commit();
    }
    if constexpr (NBUF > 1) cur = cur + 1 == NBUF ? 0 : cur + 1;
  }
};

// ------------------------------------------------------------------------------------------------- wave sync
// Persistent CTA pairs drift apart over a long launch; the pairs that share an A or B panel then fetch it at
// different times, the panel has to survive in L2 for the whole skew, and DRAM reads grow to several times the
// unique bytes (measured: 4.5 GB instead of 2-3 GB per C4 GEMM).  So the producers of all
// clusters line up at every tile boundary: a cluster announces that the loads of its tile i are issued, and starts
// the loads of tile i + 1 only when every cluster has announced tile i.  Tiles are equal work, so the wait is short,
// and with MT = 2 it falls under the exposed epilogue.  In step, sharers hit L2 together (near-simultaneous
// requests for a line are merged there) and DRAM reads fall to the unique bytes of a wave.
// One counter per launch in flight; the cluster that makes the last announcement of a launch resets it to zero.
constexpr int kWaveSyncSlots = 256;
__device__ unsigned int g_wave_sync[kWaveSyncSlots];

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
  unsigned int v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ unsigned int atom_add_release_gpu(unsigned int* p, unsigned int x) {
  unsigned int old;
  asm volatile("atom.add.release.gpu.global.u32 %0, [%1], %2;" : "=r"(old) : "l"(p), "r"(x) : "memory");
  return old;
}
// The sync is a performance hint, never a correctness requirement, and it must not become a deadlock: two such
// launches running concurrently on different streams can each hold SMs the other one's missing CTAs need.  So a
// wait gives up after ~200 us (tiles take 50-120 us; a healthy wait is a few us) and returns false; the caller
// then stops waiting for the rest of the launch but keeps announcing, so the counter still balances.
__device__ __forceinline__ bool wave_wait(const unsigned int* ctr, unsigned int target) {
  if (ld_acquire_gpu(ctr) >= target) return true;
  const uint64_t t0 = global_timer_ns();
  uint32_t spins = 0;
  while (ld_acquire_gpu(ctr) < target) {
    __nanosleep(64);
    if ((++spins & 0x3Fu) == 0 && global_timer_ns() - t0 > 200ull * 1000) return false;
  }
  return true;
}

// ------------------------------------------------------------------------------------------------- the kernel
struct TileCoord {
  int m_blk, n_blk;   // cluster-tile coordinates: rows m_blk * CM * 256, columns n_blk * CN * 256
};
__device__ __forceinline__ TileCoord tile_coord(int t, int num_m, int num_n, int group_m) {
  const int per_group = group_m * num_n;
  const int g = t / per_group;
  const int first_m = g * group_m;
  const int gsize = min(group_m, num_m - first_m);
  const int local = t - g * per_group;
  return {first_m + local % gsize, local / gsize};
}

// CM x CN CTA pairs form one cluster (2 * CM * CN CTAs) and compute a (CM * 256) x (CN * 256) block of C.  Pairs in
// the same cluster row need the same A rows, pairs in the same cluster column the same B columns: each CTA fetches
// 1/CN of its A tile and 1/CM of its B half-tile and TMA-multicasts it to the CTAs that share it, so L2 -> SM
// traffic per flop falls by (1/CN + 1/CM) / 2.  CM = CN = 1 is the plain pair kernel.
template <int A_MAJOR, int B_MAJOR, int EPI, int MT, int CM, int CN>
__global__ void __launch_bounds__(kThreads, 1)
gemm_bf16_sm100_kernel(const __grid_constant__ CUtensorMap tmap_a, const __grid_constant__ CUtensorMap tmap_b,
                       const __grid_constant__ CUtensorMap tmap_out0, const __grid_constant__ CUtensorMap tmap_out1,
                       const GemmShape shape, const EpiParams ep, const int group_m, unsigned int* wave_sync,
                       const int sync_kb, const int bn_arg) {
  using Cfg = TileCfg<MT, EpiTraits<EPI>::kStoreBufs>;
  constexpr int kStages = Cfg::kStages, kAccStages = Cfg::kAccStages;
  constexpr uint32_t kSmemStore = Cfg::kSmemStore;
  constexpr int kCtaM = Cfg::kCtaM, kPairM = Cfg::kPairM;
  constexpr uint32_t kAStageBytes = Cfg::kAStageBytes, kStageBytes = Cfg::kStageBytes, kSmemTiles = Cfg::kSmemTiles;
  constexpr int kPairs = CM * CN;
  constexpr int kCluster = 2 * kPairs;
  // Tile width.  256 columns, except for the dX GEMM (K-major B, plain epilogue, no multicast cluster), whose host side
  // may ask for a narrower UMMA N (a multiple of 16) when that makes the tile count a whole number of waves
  // (launch_gemm_bf16_cluster: 128 tiles of 512 x 256 on 74 pairs are 1.73 waves, 148 tiles of 512 x 224 exactly two).
  constexpr bool kVarN = (B_MAJOR == MAJOR_K && EPI == EPI_PLAIN && kPairs == 1);
  const int bn = kVarN ? bn_arg : BLOCK_N;
  const int half_n = bn / 2;
  static_assert(CM == 1 || CM == 2, "CM");
  static_assert(CN == 1 || CN == 2, "CN");
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;   // 128B swizzle atoms need 1024 B alignment
  const uint32_t smem_a = smem_base;
  const uint32_t smem_b = smem_base + kStages * kAStageBytes;
  const uint32_t smem_store = smem_base + kSmemTiles;
  const uint32_t bars = smem_store + kSmemStore;
  const uint32_t full_bar = bars;                                  // [kStages]   (used in each pair's leader CTA)
  const uint32_t empty_bar = bars + 8 * kStages;                   // [kStages]   (one per CTA, multicast arrive)
  const uint32_t tfull_bar = bars + 16 * kStages;                  // [kAccStages] (one per CTA, multicast arrive)
  const uint32_t tempty_bar = bars + 16 * kStages + 8 * kAccStages;   // [kAccStages] (used in each pair's leader CTA)
  const uint32_t tmem_slot = bars + 16 * kStages + 16 * kAccStages;   // uint32
  uint32_t* tmem_slot_ptr = reinterpret_cast<uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

  const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
  const uint32_t crank = cluster_ctarank();
  const uint32_t rank = crank & 1u;                 // 0 = leader of its pair
  const bool leader = rank == 0;
  const uint32_t leader_crank = crank & ~1u;
  const int pi = (int)(crank >> 1) / CN, pj = (int)(crank >> 1) % CN;   // this pair's position in the cluster
  const int cluster_id = blockIdx.x / kCluster, num_clusters = gridDim.x / kCluster;
  const int num_m = (shape.M + kPairM - 1) / kPairM, num_n = (shape.N + bn - 1) / bn;   // pair tiles
  const int num_cm = (num_m + CM - 1) / CM, num_cn = (num_n + CN - 1) / CN;                         // cluster tiles
  const int num_tiles = num_cm * num_cn;
  const int num_kb = (shape.K + BLOCK_K - 1) / BLOCK_K;

  if (warp == 0 && lane == 0) {
    tma_prefetch_desc(&tmap_a);
    tma_prefetch_desc(&tmap_b);
    tma_prefetch_desc(&tmap_out0);
    if constexpr (EPI == EPI_BIAS_GELU_DUAL) tma_prefetch_desc(&tmap_out1);
  }
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < kStages; ++i) {
      mbar_init(full_bar + 8 * i, 1);                      // the leader's producer arrives (+ expect_tx of both CTAs' bytes)
      mbar_init(empty_bar + 8 * i, kPairs);                // one multicast tcgen05.commit per pair of the cluster
    }
    for (int i = 0; i < kAccStages; ++i) {
      mbar_init(tfull_bar + 8 * i, 1);                     // one multicast tcgen05.commit
      mbar_init(tempty_bar + 8 * i, 2 * kNumEpiWarps);     // the epilogue warps of both CTAs
    }
    fence_barrier_init();
  }
  if (warp == 2) {
    tmem_alloc(tmem_slot, kTmemCols);
    tmem_relinquish();
  }
  tc_fence_before();
  cluster_sync();            // every CTA's barriers are initialised and TMEM is allocated before anyone proceeds
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;
  // Programmatic dependent launch: everything above overlapped the tail of the previous kernel of the stream; from
  // here on this kernel reads and writes memory that kernel may still be using.  The next kernel may start its own
  // set-up as soon as SMs free up.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

  if (warp == 0) {
    // ================================================================== TMA producer (every CTA)
    // multicast destinations: the CTAs of equal pair-rank in this cluster row (A) / cluster column (B)
    uint16_t mask_a = 0, mask_b = 0;
#pragma unroll
    for (int j = 0; j < CN; ++j) mask_a |= (uint16_t)(1u << (2 * (pi * CN + j) + (int)rank));
#pragma unroll
    for (int i = 0; i < CM; ++i) mask_b |= (uint16_t)(1u << (2 * (i * CN + pj) + (int)rank));
    // Tiles walk along n inside a band of group_m cluster-tile rows: the band's A rows are re-used by every wave
    // of the band (keep them in L2), B streams through once per band (let it go first).
    constexpr uint64_t pol_a = kEvictNormal, pol_b = kEvictNormal;
    constexpr int kARows = kCtaM / CN;     // A rows (K-major) this CTA fetches; it is part pj of the tile
    constexpr int kBRows = HALF_N / CM;    // B columns this CTA fetches; it is part pi of the half-tile
    int stage = 0;
    uint32_t phase = 0;
    int it = 0;
    bool waiting = true;   // false once a wait has timed out (see wave_wait)
    for (int t = cluster_id; t < num_tiles; t += num_clusters, ++it) {
      // Sync points of a tile: before k-blocks sync_kb, 2 sync_kb, ... (if sync_kb > 0) and after the last one.
      const unsigned int syncs_per_tile = 1u + (sync_kb > 0 ? (unsigned int)((num_kb - 1) / sync_kb) : 0u);
      const unsigned int sync_base = (unsigned int)it * syncs_per_tile * (unsigned int)num_clusters;   // earlier waves were full
      const unsigned int active = (unsigned int)min(num_clusters, num_tiles - it * num_clusters);       // clusters in this wave
      if (wave_sync != nullptr && waiting && it > 0) {   // every cluster has issued the loads of its previous tile
        waiting = __shfl_sync(0xFFFFFFFFu, lane == 0 ? (int)wave_wait(wave_sync, sync_base) : 0, 0) != 0;
      }
      const TileCoord tc = tile_coord(t, num_cm, num_cn, group_m);
      const int m0 = (tc.m_blk * CM + pi) * kPairM + (int)rank * kCtaM;       // this CTA's rows of A
      const int n0 = (tc.n_blk * CN + pj) * bn + (int)rank * half_n;     // this CTA's half of the B tile
      for (int kb = 0; kb < num_kb; ++kb) {
        if (wave_sync != nullptr && sync_kb > 0 && kb > 0 && kb % sync_kb == 0) {   // stay in step inside the tile too
          int ok = 1;
          if (lane == 0) {
            if (crank == 0) atom_add_release_gpu(wave_sync, 1u);
            if (waiting) ok = (int)wave_wait(wave_sync, sync_base + (unsigned int)(kb / sync_kb) * active);
          }
          waiting = waiting && __shfl_sync(0xFFFFFFFFu, ok, 0) != 0;
        }
        mbar_wait(empty_bar + 8 * stage, phase ^ 1);   // the slot is free in every CTA of the cluster
        if (lane == 0) {
          const uint32_t fb_local = full_bar + 8 * stage;
          const uint32_t fb = mapa(fb_local, leader_crank);     // the pair leader's barrier receives both CTAs' bytes
          const uint32_t sa = smem_a + stage * kAStageBytes, sb = smem_b + stage * kBStageBytes;
          const int k0 = kb * BLOCK_K;
          if (leader) mbar_expect_tx(fb_local, kVarN ? 2u * (kAStageBytes + (uint32_t)half_n * (BLOCK_K * 2)) : 2 * kStageBytes);
          if constexpr (kPairs == 1) {
            if constexpr (A_MAJOR == MAJOR_K) {
              tma_load_2d(sa, &tmap_a, fb, k0, m0, pol_a);
            } else {
#pragma unroll
              for (int c = 0; c < kCtaM / 64; ++c) tma_load_2d(sa + c * (BLOCK_K * 128), &tmap_a, fb, m0 + 64 * c, k0, pol_a);
            }
            if constexpr (B_MAJOR == MAJOR_K) {
              tma_load_2d(sb, &tmap_b, fb, k0, n0, pol_b);
            } else {
#pragma unroll
              for (int c = 0; c < HALF_N / 64; ++c) tma_load_2d(sb + c * (BLOCK_K * 128), &tmap_b, fb, n0 + 64 * c, k0, pol_b);
            }
          } else {
            if constexpr (A_MAJOR == MAJOR_K) {
              tma_load_2d_mc(sa + pj * (kARows * 128), &tmap_a, fb, k0, m0 + pj * kARows, mask_a, pol_a);
            } else {
#pragma unroll
              for (int c = pj * (kARows / 64); c < (pj + 1) * (kARows / 64); ++c)
                tma_load_2d_mc(sa + c * (BLOCK_K * 128), &tmap_a, fb, m0 + 64 * c, k0, mask_a, pol_a);
            }
            if constexpr (B_MAJOR == MAJOR_K) {
              tma_load_2d_mc(sb + pi * (kBRows * 128), &tmap_b, fb, k0, n0 + pi * kBRows, mask_b, pol_b);
            } else {
#pragma unroll
              for (int c = pi * (kBRows / 64); c < (pi + 1) * (kBRows / 64); ++c)
                tma_load_2d_mc(sb + c * (BLOCK_K * 128), &tmap_b, fb, n0 + 64 * c, k0, mask_b, pol_b);
            }
          }
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
      if (wave_sync != nullptr && crank == 0 && lane == 0) {
        if (atom_add_release_gpu(wave_sync, 1u) == (unsigned int)num_tiles * syncs_per_tile - 1u)
          *reinterpret_cast<volatile unsigned int*>(wave_sync) = 0u;   // last announcement of the launch: nobody waits any more
      }
    }
  } else if (warp == 1 && leader) {
    // ================================================================== MMA issuer (each pair's leader CTA)
    const uint32_t idesc = kVarN ? ((make_idesc<A_MAJOR, B_MAJOR>() & ~(0x3Fu << 17)) | ((uint32_t)(bn >> 3) << 17))
                                 : make_idesc<A_MAJOR, B_MAJOR>();
    constexpr uint16_t mask_cluster = (uint16_t)((1u << kCluster) - 1u);
    const uint16_t mask_pair = (uint16_t)(3u << leader_crank);
    int stage = 0;
    uint32_t phase = 0;
    int it = 0;
    for (int t = cluster_id; t < num_tiles; t += num_clusters, ++it) {
      const TileCoord tc = tile_coord(t, num_cm, num_cn, group_m);
      // a pair whose tile lies outside C (odd tile counts) still takes part in the loads, but skips the math
      const bool valid = (tc.m_blk * CM + pi) < num_m && (tc.n_blk * CN + pj) < num_n;
      const int as = it % kAccStages;
      const uint32_t aphase = (it / kAccStages) & 1;
      mbar_wait(tempty_bar + 8 * as, aphase ^ 1);   // both CTAs' epilogues have drained this accumulator stage
      tc_fence_after();
      const uint32_t tmem_d = tmem_base + as * (MT * BLOCK_N);   // M-half h accumulates in columns [256 h, 256 h + 256)
      for (int kb = 0; kb < num_kb; ++kb) {
        mbar_wait(full_bar + 8 * stage, phase);      // both CTAs' TMA bytes have landed
        tc_fence_after();
        if (lane == 0) {
          const uint32_t sa = smem_a + stage * kAStageBytes, sb = smem_b + stage * kBStageBytes;
          if (valid) {
#pragma unroll
            for (int k = 0; k < BLOCK_K / UMMA_K; ++k) {
              const uint64_t bdesc = operand_desc<B_MAJOR>(sb, k);
#pragma unroll
              for (int h = 0; h < MT; ++h)
                umma_bf16(tmem_d + h * BLOCK_N, operand_desc<A_MAJOR>(sa + h * (BLOCK_M * BLOCK_K * 2), k), bdesc, idesc,
                          (kb | k) != 0);
            }
          }
          umma_commit(empty_bar + 8 * stage, mask_cluster);   // slot free (for this pair) in every CTA that may refill it
          if (kb == num_kb - 1) umma_commit(tfull_bar + 8 * as, mask_pair);   // accumulator complete (both CTAs)
        }
        __syncwarp();
        if (++stage == kStages) { stage = 0; phase ^= 1; }
      }
    }
  } else if (warp >= kEpiWarp0) {
    // ================================================================== epilogue (both CTAs, own rows)
    using Tr = EpiTraits<EPI>;
    constexpr int kChunk = Tr::kChunkCols;
    const int q = warp % 4;                    // TMEM lane quarter this warp may access
    const int cg = (warp - kEpiWarp0) / 4;     // which of the two warps of that quarter: takes chunks cg, cg + 2, ...
    StorePipe<Cfg::kStoreBufs> pipe{smem_store + (uint32_t)(warp - kEpiWarp0) * (Cfg::kStoreBufs * kStoreBufBytes), lane};
    const uint32_t tempty_leader = mapa(tempty_bar, leader_crank);
    const __nv_bfloat16* bias = reinterpret_cast<const __nv_bfloat16*>(ep.bias);
    constexpr bool kHasBias = (EPI == EPI_BIAS_GELU || EPI == EPI_BIAS || EPI == EPI_BIAS_GELU_DUAL);
    // The bias of a warp's column chunks is fetched BEFORE the wait for the accumulator (a global load inside the
    // chunk loop costs ~1.3 us per chunk on the exposed path): lane l keeps columns 2 l, 2 l + 1 of chunk ci in
    // bias_reg[ci]; the chunk loop reads them back with shuffles.  Both row halves of an MT = 2 tile use the same columns.
    constexpr int kBiasChunks = BLOCK_N / (2 * 64);   // chunks of 64 columns this warp owns per tile (bf16 outputs)
    uint32_t bias_reg[kBiasChunks] = {};
    // 8 consecutive accumulator columns (+ bias) -> fp32 values; j = index of the 8-column group inside chunk ci
    static_assert(kBiasChunks == 2, "bias registers: two column chunks per epilogue warp");
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
    int it = 0;
    for (int t = cluster_id; t < num_tiles; t += num_clusters, ++it) {
      const TileCoord tc = tile_coord(t, num_cm, num_cn, group_m);
      const int as = it % kAccStages;
      const uint32_t aphase = (it / kAccStages) & 1;
      const int n0 = (tc.n_blk * CN + pj) * bn;
      const int n_end = min(n0 + bn, shape.N);
      if constexpr (kHasBias) {
#pragma unroll
        for (int ci = 0; ci < kBiasChunks; ++ci) {
          const int c = n0 + (cg + 2 * ci) * 64 + 2 * lane;
          bias_reg[ci] = c < shape.N ? __ldg(reinterpret_cast<const uint32_t*>(bias + c)) : 0u;   // N is even
        }
      }
      if constexpr (Tr::kF32Out) {
        // Cross-slice accumulation (beta = 1) is a reduce-add performed AT L2; on a miss L2 first fetches the old line
        // from DRAM, and a warp's next chunk waits behind that (one staging buffer), so the drain of a tile runs at the
        // DRAM latency: ~2.8 k cycles per 4 KiB chunk (ncu, C4).  With short slices (K = T_s <= 1024) the main loop is too
        // short to hide that, so the warp asks for its chunks of the old dW tile while the main loop is still running and
        // the reduce-adds hit in L2: +3.7 % per step at C4 k = 16.  For longer K the drain is hidden anyway and the
        // prefetch only costs L2 space (-0.5 ... -1.5 % at K = 2048), so it is limited to short K.
        if (ep.beta != 0 && shape.K <= kPrefetchMaxK && lane == 0) {
#pragma unroll 1
          for (int h = 0; h < MT; ++h) {
            const int prow0 = (tc.m_blk * CM + pi) * kPairM + (int)rank * kCtaM + h * BLOCK_M + q * 32;
            if (prow0 >= shape.M) continue;
            for (int n = n0 + cg * kChunk; n < n_end; n += 2 * kChunk) tma_prefetch_l2_2d(&tmap_out0, n, prow0);
          }
        }
      }
      mbar_wait(tfull_bar + 8 * as, aphase);
      tc_fence_after();
      bool released = false;   // the accumulator stage goes back to the MMA warp right after this warp's last tcgen05.ld
      // ... if a later tile of this cluster will wait for it.  A hand-back that nobody consumes is a remote arrive that
      // may still be in flight when the leader CTA has exited (the teardown rendezvous is relaxed): it would then land
      // in the barriers of the NEXT kernel's CTA on that SM as a spurious arrival (seen in slice_sm100.cuh).
      const bool hand_back = t + kAccStages * num_clusters < num_tiles;
#pragma unroll 1
      for (int h = 0; h < MT; ++h) {
        const int row0 = (tc.m_blk * CM + pi) * kPairM + (int)rank * kCtaM + h * BLOCK_M + q * 32;   // this warp's 32-row band
        const int64_t row = row0 + lane;
        const bool row_ok = row < shape.M;
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * (MT * BLOCK_N) + h * BLOCK_N;
        if (row0 >= shape.M) continue;   // nothing of this warp's band lies inside C (warp-uniform)
#pragma unroll 1
        for (int n = n0 + cg * kChunk; n < n_end; n += 2 * kChunk) {
          uint32_t acc[kChunk];
          [[maybe_unused]] uint4 zraw[8];
          if constexpr (EPI == EPI_DGELU) {   // stored Z_s of this chunk: issue the loads before waiting on TMEM
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              zraw[j] = make_uint4(0, 0, 0, 0);
              if (row_ok && n + 8 * j < shape.N)
                zraw[j] = *reinterpret_cast<const uint4*>((const __nv_bfloat16*)ep.aux + row * ep.ldo + n + 8 * j);
            }
          }
#pragma unroll
          for (int i = 0; i < kChunk / 32; ++i)
            tmem_ld_32x32(taddr + (n - n0) + 32 * i, *reinterpret_cast<uint32_t(*)[32]>(&acc[32 * i]));
          tmem_ld_wait();
          if (h == MT - 1 && n + 2 * kChunk >= n_end) {   // this warp's last read of the accumulator stage
            tc_fence_before();
            __syncwarp();
            if (lane == 0 && hand_back) mbar_arrive_cluster(tempty_leader + 8 * as);
            released = true;
          }
          [[maybe_unused]] const uint32_t bias_cur = (n - n0) >= 2 * kChunk ? bias_reg[1] : bias_reg[0];
          if constexpr (Tr::kF32Out) {
            pipe.begin();
#pragma unroll
            for (int j = 0; j < 8; ++j) pipe.put(j, make_uint4(acc[4 * j], acc[4 * j + 1], acc[4 * j + 2], acc[4 * j + 3]));
            pipe.commit(&tmap_out0, n, row0, ep.beta != 0);
          } else {
            if constexpr (EPI == EPI_BIAS_GELU_DUAL) {   // first pass: Z_s = acc + bias
              pipe.begin();
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                float v[8];
                load8(&acc[8 * j], bias_cur, j, v);
                pipe.put(j, pack8(v));
              }
              pipe.commit(&tmap_out0, n, row0, false);
            }
            if constexpr (kVarN) {
              // a tile narrower than 256 columns ends inside this warp's last 64-column chunk: the 64-column TMA box would
              // run over into the next tile's columns, so the chunk's 16 / 32 / 48 columns go out as 16-byte stores
              if (n + kChunk > n0 + bn && n0 + bn < shape.N) {
                if (row_ok) {
                  __nv_bfloat16* dst = reinterpret_cast<__nv_bfloat16*>(ep.out0) + row * ep.ldo + n;
#pragma unroll
                  for (int j = 0; j < 8; ++j) {
                    if (n + 8 * j < n_end) {
                      float v[8];
                      load8(&acc[8 * j], bias_cur, j, v);
                      *reinterpret_cast<uint4*>(dst + 8 * j) = pack8(v);
                    }
                  }
                }
                continue;
              }
            }
            pipe.begin();
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              float v[8];
              load8(&acc[8 * j], bias_cur, j, v);
              if constexpr (EPI == EPI_BIAS_GELU || EPI == EPI_BIAS_GELU_DUAL) {
#pragma unroll
                for (int i = 0; i < 8; ++i) v[i] = gelu_fwd<false>(v[i]);
              }
              if constexpr (EPI == EPI_DGELU) {
                const uint32_t zw[4] = {zraw[j].x, zraw[j].y, zraw[j].z, zraw[j].w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  v[2 * i] *= gelu_bwd<false>(bf16_lo(zw[i]));
                  v[2 * i + 1] *= gelu_bwd<false>(bf16_hi(zw[i]));
                }
              }
              pipe.put(j, pack8(v));
            }
            pipe.commit(EPI == EPI_BIAS_GELU_DUAL ? &tmap_out1 : &tmap_out0, n, row0, false);
            if constexpr (EPI == EPI_DGELU) {
              // db1 (step A4 of SURVEY.md section 8(a)): column sums of this warp's 32 rows x 64 columns of dZ_s, taken
              // from the staged bf16 values (exactly what is stored).  Lane l owns columns 2l and 2l + 1 and walks the
              // 32 rows in order (word l of every 128-byte row: conflict-free under the 128B swizzle); rows outside M hold
              // zeros (zero-filled operand rows).  One 256-byte store per chunk into the band-partials scratch; the
              // fixed-order sum over bands is colsum_final_kernel's.
              if (ep.colsum != nullptr) {
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
                if (c < shape.N)
                  *reinterpret_cast<float2*>(ep.colsum + (int64_t)(row0 >> 5) * ep.ld_colsum + c) = make_float2(s0, s1);
              }
            }
          }
        }
      }   // h
      if (!released) {
        tc_fence_before();
        __syncwarp();
        if (lane == 0 && hand_back) mbar_arrive_cluster(tempty_leader + 8 * as);
      }
    }
    if (lane == 0) bulk_wait<0>();   // all of this warp's stores have completed before the CTA's smem goes away
    __syncwarp();
  }

  // No CTA may exit (or free TMEM) while a peer can still signal its barriers, write its smem or run UMMAs on its TMEM.
  tc_fence_before();
  cluster_sync_relaxed();
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

// Per-device launch state.  A process may drive several GPUs from several host threads (one device current per
// thread), so nothing about a device is cached in a plain static: the SM count, the wave-sync counters (a __device__
// array has one instance per device) and, per kernel instantiation, the shared-memory opt-in and the resident cluster
// count are all kept per device ordinal and initialised under a mutex (osdp_api.cu).
constexpr int kMaxDevices = 64;
struct DeviceInfo {
  int ordinal;
  int sms;
};
int current_device(DeviceInfo* out);   // osdp_api.cu; OSDP_OK / OSDP_ERR_CUDA / OSDP_ERR_ARG (ordinal >= kMaxDevices)
std::mutex& launch_setup_mutex();      // osdp_api.cu

// Matrix stored row-major [outer x inner] with `ld` elements between rows; 128B-swizzled box.
// cuTensorMapEncodeTiled is a pure function of its arguments and costs about a microsecond; a slice loop re-creates
// the same few maps call after call (launch-bound shapes feel it), so each host thread keeps the last encodings in a
// small direct-mapped cache keyed on every argument.
struct TmapKey {
  const void* ptr;
  int64_t inner, outer, ld;
  int box_inner, box_outer, f32;
  bool operator==(const TmapKey& o) const {
    return ptr == o.ptr && inner == o.inner && outer == o.outer && ld == o.ld && box_inner == o.box_inner &&
           box_outer == o.box_outer && f32 == o.f32;
  }
};
struct TmapCache {
  static constexpr int kSlots = 256;
  struct Slot {
    TmapKey key;
    CUtensorMap map;
    bool used;
  };
  Slot slots[kSlots] = {};
  static size_t slot_of(const TmapKey& k) {
    uint64_t h = (uint64_t)(uintptr_t)k.ptr * 0x9E3779B97F4A7C15ull;
    h ^= (uint64_t)k.inner * 0xBF58476D1CE4E5B9ull + (uint64_t)k.outer * 0x94D049BB133111EBull + (uint64_t)k.ld;
    h ^= ((uint64_t)k.box_inner << 40) ^ ((uint64_t)k.box_outer << 20) ^ (uint64_t)k.f32;
    h ^= h >> 29;
    return (size_t)(h % kSlots);
  }
};
inline int make_tmap(CUtensorMap* map, const void* ptr, int64_t inner, int64_t outer, int64_t ld, int box_inner,
                     int box_outer, bool f32 = false) {
  static thread_local TmapCache cache;
  const TmapKey key{ptr, inner, outer, ld, box_inner, box_outer, f32 ? 1 : 0};
  TmapCache::Slot& slot = cache.slots[TmapCache::slot_of(key)];
  if (slot.used && slot.key == key) {
    *map = slot.map;
    return OSDP_OK;
  }
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return OSDP_ERR_CUDA;
  const cuuint64_t dims[2] = {(cuuint64_t)inner, (cuuint64_t)outer};
  const cuuint64_t strides[1] = {(cuuint64_t)ld * (f32 ? 4 : 2)};
  const cuuint32_t box[2] = {(cuuint32_t)box_inner, (cuuint32_t)box_outer};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = fn(map, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2,
                        const_cast<void*>(ptr), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) {
    note_cuda_error(cudaErrorInvalidValue, "cuTensorMapEncodeTiled");
    return OSDP_ERR_CUDA;
  }
  slot.key = key;
  slot.map = *map;
  slot.used = true;
  return OSDP_OK;
}

// A, B: bf16 device pointers stored as common.cuh describes for the given majorness.
template <int A_MAJOR, int B_MAJOR, int EPI, int MT, int CM, int CN>
inline int launch_gemm_bf16_cluster(const void* A, int64_t lda, const void* B, int64_t ldb, const GemmShape& s,
                                    const EpiParams& ep, cudaStream_t st) {
  using Cfg = TileCfg<MT, EpiTraits<EPI>::kStoreBufs>;
  CUtensorMap ta, tb, to0, to1;
  int rc;
  // one TMA box = what ONE CTA fetches per k-block: 1/CN of its A rows, 1/CM of its B half (MN-major: 64-wide boxes)
  if (A_MAJOR == MAJOR_K) rc = make_tmap(&ta, A, s.K, s.M, lda, BLOCK_K, Cfg::kCtaM / CN);
  else                    rc = make_tmap(&ta, A, s.M, s.K, lda, 64, BLOCK_K);
  if (rc != OSDP_OK) return rc;
  // Tile width (see kVarN in the kernel): among 256, 240, 224, 208, 192 columns the one with the least waves x width, if
  // that saves at least 5 % of the launch's tile-time.  Results do not depend on it (one owner per output element,
  // ascending-k accumulation).
  int bn = BLOCK_N;
  DeviceInfo dev;
  rc = current_device(&dev);
  if (rc != OSDP_OK) return rc;
  if (B_MAJOR == MAJOR_K && EPI == EPI_PLAIN && CM * CN == 1 && tuning().balance_n.load() != 0) {
    const int64_t pairs = dev.sms / 2, nm = (s.M + Cfg::kPairM - 1) / Cfg::kPairM;
    auto cost = [&](int w) { return ((nm * ((s.N + w - 1) / w) + pairs - 1) / pairs) * (int64_t)w; };
    int64_t best = cost(BLOCK_N);
    for (int w = BLOCK_N - 16; w >= 192; w -= 16)
      if (cost(w) < best) { best = cost(w); bn = w; }
    if (20 * best > 19 * cost(BLOCK_N)) bn = BLOCK_N;
  }
  if (B_MAJOR == MAJOR_K) rc = make_tmap(&tb, B, s.K, s.N, ldb, BLOCK_K, (bn / 2) / CM);
  else                    rc = make_tmap(&tb, B, s.N, s.K, ldb, 64, BLOCK_K);
  if (rc != OSDP_OK) return rc;
  // outputs: [M x N] row-major, leading dimension ldo; one store = 32 rows x 128 bytes
  constexpr bool f32out = EpiTraits<EPI>::kF32Out;
  rc = make_tmap(&to0, ep.out0, s.N, s.M, ep.ldo, EpiTraits<EPI>::kChunkCols, 32, f32out);
  if (rc != OSDP_OK) return rc;
  to1 = to0;
  if (EPI == EPI_BIAS_GELU_DUAL) {
    rc = make_tmap(&to1, ep.out1, s.N, s.M, ep.ldo, EpiTraits<EPI>::kChunkCols, 32, false);
    if (rc != OSDP_OK) return rc;
  }

  constexpr int kCluster = 2 * CM * CN;
  auto kernel = gemm_bf16_sm100_kernel<A_MAJOR, B_MAJOR, EPI, MT, CM, CN>;
  cudaLaunchConfig_t cfg = {};
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = Cfg::kSmemBytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = kCluster;
  attr[0].val.clusterDim.y = 1;
  attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see griddepcontrol in the kernel
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  // per (kernel instantiation, device): the dynamic shared-memory opt-in and the number of co-resident clusters
  static std::atomic<int> max_clusters_of[kMaxDevices];
  int max_clusters = max_clusters_of[dev.ordinal].load(std::memory_order_acquire);
  if (max_clusters == 0) {
    std::lock_guard<std::mutex> lock(launch_setup_mutex());
    OSDP_CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Cfg::kSmemBytes));
    int n = 0;
    cfg.gridDim = dim3(kCluster * 64);
    if (kCluster == 2) n = dev.sms / 2;   // one CTA pair per TPC
    else OSDP_CUDA_TRY(cudaOccupancyMaxActiveClusters(&n, kernel, &cfg));
    if (n < 1) {
      note_cuda_error(cudaErrorInvalidConfiguration, "cudaOccupancyMaxActiveClusters");
      return OSDP_ERR_CUDA;
    }
    max_clusters = n;
    max_clusters_of[dev.ordinal].store(n, std::memory_order_release);
  }
  const int num_m = (s.M + Cfg::kPairM - 1) / Cfg::kPairM, num_n = (s.N + bn - 1) / bn;   // pair tiles
  const int tiles = ((num_m + CM - 1) / CM) * ((num_n + CN - 1) / CN);                      // cluster tiles
  cfg.gridDim = dim3(kCluster * (tiles < max_clusters ? tiles : max_clusters));
  // Raster band = group_m tile rows; inside a band tiles walk m fastest, then n, so one wave of P resident clusters
  // covers group_m tile rows x P / group_m tile columns.  All clusters of a wave sweep K in step (wave sync, or simply
  // equal work), so what a wave pulls from DRAM is its UNIQUE operand rows and columns, about
  // (group_m * rows_per_tile + P / group_m * cols_per_tile) * K elements: least for a square-ish wave,
  // group_m = sqrt(P * cols_per_tile / rows_per_tile), whatever K is.  (Round 1 sized the band so that its A rows fit an
  // L2 budget; for long K that degenerates to one tile row per band and B is re-read per row: 1.24 GB instead of
  // 0.67 GB for the A2 / A7 launches of C4 k = 4.  OSDP_TUNE_BAND_MIB > 0 brings that rule back.)
  int64_t group_m;
  const int64_t band_mib = tuning().band_mib.load();
  if (band_mib > 0) {
    const int64_t row_bytes = (int64_t)CM * Cfg::kPairM * s.K * 2;
    group_m = (band_mib << 20) / row_bytes;
  } else {
    const int num_cm = (num_m + CM - 1) / CM;
    const double ideal = std::sqrt((double)max_clusters * (CN * BLOCK_N) / (double)(CM * Cfg::kPairM));
    int64_t g = (int64_t)(ideal + 0.5);
    if (g < 1) g = 1;
    const int64_t bands = (num_cm + g - 1) / g;          // equal bands: no thin last band
    group_m = (num_cm + bands - 1) / bands;
  }
  if (group_m < 1) group_m = 1;
  if (group_m > (1 << 20)) group_m = 1 << 20;
  // wave sync only when there is more than one wave, and only with a fully resident grid
  unsigned int* wave_sync = nullptr;
  const int64_t sync_mode = tuning().wave_sync.load();   // 0 off, 1 tile boundaries, q > 1: also every q k-blocks
  // (MT = 1 overlaps its epilogue with the next main loop, so a wait at the tile boundary would be exposed)
  if (MT == 2 && tiles > max_clusters && sync_mode != 0) {
    static std::atomic<unsigned int*> base_of[kMaxDevices];   // this device's instance of g_wave_sync
    static std::atomic<unsigned int> seq{0};
    unsigned int* base = base_of[dev.ordinal].load(std::memory_order_acquire);
    if (!base) {
      OSDP_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&base), g_wave_sync));
      base_of[dev.ordinal].store(base, std::memory_order_release);
    }
    wave_sync = base + (seq.fetch_add(1) % kWaveSyncSlots);
  }
  cudaError_t err;
  {
    LaunchTrace tr(st);
    err = cudaLaunchKernelEx(&cfg, kernel, ta, tb, to0, to1, s, ep, (int)group_m, wave_sync,
                             sync_mode > 1 ? (int)sync_mode : 0, bn);
  }
  OSDP_CUDA_TRY(err);
  OSDP_CUDA_TRY(cudaGetLastError());
  return OSDP_OK;
}

// Tile shape and cluster shape per launch.
//  * MT = 2 (512 x 256 pair tiles, 25 % less operand traffic, exposed epilogue) for long contractions, where the
//    main loop of a tile dwarfs its epilogue; MT = 1 (256 x 256, overlapped epilogue) otherwise.
//  * Multicast clusters: OSDP_TUNE_CLUSTER_MIN_TILES = n > 0 takes clusters of OSDP_CM x OSDP_CN pairs (default 1 x 2: the two
//    pairs of a cluster share their A rows) for launches of at least that many pair tiles (0 = never).
//    Off by default: clusters of more than 2 CTAs can use at most 132 of the 148 SMs, which costs more than the
//    saved L2 -> SM traffic returns.  Other cluster shapes: -DOSDP_CM / -DOSDP_CN.
#ifndef OSDP_CM
#define OSDP_CM 1
#endif
#ifndef OSDP_CN
#define OSDP_CN 2
#endif
template <int A_MAJOR, int B_MAJOR, int EPI, int MT>
inline int launch_gemm_bf16_mt(const void* A, int64_t lda, const void* B, int64_t ldb, const GemmShape& s,
                               const EpiParams& ep, cudaStream_t st) {
  const int64_t num_m = (s.M + (2 * MT * BLOCK_M) - 1) / (2 * MT * BLOCK_M), num_n = (s.N + BLOCK_N - 1) / BLOCK_N;
  const int64_t cluster_min_tiles = tuning().cluster_min_tiles.load();   // 0 = never
  if (OSDP_CM * OSDP_CN > 1 && cluster_min_tiles > 0 && num_m * num_n >= cluster_min_tiles)
    return launch_gemm_bf16_cluster<A_MAJOR, B_MAJOR, EPI, MT, OSDP_CM, OSDP_CN>(A, lda, B, ldb, s, ep, st);
  return launch_gemm_bf16_cluster<A_MAJOR, B_MAJOR, EPI, MT, 1, 1>(A, lda, B, ldb, s, ep, st);
}
// Fraction of the machine's MMA slots that do useful work for pair tiles of pair_m rows: padding of M to whole
// tiles (N is a multiple of 256 in every workload; its padding is the same for both shapes) times the fill of
// the last wave.
inline double tile_efficiency(const GemmShape& s, int pair_m, int sms) {
  const int64_t num_m = (s.M + pair_m - 1) / pair_m, num_n = (s.N + BLOCK_N - 1) / BLOCK_N;
  const int64_t tiles = num_m * num_n, pairs = sms / 2;
  const int64_t waves = (tiles + pairs - 1) / pairs;
  return ((double)s.M / (double)(num_m * pair_m)) * ((double)tiles / (double)(waves * pairs));
}

template <int A_MAJOR, int B_MAJOR, int EPI>
inline int launch_gemm_bf16(const void* A, int64_t lda, const void* B, int64_t ldb, const GemmShape& s,
                            const EpiParams& ep, cudaStream_t st) {
  const int64_t tiles2 = ((s.M + 511) / 512) * ((s.N + BLOCK_N - 1) / BLOCK_N);
  const int64_t min_tiles = tuning().mt2_min_tiles.load();
  // MT = 2 saves a quarter of the operand traffic; it is not worth more than ~10 % of idle MMA slots (padding of M
  // to 512 rows, fill of the last wave).  A positive OSDP_TUNE_MT2_MIN_TILES replaces that rule by a plain tile-count
  // threshold (tests use it to force MT = 2 on small shapes).
  DeviceInfo dev;
  const int drc = current_device(&dev);
  if (drc != OSDP_OK) return drc;
  const bool fits = min_tiles > 0 ? tiles2 >= min_tiles : tile_efficiency(s, 512, dev.sms) >= 0.9 * tile_efficiency(s, 256, dev.sms);
  const int64_t min_k = EpiTraits<EPI>::kF32Out ? tuning().mt2_min_k_acc.load() : tuning().mt2_min_k.load();
  if (s.K >= min_k && fits)
    return launch_gemm_bf16_mt<A_MAJOR, B_MAJOR, EPI, 2>(A, lda, B, ldb, s, ep, st);
  return launch_gemm_bf16_mt<A_MAJOR, B_MAJOR, EPI, 1>(A, lda, B, ldb, s, ep, st);
}

}  // namespace sm100
}  // namespace osdp
