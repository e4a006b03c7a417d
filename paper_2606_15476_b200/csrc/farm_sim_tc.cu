// farm_sim_tc.cu -- step 4 on the 5th-generation tensor cores (sm_100a: tcgen05.mma + TMEM + TMA).
//
//   cos(a_d, b_o) for every detection d and every object o of the entry snapshot (R14-R16; PAPER.md:350
//   "a single batched detection-by-entity similarity matrix").  A = detection rows [M, D], B = the map's
//   storage-dtype shadows [N, D], both K-major (D contiguous), bf16 or fp16 in, fp32 accumulate in TMEM.
//   The M x N result is never written: the epilogue scales every accumulator column by 1/|b_o|, keeps the
//   row maximum and its lowest-id argmax, and publishes clamp(max/|a_d|) with one atomicMax per row and
//   tile (R15, R18 tie rule, R19).
//
// Shape of the kernel (persistent, one CTA per SM, 256 threads):
//   warp 0      TMA producer: A tile 128 x 64 and B tile 256 x 64 per stage, SWIZZLE_128B, 4-stage mbarrier ring
//   warp 1      MMA issuer: one elected thread, tcgen05.mma.cta_group::1.kind::f16, UMMA 128 x 256 x 16
//   warp 2      TMEM allocator (512 columns = two 128 x 256 fp32 accumulators, double buffered)
//   warps 4-7   epilogue: tcgen05.ld 32 lanes x 32 columns at a time, one detection row per lane, four independent
//               (max, argmax) chains per thread so that the compare/select dependency chain stays short
//               (EPI_SPLIT = 2 puts two warps on each TMEM lane quadrant, each scanning half of the columns)
// Detections sit on the UMMA M axis (TMEM lanes) so that the per-detection max over objects is a scan
// along TMEM columns inside one thread -- no cross-thread reduction.
// N is read from device memory (no host sync); tiles are enumerated m-fastest so that concurrently
// running CTAs share the B tile in L2.
#include <cuda.h>

#include "farm_internal.cuh"

namespace farm {
FARM_TRACE_TABLE(farm_trace_clock)  // CTA 0 of the call's similarity kernel: [0] SM cycles, [1] nanoseconds of its lifetime
FARM_TRACE_TABLE(farm_trace_tiles)  // CTA 0: time its MMA issuer starts tile 0, 3, 6, ... (odd slots), epilogue done with tile 0, 6, 12, 18 (even)
FARM_TRACE_TABLE(farm_trace_sim)  // 0 first CTA start, 1 last prep wait over, 3 last scan wait over, 2 first phase-2 wait, 5 last phase-2 wait over, 7 end
namespace {

constexpr int BLOCK_M = 128;  // detections per tile (UMMA M)
constexpr int BLOCK_N = 256;  // objects per tile (UMMA N)
constexpr int BLOCK_K = 64;   // 64 x 16-bit = one 128-byte swizzle row
constexpr int UMMA_K = 16;
constexpr int STAGES = 4;
constexpr int EPI_SPLIT = 1;    // epilogue warps per TMEM lane quadrant (each scans BLOCK_N / EPI_SPLIT columns)
constexpr int EPI_THREADS = 128 * EPI_SPLIT;
constexpr int TC_THREADS = 128 + EPI_THREADS;  // warps 0-2 producer / MMA / TMEM, warp 3 idle, then the epilogue warps
constexpr uint32_t A_BYTES = BLOCK_M * BLOCK_K * 2;  // 16 KB
constexpr uint32_t B_BYTES = BLOCK_N * BLOCK_K * 2;  // 32 KB
constexpr uint32_t STAGE_BYTES = A_BYTES + B_BYTES;
constexpr uint32_t TMEM_COLS = 512;
constexpr size_t SMEM_BYTES = 1024 /*align slack*/ + STAGES * STAGE_BYTES + 2 * BLOCK_N * 4 + 256;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done, polls = 0;
  do {
    if (++polls == (1u << 28)) __trap();  // a protocol error must end the kernel, not hang the device
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
      "l"(map), "r"(bar), "r"(c0), "r"(c1)
      : "memory");
}
// ---- CTA-pair (cta_group::2) variants: a cluster of two CTAs computes a 256 x 256 tile, each CTA loading its own 128 rows of
// A and HALF of the B tile (the tensor cores of the pair share B), all transfers signalling the leader CTA's barrier
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t leader_addr(uint32_t local) {  // the same location in the shared memory of cluster rank 0
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, 0;" : "=r"(r) : "r"(local));
  return r;
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void tma_load_2d_pair(uint32_t dst, const CUtensorMap *map, uint32_t leader_bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
      "l"(map), "r"(leader_bar), "r"(c0), "r"(c1)
      : "memory");
}
__device__ __forceinline__ void umma_f16_pair(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit_pair(uint32_t bar) {  // arrives on the barrier at this offset in BOTH CTAs
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
               "h"((uint16_t)3)
               : "memory");
}

__device__ __forceinline__ void tcgen05_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tcgen05_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// shared-memory matrix descriptor: K-major operand, SWIZZLE_128B, rows of 128 bytes, 8-row groups 1024 B apart
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);  // start address, 16-byte units
  d |= (uint64_t)1 << 16;                   // leading byte offset (unused for swizzled K-major), 16-byte units
  d |= (uint64_t)(1024 >> 4) << 32;         // stride byte offset between 8-row core groups
  d |= (uint64_t)1 << 46;                   // descriptor version (sm_100)
  d |= (uint64_t)2 << 61;                   // SWIZZLE_128B
  return d;
}

__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}\n" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// 80 registers per thread (no spills): 256 x 80 leaves room for four 128 x 80 lift CTAs on the same SM
// NCTA = 2: CTA pairs (cluster of 2, tcgen05 cta_group::2, UMMA 256 x 256 x 16): per stage a CTA holds its A tile and half
// of the B tile (32 KB instead of 48 KB: six stages instead of four in the same shared memory, a third less L2 traffic).
//
// SPLIT (FARM_OPT_INPUTS_READY): the kernel of call c is enqueued with no dependency on the main stream and
// starts when the kernel of call c-1 ends, while that call's decision scan and merge are still to run.  R2 (every detection of
// call c sees the map as call c-1 left it) is kept by splitting the columns:
//   phase 1  the rows that existed at the entry of call c-1, n1 = n_hist[(seq-1)&1] of them, read as they are; the columns of
//            the objects call c-1 merges into (touch_seq[o] == seq-1, final once its scan is done: dm.scan_done) are masked
//            -- their rows may be half rewritten --, every other row is the same before and after that merge;
//   phase 2  once call c-1's merge warps are done (dm.merge_done): the rows they wrote -- merged old objects and new objects
//            -- which they also copied, with id and inverse norm, into dm.delta_*; extra tiles with the delta buffer as B.
// Both phases feed the same packed atomicMax per row, so the result is the row max / lowest-id argmax over exactly the rows of
// the map after call c-1.  The kernel also does the similarity's share of prep (row norms of A, cleared best_dense words).
struct SplitArgs {
  const void *A;  // the detection rows (what map_a describes)
  uint32_t seq, scan_target, merge_target;
};
template <bool EMIT, int NCTA, bool SPLIT>  // EMIT: pairs whose cosine exceeds m.dense_thr also go to the dense list (H1 prefilter / U1 edges)
__global__ void __maxnreg__(80)
similarity_tc_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b,
                     const __grid_constant__ CUtensorMap map_d, DevMap m, int M, uint32_t idesc, uint32_t prep_target, SplitArgs sp) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t *smem = (uint8_t *)(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);  // SWIZZLE_128B needs 1024-byte alignment
  constexpr int NSTAGES = NCTA == 2 ? 6 : STAGES;
  constexpr uint32_t B_LOAD_BYTES = B_BYTES / NCTA;              // B rows this CTA loads per stage
  constexpr uint32_t STG_BYTES = A_BYTES + B_LOAD_BYTES;         // 48 KB, or 32 KB for a CTA of a pair
  static_assert(NSTAGES * STG_BYTES == STAGES * STAGE_BYTES, "both variants use the same shared memory");
  float *ib_s = (float *)(smem + STAGES * STAGE_BYTES);                         // [2][BLOCK_N] inverse norms of B
  uint64_t *bars = (uint64_t *)(ib_s + 2 * BLOCK_N);
  uint64_t *full_bar = bars, *empty_bar = bars + NSTAGES, *tfull_bar = bars + 2 * NSTAGES, *tempty_bar = bars + 2 * NSTAGES + 2;
  uint32_t *tmem_slot = (uint32_t *)(bars + 2 * NSTAGES + 4);
  // Tile schedule of the CTA: static round-robin (tile = unit, unit + n_units, ...; a device-wide tile counter was measured
  // 1 % slower: the other kernels of a call slow all SMs alike).  With the split schedule the number of tiles is known only
  // when the previous call's merge is done, so the producer thread decides where the sequence ends and publishes the tiles,
  // tagged with their ordinal, in this ring; the MMA issuer and the epilogue follow it.  The producer is at most two accumulators
  // plus one shared-memory ring ahead of the epilogue, far less than the 8 entries.
  volatile unsigned long long *ring = (volatile unsigned long long *)(bars + 2 * NSTAGES + 6);
  static_assert((2 * 6 + 6 + 8) * 8 <= 256, "barriers, TMEM slot and tile ring fit the 256 bytes reserved for them");
  auto ring_get = [&](uint32_t k) -> int {
    unsigned long long e;
    do e = ring[k & 7]; while ((uint32_t)(e >> 32) != k + 1);
    return (int)(uint32_t)e;  // -1: no more tiles
  };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int N = SPLIT ? (int)__ldcg(&m.n_hist[(sp.seq - 1) & 1]) : (int)*m.n_objects;
  const int rank = NCTA == 2 ? (int)cluster_ctarank() : 0;       // rank 0 = leader: issues the MMAs of the pair
  const int unit = blockIdx.x / NCTA, n_units = gridDim.x / NCTA; // a unit = one CTA, or one CTA pair
  // tiles_m counts tiles of BLOCK_M * NCTA rows; CTA `rank` of a pair owns rows [tm * 256 + rank * 128, + 128)
  const int tiles_m = (M + BLOCK_M * NCTA - 1) / (BLOCK_M * NCTA), tiles_n = (N + BLOCK_N - 1) / BLOCK_N;
  const int n_tiles = tiles_m * tiles_n;
  const int k_blocks = (m.D + BLOCK_K - 1) / BLOCK_K;
  // SPLIT: number of tiles of both phases, known once call c-1's merge warps are done; every role asks when it gets there
  auto all_tiles = [&]() -> int {
    spin_until(m.merge_done, sp.merge_target, m.err);
    const int nd = (int)min(__ldcg(&m.delta_cnt[(sp.seq - 1) & 1]), m.max_det);
    return n_tiles + tiles_m * ((nd + BLOCK_N - 1) / BLOCK_N);
  };

  if (SPLIT && threadIdx.x == 0) TRACE_MIN(farm_trace_sim, sp.seq, 0), TRACE_MAX(farm_trace_sim, sp.seq, 1);
#ifdef FARM_TRACE
  long long trace_c0 = 0;
  unsigned long long trace_t0 = 0;
  if (blockIdx.x == 0 && threadIdx.x == 0) trace_c0 = clock64(), trace_t0 = gtime();
#endif
  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&map_a) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&map_b) : "memory");
    if (SPLIT) asm volatile("prefetch.tensormap [%0];" ::"l"(&map_d) : "memory");
  }
  if (threadIdx.x < 8) ring[threadIdx.x] = 0ull;
  if (warp == 1 && lane == 0) {
    for (int i = 0; i < NSTAGES; ++i) {
      mbar_init(smem_u32(&full_bar[i]), 1);
      mbar_init(smem_u32(&empty_bar[i]), 1);
    }
    for (int i = 0; i < 2; ++i) {
      mbar_init(smem_u32(&tfull_bar[i]), 1);
      mbar_init(smem_u32(&tempty_bar[i]), NCTA * EPI_THREADS / 32);  // the epilogue warps of BOTH CTAs of a pair
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 2) {
    if (NCTA == 2) {  // issued by the same warp of both CTAs of the pair
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(TMEM_COLS));
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(TMEM_COLS));
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
  }
  tcgen05_fence_before();
  __syncthreads();
  if (NCTA == 2) cluster_sync_all();  // the peer's barriers are initialised before anything signals them
  tcgen05_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      int n_all = SPLIT ? -1 : n_tiles;
      int cur = unit;
      for (uint32_t k = 0;; ++k) {
        int tile = cur;
        if (tile >= n_tiles) {
          if (SPLIT && n_all < 0) {
            n_all = all_tiles();
            asm volatile("fence.proxy.async;" ::: "memory");  // the delta rows were written through the generic proxy; TMA reads them
            // Split kernels are launched with programmatic stream serialisation and never wait for their predecessor (nothing
            // they read comes from it; the counters that tell calls apart are indexed by call parity): once every CTA is here,
            // CTAs of the next call's kernel take over the SMs as this kernel's CTAs exit -- many have no phase-2 tile -- instead
            // of after the whole grid plus a launch latency.  Not earlier than this point: a pending grid on the high-priority
            // stream keeps the other streams' grids from being dispatched, and until here this kernel still waits for one of
            // them (the previous call's merge).
            // Skinny call on a large map (one row tile, several rounds): no early trigger either -- the next call's CTAs cannot
            // all be resident beside this kernel's and would stay pending, in front of this call's probe kernel.
            if (!(tiles_m == 1 && n_tiles > n_units)) pdl_trigger();
          }
          if (tile >= n_all) tile = -1;
        }
        ring[k & 7] = ((unsigned long long)(k + 1) << 32) | (uint32_t)tile;
        if (tile < 0) break;
        cur += n_units;
        const bool ph2 = SPLIT && tile >= n_tiles;
        if (ph2) TRACE_MIN(farm_trace_tiles, sp.seq, 6), TRACE_MAX(farm_trace_tiles, sp.seq, 7);  // producer starts a phase-2 tile
        const int t2 = ph2 ? tile - n_tiles : tile;
        const int tm = t2 % tiles_m, tn = t2 / tiles_m;
        const CUtensorMap *mb = ph2 ? &map_d : &map_b;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(smem_u32(&empty_bar[stage]), phase ^ 1);
          const uint32_t fb = smem_u32(&full_bar[stage]);
          const uint32_t sa = smem_u32(smem + stage * STG_BYTES);
          if (NCTA == 2) {
            // the leader's barrier collects the bytes of both CTAs; the peer only issues its loads
            if (rank == 0) mbar_expect_tx(fb, 2 * STG_BYTES);
            const uint32_t lb = fb & 0xFEFFFFFFu;  // shared::cluster address of the same barrier in the pair's even CTA
            tma_load_2d_pair(sa, &map_a, lb, kb * BLOCK_K, (tm * NCTA + rank) * BLOCK_M);
            tma_load_2d_pair(sa + A_BYTES, &map_b, lb, kb * BLOCK_K, tn * BLOCK_N + rank * (BLOCK_N / NCTA));
          } else {
            mbar_expect_tx(fb, STG_BYTES);
            tma_load_2d(sa, &map_a, fb, kb * BLOCK_K, tm * BLOCK_M);
            tma_load_2d(sa + A_BYTES, mb, fb, kb * BLOCK_K, tn * BLOCK_N);
          }
          if (++stage == NSTAGES) stage = 0, phase ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0 && rank == 0) {  // a pair's MMAs are issued by its leader CTA alone
      uint32_t stage = 0, phase = 0, as = 0, aphase = 0;
      for (uint32_t k = 0;; ++k) {
        const int tile = ring_get(k);
        if (tile < 0) break;
        mbar_wait(smem_u32(&tempty_bar[as]), aphase ^ 1);  // epilogue has drained this accumulator (in both CTAs of a pair)
        tcgen05_fence_after();
#ifdef FARM_TRACE
        if (SPLIT && tile >= n_tiles) TRACE_MIN(farm_trace_tiles, sp.seq, 0), TRACE_MAX(farm_trace_tiles, sp.seq, 1);  // MMA of a phase-2 tile starts
#endif
        const uint32_t tmem_d = tmem_base + as * BLOCK_N;
        for (int kb = 0; kb < k_blocks; ++kb) {
          mbar_wait(smem_u32(&full_bar[stage]), phase);
          tcgen05_fence_after();
          const uint32_t sa = smem_u32(smem + stage * STG_BYTES);
          const uint64_t adesc = make_smem_desc(sa), bdesc = make_smem_desc(sa + A_BYTES);
#pragma unroll
          for (int k = 0; k < BLOCK_K / UMMA_K; ++k) {
            // advance 32 bytes (16 elements) along K inside the 128-byte swizzle row: +2 in 16-byte units
            if (NCTA == 2)
              umma_f16_pair(tmem_d, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (kb | k) != 0);
            else
              umma_f16(tmem_d, adesc + (uint64_t)(2 * k), bdesc + (uint64_t)(2 * k), idesc, (kb | k) != 0);
          }
          // frees the smem stage (in both CTAs of a pair) when these MMAs retire
          if (NCTA == 2) umma_commit_pair(smem_u32(&empty_bar[stage])); else umma_commit(smem_u32(&empty_bar[stage]));
          if (++stage == NSTAGES) stage = 0, phase ^= 1;
        }
        if (NCTA == 2) umma_commit_pair(smem_u32(&tfull_bar[as])); else umma_commit(smem_u32(&tfull_bar[as]));  // accumulator complete
        if (++as == 2) as = 0, aphase ^= 1;
      }
    }
  } else if (warp >= 4) {
    // ===== epilogue: one detection row per lane, half of the tile's columns per warp =====
    const int q = warp & 3;            // TMEM lane quadrant this warp may access
    const int half = (warp - 4) >> 2;  // which BLOCK_N / EPI_SPLIT column range of the tile this warp scans
    const int row_in_tile = q * 32 + lane;
    const int et = threadIdx.x - 128;  // 0..EPI_THREADS-1
    uint32_t as = 0, aphase = 0;
    if (SPLIT) {
      // the similarity's share of prep_kernel, with its arithmetic (same summation order: bit-identical norms): one warp per
      // row, rows unit, unit + n_units, ... of A; the main-stream prep skips them (CallArgs.split)
      const uint16_t *A16 = (const uint16_t *)sp.A;
      for (int r = unit + n_units * (warp - 4); r < M; r += n_units * (EPI_THREADS / 32)) {
        float s = 0.f;
        for (int i0 = lane * 8; i0 < m.D; i0 += 1024) {  // four loads in flight, then the sums in prep_kernel's order
          uint4 w4[4];
#pragma unroll
          for (int u = 0; u < 4; ++u)
            if (i0 + 256 * u < m.D) w4[u] = __ldg(reinterpret_cast<const uint4 *>(A16 + (size_t)r * m.D + i0 + 256 * u));
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (i0 + 256 * u < m.D) {
              const uint16_t *e = reinterpret_cast<const uint16_t *>(&w4[u]);
#pragma unroll
              for (int k = 0; k < 8; ++k) {
                const float x = m.dtype == FARM_DTYPE_F16 ? __half2float(__ushort_as_half(e[k])) : __uint_as_float((uint32_t)e[k] << 16);
                s = fmaf(x, x, s);
              }
            }
          }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
        if (lane == 0) m.det_inv_norm[r] = s > 0.f ? 1.0f / sqrtf(s) : 0.f, m.best_dense[r] = 0ull;
      }
      __threadfence();
      asm volatile("bar.sync 1, %0;" ::"n"(EPI_THREADS) : "memory");
      if (et == 0) TRACE_MAX(farm_trace_sim, sp.seq, 3), TRACE_MIN(farm_trace_sim, sp.seq, 6);
      if (et == 0) atomicAdd(m.prep_done, 1u);
    }
    // prep_kernel (main stream) may still be running: its row norms and the zeroed best_dense words are first
    // needed here, one tile of MMAs after the kernel started
    spin_until(m.prep_done, prep_target, m.err);  // bounded: sticky ERR_SYNC_TIMEOUT instead of a hang
    if (SPLIT) spin_until(m.scan_done, sp.scan_target, m.err);  // touch_seq of call c-1 is final
    const uint32_t tempty_leader0 = NCTA == 2 ? leader_addr(smem_u32(&tempty_bar[0])) : 0u;
    for (uint32_t k = 0;; ++k) {
      const int tile = ring_get(k);
      if (tile < 0) break;
      if (SPLIT && tile >= n_tiles) {
        if (et == 0) TRACE_MIN(farm_trace_sim, sp.seq, 2), TRACE_MAX(farm_trace_sim, sp.seq, 5);
        // ---- phase 2: B = the delta rows of call c-1; column k of the tile is object delta_id[n0 + k].  The ids are in no
        // order, so R15 / R18 are applied literally: clamp first, then larger cosine wins, equal cosines -> lower id.
        const int t2 = tile - n_tiles;
        const int tm = t2 % tiles_m, n0 = (t2 / tiles_m) * BLOCK_N;
        const int ncols = min(BLOCK_N, (int)min(__ldcg(&m.delta_cnt[(sp.seq - 1) & 1]), m.max_det) - n0);
        float *ib = ib_s + as * BLOCK_N;
#pragma unroll
        for (int c = et; c < BLOCK_N; c += EPI_THREADS) ib[c] = c < ncols ? __ldcg(&m.delta_inv[n0 + c]) : 0.f;
        const int row = tm * BLOCK_M + row_in_tile;
        const bool row_ok = row < M;
        const float ia = row_ok ? m.det_inv_norm[row] : 0.f;
        asm volatile("bar.sync 1, %0;" ::"n"(EPI_THREADS) : "memory");
        mbar_wait(smem_u32(&tfull_bar[as]), aphase);
        tcgen05_fence_after();
        if (et == 0) TRACE_MIN(farm_trace_tiles, sp.seq, 2), TRACE_MAX(farm_trace_tiles, sp.seq, 3);  // accumulator of a phase-2 tile complete
        // the id of a column is needed only to break an exact tie (or for a zero-norm row, which ties everywhere): the common
        // path keeps the column and looks the id up once at the end
        float best = -3.0e38f;
        int bcol = -1;
        bool tie = false;  // some column equals the running maximum: decided by id in a second pass (rare: duplicate rows)
        const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BLOCK_N;
        const bool scan_row = row_ok && ia != 0.f;
#pragma unroll 1
        for (int c0 = 0; c0 < ncols; c0 += 32) {
          uint32_t r[32];
          tmem_ld32(taddr + c0, r);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float cs = fminf(1.f, fmaxf(-1.f, __uint_as_float(r[i]) * ib[c0 + i] * ia));
            const bool in = c0 + i < ncols;
            tie = (in && cs == best) ? true : ((in && cs > best) ? false : tie);
            if (in && cs > best) best = cs, bcol = c0 + i;
          }
        }
        if (__any_sync(0xFFFFFFFFu, scan_row && tie)) {  // lowest id among the columns that reach the maximum
          uint32_t low = bcol >= 0 ? __ldcg(&m.delta_id[n0 + bcol]) : 0xFFFFFFFFu;
#pragma unroll 1
          for (int c0 = 0; c0 < ncols; c0 += 32) {
            uint32_t r[32];
            tmem_ld32(taddr + c0, r);
            tmem_ld_wait();
#pragma unroll 1
            for (int i = 0; i < 32; ++i) {
              const float cs = fminf(1.f, fmaxf(-1.f, __uint_as_float(r[i]) * ib[c0 + i] * ia));
              if (scan_row && tie && c0 + i < ncols && cs == best) {
                const uint32_t id = __ldcg(&m.delta_id[n0 + c0 + i]);
                if (id < low) low = id, bcol = c0 + i;
              }
            }
          }
        }
        if (!scan_row) bcol = -1;
        uint32_t best_id = bcol >= 0 ? __ldcg(&m.delta_id[n0 + bcol]) : 0xFFFFFFFFu;
        if (row_ok && ia == 0.f) {  // cosine 0 with every object: the lowest id of the tile
          best = 0.f;
          for (int c = 0; c < ncols; ++c) best_id = min(best_id, __ldcg(&m.delta_id[n0 + c]));
        }
        tcgen05_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(smem_u32(&tempty_bar[as]));
        if (row_ok && best_id != 0xFFFFFFFFu) atomicMax(&m.best_dense[row], pack_score(best, best_id));
        if (et == 0) TRACE_MIN(farm_trace_tiles, sp.seq, 4), TRACE_MAX(farm_trace_tiles, sp.seq, 5);  // epilogue of a phase-2 tile done
        if (++as == 2) as = 0, aphase ^= 1;
        continue;
      }
      const int tm = (tile % tiles_m) * NCTA + rank, tn = tile / tiles_m;
      const int n0 = tn * BLOCK_N;
      const int ncols = min(BLOCK_N, N - n0);
      float *ib = ib_s + as * BLOCK_N;
      if (SPLIT) {  // a column whose object call c-1 merges into: NaN never wins a comparison below; phase 2 brings its new row
        const float masked = __int_as_float(0x7FC00000);
#pragma unroll
        for (int c = et; c < BLOCK_N; c += EPI_THREADS)
          ib[c] = c < ncols ? (__ldcg(&m.touch_seq[n0 + c]) == sp.seq - 1 ? masked : m.inv_norm[n0 + c]) : 0.f;
      } else {
#pragma unroll
        for (int c = et; c < BLOCK_N; c += EPI_THREADS) ib[c] = c < ncols ? m.inv_norm[n0 + c] : 0.f;
      }
      const int cbeg = half * (BLOCK_N / EPI_SPLIT);
      const int row = tm * BLOCK_M + row_in_tile;
      const bool row_ok = row < M && cbeg < ncols;
      const float ia = row_ok ? m.det_inv_norm[row] : 0.f;  // requested before the wait for the accumulator
      asm volatile("bar.sync 1, %0;" ::"n"(EPI_THREADS) : "memory");
      mbar_wait(smem_u32(&tfull_bar[as]), aphase);
      tcgen05_fence_after();
      // four interleaved chains (columns = chain mod 4): strict > keeps the lowest column inside a chain
      float bv[4] = {-3.0e38f, -3.0e38f, -3.0e38f, -3.0e38f};
      int bc[4] = {0, 1, 2, 3};
      // raw threshold of the row: acc * ib > thr / ia  <=>  cos > thr (slightly low: the exact test follows in the emit)
      const float thr_t = m.dense_thr / ia;
      const float thr_row = (EMIT && row_ok && ia > 0.f) ? thr_t - fabsf(thr_t) * 1e-5f - 1e-30f : 3.0e38f;
      const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + as * BLOCK_N;
#pragma unroll 1
      for (int c0 = cbeg; c0 < cbeg + BLOCK_N / EPI_SPLIT; c0 += 32) {
        if (c0 >= ncols) break;
        uint32_t r[32];
        tmem_ld32(taddr + c0, r);
        tmem_ld_wait();
        if (c0 + 32 <= ncols) {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float v = __uint_as_float(r[i]) * ib[c0 + i];
            if (v > bv[i & 3]) bv[i & 3] = v, bc[i & 3] = c0 + i;
            if (EMIT && v > thr_row) {
              const float cs = fminf(1.f, fmaxf(-1.f, v * ia));
              if (cs > m.dense_thr) dense_emit(m, (uint32_t)row, (uint32_t)(n0 + c0 + i), cs);
            }
          }
        } else {
#pragma unroll
          for (int i = 0; i < 32; ++i) {
            const float v = __uint_as_float(r[i]) * ib[c0 + i];
            if (c0 + i < ncols && v > bv[i & 3]) bv[i & 3] = v, bc[i & 3] = c0 + i;
            if (EMIT && c0 + i < ncols && v > thr_row) {
              const float cs = fminf(1.f, fmaxf(-1.f, v * ia));
              if (cs > m.dense_thr) dense_emit(m, (uint32_t)row, (uint32_t)(n0 + c0 + i), cs);
            }
          }
        }
      }
      // combine the chains: larger value wins, equal values -> lower column (R18 tie rule)
      float best = bv[0];
      int best_c = bc[0];
#pragma unroll
      for (int k = 1; k < 4; ++k)
        if (bv[k] > best || (bv[k] == best && bc[k] < best_c)) best = bv[k], best_c = bc[k];
      float cs = best * ia;
      // R15 clamps before R18 compares: every column whose cosine reaches 1 ties at exactly 1.0 and the lowest id wins.
      // Rare (duplicates of the detection in the map): the warp re-scans its accumulator for the first such column.
      const bool sat = row_ok && cs >= 1.0f;
      if (__any_sync(0xFFFFFFFFu, sat)) {
        int first = best_c;
#pragma unroll 1
        for (int c0 = cbeg; c0 < cbeg + BLOCK_N / EPI_SPLIT; c0 += 32) {
          if (c0 >= ncols) break;
          uint32_t r[32];
          tmem_ld32(taddr + c0, r);
          tmem_ld_wait();
#pragma unroll
          for (int i = 0; i < 32; ++i)
            if (sat && c0 + i < ncols && c0 + i < first && __uint_as_float(r[i]) * ib[c0 + i] * ia >= 1.0f) first = c0 + i;
        }
        best_c = first;
      }
      tcgen05_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (NCTA == 2) mbar_arrive_remote(tempty_leader0 + as * 8u); else mbar_arrive(smem_u32(&tempty_bar[as]));
      }
      if (row_ok && (!SPLIT || best > -2.0e38f || ia == 0.f)) {  // SPLIT: a row of a tile whose columns are all masked has nothing to say
        cs = fminf(1.f, fmaxf(-1.f, cs));                    // R15 clamp
        if (ia == 0.f) cs = 0.f, best_c = 0;                 // zero-norm detection: cos = 0 for every object
        atomicMax(&m.best_dense[row], pack_score(cs, (uint32_t)(n0 + best_c)));
      }
      if (++as == 2) as = 0, aphase ^= 1;

    }
  }
  tcgen05_fence_before();
  __threadfence();  // the epilogue's atomicMax results precede the completion count below
  __syncthreads();
  if (SPLIT && threadIdx.x == 0) TRACE_MAX(farm_trace_sim, sp.seq, 7);
#ifdef FARM_TRACE
  if (blockIdx.x == 0 && threadIdx.x == 0) {  // SM clock of CTA 0 over its lifetime: cycles and nanoseconds
    farm_trace_clock[sp.seq & 15][0] = (unsigned long long)(clock64() - trace_c0);
    farm_trace_clock[sp.seq & 15][1] = gtime() - trace_t0;
  }
#endif
  if (threadIdx.x == 0) atomicAdd(m.sim_done + (sp.seq & 1), 1u);  // cand_associate's decision scan waits for every CTA of this grid
  if (NCTA == 2) cluster_sync_all();  // no CTA of a pair leaves (or frees TMEM) while its peer still uses the pair's resources
  if (warp == 2) {
    tcgen05_fence_after();
    if (NCTA == 2)
      asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS));
    else
      asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS));
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TcState {
  EncodeTiledFn encode = nullptr;
  CUtensorMap map_a, map_b;  // map_a is re-encoded per call by tc_prepare (host work only)
  CUtensorMap map_b_half;    // CTA pairs: each CTA loads half of the B tile
  CUtensorMap map_d;         // split schedule: the delta rows (phase 2)
  bool has_delta = false;
  uint32_t idesc_pair = 0;
  int pair = 0;              // 1: launch CTA pairs (cluster of 2, cta_group::2)
  CUtensorMapDataType dt;
  uint32_t idesc;
  bool ok = false;
};

bool encode_2d(TcState *st, CUtensorMap *map, const void *base, uint64_t rows, uint64_t cols, uint32_t box_rows) {
  const cuuint64_t gdim[2] = {cols, rows};
  const cuuint64_t gstride[1] = {cols * 2};
  const cuuint32_t box[2] = {(cuuint32_t)BLOCK_K, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  return st->encode(map, st->dt, 2, const_cast<void *>(base), gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

bool tc_supported(const DevMap &m) { return m.dtype != FARM_DTYPE_F32 && m.D % 8 == 0 && m.D >= 8; }

void *tc_state_create(const DevMap &m) {
  TcState *st = new TcState();
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    delete st;
    return nullptr;
  }
  st->encode = (EncodeTiledFn)fn;
  st->dt = m.dtype == FARM_DTYPE_F16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_BFLOAT16;
  const uint32_t fmt = m.dtype == FARM_DTYPE_F16 ? 0u : 1u;
  // instruction descriptor, kind::f16: D = fp32, A/B = fmt, both K-major, N = 256, M = 128
  st->idesc = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(BLOCK_N >> 3) << 17) | ((uint32_t)(BLOCK_M >> 4) << 24);
  st->idesc_pair = (1u << 4) | (fmt << 7) | (fmt << 10) | ((uint32_t)(BLOCK_N >> 3) << 17) | ((uint32_t)((2 * BLOCK_M) >> 4) << 24);
  if (!encode_2d(st, &st->map_b, m.desc_shadow, m.max_objects, (uint64_t)m.D, BLOCK_N) ||
      !encode_2d(st, &st->map_b_half, m.desc_shadow, m.max_objects, (uint64_t)m.D, BLOCK_N / 2)) {
    delete st;
    return nullptr;
  }
  if (m.delta_rows) {
    if (!encode_2d(st, &st->map_d, m.delta_rows, m.max_det, (uint64_t)m.D, BLOCK_N)) {
      delete st;
      return nullptr;
    }
    st->has_delta = true;
  } else {
    st->map_d = st->map_b;  // never read
  }
  if (cudaFuncSetAttribute(similarity_tc_kernel<false, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<true, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<false, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<true, 2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<false, 1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess) {
    delete st;
    return nullptr;
  }
  st->ok = true;
  return st;
}

void tc_state_destroy(void *p) { delete (TcState *)p; }
void tc_state_set_pair(void *p, int pair) { ((TcState *)p)->pair = pair; }

// Encode the call's A operand (detection rows).  Called before anything of the call is enqueued, so that a
// descriptor pointer TMA cannot address (not 16-byte aligned) fails the call with the map untouched.
bool tc_prepare(void *state, const DevMap &m, const CallArgs &a) {
  TcState *st = (TcState *)state;
  if (a.M == 0) return true;
  if (((uintptr_t)a.desc & 15) != 0) return false;
  return encode_2d(st, &st->map_a, a.desc, (uint64_t)a.M, (uint64_t)m.D, BLOCK_M);
}

// prep_target: value dm.prep_done has when prep_kernel's CTAs of this call are done; with the split schedule (a.split) the
// kernel does that share itself and the value becomes prep_target + its own CTAs (returned through *prep_after).
int launch_similarity_tc(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s, void *state, uint32_t prep_target,
                         int *n_ctas, uint32_t *prep_after) {
  TcState *st = (TcState *)state;
  if (prep_after) *prep_after = prep_target;
  if (a.M == 0 || n_upper == 0) return 0;
  const CUtensorMap &map_a = st->map_a;
  const bool emit = m.dense_d && m.dense_thr < 2.0f;
  SplitArgs sp = {a.desc, a.seq, a.scan_target, a.merge_target};
  int grid;
  if (st->pair) {  // CTA pairs: one cluster of two CTAs per 256 x 256 tile
    const long long tiles = (long long)((a.M + 2 * BLOCK_M - 1) / (2 * BLOCK_M)) * ((n_upper + BLOCK_N - 1) / BLOCK_N);
    grid = 2 * (int)(tiles < m.num_sms / 2 ? tiles : m.num_sms / 2);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid), cfg.blockDim = dim3(TC_THREADS), cfg.dynamicSmemBytes = SMEM_BYTES, cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2, attr[0].val.clusterDim.y = 1, attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr, cfg.numAttrs = 1;
    const cudaError_t e =
        emit ? cudaLaunchKernelEx(&cfg, similarity_tc_kernel<true, 2, false>, map_a, st->map_b_half, st->map_d, m, a.M, st->idesc_pair, prep_target, sp)
             : cudaLaunchKernelEx(&cfg, similarity_tc_kernel<false, 2, false>, map_a, st->map_b_half, st->map_d, m, a.M, st->idesc_pair, prep_target, sp);
    if (e != cudaSuccess) return -1;
  } else {
    // split: phase 2 adds up to ceil(max touched rows / 256) column tiles; the grid is sized on the rows known to the host
    const long long tiles = (long long)((a.M + BLOCK_M - 1) / BLOCK_M) * ((n_upper + BLOCK_N - 1) / BLOCK_N);
    grid = (int)(tiles < m.num_sms ? tiles : m.num_sms);
    if (a.M <= BLOCK_M && tiles > m.num_sms) {
      // Skinny call on a large map (one row tile, more column tiles than SMs): every B tile is streamed from HBM once, and a last
      // round with a few CTAs cannot keep enough loads in flight to use the bandwidth.  Same number of rounds for every CTA.
      const long long rounds = (tiles + m.num_sms - 1) / m.num_sms;
      grid = (int)((tiles + rounds - 1) / rounds);
    }
    if (a.split) {
      if (prep_after) *prep_after = prep_target + (uint32_t)grid;
      if (launch_pdl(similarity_tc_kernel<false, 1, true>, dim3(grid), dim3(TC_THREADS), SMEM_BYTES, s, map_a, st->map_b, st->map_d, m, a.M,
                     st->idesc, prep_target + (uint32_t)grid, sp) != cudaSuccess)
        return -1;
    } else if (emit) {
      similarity_tc_kernel<true, 1, false><<<grid, TC_THREADS, SMEM_BYTES, s>>>(map_a, st->map_b, st->map_d, m, a.M, st->idesc, prep_target, sp);
    } else {
      similarity_tc_kernel<false, 1, false><<<grid, TC_THREADS, SMEM_BYTES, s>>>(map_a, st->map_b, st->map_d, m, a.M, st->idesc, prep_target, sp);
    }
  }
  if (n_ctas) *n_ctas = grid;
  return 1;
}

bool tc_can_split(void *state) { return state && ((TcState *)state)->has_delta && !((TcState *)state)->pair; }

}  // namespace farm
