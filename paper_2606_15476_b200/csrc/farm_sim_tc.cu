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
template <bool EMIT, int NCTA>  // EMIT: pairs whose cosine exceeds m.dense_thr also go to the dense list (H1 prefilter / U1 edges)
__global__ void __maxnreg__(80)
similarity_tc_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b, DevMap m,
                     int M, uint32_t idesc, uint32_t prep_target) {
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

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int N = (int)*m.n_objects;
  const int rank = NCTA == 2 ? (int)cluster_ctarank() : 0;       // rank 0 = leader: issues the MMAs of the pair
  const int unit = blockIdx.x / NCTA, n_units = gridDim.x / NCTA; // a unit = one CTA, or one CTA pair
  // tiles_m counts tiles of BLOCK_M * NCTA rows; CTA `rank` of a pair owns rows [tm * 256 + rank * 128, + 128)
  const int tiles_m = (M + BLOCK_M * NCTA - 1) / (BLOCK_M * NCTA), tiles_n = (N + BLOCK_N - 1) / BLOCK_N;
  const int n_tiles = tiles_m * tiles_n;
  const int k_blocks = (m.D + BLOCK_K - 1) / BLOCK_K;

  if (warp == 0 && lane == 0) {
    asm volatile("prefetch.tensormap [%0];" ::"l"(&map_a) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&map_b) : "memory");
  }
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
      for (int tile = unit; tile < n_tiles; tile += n_units) {
        const int tm = tile % tiles_m, tn = tile / tiles_m;
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
            tma_load_2d(sa + A_BYTES, &map_b, fb, kb * BLOCK_K, tn * BLOCK_N);
          }
          if (++stage == NSTAGES) stage = 0, phase ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer =====
    if (lane == 0 && rank == 0) {  // a pair's MMAs are issued by its leader CTA alone
      uint32_t stage = 0, phase = 0, as = 0, aphase = 0;
      for (int tile = unit; tile < n_tiles; tile += n_units) {
        mbar_wait(smem_u32(&tempty_bar[as]), aphase ^ 1);  // epilogue has drained this accumulator (in both CTAs of a pair)
        tcgen05_fence_after();
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
    // prep_kernel (main stream) may still be running: its row norms and the zeroed best_dense words are first
    // needed here, one tile of MMAs after the kernel started
    spin_until(m.prep_done, prep_target, m.err);  // bounded: sticky ERR_SYNC_TIMEOUT instead of a hang
    const uint32_t tempty_leader0 = NCTA == 2 ? leader_addr(smem_u32(&tempty_bar[0])) : 0u;
    for (int tile = unit; tile < n_tiles; tile += n_units) {
      const int tm = (tile % tiles_m) * NCTA + rank, tn = tile / tiles_m;
      const int n0 = tn * BLOCK_N;
      const int ncols = min(BLOCK_N, N - n0);
      float *ib = ib_s + as * BLOCK_N;
#pragma unroll
      for (int c = et; c < BLOCK_N; c += EPI_THREADS) ib[c] = c < ncols ? m.inv_norm[n0 + c] : 0.f;
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
      if (row_ok) {
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
  if (threadIdx.x == 0) atomicAdd(m.sim_done, 1u);  // cand_associate's decision scan waits for every CTA of this grid
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
  if (cudaFuncSetAttribute(similarity_tc_kernel<false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess ||
      cudaFuncSetAttribute(similarity_tc_kernel<true, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_BYTES) != cudaSuccess) {
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

int launch_similarity_tc(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s, void *state, uint32_t prep_target,
                         int *n_ctas) {
  TcState *st = (TcState *)state;
  if (a.M == 0 || n_upper == 0) return 0;
  const CUtensorMap &map_a = st->map_a;
  const bool emit = m.dense_d && m.dense_thr < 2.0f;
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
    const cudaError_t e = emit ? cudaLaunchKernelEx(&cfg, similarity_tc_kernel<true, 2>, map_a, st->map_b_half, m, a.M, st->idesc_pair, prep_target)
                               : cudaLaunchKernelEx(&cfg, similarity_tc_kernel<false, 2>, map_a, st->map_b_half, m, a.M, st->idesc_pair, prep_target);
    if (e != cudaSuccess) return -1;
  } else {
    const long long tiles = (long long)((a.M + BLOCK_M - 1) / BLOCK_M) * ((n_upper + BLOCK_N - 1) / BLOCK_N);
    grid = (int)(tiles < m.num_sms ? tiles : m.num_sms);
    if (emit)
      similarity_tc_kernel<true, 1><<<grid, TC_THREADS, SMEM_BYTES, s>>>(map_a, st->map_b, m, a.M, st->idesc, prep_target);
    else
      similarity_tc_kernel<false, 1><<<grid, TC_THREADS, SMEM_BYTES, s>>>(map_a, st->map_b, m, a.M, st->idesc, prep_target);
  }
  if (n_ctas) *n_ctas = grid;
  return 1;
}

}  // namespace farm
