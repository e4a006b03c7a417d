// farm_lift.cu -- steps 1-3 of the hot path:
//   lift_voxelise_kernel  back-project masked pixels (R5), quantise to voxel keys (R6), aggregate the keys of
//                         a pixel tile per (detection, 4x4x4 voxel block) into 64-bit voxel masks (R7)
//   probe_kernel          find / insert the blocks in the global voxel-block hash (R11, R12 pass 1), make the
//                         (detection, voxel) pairs exact and build the sparse overlap histogram (R9)
// BASELINE.json north_star steps (1)-(3); PAPER.md:65, 347 ("masked depth points").
//
// The mandatory traffic is 6 B/pixel of depth+mask (128-bit loads) plus, per distinct (detection, block)
// pair, one 8-byte key probe and the 32-byte owner sectors of the voxels the detection touches.
#include "farm_internal.cuh"

namespace farm {
FARM_TRACE_TABLE(farm_trace_probe)  // probe kernel: 0 first CTA resident; last warp with records past 1 its record loads, 3 the block hash, 5 the pair set, 7 phase B
FARM_TRACE_TABLE(farm_trace_lift)  // 0 / 1 lift first CTA start / last CTA end, 2 / 3 probe first CTA past its wait / last CTA end, 4 prep start

namespace {

constexpr int TILE_W = 64;        // 8 threads x 8 pixels per row
constexpr int TILE_H = 16;
constexpr int LIFT_THREADS = 128;
constexpr int LIFT_WARPS = LIFT_THREADS / 32;
constexpr int TILE_ENT = 128;     // (detection, block) entries per tile; overflow goes straight to the global queue
constexpr int STAGE_PX = 128;     // compacted pixels per warp and round (4 of a lane's 8 pixels)
constexpr int MAX_LABELS = 32;    // per-tile detection accumulators (the entry tag holds a 5-bit label slot)
constexpr int LABEL_SHIFT = 57;   // block keys use bits 0..56
constexpr uint32_t NONE32 = 0xFFFFFFFFu;

struct Camera {
  float inv_fx, inv_fy, cx, cy;
  float r[9], t[3];
};

__device__ __forceinline__ Camera load_camera(const float *__restrict__ K, const float *__restrict__ T) {
  Camera c;
  c.inv_fx = __fdiv_rn(1.0f, __ldg(K + 0));  // R5: IEEE fp32 reciprocal, once per frame
  c.inv_fy = __fdiv_rn(1.0f, __ldg(K + 4));
  c.cx = __ldg(K + 2);
  c.cy = __ldg(K + 5);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    c.r[3 * i + 0] = __ldg(T + 4 * i + 0);
    c.r[3 * i + 1] = __ldg(T + 4 * i + 1);
    c.r[3 * i + 2] = __ldg(T + 4 * i + 2);
    c.t[i] = __ldg(T + 4 * i + 3);
  }
  return c;
}

// R5: every multiply and add individually rounded (the _rn intrinsics are never contracted into FMA).
__device__ __forceinline__ void backproject(const Camera &c, int u, int v, float z, float p[3]) {
  const float xn = __fmul_rn(__fsub_rn((float)u, c.cx), c.inv_fx);
  const float yn = __fmul_rn(__fsub_rn((float)v, c.cy), c.inv_fy);
  const float xc = __fmul_rn(xn, z), yc = __fmul_rn(yn, z);
#pragma unroll
  for (int i = 0; i < 3; ++i)
    p[i] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c.r[3 * i], xc), __fmul_rn(c.r[3 * i + 1], yc)),
                               __fmul_rn(c.r[3 * i + 2], z)),
                     c.t[i]);
}

// R6: index = floor(fp32(X * inv_vs)) per axis, valid iff in [-2^20, 2^20).  cvt.rmi (round towards -inf,
// saturating) is floor-then-convert in one instruction; the float pre-test rejects NaN and anything the
// saturation would alias.
__device__ __forceinline__ bool voxel_index(const float p[3], float inv_vs, uint32_t &ix, uint32_t &iy, uint32_t &iz) {
  const float fx = __fmul_rn(p[0], inv_vs), fy = __fmul_rn(p[1], inv_vs), fz = __fmul_rn(p[2], inv_vs);
  const bool finite = fabsf(fx) < 2.0e6f && fabsf(fy) < 2.0e6f && fabsf(fz) < 2.0e6f;
  ix = (uint32_t)(__float2int_rd(fx) + KEY_BIAS), iy = (uint32_t)(__float2int_rd(fy) + KEY_BIAS),
  iz = (uint32_t)(__float2int_rd(fz) + KEY_BIAS);
  return finite && ((ix | iy | iz) >> 21) == 0;
}
__device__ __forceinline__ bool voxel_key(const float p[3], float inv_vs, unsigned long long *key) {
  uint32_t ix, iy, iz;
  if (!voxel_index(p, inv_vs, ix, iy, iz)) return false;
  const uint32_t lo = iz | (iy << 21), hi = (iy >> 11) | (ix << 10);
  *key = ((unsigned long long)hi << 32) | lo;
  return true;
}

__device__ __forceinline__ bool depth_valid(float z, float z_min, float z_max) {
  return (fabsf(z) <= 3.402823466e+38f) && z > z_min && z <= z_max;  // finite, in (z_min, z_max]  (R4)
}

// ---------------------------------------------------------------------------------------------------
// prep: reset per-call state and compute detection row norms (operand A of step 4).  One warp per row.
// With the split schedule (CallArgs.split) the kernel runs on the lift's stream ahead of the previous call's tail -- everything it
// resets is double buffered by call parity -- and leaves the row norms and best_dense to the similarity kernel.
template <typename T>
__global__ void prep_kernel(DevMap m, CallArgs a) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    TRACE_MIN(farm_trace_lift, a.seq, 4);
    m.counters[0] = 0;
    m.counters[1] = 0;
    m.counters[4] = 0, m.counters[5] = 0, m.counters[6] = 0, m.counters[7] = 0, m.counters[8] = 0;
    *m.surv_cnt = 0;
    CallStats z = {};
    z.n_det = (uint32_t)a.M;
    *m.stats = z;
  }
  if (blockIdx.x == 0 && (int)threadIdx.x < a.F) {  // per-frame camera block of the lift kernel (R5 reciprocals)
    const Camera c = load_camera(a.K + 9 * threadIdx.x, a.T + 16 * threadIdx.x);
    float *o = m.cam + 16 * threadIdx.x;
    o[0] = c.inv_fx, o[1] = c.inv_fy, o[2] = c.cx, o[3] = c.cy;
#pragma unroll
    for (int i = 0; i < 3; ++i) o[4 + 4 * i] = c.r[3 * i], o[5 + 4 * i] = c.r[3 * i + 1], o[6 + 4 * i] = c.r[3 * i + 2], o[7 + 4 * i] = c.t[i];
  }
  if (warp < a.M) {
    const T *row = (const T *)a.desc + (size_t)warp * m.D;
    float s = 0.f;
    if (a.split) {
      // the similarity kernel (split schedule) computes the row norms and clears best_dense itself
    } else if (sizeof(T) == 2 && (m.D & 7) == 0 && (((uintptr_t)a.desc) & 15) == 0) {  // 128-bit loads, 8 elements each
      for (int i = lane * 8; i < m.D; i += 256) {
        const uint4 w = __ldg(reinterpret_cast<const uint4 *>(row + i));
        const T *e = reinterpret_cast<const T *>(&w);
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const float x = to_f32<T>(e[q]);
          s = fmaf(x, x, s);
        }
      }
    } else {
      for (int i = lane; i < m.D; i += 32) {
        const float x = to_f32<T>(row[i]);
        s = fmaf(x, x, s);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
    if (lane == 0) {
      if (!a.split) m.det_inv_norm[warp] = s > 0.f ? 1.0f / sqrtf(s) : 0.f, m.best_dense[warp] = 0ull;
      m.det_nv[warp] = 0;
      m.det_npx[warp] = 0;
      m.best_cand[warp] = 0ull;
      m.assoc[warp] = -1;
      m.is_new[warp] = 0;
      m.best_score[warp] = 0.f;
      if (m.det_flags) m.det_flags[warp] = 0;
    }
    if (lane < 6) m.det_box[warp * 6 + lane] = lane < 3 ? 0x7FFFFFFF : (int)0x80000000;
    if (m.det_gm) {
      if (lane < 9) m.det_gm[(size_t)warp * 9 + lane] = 0.0;
      if (lane == 9) m.hell[warp] = -1.f;
    }
  }
  // publish: the similarity kernel runs on another stream and waits for every prep CTA before its first epilogue
  if (a.split) return;  // nothing of this kernel is awaited through prep_done then
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(m.prep_done, 1u);
  }
}


// ---------------------------------------------------------------------------------------------------
// per-call scratch helpers

// epoch-tagged set/map insert: entries whose epoch field differs from `epoch` count as free.
// returns 1 = newly inserted, 0 = already present, -1 = table full.
__device__ __forceinline__ int epoch_insert(unsigned long long *tab, uint32_t mask, unsigned long long v,
                                            uint32_t epoch, uint32_t *slot) {
  uint32_t h = hash32((uint32_t)v, (uint32_t)(v >> 32) * 0x632BE5ABu) & mask;
  for (uint32_t probe = 0; probe <= mask; ++probe) {
    unsigned long long cur = __ldcg(&tab[h]);
    for (;;) {
      if (cur == v) {
        *slot = h;
        return 0;
      }
      if ((uint32_t)(cur >> 48) == epoch) break;  // live entry of another pair
      const unsigned long long old = atomicCAS(&tab[h], cur, v);
      if (old == cur) {
        *slot = h;
        return 1;
      }
      cur = old;
    }
    h = (h + 1) & mask;
    if (probe > 8192) break;
  }
  return -1;
}

// write one (block, detection, voxel bits) record of the call's survivor queue
__device__ __forceinline__ void survivor_store(const DevMap &m, uint32_t pos, unsigned long long bkey, uint32_t j,
                                               uint32_t lo, uint32_t hi) {
  if (pos < m.surv_cap) {
    m.surv_key[pos] = bkey;
    m.surv_bits[pos] = ((unsigned long long)hi << 32) | lo;
    m.surv_j[pos] = j;
  } else {
    atomicOr(m.err, ERR_PAIR_TABLE_FULL);
  }
}

struct TileSmem {
  unsigned long long tag[TILE_ENT];       // block key | label slot << 57, BLK_EMPTY when free
  uint32_t mlo[TILE_ENT], mhi[TILE_ENT];  // voxel bits of the block seen for that detection inside the tile
  unsigned long long stage[LIFT_WARPS][STAGE_PX + 1];  // per warp, the compacted masked pixels of one round (+ a dump slot):
                                                   // (label << 16 | row in tile << 8 | column in tile) << 32 | depth bits
  uint32_t q_count;                       // entries flushed by the tile that just finished
  uint32_t cur_pos, cur_end;              // the CTA's current chunk of the survivor queue
  uint32_t next_base, next_valid;         // the chunk reserved after it
  uint32_t n_valid, n_dropped, n_ignored;
};

// slot of detection j in the tile's label table (-1 when more than MAX_LABELS detections meet in one tile)
__device__ __forceinline__ int tile_label_slot_in(uint32_t *lab_j, uint32_t j) {
  uint32_t h = j % MAX_LABELS;
  for (int probe = 0; probe < MAX_LABELS; ++probe) {
    uint32_t l = *(volatile uint32_t *)&lab_j[h];
    if (l == NONE32) {
      l = atomicCAS(&lab_j[h], NONE32, j);
      if (l == NONE32) l = j;
    }
    if (l == j) return (int)h;
    h = (h + 1) % MAX_LABELS;
  }
  return -1;
}

// OR the voxel bits (lo, hi) of block `bkey` into the tile's entry of (label slot li, block).  Exact: the tag
// holds the whole block key and the label slot.  When the tile table is full the record goes straight to the
// global queue (the probe kernel's pair set keeps the result exact).
__device__ __forceinline__ bool tile_block_add(TileSmem &s, int li, unsigned long long bkey, uint32_t lo, uint32_t hi) {
  const unsigned long long tag = bkey | ((unsigned long long)li << LABEL_SHIFT);
  // multiplicative hash of the 64-bit tag, top bits (neighbouring blocks differ in the low bits of the key fields)
  uint32_t h = (((uint32_t)tag * 0x9E3779B1u) ^ ((uint32_t)(tag >> 32) * 0x85EBCA77u)) >> (32 - 7);
  static_assert(TILE_ENT == 128, "hash width");
  for (int probe = 0; probe < 16; ++probe) {  // a short probe sequence: a miss only costs one more queue record
    unsigned long long cur = *(volatile unsigned long long *)&s.tag[h];
    if (cur == BLK_EMPTY) {
      cur = atomicCAS(&s.tag[h], BLK_EMPTY, tag);
      if (cur == BLK_EMPTY) cur = tag;
    }
    if (cur == tag) {
      if (lo) atomicOr(&s.mlo[h], lo);
      if (hi) atomicOr(&s.mhi[h], hi);
      return true;
    }
    h = (h + 1) & (TILE_ENT - 1);
  }
  return false;
}

// Records the tile table could not absorb (no label slot, table full: far, noisy surfaces put every pixel into its
// own block) go straight to the global queue -- one atomicAdd per warp, not per lane.  Warp-synchronous.
__device__ __forceinline__ void emit_overflow(const DevMap &m, bool ovf, unsigned long long bkey, uint32_t j, uint32_t lo, uint32_t hi) {
  const unsigned b = __ballot_sync(0xFFFFFFFFu, ovf);
  if (!b) return;
  const int lane = threadIdx.x & 31;
  uint32_t base = 0;
  if (lane == __ffs(b) - 1) base = atomicAdd(m.surv_cnt, (uint32_t)__popc(b));
  base = __shfl_sync(0xFFFFFFFFu, base, __ffs(b) - 1);
  if (ovf) survivor_store(m, base + __popc(b & ((1u << lane) - 1)), bkey, j, lo, hi);
}

// raw registers of one thread's 8 pixels (2 x 128-bit depth + 1 x 128-bit mask)
struct TileRegs {
  float4 d0, d1;
  uint4 mk;
};

// A warp owns a 16-column x 16-row patch of the tile: lane -> row = lane >> 1, 8 consecutive pixels at column
// 16 * warp + 8 * (lane & 1)  (32 contiguous bytes of depth and 16 of mask per lane: whole DRAM sectors).
// (f, ty, tx) = frame and tile coordinates.
template <bool VEC>
__device__ __forceinline__ TileRegs load_tile(const DevMap &m, const CallArgs &a, int f, int ty, int tx, int row, int cg) {
  const int v = ty * TILE_H + row;
  const int u0 = tx * TILE_W + cg * 8;
  const bool row_ok = v < m.H;
  const size_t off = ((size_t)f * m.H + v) * m.W + u0;
  TileRegs r;
  if (VEC && row_ok && u0 + 7 < m.W) {
    r.d0 = __ldcs(reinterpret_cast<const float4 *>(a.depth + off));
    r.d1 = __ldcs(reinterpret_cast<const float4 *>(a.depth + off + 4));
    r.mk = __ldcs(reinterpret_cast<const uint4 *>(a.mask + off));
  } else {
    float z[8];
    uint32_t lab[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool ok = row_ok && u0 + i < m.W;
      lab[i] = ok ? (uint32_t)__ldcs(a.mask + off + i) : 0u;
      z[i] = ok ? __ldcs(a.depth + off + i) : 0.f;
    }
    r.d0 = make_float4(z[0], z[1], z[2], z[3]);
    r.d1 = make_float4(z[4], z[5], z[6], z[7]);
    r.mk = make_uint4(lab[0] | (lab[1] << 16), lab[2] | (lab[3] << 16), lab[4] | (lab[5] << 16), lab[6] | (lab[7] << 16));
  }
  return r;
}

// per-lane running evidence of the detection and voxel block the lane is currently looking at
// (R7: voxel bits of the block, pixel count, point box; G1: moments)
template <bool GAUSS>
struct LaneAcc {
  uint32_t j, cnt;          // detection (NONE32 = none yet in this tile) and its pixels seen by the lane
  int li;                   // its label slot in the tile (-1: none left)
  uint32_t klo, khi;        // current block key (64 bit, two halves) and
  uint32_t mlo, mhi;        //   the voxel bits of that block seen by the lane
  float mn0, mn1, mn2, mx0, mx1, mx2;
  float gc0, gc1, gc2, g1x, g1y, g1z, gxx, gxy, gxz, gyy, gyz, gzz;  // G1, about the lane's first point (GAUSS only)
};

// G1: raw moments in double from the lane's centred fp32 sums (parallel-axis shift)
template <bool GAUSS>
__device__ __forceinline__ void lane_raw_moments(const LaneAcc<GAUSS> &c, double g[9]) {
  const double n = (double)c.cnt, c0 = c.gc0, c1 = c.gc1, c2 = c.gc2, sx = c.g1x, sy = c.g1y, sz = c.g1z;
  g[0] = sx + n * c0, g[1] = sy + n * c1, g[2] = sz + n * c2;
  g[3] = c.gxx + 2.0 * c0 * sx + n * c0 * c0, g[4] = c.gxy + c0 * sy + c1 * sx + n * c0 * c1, g[5] = c.gxz + c0 * sz + c2 * sx + n * c0 * c2;
  g[6] = c.gyy + 2.0 * c1 * sy + n * c1 * c1, g[7] = c.gyz + c1 * sz + c2 * sy + n * c1 * c2, g[8] = c.gzz + 2.0 * c2 * sz + n * c2 * c2;
}

// rare: the lane's detection changes inside a patch -- its partial evidence goes to the detection on its own
template <bool GAUSS>
__device__ __forceinline__ void lane_flush_own(const DevMap &m, const LaneAcc<GAUSS> &c) {
  const uint32_t j = c.j;
  atomicAdd(&m.det_npx[j], c.cnt);
  atomicMin(&m.det_box[j * 6 + 0], f2ord(c.mn0)), atomicMin(&m.det_box[j * 6 + 1], f2ord(c.mn1)), atomicMin(&m.det_box[j * 6 + 2], f2ord(c.mn2));
  atomicMax(&m.det_box[j * 6 + 3], f2ord(c.mx0)), atomicMax(&m.det_box[j * 6 + 4], f2ord(c.mx1)), atomicMax(&m.det_box[j * 6 + 5], f2ord(c.mx2));
  if (GAUSS) {
    double g[9];
    lane_raw_moments<GAUSS>(c, g);
#pragma unroll
    for (int k = 0; k < 9; ++k) atomicAdd(m.det_gm + (size_t)j * 9 + k, g[k]);
  }
}

// the lane's voxel bits of its current (detection, block) -> the tile's table; to the global queue when the table
// cannot take them (no label slot, table full).  Called when the lane moves on to another block.
template <bool GAUSS>
__device__ __forceinline__ void lane_flush_block(const DevMap &m, TileSmem &s, const LaneAcc<GAUSS> &c) {
  const unsigned long long bkey = ((unsigned long long)c.khi << 32) | c.klo;
  if (c.li >= 0 && tile_block_add(s, c.li, bkey, c.mlo, c.mhi)) return;
  survivor_store(m, atomicAdd(m.surv_cnt, 1u), bkey, c.j, c.mlo, c.mhi);
}

// ---------------------------------------------------------------------------------------------------
// lift kernel (steps 1-2).  Persistent CTAs; one 64x16 pixel tile per iteration; each warp owns a 16x16 patch of
// it and each lane 8 consecutive pixels of one row (2 x 128-bit depth loads + 1 x 128-bit mask load, issued one
// tile ahead).
//   Compaction (BASELINE.json: "warp-ballot compaction of masked pixels"): the lanes mark their valid masked
//     pixels (R3, R4); per pixel position one ballot gives every valid pixel its dense slot (prefix popcount), and
//     depth + (label, row, column) go to the warp's staging area in shared memory as one 64-bit word, 4 of a lane's 8
//     pixels per round.  The arithmetic below then runs over DENSE slots -- one pixel per lane, every lane busy
//     except in the last iteration of a round.
//   Per pixel (straight-line fp32/int code): back-projection (R5, every operation individually rounded), voxel
//     index (R6; floor by a round-down add of 1.5 * 2^23, exact for |x| < 2^22), block key + voxel bit.
//   Dedupe (R7): the voxel of a pixel is one bit of its block's 64-bit mask.  A lane ORs the bits of consecutive
//     pixels that fall into the same (detection, block) in registers (neighbouring pixels nearly always do), together
//     with the pixel count and point box (and G1 moments) of the detection; when it moves on to another block the bits go
//     to the tile's shared-memory table (atomicOr), and at the end of the patch the lanes holding the same
//     (detection, block) combine theirs first (match.any + redux.or).  No per-pixel warp-collective work.
//   Flush: one (block, detection, voxel bits) record per table entry goes to the call's survivor queue.  The CTA
//     reserves queue space in chunks of TILE_ENT records one tile ahead, so no thread ever waits for a global
//     atomic; the unused tail of the last chunk is padded with empty records (bits == 0).  The lanes' pixel counts
//     and boxes are combined per detection over the warp (REDUX) and leave as one set of global atomics per
//     (warp patch, detection).
// Two barriers per tile.
// 6 CTAs per SM = at most 80 registers, for both variants: the grid's 4 CTAs per SM must ALL be resident beside the
// similarity CTA (256 threads x 80 registers), otherwise the statically assigned tiles of the late CTAs run as a second
// wave (measured with the Gaussian variant at 96 registers: 3 resident, lift 194 us instead of 139 us in the step; its
// 84 bytes of spill at 80 registers cost less than that).
template <bool VEC, bool GAUSS>
__global__ void __launch_bounds__(LIFT_THREADS, 6) lift_voxelise_kernel(DevMap m, CallArgs a, int tiles_x, int tiles_y) {
  pdl_trigger();  // the probe kernel may become resident as soon as CTAs of this grid retire
  if (threadIdx.x == 0) TRACE_MIN(farm_trace_lift, a.seq, 0);
  __shared__ TileSmem s;
  __shared__ uint32_t lab_j2[2][MAX_LABELS];  // label tables are double buffered: the flush of tile t reads its copy
                                              // while tile t+1 initialises the other
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int tiles_xy = tiles_x * tiles_y;
  const int n_tiles = tiles_xy * a.F;
  const float inv_vs = m.inv_vs, z_min = m.z_min;
  const float z_max = fminf(m.z_max, 3.402823466e+38f);  // z <= z_max then also rejects +inf and NaN (R4: finite)
  const float INF = __int_as_float(0x7F800000);
  constexpr unsigned FULL = 0xFFFFFFFFu;
  const unsigned lt_mask = (1u << lane) - 1u;
  for (int i = tid; i < TILE_ENT; i += LIFT_THREADS) {
    s.tag[i] = BLK_EMPTY;
    s.mlo[i] = 0;
    s.mhi[i] = 0;
  }
  if (tid == 0) {
    s.q_count = 0, s.cur_pos = 0, s.cur_end = 0, s.next_base = 0, s.next_valid = 0;
    s.n_valid = 0, s.n_dropped = 0, s.n_ignored = 0;
  }
  uint32_t acc_valid = 0, acc_dropped = 0, acc_ignored = 0;  // per-thread counters over all tiles
  const int row = lane >> 1, cg = warp * 2 + (lane & 1);     // the lane's row and 8-pixel column group inside a tile
  unsigned long long *stage = s.stage[warp];
  // tile coordinates advance incrementally (no per-tile divisions): this CTA's tiles are blockIdx.x + k * gridDim.x
  int f = blockIdx.x / tiles_xy, ty = (blockIdx.x - f * tiles_xy) / tiles_x, tx = blockIdx.x - f * tiles_xy - ty * tiles_x;
  const int df = gridDim.x / tiles_xy, dty = (gridDim.x - df * tiles_xy) / tiles_x, dtx = gridDim.x - df * tiles_xy - dty * tiles_x;
  auto advance = [&](int &ff, int &yy, int &xx) {
    xx += dtx;
    if (xx >= tiles_x) xx -= tiles_x, ++yy;
    yy += dty;
    if (yy >= tiles_y) yy -= tiles_y, ++ff;
    ff += df;
  };
  int par = 0;
  TileRegs cur = load_tile<VEC>(m, a, f, ty, tx, row, cg);
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, par ^= 1) {
    int nf = f, nty = ty, ntx = tx;
    advance(nf, nty, ntx);
    TileRegs nxt = cur;
    if (tile + (int)gridDim.x < n_tiles) nxt = load_tile<VEC>(m, a, nf, nty, ntx, row, cg);
    // (float)u = as_float(0x4B000000 | u) - 2^23 for u < 2^23: the tile origin is folded into the integer constant
    const uint32_t v_magic = 0x4B000000u + (uint32_t)(ty * TILE_H), u_magic = 0x4B000000u + (uint32_t)(tx * TILE_W);
    // camera of the frame, prepared by prep_kernel: (inv_fx, inv_fy, cx, cy), (r00 r01 r02 tx), (r10 ..), (r20 ..)
    const float4 *cp = reinterpret_cast<const float4 *>(m.cam + 16 * f);
    const float4 c0 = __ldg(cp), c1 = __ldg(cp + 1), c2 = __ldg(cp + 2), c3 = __ldg(cp + 3);
    const int det_base = a.base[f];
    const uint32_t n_det_f = (uint32_t)(a.base[f + 1] - det_base);
    uint32_t *lab_j = lab_j2[par];
    if (tid < MAX_LABELS) lab_j[tid] = NONE32;
    __syncthreads();  // B1: label table ready; every warp has finished the flush of the previous tile
    if (tid == 0) {
      // account for the records the previous tile flushed; reserve the next queue chunk one tile ahead
      uint32_t pos = s.cur_pos + s.q_count;
      s.q_count = 0;
      if (pos >= s.cur_end && s.next_valid) {
        pos = s.next_base + (pos - s.cur_end);
        s.cur_end = s.next_base + TILE_ENT;
        s.next_valid = 0;
      }
      s.cur_pos = pos;
      if (s.cur_end - pos < (uint32_t)TILE_ENT && !s.next_valid) {
        s.next_base = atomicAdd(m.surv_cnt, (uint32_t)TILE_ENT);
        s.next_valid = 1;
      }
    }

    // ---- validity of the lane's 8 pixels (R3, R4)
    const float z8[8] = {cur.d0.x, cur.d0.y, cur.d0.z, cur.d0.w, cur.d1.x, cur.d1.y, cur.d1.z, cur.d1.w};
    const uint32_t lab8[8] = {cur.mk.x & 0xFFFF, cur.mk.x >> 16, cur.mk.y & 0xFFFF, cur.mk.y >> 16,
                              cur.mk.z & 0xFFFF, cur.mk.z >> 16, cur.mk.w & 0xFFFF, cur.mk.w >> 16};
    uint32_t vm = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i)
      if (lab8[i] - 1u < n_det_f && z8[i] > z_min && z8[i] <= z_max) vm |= 1u << i;   // 1 <= label <= n_det, depth valid
    // labels without a descriptor row (R3: ignored, counted) are rare: look for them only where the packed words say so
    const uint32_t lab_max2 = __vmaxu2(__vmaxu2(cur.mk.x, cur.mk.y), __vmaxu2(cur.mk.z, cur.mk.w));  // per 16-bit half
    if (max(lab_max2 & 0xFFFFu, lab_max2 >> 16) > n_det_f) {
#pragma unroll
      for (int i = 0; i < 8; ++i) acc_ignored += lab8[i] > n_det_f ? 1u : 0u;
    }
    LaneAcc<GAUSS> ac;
    ac.j = NONE32, ac.cnt = 0, ac.li = -1, ac.klo = ac.khi = 0xFFFFFFFFu, ac.mlo = ac.mhi = 0;
    ac.mn0 = INF, ac.mn1 = INF, ac.mn2 = INF, ac.mx0 = -INF, ac.mx1 = -INF, ac.mx2 = -INF;
    ac.gc0 = ac.gc1 = ac.gc2 = ac.g1x = ac.g1y = ac.g1z = ac.gxx = ac.gxy = ac.gxz = ac.gyy = ac.gyz = ac.gzz = 0.f;

    if (__any_sync(FULL, vm != 0)) {
#pragma unroll
      for (int r = 0; r < 2; ++r) {
        // ---- compaction of pixels 4r .. 4r+3 of every lane into dense slots: slot = pixels before it in (i, lane) order
        // (invalid pixels are written to the dump slot: no divergent branch)
        const uint32_t meta0 = ((uint32_t)row << 8) | (uint32_t)(cg * 8 + 4 * r);
        uint32_t n = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          const bool on_i = (vm >> (4 * r + i)) & 1u;
          const unsigned b = __ballot_sync(FULL, on_i);
          const uint2 val = make_uint2(__float_as_uint(z8[4 * r + i]), (lab8[4 * r + i] << 16) | (meta0 + i));
          *reinterpret_cast<uint2 *>(&stage[on_i ? n + __popc(b & lt_mask) : STAGE_PX]) = val;
          n += __popc(b);
        }
        if (n == 0) continue;  // warp-uniform
        __syncwarp();
        // ---- dense pass: one pixel per lane
#pragma unroll 1
        for (uint32_t base = 0; base < n; base += 32) {
          const uint32_t slot = base + lane;
          const bool on = slot < n;
          const uint2 sv = *reinterpret_cast<const uint2 *>(&stage[on ? slot : 0]);
          const float z = __uint_as_float(sv.x);
          const uint32_t meta = sv.y;
          const uint32_t j = (uint32_t)det_base + (meta >> 16) - 1u;
          // (float)u, (float)v exactly (integers below 2^23), then R5 in its fixed order
          const float uf = __fsub_rn(__uint_as_float(u_magic + (meta & 0xFFu)), 8388608.0f);
          const float vf = __fsub_rn(__uint_as_float(v_magic + ((meta >> 8) & 0xFFu)), 8388608.0f);
          const float xn = __fmul_rn(__fsub_rn(uf, c0.z), c0.x), yn = __fmul_rn(__fsub_rn(vf, c0.w), c0.y);
          const float xc = __fmul_rn(xn, z), yc = __fmul_rn(yn, z);
          const float p0 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c1.x, xc), __fmul_rn(c1.y, yc)), __fmul_rn(c1.z, z)), c1.w);
          const float p1 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c2.x, xc), __fmul_rn(c2.y, yc)), __fmul_rn(c2.z, z)), c2.w);
          const float p2 = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c3.x, xc), __fmul_rn(c3.y, yc)), __fmul_rn(c3.z, z)), c3.w);
          // R6: floor(fp32(X * inv_vs)) by a round-down add of 1.5 * 2^23 (exact for |x| < 2^22; the pre-test keeps
          // |x| < 2e6 and rejects NaN / inf), biased by 2^20
          const float fx = __fmul_rn(p0, inv_vs), fy = __fmul_rn(p1, inv_vs), fz = __fmul_rn(p2, inv_vs);
          const bool finite = fabsf(fx) < 2.0e6f && fabsf(fy) < 2.0e6f && fabsf(fz) < 2.0e6f;
          constexpr int UNBIAS = 0x4B400000 - KEY_BIAS;
          const uint32_t ix = (uint32_t)(__float_as_int(__fadd_rd(fx, 12582912.0f)) - UNBIAS);
          const uint32_t iy = (uint32_t)(__float_as_int(__fadd_rd(fy, 12582912.0f)) - UNBIAS);
          const uint32_t iz = (uint32_t)(__float_as_int(__fadd_rd(fz, 12582912.0f)) - UNBIAS);
          const bool ok = on && finite && ((ix | iy | iz) >> 21) == 0;
          acc_dropped += (on && !ok) ? 1u : 0u;
          acc_valid += ok ? 1u : 0u;
          // block key halves (bx << 38 | by << 19 | bz with b = i >> 2) and the voxel's bit inside the block
          const uint32_t bx = ix >> 2, by = iy >> 2, bz = iz >> 2;
          const uint32_t klo = bz | (by << 19), khi = (by >> 13) | (bx << 6);
          const uint32_t bit = ((ix & 3u) << 4) | ((iy & 3u) << 2) | (iz & 3u);
          if (ok) {
            if (klo != ac.klo || khi != ac.khi || j != ac.j) {  // the lane moves on to another block (or detection)
              if (ac.mlo | ac.mhi) lane_flush_block<GAUSS>(m, s, ac);
              ac.klo = klo, ac.khi = khi, ac.mlo = 0, ac.mhi = 0;
              if (j != ac.j) {  // first pixel of the lane in this tile, or (rare) another detection
                if (ac.cnt) lane_flush_own<GAUSS>(m, ac);
                ac.j = j, ac.cnt = 0;
                ac.li = tile_label_slot_in(lab_j, j);
                ac.mn0 = INF, ac.mn1 = INF, ac.mn2 = INF, ac.mx0 = -INF, ac.mx1 = -INF, ac.mx2 = -INF;
                if (GAUSS) {
                  ac.gc0 = p0, ac.gc1 = p1, ac.gc2 = p2;
                  ac.g1x = ac.g1y = ac.g1z = ac.gxx = ac.gxy = ac.gxz = ac.gyy = ac.gyz = ac.gzz = 0.f;
                }
              }
            }
            const uint32_t one = 1u << (bit & 31);
            ac.mlo |= (bit & 32) ? 0u : one, ac.mhi |= (bit & 32) ? one : 0u;
            ac.cnt++;
            ac.mn0 = fminf(ac.mn0, p0), ac.mn1 = fminf(ac.mn1, p1), ac.mn2 = fminf(ac.mn2, p2);
            ac.mx0 = fmaxf(ac.mx0, p0), ac.mx1 = fmaxf(ac.mx1, p1), ac.mx2 = fmaxf(ac.mx2, p2);
            if (GAUSS) {
              const float dx = p0 - ac.gc0, dy = p1 - ac.gc1, dz = p2 - ac.gc2;
              ac.g1x += dx, ac.g1y += dy, ac.g1z += dz;
              ac.gxx = fmaf(dx, dx, ac.gxx), ac.gxy = fmaf(dx, dy, ac.gxy), ac.gxz = fmaf(dx, dz, ac.gxz);
              ac.gyy = fmaf(dy, dy, ac.gyy), ac.gyz = fmaf(dy, dz, ac.gyz), ac.gzz = fmaf(dz, dz, ac.gzz);
            }
          }
        }
        __syncwarp();  // the staging area is rewritten by the next round
      }
      // ---- end of the patch: the lanes' last blocks, combined over the lanes that hold the same (detection, block)
      {
        const bool has = (ac.mlo | ac.mhi) != 0;
        const bool tab = has && ac.li >= 0;
        const unsigned long long bkey = ((unsigned long long)ac.khi << 32) | ac.klo;
        const unsigned long long tag = tab ? (bkey | ((unsigned long long)ac.li << LABEL_SHIFT)) : BLK_EMPTY;
        const unsigned same = __match_any_sync(FULL, tag);
        const uint32_t lo = __reduce_or_sync(same, ac.mlo), hi = __reduce_or_sync(same, ac.mhi);
        bool ovf = has && ac.li < 0;  // no label slot: the lane's record goes to the global queue on its own
        if (tab && lane == __ffs(same) - 1) ovf = !tile_block_add(s, ac.li, bkey, lo, hi);
        emit_overflow(m, ovf, bkey, ac.j, tab ? lo : ac.mlo, tab ? hi : ac.mhi);
      }
      // ---- the lanes' evidence per detection (R7): combined over the warp, one set of global atomics per detection
      {
        const uint32_t key = ac.cnt ? ac.j : NONE32;
        const unsigned grp = __match_any_sync(FULL, key);
        const uint32_t tot = __reduce_add_sync(grp, ac.cnt);
        const int r0 = __reduce_min_sync(grp, f2ord(ac.mn0)), r1 = __reduce_min_sync(grp, f2ord(ac.mn1)),
                  r2 = __reduce_min_sync(grp, f2ord(ac.mn2)), r3 = __reduce_max_sync(grp, f2ord(ac.mx0)),
                  r4 = __reduce_max_sync(grp, f2ord(ac.mx1)), r5 = __reduce_max_sync(grp, f2ord(ac.mx2));
        if (ac.cnt && lane == __ffs(grp) - 1) {
          atomicAdd(&m.det_npx[key], tot);
          atomicMin(&m.det_box[key * 6 + 0], r0), atomicMin(&m.det_box[key * 6 + 1], r1), atomicMin(&m.det_box[key * 6 + 2], r2);
          atomicMax(&m.det_box[key * 6 + 3], r3), atomicMax(&m.det_box[key * 6 + 4], r4), atomicMax(&m.det_box[key * 6 + 5], r5);
        }
        if (GAUSS) {  // G1: raw moments in double, one set of atomics per warp when it holds one detection
          double g[9];
          lane_raw_moments<GAUSS>(ac, g);
          const unsigned hasg = __ballot_sync(FULL, ac.cnt != 0);
          if (hasg) {
            const uint32_t lead_j = __shfl_sync(FULL, ac.j, __ffs(hasg) - 1);
            if (__all_sync(FULL, ac.cnt == 0 || ac.j == lead_j)) {
#pragma unroll
              for (int k = 0; k < 9; ++k) {
                if (!ac.cnt) g[k] = 0.0;
#pragma unroll
                for (int sft = 16; sft; sft >>= 1) g[k] += __shfl_xor_sync(FULL, g[k], sft);
              }
              if (lane < 9) {
                double v = g[0];
#pragma unroll
                for (int k = 1; k < 9; ++k) v = lane == k ? g[k] : v;
                atomicAdd(m.det_gm + (size_t)lead_j * 9 + lane, v);
              }
            } else if (ac.cnt) {
#pragma unroll
              for (int k = 0; k < 9; ++k) atomicAdd(m.det_gm + (size_t)ac.j * 9 + k, g[k]);
            }
          }
        }
      }
    }
    __syncthreads();  // B2: the tile's table is complete; thread 0 has published the queue chunk

    // ---- flush: table entries -> survivor queue (positions inside the CTA's reserved chunks), then clear them
    {
      const uint32_t cpos = s.cur_pos, cend = s.cur_end, nbase = s.next_base;
#pragma unroll
      for (int r = 0; r < TILE_ENT / LIFT_THREADS; ++r) {
        const int e = tid + r * LIFT_THREADS;
        const unsigned long long tag = s.tag[e];
        const bool has = tag != BLK_EMPTY;
        const unsigned b = __ballot_sync(FULL, has);
        uint32_t base = 0;
        if (lane == 0 && b) base = atomicAdd(&s.q_count, (uint32_t)__popc(b));
        base = __shfl_sync(FULL, base, 0);
        if (has) {
          uint32_t pos = cpos + base + __popc(b & lt_mask);
          if (pos >= cend) pos = nbase + (pos - cend);
          survivor_store(m, pos, tag & ((1ull << LABEL_SHIFT) - 1), lab_j[(uint32_t)(tag >> LABEL_SHIFT)], s.mlo[e], s.mhi[e]);
          s.tag[e] = BLK_EMPTY;
          s.mlo[e] = 0;
          s.mhi[e] = 0;
        }
      }
    }
    cur = nxt;
    f = nf, ty = nty, tx = ntx;
  }
  // ---- end of the CTA's tiles: statistics, and empty records over the unused part of the reserved chunks
  acc_valid = __reduce_add_sync(FULL, acc_valid);
  acc_dropped = __reduce_add_sync(FULL, acc_dropped);
  acc_ignored = __reduce_add_sync(FULL, acc_ignored);
  if (lane == 0) {
    if (acc_valid) atomicAdd(&s.n_valid, acc_valid);
    if (acc_dropped) atomicAdd(&s.n_dropped, acc_dropped);
    if (acc_ignored) atomicAdd(&s.n_ignored, acc_ignored);
  }
  __syncthreads();
  if (tid == 0) {
    if (s.n_valid) atomicAdd(&m.stats->valid_points, (unsigned long long)s.n_valid);
    if (s.n_dropped) atomicAdd(&m.stats->dropped_points, (unsigned long long)s.n_dropped);
    if (s.n_ignored) atomicAdd(&m.stats->ignored_pixels, (unsigned long long)s.n_ignored);
  }
  {
    uint32_t pos = s.cur_pos + s.q_count, end = s.cur_end;
    if (pos >= end && s.next_valid) {
      pos = s.next_base + (pos - end);
      end = s.next_base + TILE_ENT;
    } else if (s.next_valid) {  // a reserved chunk that was never reached
      for (uint32_t p = s.next_base + tid; p < s.next_base + TILE_ENT; p += LIFT_THREADS) survivor_store(m, p, 0ull, 0u, 0u, 0u);
    }
    for (uint32_t p = pos + tid; p < end; p += LIFT_THREADS) survivor_store(m, p, 0ull, 0u, 0u, 0u);
  }
  if (tid == 0) TRACE_MAX(farm_trace_lift, a.seq, 1);
}

// ---------------------------------------------------------------------------------------------------
// probe kernel (step 3 and R12 pass 1).  Each warp takes 32 survivor records.
// Phase A, one lane per record: find or insert the block in the global hash, then OR the record's voxel bits
//   into the per-call pair set entry of (detection, block): the bits that were not set before are the
//   detection's NEW voxels -- exactly one record wins each (detection, voxel) pair, whatever the tiling.
// Phase B, eight lanes per record (one 32-byte owner sector each): for every new voxel read its owner;
//   owned at entry -> overlap c[d][owner] += 1 (R9), else claim = min(claim, d) (R12, lowest index wins).
//   |V_d| += popc(new bits); the (detection, block, new bits) event is appended to the event list for the
//   commit pass.  Overlap counts are aggregated over the lanes of a warp (match.any + redux.add).
constexpr int PROBE_THREADS = 256;
constexpr uint32_t PROBE_DIAGONAL_MAX = 1u << 16;  // records; above this the queue is read in order

__global__ void __launch_bounds__(PROBE_THREADS) probe_kernel(DevMap m, CallArgs a) {
  __shared__ uint8_t s_pairs[PROBE_THREADS / 32][256];  // per warp: (record lane << 3 | sector) of the sectors with new voxels
  if (threadIdx.x == 0) TRACE_MIN(farm_trace_probe, a.seq, 0);
  pdl_trigger();  // cand_associate may become resident behind this grid
  pdl_wait();     // launched with PDL behind the lift kernel: its survivor queue is complete from here on
  if (threadIdx.x == 0) TRACE_MIN(farm_trace_lift, a.seq, 2);
#ifdef FARM_TRACE
  struct ProbeEnd {
    uint32_t seq;
    __device__ ~ProbeEnd() {
      if (threadIdx.x == 0) TRACE_MAX(farm_trace_lift, seq, 3);
    }
  } probe_end{a.seq};
#endif
  const uint32_t nq = min(__ldcg(m.surv_cnt), m.surv_cap);
  const int lane = threadIdx.x & 31;
  const uint32_t stride = gridDim.x * blockDim.x;
  // Small queues (single-frame calls) are read along a diagonal: the real records sit at the start of each 128-record chunk that
  // a lift CTA reserved, so a warp that took 32 consecutive records would hold either 32 real ones (and run phase B's dependent
  // rounds seven or eight times) or none.  Lane l of warp task (g, k) takes record (k + 4 l) mod 128 of chunk 32 g + l instead:
  // a bijection on [0, 4096) per group, every warp samples all chunk positions and gets the average fill.  Large queues (batches)
  // keep the coalesced order -- their warps are all busy and the uncoalesced record loads would cost bandwidth.
  const bool diagonal = nq <= PROBE_DIAGONAL_MAX;
  const uint32_t n_end = diagonal ? (nq + 4095u) & ~4095u : nq;
  for (uint32_t i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u; i0 < n_end; i0 += stride) {
    const uint32_t wt = i0 >> 5;
    const uint32_t i = diagonal ? ((wt >> 7) << 12) + ((uint32_t)lane << 7) + (((wt & 127u) + 4u * lane) & 127u) : i0 + lane;
    // ---- phase A
    uint32_t j = 0, slot = NONE32, ps = 0;
    unsigned long long nb = 0;
    if (i < nq) {
      const unsigned long long bkey = __ldcg(&m.surv_key[i]);
      const unsigned long long bits = __ldcg(&m.surv_bits[i]);
      j = __ldcg(&m.surv_j[i]);
#ifdef FARM_TRACE
      if (bits && lane == __ffs(__activemask()) - 1) TRACE_MAX(farm_trace_probe, a.seq, 1);
#endif
      if (bits) slot = block_find_or_insert(m, bkey);  // bits == 0: padding of a reserved queue chunk
#ifdef FARM_TRACE
      if (bits && lane == __ffs(__activemask()) - 1) TRACE_MAX(farm_trace_probe, a.seq, 3);
#endif
      if (slot != NONE32) {
        const unsigned long long pv = ((unsigned long long)((a.epoch << 16) | j) << 32) | slot;
        const int r = epoch_insert(m.pair_set, m.pair_mask, pv, a.epoch, &ps);
        if (r < 0) {
          atomicOr(m.err, ERR_PAIR_TABLE_FULL);
        } else {
          const unsigned long long old = atomicOr(&m.pair_bits[ps], bits);
          nb = bits & ~old;
        }
      }
    }
    const unsigned act = __ballot_sync(0xFFFFFFFFu, nb != 0);
    if (!act) continue;
    if (lane == 0) TRACE_MAX(farm_trace_probe, a.seq, 5);
    // |V_d| += new voxels (aggregated over the lanes of the same detection)
    if (nb) {
      const unsigned same = __match_any_sync(act, j);
      const uint32_t tot = __reduce_add_sync(same, (uint32_t)__popcll(nb));
      if (lane == __ffs(same) - 1) atomicAdd(&m.det_nv[j], tot);
    }
    // event list slots (one atomic per warp)
    uint32_t ev = 0;
    if (lane == 0) ev = atomicAdd(&m.counters[0], (uint32_t)__popc(act));
    ev = __shfl_sync(0xFFFFFFFFu, ev, 0) + __popc(act & ((1u << lane) - 1));
    // ---- phase B: one lane per (record, owner sector) that holds a new voxel.  The non-empty sectors of the warp's 32
    // records are compacted (prefix sum of the per-record sector counts, list in shared memory), so that a round handles
    // 32 of them whatever their spread over the records: a sparse warp (single-frame calls: a few real records among the
    // padding of the queue) needs one round of dependent memory accesses, not one per group of four records.
    uint32_t smask = 0;  // sectors (bytes of nb) with a new voxel
#pragma unroll
    for (int sc = 0; sc < 8; ++sc) smask |= ((uint32_t)(nb >> (8 * sc)) & 0xFFu) ? 1u << sc : 0u;
    const uint32_t cnt_s = __popc(smask);
    uint32_t incl = cnt_s;
#pragma unroll
    for (int sft = 1; sft < 32; sft <<= 1) {
      const uint32_t up = __shfl_up_sync(0xFFFFFFFFu, incl, sft);
      if (lane >= sft) incl += up;
    }
    const uint32_t n_pairs = __shfl_sync(0xFFFFFFFFu, incl, 31), off_s = incl - cnt_s;
    uint8_t *plist = s_pairs[threadIdx.x >> 5];
    {
      uint32_t pos = off_s;
      for (uint32_t sm = smask; sm; sm &= sm - 1) plist[pos++] = (uint8_t)((lane << 3) | (__ffs(sm) - 1));
    }
    __syncwarp();
    uint32_t pend_mine = 0;  // lane r: does record r have a voxel that was unowned at entry
#pragma unroll 1
    for (uint32_t p0 = 0; p0 < n_pairs; p0 += 32) {
      const bool on = p0 + lane < n_pairs;
      const uint32_t pr = on ? plist[p0 + lane] : 0u;
      const int src = pr >> 3, sec = pr & 7;
      const unsigned long long rnb = __shfl_sync(0xFFFFFFFFu, nb, src);
      const uint32_t rslot = __shfl_sync(0xFFFFFFFFu, slot, src);
      const uint32_t rj = __shfl_sync(0xFFFFFFFFu, j, src);
      const uint32_t byte = on ? (uint32_t)(rnb >> (8 * sec)) & 0xFFu : 0u;
      uint32_t own[8];
      bool unowned = false;
      uint32_t o1 = NONE32, c1 = 0;  // first owner seen by this lane and how many of its voxels have it
      if (byte) {
        uint32_t *base = m.blk_owner + (size_t)rslot * BLK_VOXELS + sec * 8;
        const uint4 w0 = __ldcg(reinterpret_cast<const uint4 *>(base));
        const uint4 w1 = __ldcg(reinterpret_cast<const uint4 *>(base) + 1);
        own[0] = w0.x, own[1] = w0.y, own[2] = w0.z, own[3] = w0.w, own[4] = w1.x, own[5] = w1.y, own[6] = w1.z, own[7] = w1.w;
#pragma unroll
        for (int b = 0; b < 8; ++b) {
          if (!((byte >> b) & 1u)) continue;
          uint32_t o = own[b];
          if (o < OWNER_PENDING && m.alias) o = __ldg(&m.alias[o]);  // U4: voxels of an absorbed entity count for its winner
          if (o >= OWNER_PENDING) {  // unowned at entry (free, or claimed by a detection of this call)
            unowned = true;
            atomicMin(base + b, OWNER_PENDING | rj);  // R12: lowest detection index wins
          } else if (o1 == NONE32 || o == o1) {
            o1 = o, c1++;
          } else {  // a second owner inside one sector: rare, counted on its own
            const unsigned long long ov = ((unsigned long long)a.epoch << 48) | ((unsigned long long)rj << 32) | o;
            uint32_t os;
            const int r = epoch_insert(m.ov_keys, m.ov_mask, ov, a.epoch, &os);
            if (r < 0) {
              atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
            } else {
              if (r == 1) {
                const uint32_t c = atomicAdd(&m.counters[1], 1u);
                if (c < m.cand_cap) m.cand_slot[c] = os, m.cand_key[c] = ov; else atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
              }
              atomicAdd(&m.ov_cnt[os], 1u);
            }
          }
        }
      }
      // overlap histogram c[j][owner] += count, aggregated over the lanes with the same (j, owner)
      const unsigned oact = __ballot_sync(0xFFFFFFFFu, c1 != 0);
      if (c1) {
        const unsigned long long jo = ((unsigned long long)rj << 32) | o1;
        const unsigned same = __match_any_sync(oact, jo);
        const uint32_t tot = __reduce_add_sync(same, c1);
        if (lane == __ffs(same) - 1) {
          const unsigned long long ov = ((unsigned long long)a.epoch << 48) | jo;
          uint32_t os;
          const int r = epoch_insert(m.ov_keys, m.ov_mask, ov, a.epoch, &os);
          if (r < 0) {
            atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
          } else {
            if (r == 1) {
              const uint32_t c = atomicAdd(&m.counters[1], 1u);
              if (c < m.cand_cap) m.cand_slot[c] = os, m.cand_key[c] = ov; else atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
            }
            atomicAdd(&m.ov_cnt[os], tot);
          }
        }
      }
      // the sectors of record `lane` occupy list positions off_s .. off_s + cnt_s - 1: those that fall into this round
      const unsigned ub = __ballot_sync(0xFFFFFFFFu, unowned);
      const int lo = max((int)off_s - (int)p0, 0), hi = min((int)(off_s + cnt_s) - (int)p0, 32);
      if (hi > lo) pend_mine |= ub & ((hi - lo == 32 ? 0xFFFFFFFFu : ((1u << (hi - lo)) - 1u)) << lo);
    }
    __syncwarp();  // the list is rewritten by the warp's next 32 records
    if (lane == 0) TRACE_MAX(farm_trace_probe, a.seq, 7);
    if (nb) {
      if (ev < m.pair_cap) {
        m.pl_bits[ev] = nb;
        m.pl_slot[ev] = slot;
        m.pl_j[ev] = j | (pend_mine ? 0x80000000u : 0u);
        m.pl_ps[ev] = ps;
      } else {
        atomicOr(m.err, ERR_PAIR_TABLE_FULL);
      }
    }
  }
}

// U2 (detection-detection overlap, only with FARM_OPT_CORRESPONDENCE): after every probe has run, the owner word of a
// voxel that was unowned at entry holds OWNER_PENDING | e, e = the lowest-index detection of the call containing it
// (the R12 claimant).  For every event (detection j, block, new voxel bits) the voxels claimed by another detection
// e != j are counted into the overlap map under the key (j, DD_FLAG | e): c_dd(j, e).  Eight lanes per event.
__global__ void __launch_bounds__(256) dd_overlap_kernel(DevMap m, CallArgs a) {
  pdl_wait();
  const uint32_t n = min(m.counters[0], m.pair_cap);
  const int lane = threadIdx.x & 31, sec = lane & 7;
  const uint32_t per_pass = (gridDim.x * blockDim.x) >> 3;
  const uint32_t n_pad = (n + 3u) & ~3u;  // whole groups of 4 events per warp
  for (uint32_t e0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 3; e0 < n_pad; e0 += per_pass) {
    const bool act = e0 < n;
    const uint32_t jp = act ? m.pl_j[e0] : 0u;
    const uint32_t j = jp & 0x7FFFFFFFu;
    const uint32_t byte = (act && (jp >> 31)) ? (uint32_t)(m.pl_bits[e0] >> (8 * sec)) & 0xFFu : 0u;
    uint32_t e1 = NONE32, c1 = 0;
    if (byte) {
      const uint32_t *base = m.blk_owner + (size_t)m.pl_slot[e0] * BLK_VOXELS + sec * 8;
      const uint4 w0 = __ldcg(reinterpret_cast<const uint4 *>(base)), w1 = __ldcg(reinterpret_cast<const uint4 *>(base) + 1);
      const uint32_t own[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
      for (int b = 0; b < 8; ++b) {
        if (!((byte >> b) & 1u) || own[b] < OWNER_PENDING) continue;
        const uint32_t e = own[b] & 0x7FFFFFFFu;
        if (e == j) continue;
        if (e1 == NONE32 || e == e1) {
          e1 = e, c1++;
        } else {  // a second claimant inside one sector: counted on its own
          const unsigned long long ov = ((unsigned long long)a.epoch << 48) | ((unsigned long long)j << 32) | (DD_FLAG | e);
          uint32_t os;
          const int r = epoch_insert(m.ov_keys, m.ov_mask, ov, a.epoch, &os);
          if (r < 0) { atomicOr(m.err, ERR_OVERLAP_TABLE_FULL); continue; }
          if (r == 1) {
            const uint32_t c = atomicAdd(&m.counters[1], 1u);
            if (c < m.cand_cap) m.cand_slot[c] = os, m.cand_key[c] = ov; else atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
          }
          atomicAdd(&m.ov_cnt[os], 1u);
        }
      }
    }
    const unsigned oact = __ballot_sync(0xFFFFFFFFu, c1 != 0);
    if (c1) {
      const unsigned long long je = ((unsigned long long)j << 32) | (DD_FLAG | e1);
      const unsigned same = __match_any_sync(oact, je);
      const uint32_t tot = __reduce_add_sync(same, c1);
      if (lane == __ffs(same) - 1) {
        const unsigned long long ov = ((unsigned long long)a.epoch << 48) | je;
        uint32_t os;
        const int r = epoch_insert(m.ov_keys, m.ov_mask, ov, a.epoch, &os);
        if (r < 0) {
          atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
        } else {
          if (r == 1) {
            const uint32_t c = atomicAdd(&m.counters[1], 1u);
            if (c < m.cand_cap) m.cand_slot[c] = os, m.cand_key[c] = ov; else atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
          }
          atomicAdd(&m.ov_cnt[os], tot);
        }
      }
    }
  }
}

// U4: after the merges of a call, every id that pointed at an absorbed entity points at the entity that absorbed it
__global__ void alias_compress_kernel(DevMap m, uint32_t n_upper) {
  pdl_wait();
  if (m.counters[7] == 0) return;
  const uint32_t N = min(*m.n_objects, n_upper);
  for (uint32_t o = blockIdx.x * blockDim.x + threadIdx.x; o < N; o += gridDim.x * blockDim.x) {
    uint32_t r = m.alias[o];
    for (int hop = 0; hop < 64 && m.alias[r] != r; ++hop) r = m.alias[r];
    if (r != m.alias[o]) m.alias[o] = r;
  }
}

__global__ void debug_backproject_kernel(DevMap m, const float *__restrict__ depth, const uint16_t *__restrict__ mask,
                                         const float *__restrict__ K, const float *__restrict__ T, int n_det,
                                         float *__restrict__ xyz, unsigned long long *__restrict__ keys) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m.H * m.W) return;
  const Camera cam = load_camera(K, T);
  const int v = i / m.W, u = i - v * m.W;
  float p[3] = {__int_as_float(0x7FC00000), __int_as_float(0x7FC00000), __int_as_float(0x7FC00000)};
  unsigned long long key = KEY_EMPTY;
  const uint32_t l = mask[i];
  const float z = depth[i];
  if (l != 0 && (int)l <= n_det && depth_valid(z, m.z_min, m.z_max)) {
    backproject(cam, u, v, z, p);
    if (!voxel_key(p, m.inv_vs, &key)) key = KEY_EMPTY;
  }
  xyz[3 * (size_t)i] = p[0], xyz[3 * (size_t)i + 1] = p[1], xyz[3 * (size_t)i + 2] = p[2];
  keys[i] = key;
}

template <typename K>
void max_shared_carveout(K kernel) {
  cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
}

}  // namespace

void configure_lift_kernels() {
  max_shared_carveout(prep_kernel<float>);
  max_shared_carveout(prep_kernel<__half>);
  max_shared_carveout(prep_kernel<__nv_bfloat16>);
  max_shared_carveout(lift_voxelise_kernel<true, false>);
  max_shared_carveout(lift_voxelise_kernel<false, false>);
  max_shared_carveout(lift_voxelise_kernel<true, true>);
  max_shared_carveout(lift_voxelise_kernel<false, true>);
  max_shared_carveout(probe_kernel);
}

int launch_prep(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  const int blocks = a.M > 0 ? (a.M + 3) / 4 : 1;
  if (m.dtype == FARM_DTYPE_F32)
    prep_kernel<float><<<blocks, 128, 0, s>>>(m, a);
  else if (m.dtype == FARM_DTYPE_F16)
    prep_kernel<__half><<<blocks, 128, 0, s>>>(m, a);
  else
    prep_kernel<__nv_bfloat16><<<blocks, 128, 0, s>>>(m, a);
  return a.split ? 0 : blocks;
}

int launch_lift(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  const int tiles_x = (m.W + TILE_W - 1) / TILE_W, tiles_y = (m.H + TILE_H - 1) / TILE_H;
  const int n_tiles = tiles_x * tiles_y * a.F;
  // persistent, 4 CTAs per SM: 4 x 128 x 80 registers fit beside the similarity CTA (256 x 80) in the 64 K register file
  const int grid = n_tiles < m.num_sms * 4 ? n_tiles : m.num_sms * 4;
  const bool vec = (m.W % 8 == 0) && ((uintptr_t)a.depth % 16 == 0) && ((uintptr_t)a.mask % 16 == 0);
  if (m.det_gm) {
    if (vec)
      lift_voxelise_kernel<true, true><<<grid, LIFT_THREADS, 0, s>>>(m, a, tiles_x, tiles_y);
    else
      lift_voxelise_kernel<false, true><<<grid, LIFT_THREADS, 0, s>>>(m, a, tiles_x, tiles_y);
  } else if (vec) {
    lift_voxelise_kernel<true, false><<<grid, LIFT_THREADS, 0, s>>>(m, a, tiles_x, tiles_y);
  } else {
    lift_voxelise_kernel<false, false><<<grid, LIFT_THREADS, 0, s>>>(m, a, tiles_x, tiles_y);
  }
  return 1;
}

int launch_probe(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  launch_pdl(probe_kernel, dim3(m.num_sms * 4), dim3(PROBE_THREADS), 0, s, m, a);
  return 1;
}

int launch_dd_overlap(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  if (!m.corr || a.M == 0) return 0;
  launch_pdl(dd_overlap_kernel, dim3(m.num_sms * 2), dim3(256), 0, s, m, a);
  return 1;
}

int launch_alias_compress(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s) {
  if (!m.corr || a.M == 0) return 0;
  launch_pdl(alias_compress_kernel, dim3(m.num_sms), dim3(256), 0, s, m, n_upper);
  return 1;
}

int launch_debug_backproject(const DevMap &m, const float *depth, const uint16_t *mask, const float *K, const float *T,
                             int n_det, float *xyz, unsigned long long *keys, cudaStream_t s) {
  const int n = m.H * m.W;
  debug_backproject_kernel<<<(n + 255) / 256, 256, 0, s>>>(m, depth, mask, K, T, n_det, xyz, keys);
  return 1;
}

}  // namespace farm
