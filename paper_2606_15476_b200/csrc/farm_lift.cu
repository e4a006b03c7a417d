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

namespace {

constexpr int TILE_W = 64;        // 8 threads x 8 pixels per row
constexpr int TILE_H = 16;
constexpr int LIFT_THREADS = 128;
constexpr int TILE_ENT = 256;     // (detection, block) entries per tile; overflow goes straight to the global queue
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
template <typename T>
__global__ void prep_kernel(DevMap m, CallArgs a) {
  const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    m.counters[0] = 0;
    m.counters[1] = 0;
    m.counters[2] = 0;
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
  if (sizeof(T) == 2 && (m.D & 7) == 0 && (((uintptr_t)a.desc) & 15) == 0) {  // 128-bit loads, 8 elements each
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
    m.det_inv_norm[warp] = s > 0.f ? 1.0f / sqrtf(s) : 0.f;
    m.det_nv[warp] = 0;
    m.det_npx[warp] = 0;
    m.best_cand[warp] = 0ull;
    m.best_dense[warp] = 0ull;
    m.assoc[warp] = -1;
    m.is_new[warp] = 0;
    m.best_score[warp] = 0.f;
  }
  if (lane < 6) m.det_box[warp * 6 + lane] = lane < 3 ? 0x7FFFFFFF : (int)0x80000000;
  if (m.det_gm) {
    if (lane < 9) m.det_gm[(size_t)warp * 9 + lane] = 0.0;
    if (lane == 9) m.hell[warp] = -1.f;
  }
  }
  // publish: the similarity kernel runs on another stream and waits for every prep CTA before its first epilogue
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

// accumulate cnt pixels and their box (ordered ints) of detection j into the tile's per-detection accumulators
__device__ __forceinline__ void label_add_in(uint32_t *lab_cnt, int (*lab_box)[6], const DevMap &m, int li, uint32_t j,
                                             uint32_t cnt, int mn0, int mn1, int mn2, int mx0, int mx1, int mx2) {
  if (li >= 0) {
    atomicAdd(&lab_cnt[li], cnt);
    atomicMin(&lab_box[li][0], mn0), atomicMin(&lab_box[li][1], mn1), atomicMin(&lab_box[li][2], mn2);
    atomicMax(&lab_box[li][3], mx0), atomicMax(&lab_box[li][4], mx1), atomicMax(&lab_box[li][5], mx2);
    return;
  }
  atomicAdd(&m.det_npx[j], cnt);
  atomicMin(&m.det_box[j * 6 + 0], mn0), atomicMin(&m.det_box[j * 6 + 1], mn1), atomicMin(&m.det_box[j * 6 + 2], mn2);
  atomicMax(&m.det_box[j * 6 + 3], mx0), atomicMax(&m.det_box[j * 6 + 4], mx1), atomicMax(&m.det_box[j * 6 + 5], mx2);
}

// OR the voxel bits (lo, hi) of block `bkey` into the tile's entry of (label slot li, block).  Exact: the tag
// holds the whole block key and the label slot.  Without a label slot, or when the tile table is full, the
// record goes straight to the global queue (the probe kernel's pair set keeps the result exact).
__device__ __forceinline__ bool tile_block_add(TileSmem &s, int li, unsigned long long bkey, uint32_t lo, uint32_t hi) {
  if (li < 0) return false;
  const unsigned long long tag = bkey | ((unsigned long long)li << LABEL_SHIFT);
  uint32_t h = hash32((uint32_t)tag, (uint32_t)(tag >> 32)) & (TILE_ENT - 1);
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
  if (lane == __ffs(b) - 1) base = atomicAdd(&m.counters[2], (uint32_t)__popc(b));
  base = __shfl_sync(0xFFFFFFFFu, base, __ffs(b) - 1);
  if (ovf) survivor_store(m, base + __popc(b & ((1u << lane) - 1)), bkey, j, lo, hi);
}

// raw registers of one thread's 8 pixels (2 x 128-bit depth + 1 x 128-bit mask)
struct TileRegs {
  float4 d0, d1;
  uint4 mk;
};

template <bool VEC>
__device__ __forceinline__ TileRegs load_tile(const DevMap &m, const CallArgs &a, int tile, int tiles_x, int tiles_xy, int tid) {
  const int f = tile / tiles_xy;
  const int trem = tile - f * tiles_xy;
  const int ty = trem / tiles_x, tx = trem - ty * tiles_x;
  const int v = ty * TILE_H + (tid >> 3);
  const int u0 = tx * TILE_W + (tid & 7) * 8;
  const size_t frame_off = (size_t)f * m.H * m.W;
  const bool row_ok = v < m.H;
  TileRegs r;
  if (VEC && row_ok && u0 + 7 < m.W) {
    const size_t off = frame_off + (size_t)v * m.W + u0;
    r.d0 = __ldcs(reinterpret_cast<const float4 *>(a.depth + off));
    r.d1 = __ldcs(reinterpret_cast<const float4 *>(a.depth + off + 4));
    r.mk = __ldcs(reinterpret_cast<const uint4 *>(a.mask + off));
  } else {
    float z[8];
    uint32_t lab[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool ok = row_ok && u0 + i < m.W;
      const size_t off = frame_off + (size_t)v * m.W + u0 + i;
      lab[i] = ok ? (uint32_t)__ldcs(a.mask + off) : 0u;
      z[i] = ok ? __ldcs(a.depth + off) : 0.f;
    }
    r.d0 = make_float4(z[0], z[1], z[2], z[3]);
    r.d1 = make_float4(z[4], z[5], z[6], z[7]);
    r.mk = make_uint4(lab[0] | (lab[1] << 16), lab[2] | (lab[3] << 16), lab[4] | (lab[5] << 16), lab[6] | (lab[7] << 16));
  }
  return r;
}

// Rare path of the lift kernel: one pixel whose detection differs from the first detection of its thread.  It
// is added on its own: count 1, box = the point, one voxel bit of its block.
__device__ __noinline__ void stray_pixel(TileSmem &s, uint32_t *lab_j, uint32_t *lab_cnt, int (*lab_box)[6], uint32_t *det_npx,
                                         int *det_box, unsigned long long *surv_key, unsigned long long *surv_bits,
                                         uint32_t *surv_j, uint32_t surv_cap, uint32_t *counters, uint32_t *err, double *det_gm,
                                         uint32_t j, unsigned long long bkey, uint32_t bit, float p0, float p1, float p2) {
  if (det_gm) {  // G1: the point's contribution to the detection's moments
    double *g = det_gm + (size_t)j * 9;
    const double x = p0, y = p1, z = p2;
    atomicAdd(g + 0, x), atomicAdd(g + 1, y), atomicAdd(g + 2, z);
    atomicAdd(g + 3, x * x), atomicAdd(g + 4, x * y), atomicAdd(g + 5, x * z);
    atomicAdd(g + 6, y * y), atomicAdd(g + 7, y * z), atomicAdd(g + 8, z * z);
  }
  const int li = tile_label_slot_in(lab_j, j);
  const int o0 = f2ord(p0), o1 = f2ord(p1), o2 = f2ord(p2);
  const uint32_t lo = (bit & 32) ? 0u : 1u << (bit & 31), hi = (bit & 32) ? 1u << (bit & 31) : 0u;
  if (li >= 0) {
    atomicAdd(&lab_cnt[li], 1u);
    atomicMin(&lab_box[li][0], o0), atomicMin(&lab_box[li][1], o1), atomicMin(&lab_box[li][2], o2);
    atomicMax(&lab_box[li][3], o0), atomicMax(&lab_box[li][4], o1), atomicMax(&lab_box[li][5], o2);
    const unsigned long long tag = bkey | ((unsigned long long)li << LABEL_SHIFT);
    uint32_t h = hash32((uint32_t)tag, (uint32_t)(tag >> 32)) & (TILE_ENT - 1);
    for (int probe = 0; probe < TILE_ENT; ++probe) {
      unsigned long long cur = *(volatile unsigned long long *)&s.tag[h];
      if (cur == BLK_EMPTY) {
        cur = atomicCAS(&s.tag[h], BLK_EMPTY, tag);
        if (cur == BLK_EMPTY) cur = tag;
      }
      if (cur == tag) {
        if (lo) atomicOr(&s.mlo[h], lo);
        if (hi) atomicOr(&s.mhi[h], hi);
        return;
      }
      h = (h + 1) & (TILE_ENT - 1);
    }
  } else {
    atomicAdd(&det_npx[j], 1u);
    atomicMin(&det_box[j * 6 + 0], o0), atomicMin(&det_box[j * 6 + 1], o1), atomicMin(&det_box[j * 6 + 2], o2);
    atomicMax(&det_box[j * 6 + 3], o0), atomicMax(&det_box[j * 6 + 4], o1), atomicMax(&det_box[j * 6 + 5], o2);
  }
  const uint32_t pos = atomicAdd(&counters[2], 1u);
  if (pos < surv_cap) {
    surv_key[pos] = bkey;
    surv_bits[pos] = ((unsigned long long)hi << 32) | lo;
    surv_j[pos] = j;
  } else {
    atomicOr(err, ERR_PAIR_TABLE_FULL);
  }
}

// ---------------------------------------------------------------------------------------------------
// lift kernel (steps 1-2).  Persistent CTAs; one 64x16 pixel tile per iteration, each thread owns 8
// consecutive pixels of one row (2 x 128-bit depth loads + 1 x 128-bit mask load, issued one tile ahead).
//   Phase 1 (straight-line fp32/int code per pixel): validity (R3, R4), back-projection (R5), voxel index
//     (R6) -> block key + voxel bit, point box.
//   Phase 2 (warp-synchronous): the voxel of a pixel is one bit of its block's 64-bit mask, so the
//     per-detection dedupe (R7) is a bitwise OR -- over the thread's pixels of one block, over the lanes of
//     the warp that hold the same (detection, block) (match.any + redux.or), and into the tile's
//     shared-memory table (atomicOr).
//   Flush: one (block, detection, voxel bits) record per table entry goes to the call's survivor queue.  The
//     CTA reserves queue space in chunks of TILE_ENT records one tile ahead, so no thread ever waits for a
//     global atomic; the unused tail of the last chunk is padded with empty records (bits == 0).
// Two barriers per tile.  Per-detection pixel counts and point boxes go through shared-memory
// accumulators (REDUX fast path when a warp holds one detection) to one set of global atomics per
// (tile, detection).
template <bool VEC, bool GAUSS>
__global__ void __launch_bounds__(LIFT_THREADS, GAUSS ? 4 : 6) lift_voxelise_kernel(DevMap m, CallArgs a, int tiles_x, int tiles_y) {
  pdl_trigger();  // the probe kernel may become resident as soon as CTAs of this grid retire
  __shared__ TileSmem s;
  __shared__ uint32_t lab_j2[2][MAX_LABELS];  // label tables are double buffered: the flush of tile t reads
  __shared__ uint32_t lab_cnt2[2][MAX_LABELS];  // its copy while tile t+1 initialises the other
  __shared__ int lab_box2[2][MAX_LABELS][6];
  const int tid = threadIdx.x, lane = tid & 31;
  const int tiles_xy = tiles_x * tiles_y;
  const int n_tiles = tiles_xy * a.F;
  const float inv_vs = m.inv_vs, z_min = m.z_min, z_max = m.z_max;
  const float INF = __int_as_float(0x7F800000);
  constexpr unsigned FULL = 0xFFFFFFFFu;
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
  int par = 0;
  TileRegs cur = load_tile<VEC>(m, a, blockIdx.x, tiles_x, tiles_xy, tid);
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, par ^= 1) {
    TileRegs nxt = cur;
    if (tile + (int)gridDim.x < n_tiles) nxt = load_tile<VEC>(m, a, tile + gridDim.x, tiles_x, tiles_xy, tid);
    const int f = tile / tiles_xy;
    const int trem = tile - f * tiles_xy;
    const int ty = trem / tiles_x, tx = trem - ty * tiles_x;
    const int v = ty * TILE_H + (tid >> 3);
    const int u0 = tx * TILE_W + (tid & 7) * 8;
    // camera of the frame, prepared by prep_kernel: (inv_fx, inv_fy, cx, cy), (r00 r01 r02 tx), (r10 ..), (r20 ..)
    const float4 *cp = reinterpret_cast<const float4 *>(m.cam + 16 * f);
    const float4 c0 = __ldg(cp), c1 = __ldg(cp + 1), c2 = __ldg(cp + 2), c3 = __ldg(cp + 3);
    const int det_base = a.base[f];
    const uint32_t n_det_f = (uint32_t)(a.base[f + 1] - det_base);
    uint32_t *lab_j = lab_j2[par], *lab_cnt = lab_cnt2[par];
    int(*lab_box)[6] = lab_box2[par];
    if (tid < MAX_LABELS) {
      lab_j[tid] = NONE32;
      lab_cnt[tid] = 0;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        lab_box[tid][k] = 0x7FFFFFFF;
        lab_box[tid][3 + k] = (int)0x80000000;
      }
    }
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
        s.next_base = atomicAdd(&m.counters[2], (uint32_t)TILE_ENT);
        s.next_valid = 1;
      }
    }

    // ---- phase 1
    const float z[8] = {cur.d0.x, cur.d0.y, cur.d0.z, cur.d0.w, cur.d1.x, cur.d1.y, cur.d1.z, cur.d1.w};
    const uint32_t lab[8] = {cur.mk.x & 0xFFFF, cur.mk.x >> 16, cur.mk.y & 0xFFFF, cur.mk.y >> 16,
                             cur.mk.z & 0xFFFF, cur.mk.z >> 16, cur.mk.w & 0xFFFF, cur.mk.w >> 16};
    const float yn = __fmul_rn(__fsub_rn((float)v, c0.w), c0.y);  // R5 term shared by the thread's 8 pixels
    const float u0f = (float)u0;  // (float)(u0 + i) == u0f + (float)i exactly (integers below 2^24)
    unsigned long long ikey[8];
    uint32_t ibit_lo = 0, ibit_hi = 0;  // 6-bit voxel index inside the block, pixels 0-3 / 4-7
    uint32_t valid = 0, L0 = 0;         // pixels of the thread's first detection L0 (almost always the only one)
    float mn0 = INF, mn1 = INF, mn2 = INF, mx0 = -INF, mx1 = -INF, mx2 = -INF;
    // G1: moments of the thread's points about its first point (fp32 stays exact enough: offsets of a few cm)
    float gc0 = 0.f, gc1 = 0.f, gc2 = 0.f, g1x = 0.f, g1y = 0.f, g1z = 0.f;
    float gxx = 0.f, gxy = 0.f, gxz = 0.f, gyy = 0.f, gyz = 0.f, gzz = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      ikey[i] = BLK_EMPTY;
      const uint32_t l = lab[i];
      if (l != 0) {
        if (l > n_det_f) {
          acc_ignored++;
        } else if (depth_valid(z[i], z_min, z_max)) {
          const float xn = __fmul_rn(__fsub_rn(__fadd_rn(u0f, (float)i), c0.z), c0.x);
          const float xc = __fmul_rn(xn, z[i]), yc = __fmul_rn(yn, z[i]);
          float p[3];
          p[0] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c1.x, xc), __fmul_rn(c1.y, yc)), __fmul_rn(c1.z, z[i])), c1.w);
          p[1] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c2.x, xc), __fmul_rn(c2.y, yc)), __fmul_rn(c2.z, z[i])), c2.w);
          p[2] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(c3.x, xc), __fmul_rn(c3.y, yc)), __fmul_rn(c3.z, z[i])), c3.w);
          uint32_t ix, iy, iz;
          if (voxel_index(p, inv_vs, ix, iy, iz)) {
            acc_valid++;
            const unsigned long long bk = block_key(ix, iy, iz);
            const uint32_t bit = block_bit(ix, iy, iz);
            if (L0 == 0) L0 = l;
            if (l == L0) {
              valid |= 1u << i;
              ikey[i] = bk;
              if (i < 4) ibit_lo |= bit << (6 * i); else ibit_hi |= bit << (6 * (i - 4));
              mn0 = fminf(mn0, p[0]), mn1 = fminf(mn1, p[1]), mn2 = fminf(mn2, p[2]);
              mx0 = fmaxf(mx0, p[0]), mx1 = fmaxf(mx1, p[1]), mx2 = fmaxf(mx2, p[2]);
              if (GAUSS) {
                if (valid == (1u << i)) gc0 = p[0], gc1 = p[1], gc2 = p[2];  // first point of the thread
                const float dx = p[0] - gc0, dy = p[1] - gc1, dz = p[2] - gc2;
                g1x += dx, g1y += dy, g1z += dz;
                gxx = fmaf(dx, dx, gxx), gxy = fmaf(dx, dy, gxy), gxz = fmaf(dx, dz, gxz);
                gyy = fmaf(dy, dy, gyy), gyz = fmaf(dy, dz, gyz), gzz = fmaf(dz, dz, gzz);
              }
            } else {  // rare: the thread's 8 pixels straddle two detections -- this pixel goes in on its own
              stray_pixel(s, lab_j, lab_cnt, lab_box, m.det_npx, m.det_box, m.surv_key, m.surv_bits, m.surv_j, m.surv_cap,
                          m.counters, m.err, GAUSS ? m.det_gm : nullptr, (uint32_t)det_base + l - 1, bk, bit, p[0], p[1], p[2]);
            }
          } else {
            acc_dropped++;
          }
        }
      }
    }

    // ---- phase 2 (warp-synchronous): detection L0 of every thread
    if (__any_sync(FULL, valid != 0)) {
      const uint32_t j = (uint32_t)det_base + L0 - 1;
      int li = -1;
      if (valid) li = tile_label_slot_in(lab_j, j);
      // per-detection pixel count and point AABB (R7): REDUX when the warp holds one detection
      {
        const unsigned has = __ballot_sync(FULL, valid != 0);
        const int src = __ffs(has) - 1;
        const uint32_t lead_L = __shfl_sync(FULL, L0, src);
        const int lead_li = __shfl_sync(FULL, li, src);
        const bool uniform = __all_sync(FULL, valid == 0 || L0 == lead_L);
        const int o0 = f2ord(mn0), o1 = f2ord(mn1), o2 = f2ord(mn2), o3 = f2ord(mx0), o4 = f2ord(mx1), o5 = f2ord(mx2);
        const uint32_t cnt = __popc(valid);
        if (uniform) {
          const uint32_t tot = __reduce_add_sync(FULL, cnt);
          const int r0 = __reduce_min_sync(FULL, o0), r1 = __reduce_min_sync(FULL, o1), r2 = __reduce_min_sync(FULL, o2),
                    r3 = __reduce_max_sync(FULL, o3), r4 = __reduce_max_sync(FULL, o4), r5 = __reduce_max_sync(FULL, o5);
          if (lane == 0) label_add_in(lab_cnt, lab_box, m, lead_li, (uint32_t)det_base + lead_L - 1, tot, r0, r1, r2, r3, r4, r5);
        } else if (valid) {
          label_add_in(lab_cnt, lab_box, m, li, j, cnt, o0, o1, o2, o3, o4, o5);
        }
      }
      if (GAUSS) {  // G1: raw moments in double (parallel-axis shift from the thread's centre), one set of atomics per warp
        const double n = (double)__popc(valid), c0 = gc0, c1 = gc1, c2 = gc2, sx = g1x, sy = g1y, sz = g1z;
        double g[9] = {sx + n * c0, sy + n * c1, sz + n * c2,
                       gxx + 2.0 * c0 * sx + n * c0 * c0, gxy + c0 * sy + c1 * sx + n * c0 * c1, gxz + c0 * sz + c2 * sx + n * c0 * c2,
                       gyy + 2.0 * c1 * sy + n * c1 * c1, gyz + c1 * sz + c2 * sy + n * c1 * c2, gzz + 2.0 * c2 * sz + n * c2 * c2};
        const unsigned has = __ballot_sync(FULL, valid != 0);
        const uint32_t lead_L = __shfl_sync(FULL, L0, __ffs(has) - 1);
        if (__all_sync(FULL, valid == 0 || L0 == lead_L)) {
#pragma unroll
          for (int k = 0; k < 9; ++k) {
            if (!valid) g[k] = 0.0;
#pragma unroll
            for (int sft = 16; sft; sft >>= 1) g[k] += __shfl_xor_sync(FULL, g[k], sft);
          }
          if (lane < 9) {
            double v = g[0];
#pragma unroll
            for (int k = 1; k < 9; ++k) v = lane == k ? g[k] : v;
            atomicAdd(m.det_gm + (size_t)((uint32_t)det_base + lead_L - 1) * 9 + lane, v);
          }
        } else if (valid) {
#pragma unroll
          for (int k = 0; k < 9; ++k) atomicAdd(m.det_gm + (size_t)j * 9 + k, g[k]);
        }
      }
      // blocks: one pass per distinct block among the thread's pixels
      uint32_t rem = valid;
      while (__any_sync(FULL, rem != 0)) {
        unsigned long long kb = BLK_EMPTY;
#pragma unroll
        for (int i = 7; i >= 0; --i)
          if ((rem >> i) & 1u) kb = ikey[i];
        uint32_t lo = 0, hi = 0, hit = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if (((rem >> i) & 1u) && ikey[i] == kb) {
            hit |= 1u << i;
            const uint32_t bit = ((i < 4 ? ibit_lo >> (6 * i) : ibit_hi >> (6 * (i - 4)))) & 63u;
            const uint32_t one = 1u << (bit & 31);
            lo |= (bit & 32) ? 0u : one;
            hi |= (bit & 32) ? one : 0u;
          }
        rem &= ~hit;
        bool ovf = hit && li < 0;  // no label slot
        const bool tab = hit && li >= 0;
        const unsigned act = __ballot_sync(FULL, tab);
        if (tab) {
          const unsigned long long tag = kb | ((unsigned long long)li << LABEL_SHIFT);
          const unsigned same = __match_any_sync(act, tag);
          lo = __reduce_or_sync(same, lo), hi = __reduce_or_sync(same, hi);
          if (lane == __ffs(same) - 1) ovf = !tile_block_add(s, li, kb, lo, hi);
        }
        emit_overflow(m, ovf, kb, j, lo, hi);
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
          uint32_t pos = cpos + base + __popc(b & ((1u << lane) - 1));
          if (pos >= cend) pos = nbase + (pos - cend);
          survivor_store(m, pos, tag & ((1ull << LABEL_SHIFT) - 1), lab_j[(uint32_t)(tag >> LABEL_SHIFT)], s.mlo[e], s.mhi[e]);
          s.tag[e] = BLK_EMPTY;
          s.mlo[e] = 0;
          s.mhi[e] = 0;
        }
      }
      if (tid < MAX_LABELS && lab_j[tid] != NONE32) {
        const uint32_t j = lab_j[tid];
        atomicAdd(&m.det_npx[j], lab_cnt[tid]);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
          atomicMin(&m.det_box[j * 6 + k], lab_box[tid][k]);
          atomicMax(&m.det_box[j * 6 + 3 + k], lab_box[tid][3 + k]);
        }
      }
    }
    cur = nxt;
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

__global__ void __launch_bounds__(PROBE_THREADS) probe_kernel(DevMap m, CallArgs a) {
  pdl_trigger();  // cand_associate may become resident behind this grid
  pdl_wait();     // launched with PDL behind the lift kernel: its survivor queue is complete from here on
  const uint32_t nq = min(m.counters[2], m.surv_cap);
  const int lane = threadIdx.x & 31;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u; i0 < nq; i0 += stride) {
    const uint32_t i = i0 + lane;
    // ---- phase A
    uint32_t j = 0, slot = NONE32, ps = 0;
    unsigned long long nb = 0;
    if (i < nq) {
      const unsigned long long bkey = __ldcs(&m.surv_key[i]);
      const unsigned long long bits = __ldcs(&m.surv_bits[i]);
      j = __ldcs(&m.surv_j[i]);
      if (bits) slot = block_find_or_insert(m, bkey);  // bits == 0: padding of a reserved queue chunk
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
    // ---- phase B: 4 records per step, 8 lanes (owner sectors) per record
    const int sec = lane & 7;
    uint32_t pend_mine = 0;  // lane r: does record r have a voxel that was unowned at entry
#pragma unroll 1
    for (int step = 0; step < 8; ++step) {
      if (((act >> (step * 4)) & 0xFu) == 0) continue;  // warp-uniform
      const int src = step * 4 + (lane >> 3);
      const unsigned long long rnb = __shfl_sync(0xFFFFFFFFu, nb, src);
      const uint32_t rslot = __shfl_sync(0xFFFFFFFFu, slot, src);
      const uint32_t rj = __shfl_sync(0xFFFFFFFFu, j, src);
      const uint32_t byte = (uint32_t)(rnb >> (8 * sec)) & 0xFFu;
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
          const uint32_t o = own[b];
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
      const unsigned ub = __ballot_sync(0xFFFFFFFFu, unowned);
      if ((lane >> 2) == step) pend_mine = (ub >> ((lane & 3) * 8)) & 0xFFu;
    }
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
  return blocks;
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

int launch_debug_backproject(const DevMap &m, const float *depth, const uint16_t *mask, const float *K, const float *T,
                             int n_det, float *xyz, unsigned long long *keys, cudaStream_t s) {
  const int n = m.H * m.W;
  debug_backproject_kernel<<<(n + 255) / 256, 256, 0, s>>>(m, depth, mask, K, T, n_det, xyz, keys);
  return 1;
}

}  // namespace farm
