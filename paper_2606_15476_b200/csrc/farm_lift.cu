// farm_lift.cu -- steps 1-3 of the hot path in one pass over the images:
//   back-project masked pixels (R5), quantise to voxel keys (R6), per-detection dedupe (R7),
//   probe / insert the global voxel->object hash (R11, R12 pass 1) and build the sparse overlap
//   histogram (R9).  BASELINE.json north_star steps (1)-(3); PAPER.md:65, 347 ("masked depth points").
//
// HBM-bound by design: the only mandatory traffic is 6 B/pixel of depth+mask (128-bit loads) plus one
// 32-byte sector per distinct (detection, voxel) pair that survives the shared-memory tile dedupe.
#include "farm_internal.cuh"

namespace farm {

namespace {

constexpr int TILE_W = 128;
constexpr int TILE_H = 8;
constexpr int LIFT_THREADS = 128;
constexpr int TILE_PX = TILE_W * TILE_H;
constexpr int TILE_HASH = 512;   // slots of the direct-mapped tile filter
constexpr int TILE_Q = 512;      // tile queue entries in shared memory; overflow goes straight to the global queue
constexpr int MAX_LABELS = 32;   // per-tile detection accumulators
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
__device__ __forceinline__ bool voxel_key(const float p[3], float inv_vs, unsigned long long *key) {
  const float fx = __fmul_rn(p[0], inv_vs), fy = __fmul_rn(p[1], inv_vs), fz = __fmul_rn(p[2], inv_vs);
  const bool finite = fabsf(fx) < 2.0e6f && fabsf(fy) < 2.0e6f && fabsf(fz) < 2.0e6f;
  const uint32_t ix = (uint32_t)(__float2int_rd(fx) + KEY_BIAS), iy = (uint32_t)(__float2int_rd(fy) + KEY_BIAS),
                 iz = (uint32_t)(__float2int_rd(fz) + KEY_BIAS);
  if (!finite || ((ix | iy | iz) >> 21) != 0) return false;
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
  if (warp >= a.M) return;
  const T *row = (const T *)a.desc + (size_t)warp * m.D;
  float s = 0.f;
  for (int i = lane; i < m.D; i += 32) {
    const float x = to_f32<T>(row[i]);
    s = fmaf(x, x, s);
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
}

// ---------------------------------------------------------------------------------------------------
// global structures

// find-or-insert `key` in the voxel table with one 16-byte probe per slot; returns the slot index (NONE32 when the
// table is full) and the slot's owner / visit words as loaded (free slots hold OWNER_INIT / a dead epoch).
__device__ __forceinline__ uint32_t voxel_find_or_insert(const DevMap &m, unsigned long long key, uint32_t *owner,
                                                         uint32_t *visit) {
  unsigned long long h = voxel_hash(key) & m.table_mask;
  for (int probe = 0; probe < 8192; ++probe) {
    const uint4 w = __ldcg(reinterpret_cast<const uint4 *>(&m.table[h]));
    unsigned long long k = ((unsigned long long)w.y << 32) | w.x;
    if (k == KEY_EMPTY) {
      k = atomicCAS(&m.table[h].key, KEY_EMPTY, key);
      if (k == KEY_EMPTY) k = key;  // inserted: owner == OWNER_INIT already
    }
    if (k == key) {
      *owner = w.z;
      *visit = w.w;
      return (uint32_t)h;
    }
    h = (h + 1) & m.table_mask;
  }
  atomicOr(m.err, ERR_VOXEL_TABLE_FULL);
  return NONE32;
}

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

struct TileSmem {
  unsigned long long tag[TILE_HASH];   // direct-mapped filter of (key, label) pairs already queued by this tile
  unsigned long long qkey[TILE_Q];
  uint32_t qj[TILE_Q];
  uint32_t lab_j[MAX_LABELS];
  uint32_t lab_cnt[MAX_LABELS];
  int lab_box[MAX_LABELS][6];
  uint32_t q_count, q_base;
  uint32_t n_valid, n_dropped, n_ignored;
};

// accumulate a run (j, cnt, box as ordered ints) into the tile's per-detection accumulators
__device__ __noinline__ void tile_label_add(TileSmem &s, const DevMap &m, uint32_t j, uint32_t cnt, int mn0, int mn1,
                                            int mn2, int mx0, int mx1, int mx2) {
  uint32_t h = j % MAX_LABELS;
  for (int probe = 0; probe < MAX_LABELS; ++probe) {
    uint32_t l = *(volatile uint32_t *)&s.lab_j[h];
    if (l == NONE32) {
      l = atomicCAS(&s.lab_j[h], NONE32, j);
      if (l == NONE32) l = j;
    }
    if (l == j) {
      atomicAdd(&s.lab_cnt[h], cnt);
      atomicMin(&s.lab_box[h][0], mn0), atomicMin(&s.lab_box[h][1], mn1), atomicMin(&s.lab_box[h][2], mn2);
      atomicMax(&s.lab_box[h][3], mx0), atomicMax(&s.lab_box[h][4], mx1), atomicMax(&s.lab_box[h][5], mx2);
      return;
    }
    h = (h + 1) % MAX_LABELS;
  }
  // more than MAX_LABELS detections inside one tile: go to global memory directly
  atomicAdd(&m.det_npx[j], cnt);
  atomicMin(&m.det_box[j * 6 + 0], mn0), atomicMin(&m.det_box[j * 6 + 1], mn1), atomicMin(&m.det_box[j * 6 + 2], mn2);
  atomicMax(&m.det_box[j * 6 + 3], mx0), atomicMax(&m.det_box[j * 6 + 4], mx1), atomicMax(&m.det_box[j * 6 + 5], mx2);
}

// Tile-level dedupe: a direct-mapped, lock-free filter in shared memory.  The slot index carries the low 10
// bits of the label and bit 63 of the tag the 11th, so an equal tag in the same slot means the same
// (key, label) pair exactly (labels >= 2048 bypass the filter).  It may let duplicates through (evictions,
// races); it never drops a pair.  The exact set is the global pair set of probe_kernel.
__device__ __forceinline__ bool tile_filter_fresh(TileSmem &s, unsigned long long key, uint32_t l) {
  if (l >= 2048u) return true;
  const uint32_t slot = (hash32((uint32_t)key, (uint32_t)(key >> 32)) ^ l) & (TILE_HASH - 1);
  const unsigned long long tag = key | ((unsigned long long)((l >> 10) & 1u) << 63);
  if (tag == KEY_EMPTY) return true;  // indistinguishable from an empty slot: never filtered
  if (*(volatile unsigned long long *)&s.tag[slot] == tag) return false;
  *(volatile unsigned long long *)&s.tag[slot] = tag;
  return true;
}

// ---------------------------------------------------------------------------------------------------
// lift kernel (steps 1-2).  One 128x8 pixel tile per CTA; each thread owns 8 consecutive pixels of one row
// (2 x 128-bit depth loads + 1 x 128-bit mask load).  Output: per-detection pixel counts and point boxes,
// and the tile's distinct (detection, voxel key) pairs appended to the call's survivor queue.
// raw registers of one thread's 8 pixels (2 x 128-bit depth + 1 x 128-bit mask)
struct TileRegs {
  float4 d0, d1;
  uint4 mk;
};

template <bool VEC>
__device__ __forceinline__ TileRegs load_tile(const DevMap &m, const CallArgs &a, int tile, int tiles_x, int tiles_y, int tid) {
  const int f = tile / (tiles_x * tiles_y);
  const int trem = tile - f * tiles_x * tiles_y;
  const int ty = trem / tiles_x, tx = trem - ty * tiles_x;
  const int v = ty * TILE_H + (tid >> 4);
  const int u0 = tx * TILE_W + (tid & 15) * 8;
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

template <bool VEC>
__global__ void __launch_bounds__(LIFT_THREADS) lift_voxelise_kernel(DevMap m, CallArgs a, int tiles_x, int tiles_y) {
  __shared__ TileSmem s;
  const int tid = threadIdx.x, lane = tid & 31;
  const int n_tiles = tiles_x * tiles_y * a.F;
  // Each CTA walks tiles blockIdx.x, +gridDim.x, ...; the loads of the next tile are issued before the current
  // one is processed (register double buffering), so DRAM latency hides even at two resident CTAs per SM.
  TileRegs cur = load_tile<VEC>(m, a, blockIdx.x, tiles_x, tiles_y, tid);
  for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
  TileRegs nxt = cur;
  if (tile + (int)gridDim.x < n_tiles) nxt = load_tile<VEC>(m, a, tile + gridDim.x, tiles_x, tiles_y, tid);
  const int f = tile / (tiles_x * tiles_y);
  const int trem = tile - f * tiles_x * tiles_y;
  const int ty = trem / tiles_x, tx = trem - ty * tiles_x;
  const int v = ty * TILE_H + (tid >> 4);
  const int u0 = tx * TILE_W + (tid & 15) * 8;
  float z[8];
  uint32_t lab[8];
  z[0] = cur.d0.x, z[1] = cur.d0.y, z[2] = cur.d0.z, z[3] = cur.d0.w;
  z[4] = cur.d1.x, z[5] = cur.d1.y, z[6] = cur.d1.z, z[7] = cur.d1.w;
  lab[0] = cur.mk.x & 0xFFFF, lab[1] = cur.mk.x >> 16, lab[2] = cur.mk.y & 0xFFFF, lab[3] = cur.mk.y >> 16;
  lab[4] = cur.mk.z & 0xFFFF, lab[5] = cur.mk.z >> 16, lab[6] = cur.mk.w & 0xFFFF, lab[7] = cur.mk.w >> 16;
  for (int i = tid; i < TILE_HASH; i += LIFT_THREADS) s.tag[i] = KEY_EMPTY;
  if (tid < MAX_LABELS) {
    s.lab_j[tid] = NONE32;
    s.lab_cnt[tid] = 0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      s.lab_box[tid][k] = 0x7FFFFFFF;
      s.lab_box[tid][3 + k] = (int)0x80000000;
    }
  }
  if (tid == 0) s.q_count = 0, s.n_valid = 0, s.n_dropped = 0, s.n_ignored = 0;
  const Camera cam = load_camera(a.K + 9 * f, a.T + 16 * f);
  const int det_base = a.base[f];
  const uint32_t n_det_f = (uint32_t)(a.base[f + 1] - det_base);
  // R5 term shared by the thread's 8 pixels (same row)
  const float yn = __fmul_rn(__fsub_rn((float)v, cam.cy), cam.inv_fy);
  __syncthreads();

  // ---- per pixel: validity (R3, R4), back-projection (R5), key (R6), tile-level dedupe
  const float INF = __int_as_float(0x7F800000);
  uint32_t cur_l = 0, cur_cnt = 0;  // current run of equal labels (label 0 = none)
  float mn0 = INF, mn1 = INF, mn2 = INF, mx0 = -INF, mx1 = -INF, mx2 = -INF;
  unsigned long long prev_key = KEY_EMPTY;
  uint32_t prev_l = 0;
  uint32_t n_valid = 0, n_dropped = 0, n_ignored = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    bool fresh = false;
    unsigned long long key = KEY_EMPTY;
    const uint32_t l = lab[i];
    if (l != 0) {
      if (l > n_det_f) {
        n_ignored++;
      } else if (depth_valid(z[i], m.z_min, m.z_max)) {
        float p[3];
        const float xn = __fmul_rn(__fsub_rn((float)(u0 + i), cam.cx), cam.inv_fx);
        const float xc = __fmul_rn(xn, z[i]), yc = __fmul_rn(yn, z[i]);
#pragma unroll
        for (int k = 0; k < 3; ++k)
          p[k] = __fadd_rn(__fadd_rn(__fadd_rn(__fmul_rn(cam.r[3 * k], xc), __fmul_rn(cam.r[3 * k + 1], yc)),
                                     __fmul_rn(cam.r[3 * k + 2], z[i])),
                           cam.t[k]);
        if (voxel_key(p, m.inv_vs, &key)) {
          n_valid++;
          if (l != cur_l) {
            if (cur_l) tile_label_add(s, m, (uint32_t)det_base + cur_l - 1, cur_cnt, f2ord(mn0), f2ord(mn1), f2ord(mn2),
                                      f2ord(mx0), f2ord(mx1), f2ord(mx2));
            cur_l = l, cur_cnt = 0;
            mn0 = mn1 = mn2 = INF, mx0 = mx1 = mx2 = -INF;
          }
          cur_cnt++;
          mn0 = fminf(mn0, p[0]), mn1 = fminf(mn1, p[1]), mn2 = fminf(mn2, p[2]);
          mx0 = fmaxf(mx0, p[0]), mx1 = fmaxf(mx1, p[1]), mx2 = fmaxf(mx2, p[2]);
          if (!(key == prev_key && l == prev_l)) {  // thread-local dedupe of consecutive pixels
            prev_key = key, prev_l = l;
            fresh = tile_filter_fresh(s, key, l);
          }
        } else {
          n_dropped++;
        }
      }
    }
    // warp-ballot compaction of the surviving (detection, key) pairs into the tile queue
    const unsigned b = __ballot_sync(0xFFFFFFFFu, fresh);
    if (b) {
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&s.q_count, (uint32_t)__popc(b));
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      if (fresh) {
        const uint32_t pos = base + __popc(b & ((1u << lane) - 1));
        if (pos < TILE_Q) {
          s.qkey[pos] = key;
          s.qj[pos] = (uint32_t)det_base + l - 1;
        } else {  // rare: more distinct pairs in one tile than the shared queue holds
          const uint32_t gp = atomicAdd(&m.counters[2], 1u);
          if (gp < m.surv_cap) {
            m.surv_key[gp] = key;
            m.surv_j[gp] = (uint32_t)det_base + l - 1;
          } else {
            atomicOr(m.err, ERR_PAIR_TABLE_FULL);
          }
        }
      }
    }
  }
  // per-detection pixel count and point AABB (R7): warp-uniform fast path through REDUX, else per thread
  {
    const unsigned has = __ballot_sync(0xFFFFFFFFu, cur_l != 0);
    if (has) {
      const uint32_t lead_l = __shfl_sync(0xFFFFFFFFu, cur_l, __ffs(has) - 1);
      const bool uniform = __all_sync(0xFFFFFFFFu, cur_l == 0 || cur_l == lead_l);
      const int o0 = f2ord(mn0), o1 = f2ord(mn1), o2 = f2ord(mn2), o3 = f2ord(mx0), o4 = f2ord(mx1), o5 = f2ord(mx2);
      if (uniform) {
        const uint32_t cnt = __reduce_add_sync(0xFFFFFFFFu, cur_cnt);
        const int r0 = __reduce_min_sync(0xFFFFFFFFu, o0), r1 = __reduce_min_sync(0xFFFFFFFFu, o1),
                  r2 = __reduce_min_sync(0xFFFFFFFFu, o2), r3 = __reduce_max_sync(0xFFFFFFFFu, o3),
                  r4 = __reduce_max_sync(0xFFFFFFFFu, o4), r5 = __reduce_max_sync(0xFFFFFFFFu, o5);
        if (lane == 0) tile_label_add(s, m, (uint32_t)det_base + lead_l - 1, cnt, r0, r1, r2, r3, r4, r5);
      } else if (cur_l != 0) {
        tile_label_add(s, m, (uint32_t)det_base + cur_l - 1, cur_cnt, o0, o1, o2, o3, o4, o5);
      }
    }
    n_valid = __reduce_add_sync(0xFFFFFFFFu, n_valid);
    n_dropped = __reduce_add_sync(0xFFFFFFFFu, n_dropped);
    n_ignored = __reduce_add_sync(0xFFFFFFFFu, n_ignored);
    if (lane == 0) {
      if (n_valid) atomicAdd(&s.n_valid, n_valid);
      if (n_dropped) atomicAdd(&s.n_dropped, n_dropped);
      if (n_ignored) atomicAdd(&s.n_ignored, n_ignored);
    }
  }
  __syncthreads();

  // ---- append the tile queue to the call's survivor queue (one global atomic per tile, coalesced copy)
  const uint32_t nq = min(s.q_count, (uint32_t)TILE_Q);
  if (tid == 0 && nq) s.q_base = atomicAdd(&m.counters[2], nq);
  // ---- flush the tile's per-detection accumulators and counters
  if (tid < MAX_LABELS && s.lab_j[tid] != NONE32) {
    const uint32_t j = s.lab_j[tid];
    atomicAdd(&m.det_npx[j], s.lab_cnt[tid]);
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      atomicMin(&m.det_box[j * 6 + k], s.lab_box[tid][k]);
      atomicMax(&m.det_box[j * 6 + 3 + k], s.lab_box[tid][3 + k]);
    }
  }
  if (tid == 0) {
    if (s.n_valid) atomicAdd(&m.stats->valid_points, (unsigned long long)s.n_valid);
    if (s.n_dropped) atomicAdd(&m.stats->dropped_points, (unsigned long long)s.n_dropped);
    if (s.n_ignored) atomicAdd(&m.stats->ignored_pixels, (unsigned long long)s.n_ignored);
  }
  __syncthreads();
  const uint32_t qb = s.q_base;
  for (uint32_t i = tid; i < nq; i += LIFT_THREADS) {
    const uint32_t pos = qb + i;
    if (pos < m.surv_cap) {
      m.surv_key[pos] = s.qkey[i];
      m.surv_j[pos] = s.qj[i];
    } else {
      atomicOr(m.err, ERR_PAIR_TABLE_FULL);
    }
  }
  __syncthreads();  // the tile's shared state is re-initialised by the next iteration
  cur = nxt;
  }
}

// ---------------------------------------------------------------------------------------------------
// probe kernel (step 3 and R12 pass 1).  One thread per queued (detection, key) pair: find or insert the
// key in the global voxel table, make the pair exact through the per-call pair set, then
//   |V_d| += 1,  append to the pair list,  overlap c[d][owner] += 1 when the key was owned at entry (R9),
//   claim = min(claim, d) when this call inserted the key (R12).
// Atomics are aggregated over the lanes of a warp that hit the same address (__match_any_sync).
__global__ void __launch_bounds__(256) probe_kernel(DevMap m, CallArgs a) {
  const uint32_t nq = min(m.counters[2], m.surv_cap);
  const int lane = threadIdx.x & 31;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u; i0 < nq; i0 += stride) {
    const uint32_t i = i0 + lane;
    bool is_new = false, owned = false;
    uint32_t j = 0, slot = NONE32, owner = OWNER_PENDING;
    if (i < nq) {
      const unsigned long long key = __ldcs(&m.surv_key[i]);
      j = __ldcs(&m.surv_j[i]);
      uint32_t visit = 0;
      slot = voxel_find_or_insert(m, key, &owner, &visit);
      if (slot != NONE32) {
        // exactness of the (detection, key) pair: first toucher of the key in this call wins the slot's
        // visit word; a second detection on the same key (object boundaries) uses the per-call pair set
        const uint32_t mine = (a.epoch << 16) | j;
        for (;;) {
          if (visit == mine) break;                        // this pair was already counted
          if ((visit >> 16) != a.epoch) {                  // nobody touched the key in this call yet
            const uint32_t old = atomicCAS(&m.table[slot].visit, visit, mine);
            if (old == visit) {
              is_new = true;
              break;
            }
            visit = old;
            continue;
          }
          const unsigned long long pv = ((unsigned long long)mine << 32) | slot;
          uint32_t ps;
          const int r = epoch_insert(m.pair_set, m.pair_mask, pv, a.epoch, &ps);
          if (r < 0) atomicOr(m.err, ERR_PAIR_TABLE_FULL);
          is_new = r == 1;
          break;
        }
        owned = is_new && owner < OWNER_PENDING;  // owned at entry (R9); else inserted by this call (R12)
      }
    }
    const unsigned act = __ballot_sync(0xFFFFFFFFu, is_new);
    if (act) {
      // append to the pair list (one atomic per warp)
      uint32_t base = 0;
      if (lane == 0) base = atomicAdd(&m.counters[0], (uint32_t)__popc(act));
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      const unsigned oact = __ballot_sync(0xFFFFFFFFu, owned);
      if (is_new) {
        const uint32_t pos = base + __popc(act & ((1u << lane) - 1));
        if (pos < m.pair_cap)
          m.pair_list[pos] = ((unsigned long long)(owned ? 0 : 1) << 63) | ((unsigned long long)j << 32) | slot;
        else
          atomicOr(m.err, ERR_PAIR_TABLE_FULL);
        // |V_d| += 1, aggregated over the lanes of the same detection
        const unsigned same = __match_any_sync(act, j);
        if (lane == __ffs(same) - 1) atomicAdd(&m.det_nv[j], (uint32_t)__popc(same));
        if (!owned) atomicMin(&m.table[slot].owner, OWNER_PENDING | j);  // R12: lowest detection index wins
      }
      // overlap histogram c[j][owner] += 1, aggregated over lanes with the same (j, owner)
      if (owned) {
        const unsigned long long jo = ((unsigned long long)j << 32) | owner;
        const unsigned same = __match_any_sync(oact, jo);
        if (lane == __ffs(same) - 1) {
          const unsigned long long ov = ((unsigned long long)a.epoch << 48) | jo;
          uint32_t os;
          const int r = epoch_insert(m.ov_keys, m.ov_mask, ov, a.epoch, &os);
          if (r < 0) {
            atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
          } else {
            if (r == 1) {
              const uint32_t c = atomicAdd(&m.counters[1], 1u);
              if (c < m.cand_cap)
                m.cand_slot[c] = os;
              else
                atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
            }
            atomicAdd(&m.ov_cnt[os], (uint32_t)__popc(same));
          }
        }
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

}  // namespace

int launch_prep(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  const int blocks = a.M > 0 ? (a.M + 3) / 4 : 1;
  if (m.dtype == FARM_DTYPE_F32)
    prep_kernel<float><<<blocks, 128, 0, s>>>(m, a);
  else if (m.dtype == FARM_DTYPE_F16)
    prep_kernel<__half><<<blocks, 128, 0, s>>>(m, a);
  else
    prep_kernel<__nv_bfloat16><<<blocks, 128, 0, s>>>(m, a);
  return 1;
}

int launch_lift(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  const int tiles_x = (m.W + TILE_W - 1) / TILE_W, tiles_y = (m.H + TILE_H - 1) / TILE_H;
  const int n_tiles = tiles_x * tiles_y * a.F;
  const int grid = n_tiles < 148 * 8 ? n_tiles : 148 * 8;
  const bool vec = (m.W % 8 == 0) && ((uintptr_t)a.depth % 16 == 0) && ((uintptr_t)a.mask % 16 == 0);
  if (vec)
    lift_voxelise_kernel<true><<<grid, LIFT_THREADS, 0, s>>>(m, a, tiles_x, tiles_y);
  else
    lift_voxelise_kernel<false><<<grid, LIFT_THREADS, 0, s>>>(m, a, tiles_x, tiles_y);
  return 1;
}

int launch_probe(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  probe_kernel<<<148 * 8, 256, 0, s>>>(m, a);
  return 1;
}

int launch_debug_backproject(const DevMap &m, const float *depth, const uint16_t *mask, const float *K, const float *T,
                             int n_det, float *xyz, unsigned long long *keys, cudaStream_t s) {
  const int n = m.H * m.W;
  debug_backproject_kernel<<<(n + 255) / 256, 256, 0, s>>>(m, depth, mask, K, T, n_det, xyz, keys);
  return 1;
}

}  // namespace farm
