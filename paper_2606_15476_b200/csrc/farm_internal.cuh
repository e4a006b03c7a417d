// farm_internal.cuh -- device-side data layout and small helpers shared by the library's own kernels.
// (Product code.  Shares nothing with oracle/.)
#pragma once
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/farm.h"

namespace farm {

constexpr uint64_t KEY_EMPTY = 0xFFFFFFFFFFFFFFFFull;
constexpr uint32_t OWNER_PENDING = 0x80000000u;  // owner >= this: inserted by the running call, low bits = claim (R12)
constexpr uint32_t OWNER_INIT = 0xFFFFFFFFu;     // free slot: pending with no claim yet
constexpr int KEY_BIAS = 1 << 20;
constexpr int MAX_FRAMES = 64;
constexpr int EPOCH_BITS = 16;                    // per-call scratch state is epoch tagged, never cleared
constexpr int DET_BITS = 16;                      // detections per call < 2^16
constexpr uint32_t EPOCH_MAX = (1u << EPOCH_BITS) - 1;

// sticky device error bits
constexpr uint32_t ERR_VOXEL_TABLE_FULL = 1u;
constexpr uint32_t ERR_PAIR_TABLE_FULL = 2u;
constexpr uint32_t ERR_OVERLAP_TABLE_FULL = 4u;
constexpr uint32_t ERR_OBJECT_CAPACITY = 8u;
constexpr uint32_t ERR_IMPORT_DUPLICATE = 16u;
constexpr uint32_t ERR_SYNC_TIMEOUT = 32u;       // a device-side wait for another grid of the same call expired
constexpr uint32_t DD_FLAG = 0x80000000u;        // overlap-map "owner" field: DD_FLAG | e = detection e of the same call (U2)
constexpr uint32_t ERR_IMPORT_COUNT = 64u;       // import: objects[i].n_voxels differs from the voxels listed for i
constexpr uint32_t ERR_EDGE_TABLE_FULL = 128u;   // W4: the edge dictionary is full
constexpr uint32_t SPIN_LIMIT = 1u << 23;        // polls of ~0.25 us each (about 2 s) before a device-side wait gives up

// Global voxel -> object hash (R11: one owner per key), stored as a hash of 4x4x4 VOXEL BLOCKS so that the
// voxels of one surface patch share DRAM lines:
//   blk_key[slot]        57-bit block key (bx<<38 | by<<19 | bz, b = biased voxel index >> 2), BLK_EMPTY when free;
//                        8 bytes per slot: the whole key array of a 1e8-voxel map fits in L2
//   blk_owner[slot][64]  owner of voxel (lx<<4 | ly<<2 | lz) of the block: object id, OWNER_INIT = unowned;
//                        while the inserting call runs: OWNER_PENDING | lowest detection index j of that call
//                        containing the voxel (R12: that detection's object will own it).  256 bytes per block.
constexpr unsigned long long BLK_EMPTY = 0xFFFFFFFFFFFFFFFFull;
constexpr int BLK_VOXELS = 64;

__host__ __device__ __forceinline__ unsigned long long block_key(uint32_t ix, uint32_t iy, uint32_t iz) {
  return ((unsigned long long)(ix >> 2) << 38) | ((unsigned long long)(iy >> 2) << 19) | (unsigned long long)(iz >> 2);
}
__host__ __device__ __forceinline__ uint32_t block_bit(uint32_t ix, uint32_t iy, uint32_t iz) {
  return ((ix & 3u) << 4) | ((iy & 3u) << 2) | (iz & 3u);
}
// voxel key (R6 packing) of voxel `bit` of block `bkey`
__host__ __device__ __forceinline__ unsigned long long voxel_key_of(unsigned long long bkey, uint32_t bit) {
  const unsigned long long ix = (((bkey >> 38) & 0x7FFFFull) << 2) | ((bit >> 4) & 3u);
  const unsigned long long iy = (((bkey >> 19) & 0x7FFFFull) << 2) | ((bit >> 2) & 3u);
  const unsigned long long iz = ((bkey & 0x7FFFFull) << 2) | (bit & 3u);
  return (ix << 42) | (iy << 21) | iz;
}

struct CallStats {  // device mirror of farm_frame_stats
  unsigned long long valid_points, dropped_points, ignored_pixels, unique_voxels;
  uint32_t matches, spawns, skipped, n_det;
};
struct Totals {
  unsigned long long frames, calls, valid_points, unique_voxels, matches, spawns;
};

// Everything a kernel needs, passed by value.
struct DevMap {
  // parameters
  float inv_vs, w_geo, w_sem, tau, z_min, z_max;
  int D, dtype, H, W;
  int num_sms;                       // multiprocessors of the device (queried once; sizes every persistent grid)
  // objects (SoA).  HBM layout: descriptors are [max_objects, D] row-major, D contiguous.
  uint32_t max_objects;
  uint32_t *n_objects;               // device scalar N
  float *desc_master;                // fp32 masters (R21)
  void *desc_shadow;                 // storage-dtype shadows: similarity operand B (R14)
  float *inv_norm;                   // 1/|shadow_o| (0 for a zero row)
  uint32_t *n_voxels, *n_obs;
  unsigned long long *n_points;
  int *aabb;                         // [max_objects,6] order-preserving int image of fp32 min xyz, max xyz
  uint32_t *best_px;                 // best view (R23): valid pixel count, 0 = none
  unsigned long long *best_seq;      //   frame sequence number (full 64 bit) and
  uint32_t *best_det;                //   detection index inside that frame
  float *best_cam;                   // [max_objects,3]
  uint32_t *leader;                  // scratch: lowest j of the call that targets the object
  uint32_t *grp_cnt;                 // scratch: number of detections of the call that target the object
  // voxel-block hash
  unsigned long long *blk_key;       // [table_mask+1]
  uint32_t *blk_owner;               // [table_mask+1][64]
  uint32_t table_mask;               // capacity-1 (capacity is a power of two <= 2^31)
  // per-call scratch
  unsigned long long *pair_set;      // epoch-tagged map (epoch, j, block slot) -> pair_bits: voxels of the block
  unsigned long long *pair_bits;     //   already counted for detection j in this call (zero between calls)
  uint32_t pair_mask;
  unsigned long long *pl_bits;       // event list: the voxels `bits` of block `slot` are new for detection j
  uint32_t *pl_slot, *pl_j, *pl_ps;  //   pl_j = j | (1u<<31 when some voxel was unowned at entry), pl_ps = pair-set slot
  uint32_t pair_cap;
  unsigned long long *ov_keys;       // epoch-tagged map (j, owner) -> count
  uint32_t *ov_cnt;
  uint32_t ov_mask;
  uint32_t *cand_slot;               // list of overlap-map slots created this call
  unsigned long long *cand_key;      //   and their (epoch, j, owner) keys, so that scoring needs no dependent lookup
  uint32_t cand_cap;
  uint32_t *cand_j;                  // compact copy for the debug read
  int32_t *cand_o;
  uint32_t *cand_c;
  unsigned long long *surv_key;      // survivor queue of the lift kernel: (block key, voxel bits, j) after the
  unsigned long long *surv_bits;     //   tile-level aggregation
  uint32_t *surv_j;
  uint32_t surv_cap;
  uint32_t *surv_cnt;                // records reserved in the survivor queue (counters + 2, or the call-parity copy)
  uint32_t *counters;                // [0]=event_count [1]=cand_count [2]=survivor_count [3]=block ticket
                                     // [4]=dense pairs [5]=edges [6]=detection-detection edges [7]=entity merges
                                     // [8]=|S| of the call (W1)
  // per detection [max_det]
  uint32_t max_det;
  uint32_t *det_nv, *det_npx;
  int *det_box;                      // [max_det,6] ordered ints
  float *det_inv_norm;
  unsigned long long *best_cand, *best_dense;
  int32_t *assoc;
  uint8_t *is_new;
  float *best_score;
  // paper-faithful geometry carried beside the voxel rule (rules G1-G4); null when disabled
  double *det_gm;                    // [max_det,9] per detection: sum p (3), sum p p^T (6: xx xy xz yy yz zz)
  double *obj_gw, *obj_gm;           // [max_objects], [max_objects,9]: entity sufficient statistics w, M1, M2
  float *hell;                       // [max_det] Hellinger distance to the matched entity (entry snapshot), -1 if none
  float eps2;                        // voxel_size^2, added to both covariance diagonals (reading G3)
  unsigned long long *covis;         // [max_objects, covis_words] covisibility bitset (rule C1); null when disabled
  uint32_t covis_words;
  // U1-U4 correspondence by union-find with entity merges, H1-H3 Hellinger
  // distance as the geometric term; everything below is null / 0 when both are disabled
  int corr, geom;                    // FARM_OPT_CORRESPONDENCE, FARM_OPT_GEOMETRY
  float prefilter_cos, hell_budget;  // H1, H2
  float dense_thr;                   // cosine above which the similarity epilogue emits the pair (+inf: never)
  uint32_t *dense_d, *dense_o;       // emitted pairs (detection, object, clamped cosine); counters[4] = count
  float *dense_c;
  uint32_t dense_cap;
  uint32_t *alias;                   // [max_objects] the live entity every id stands for (itself while alive); U4
  uint32_t *uf_parent;               // [max_objects + max_det] union-find forest, identity between calls; node of
                                     //   detection j = max_objects + j, so that entities order before detections
  uint32_t *det_flags;               // [max_det] bit 0: the detection retained an entity (U1)
  uint32_t *det_newid;               // [max_det] id of the entity created by the component rooted at the detection
  uint32_t *edge_a, *edge_b;         // match-graph edges (node, node); counters[5] = count
  uint32_t *dd_d, *dd_e;             // detection-detection edges, used only if dd_d retained nothing (U2); counters[6]
  uint32_t edge_cap;
  uint32_t *loser, *winner;          // entity merges of the call (U4); counters[7] = count
  // V1-V2: up to views_k retained views per object; null when disabled
  farm_view *views;                  // [max_objects, views_k]
  uint32_t *view_cnt;                // [max_objects]
  int views_k;
  float view_cos, view_closer;
  // W1-W4: weighted covisibility edges; null / 0 when disabled
  int edges_k;
  float edge_decay, edge_cutoff;
  uint32_t *eg_list;                 // [max_det] S: the call's entities that carry a Gaussian (order arbitrary); counters[8]
  float4 *eg_f4;                     // [max_det] (mu, tr S) in fp32 (trace rounded up): the kNN scan's lower-bound test
  double *eg_gauss;                  // [max_det,12] per member: mu (3), tr S, S = Sigma + eps2 I (6), ln |S|, pad
  unsigned long long *ed_key;        // edge dictionary (open addressing): a << 32 | b with a < b, all ones when free
  double *ed_w;                      //   weight as of call ed_t
  uint32_t *ed_t;                    //   index (1-based) of the call that last updated the edge
  uint32_t ed_mask;
  uint32_t *ed_cnt;                  //   entries in the dictionary (persistent, unlike the per-call `counters`)
  uint32_t *sim_done;                // [2] cumulative count of finished similarity CTAs (the association scan waits on it); slot =
                                     //   parity of CallArgs.seq (0 without the split schedule): kernels of consecutive calls may overlap
  uint32_t *prep_done;               // cumulative count of finished prep_kernel CTAs (the similarity epilogue waits on it)
  // FARM_OPT_INPUTS_READY (split similarity); all null when the option is off.  The similarity kernel of
  // call c starts when that of call c-1 ends: phase 1 covers the rows that existed at the entry of call c-1 minus the rows
  // call c-1 merged into (their columns are masked), phase 2 -- after call c-1's merge warps -- the rows of `delta`.
  uint32_t *scan_done;               // cumulative count of finished decision scans (one per call)
  uint32_t *merge_done;              // cumulative count of finished merge warps
  uint32_t *touch_seq;               // [max_objects] sequence number of the last call that merged a detection into the object
  uint32_t *n_hist;                  // [2] n_hist[(s + 1) & 1] = number of objects after the call with sequence number s
  void *delta_rows;                  // [max_det, D] storage dtype: the rows written by the last call's merge (old and new objects)
  uint32_t *delta_id;                // [max_det] their object ids
  float *delta_inv;                  // [max_det] and inverse norms
  uint32_t *delta_cnt;               // [2] rows in delta, indexed by the parity of the writing call's sequence number
  float *cam;                        // [MAX_FRAMES,16] per-frame camera block written by prep_kernel
  CallStats *stats;
  Totals *totals;
  uint32_t *err;
};

struct CallArgs {
  int F, M;
  uint32_t epoch;
  uint32_t sim_target;  // value dm.sim_done reaches when this call's similarity kernel has finished
  int wait_sim;         // 1: cand_associate is launched without a stream join and waits for sim_target itself
  // FARM_OPT_INPUTS_READY
  uint32_t seq;           // sequence number of the call (1, 2, ...), the clock of touch_seq / n_hist / delta_cnt
  int split;              // 1: the similarity kernel runs the two-phase schedule and does its own share of prep
  int sim_fills_gpu;      //   1: its grid has one CTA on every SM (decides how the merge kernel is launched)
  uint32_t prep_target;   //   value dm.prep_done reaches when the row norms of this call are final (cand_associate waits)
  uint32_t scan_target;   //   value dm.scan_done reaches when the PREVIOUS call's decision scan is done
  uint32_t merge_target;  //   value dm.merge_done reaches when the PREVIOUS call's merge warps are done
  const float *depth;
  const uint16_t *mask;
  const float *K;
  const float *T;
  const void *desc;
  int base[MAX_FRAMES + 1];  // global detection index of each frame's first detection
};

// ---- order-preserving float <-> int (for atomicMin/Max on fp32 values; exact)
__device__ __forceinline__ int f2ord(float f) {
  int i = __float_as_int(f);
  return i ^ ((i >> 31) & 0x7FFFFFFF);
}
__device__ __forceinline__ float ord2f(int i) { return __int_as_float(i ^ ((i >> 31) & 0x7FFFFFFF)); }
__host__ __device__ __forceinline__ int f2ord_host(float f) {
  int i;
  memcpy(&i, &f, 4);
  return i ^ ((i >> 31) & 0x7FFFFFFF);
}

// (score, lowest id wins) packed for atomicMax
__device__ __forceinline__ unsigned long long pack_score(float s, uint32_t id) {
  uint32_t u = (uint32_t)f2ord(s) ^ 0x80000000u;  // order-preserving unsigned
  return ((unsigned long long)u << 32) | (unsigned long long)(0xFFFFFFFFu - id);
}
__device__ __forceinline__ float unpack_score(unsigned long long p) { return ord2f((int)((uint32_t)(p >> 32) ^ 0x80000000u)); }
__device__ __forceinline__ uint32_t unpack_id(unsigned long long p) { return 0xFFFFFFFFu - (uint32_t)p; }

// cheap 2-word hash (multiply-xorshift); used for the voxel table, the per-call scratch tables and the tile set
__device__ __forceinline__ uint32_t hash32(uint32_t a, uint32_t b) {
  uint32_t h = (a * 0x9E3779B1u) ^ (b * 0x85EBCA77u);
  h ^= h >> 15;
  h *= 0x2C1B3C6Du;
  h ^= h >> 12;
  h *= 0x297A2D39u;
  h ^= h >> 15;
  return h;
}
__device__ __forceinline__ uint32_t block_hash(unsigned long long bkey) { return hash32((uint32_t)bkey, (uint32_t)(bkey >> 32)); }

// find-or-insert a block key; returns the slot (0xFFFFFFFF when the table is full).  The owners of a fresh slot
// are all OWNER_INIT already (the payload of a free slot is never written).
__device__ __forceinline__ uint32_t block_find_or_insert(const DevMap &m, unsigned long long bkey) {
  uint32_t h = block_hash(bkey) & m.table_mask;
  for (int probe = 0; probe < 8192; ++probe) {
    unsigned long long k = __ldcg(&m.blk_key[h]);
    if (k == BLK_EMPTY) {
      k = atomicCAS(&m.blk_key[h], BLK_EMPTY, bkey);
      if (k == BLK_EMPTY) k = bkey;
    }
    if (k == bkey) return h;
    h = (h + 1) & m.table_mask;
  }
  atomicOr(m.err, ERR_VOXEL_TABLE_FULL);
  return 0xFFFFFFFFu;
}

template <typename T>
__device__ __forceinline__ float to_f32(T v);
template <>
__device__ __forceinline__ float to_f32<float>(float v) { return v; }
template <>
__device__ __forceinline__ float to_f32<__half>(__half v) { return __half2float(v); }
template <>
__device__ __forceinline__ float to_f32<__nv_bfloat16>(__nv_bfloat16 v) { return __bfloat162float(v); }

template <typename T>
__device__ __forceinline__ T from_f32(float v);
template <>
__device__ __forceinline__ float from_f32<float>(float v) { return v; }
template <>
__device__ __forceinline__ __half from_f32<__half>(float v) { return __float2half_rn(v); }
template <>
__device__ __forceinline__ __nv_bfloat16 from_f32<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }

// Programmatic dependent launch (PDL): a kernel launched with launch_pdl may start while its predecessor in the
// stream is still running; it must call pdl_wait() before it touches anything the predecessor wrote.  The
// predecessor calls pdl_trigger() early so that the dependent's CTAs become resident as soon as SM resources free up.
// Bounded wait until the cumulative device counter *ctr has reached `target` (another grid of the same call
// increments it).  Needs that grid to be co-resident or already finished; if it never arrives (serialised kernel
// execution, a co-tenant holding the SMs) the wait expires, sets the sticky ERR_SYNC_TIMEOUT and returns false
// instead of hanging the device.
__device__ __forceinline__ bool spin_until(const uint32_t *ctr, uint32_t target, uint32_t *err) {
  for (uint32_t it = 0; it < SPIN_LIMIT; ++it) {
    uint32_t done;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(done) : "l"(ctr) : "memory");
    if ((int)(done - target) >= 0) return true;
    __nanosleep(200);
  }
  atomicOr(err, ERR_SYNC_TIMEOUT);
  return false;
}

// -DFARM_TRACE (development builds only): %globaltimer stamps per call, one table per translation unit
#ifdef FARM_TRACE
#define FARM_TRACE_TABLE(name)                                                                               \
  static __device__ unsigned long long name[16][8];                                                          \
  extern "C" int name##_read(unsigned long long *out, int reset) {                                           \
    cudaDeviceSynchronize();                                                                                 \
    if (out && cudaMemcpyFromSymbol(out, name, sizeof(name)) != cudaSuccess) return -2;                      \
    if (reset) {                                                                                             \
      static unsigned long long init[16][8];                                                                 \
      for (int i = 0; i < 16; ++i)                                                                           \
        for (int k = 0; k < 8; ++k) init[i][k] = (k & 1) ? 0ull : ~0ull; /* even slots: minima, odd: maxima */ \
      if (cudaMemcpyToSymbol(name, init, sizeof(init)) != cudaSuccess) return -2;                            \
    }                                                                                                        \
    return 0;                                                                                                \
  }
__device__ __forceinline__ unsigned long long gtime() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
#define TRACE_MIN(tab, seq, k) atomicMin(&tab[(seq) & 15][k], gtime())
#define TRACE_MAX(tab, seq, k) atomicMax(&tab[(seq) & 15][k], gtime())
#else
#define FARM_TRACE_TABLE(name)
#define TRACE_MIN(tab, seq, k) ((void)0)
#define TRACE_MAX(tab, seq, k) ((void)0)
#endif

__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid, cfg.blockDim = block, cfg.dynamicSmemBytes = smem, cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr, cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// host-side launchers (one per translation unit); each returns the number of kernels it launched
// One-time kernel attributes.  Every kernel of the path asks for the maximum shared-memory carve-out: an SM cannot
// change its L1/shared split while CTAs are resident, so a kernel with another preference would keep the
// 197 KB similarity CTA off every SM it occupies (measured: the similarity grid then starts only when the other
// kernel has drained).
void configure_lift_kernels();
void configure_assoc_kernels();
void configure_edge_kernels();
int launch_prep(const DevMap &m, const CallArgs &a, cudaStream_t s);  // returns the number of CTAs that report to prep_done
int launch_lift(const DevMap &m, const CallArgs &a, cudaStream_t s);
int launch_probe(const DevMap &m, const CallArgs &a, cudaStream_t s);
int launch_debug_backproject(const DevMap &m, const float *depth, const uint16_t *mask, const float *K,
                             const float *T, int n_det, float *xyz, unsigned long long *keys, cudaStream_t s);
int launch_similarity_fma(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s);
int launch_cand_associate(const DevMap &m, const CallArgs &a, cudaStream_t s);
int launch_commit_merge(const DevMap &m, const CallArgs &a, unsigned long long frame_seq0, cudaStream_t s);
int launch_covisibility(const DevMap &m, const CallArgs &a, cudaStream_t s);
int launch_covis_absorb(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s);
int launch_edges(const DevMap &m, const CallArgs &a, uint32_t call, cudaStream_t s);
int launch_edge_export(const DevMap &m, uint32_t call, uint32_t *out_a, uint32_t *out_b, double *out_w, uint32_t cap, uint32_t *count,
                       cudaStream_t s);
int merge_warps_of(const CallArgs &a);  // warps of the merge kernel that report to dm.merge_done
int launch_dd_overlap(const DevMap &m, const CallArgs &a, cudaStream_t s);
int launch_alias_compress(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s);

// one pair above the similarity threshold, from the similarity epilogues (H1 prefilter / U1 dense edges)
__device__ __forceinline__ void dense_emit(const DevMap &m, uint32_t d, uint32_t o, float cs) {
  const uint32_t pos = atomicAdd(&m.counters[4], 1u);
  if (pos < m.dense_cap) {
    m.dense_d[pos] = d, m.dense_o[pos] = o, m.dense_c[pos] = cs;
  } else {
    atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
  }
}

}  // namespace farm
