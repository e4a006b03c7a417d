// farm_api.cu -- the C ABI of include/farm.h: handle, options, allocation, the per-call launch sequence,
// export / import and the debug reads.  Host logic only; every step of the path runs in the kernels of
// farm_lift.cu, farm_sim_fma.cu, farm_sim_tc.cu and farm_assoc.cu.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

#include "farm_internal.cuh"

namespace farm {
bool tc_can_split(void *tc_state);
int launch_similarity_tc(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s, void *tc_state, uint32_t prep_target,
                         int *n_ctas, uint32_t *prep_after);
int run_query(const DevMap &m, cudaStream_t st, uint32_t N, const void *const emb[3], const int dim[3], int emb_dtype, const int32_t *cls,
              const float *q_target, int target_class, int P, const int32_t *pred_type, const float *q_landmarks, int topk,
              int32_t *top_ids, float *top_scores, int32_t *landmarks, float *s_sem, float *gbar, float *s, long long *launches,
              std::string *err);
int noalloc_cosine_rowmax(const void *A, int M, const void *B, int N, int D, int dtype, float *max_cos, int32_t *argmax,
                          cudaStream_t s, std::string *err);
bool tc_prepare(void *tc_state, const DevMap &m, const CallArgs &a);
void *tc_state_create(const DevMap &m);
void tc_state_destroy(void *);
void tc_state_set_pair(void *, int pair);
bool tc_supported(const DevMap &m);
}  // namespace farm

using namespace farm;

static thread_local std::string g_err;
static int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}
#define CU(expr)                                                                                      \
  do {                                                                                                \
    cudaError_t e_ = (expr);                                                                          \
    if (e_ != cudaSuccess) return fail(FARM_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); \
  } while (0)

struct farm_map {
  float voxel_size, w_geo, w_sem, tau, z_min = 0.f, z_max = std::numeric_limits<float>::infinity();
  int D, dtype = FARM_DTYPE_F32, H = 0, W = 0;
  long long max_objects = 65536, max_voxels = 1ll << 22, max_det = 4096, max_pairs = 0, max_frames = 16, max_blocks = 0;
  int sim_path = 0, gaussian = 0, covis = 0, views_k = 0, corr = 0, geom = 0, edges_k = 0;
  float edge_decay = 0.9f, edge_cutoff = 2.0f;
  uint32_t edge_calls = 0;  // integrate calls so far: the clock of W4's decay
  // FARM_OPT_INPUTS_READY: split similarity schedule
  int inputs_ready = 0;
  uint32_t seq = 0;             // sequence number of the last integrate call (CallArgs.seq)
  long long sim_timed = 0, sim_all = 0;  // timing 1: similarity launches bracketed by events / all of them (since the last reset)
  uint32_t scan_count = 0;      // decision scans launched so far (device counter dm.scan_done)
  uint32_t merge_count = 0;     // merge warps launched so far (device counter dm.merge_done)
  // what prep resets and the lift kernel writes, double buffered by call parity: with the split schedule prep and lift of call c
  // run on their own stream while the main chain is still at call c-1 (whose scan, merge and result reads use the other set)
  struct LiftSet {
    unsigned long long *surv_key, *surv_bits;
    uint32_t *surv_j, *surv_cnt, *det_npx;
    int *det_box;
    double *det_gm;
    float *cam;
    CallStats *stats;
    uint32_t *counters, *det_nv;
    unsigned long long *best_cand;
    int32_t *assoc;
    uint8_t *is_new;
    float *best_score, *hell;
  } lset[2] = {};
  cudaStream_t early = nullptr;                 // prep (lift part) + lift of a split call
  cudaEvent_t ev_lift = nullptr, ev_end[2] = {nullptr, nullptr};
  bool ev_end_set[2] = {false, false};
  float *inv_norm2[2] = {nullptr, nullptr};               // det_inv_norm / best_dense, double buffered by call parity: the
  unsigned long long *best_dense2[2] = {nullptr, nullptr};  //   similarity kernel of call c writes them while call c-1 still reads its own
  float view_cos = 0.8660254f, view_closer = 0.8f, prefilter_cos = 0.5f, hell_budget = 1.0f;
  cudaStream_t stream = 0;
  bool finalised = false;
  DevMap dm{};
  std::vector<void *> allocs;
  long long launches = 0;
  unsigned long long frame_seq = 0;
  uint32_t epoch = 0;
  uint32_t sim_target[2] = {0, 0};  // cumulative number of similarity CTAs launched, per slot of dm.sim_done (parity of CallArgs.seq)
  uint32_t prep_target = 0;  // cumulative number of prep_kernel CTAs launched (device counter dm.prep_done)
  uint32_t n_upper = 0;  // host upper bound of N (no device sync on the integrate path)
  int last_M = 0;
  bool has_last = false;
  void *tc = nullptr;
  cudaStream_t side = nullptr;             // similarity runs here, concurrently with lift + probe
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  int overlap = 1;
  // optional per-stage timing (FARM_OPT_TIMING)
  int timing = 0;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev_pending[FARM_N_STAGES];
  std::vector<cudaEvent_t> ev_free;
  double stage_ms[FARM_N_STAGES] = {};
  long long stage_launches[FARM_N_STAGES] = {};
  // farm_map_integrate_batch_host: two device staging sets filled on a copy stream, so that the H2D copy of call
  // t+1 overlaps the kernels of call t
  struct Staging {
    float *depth = nullptr, *K = nullptr, *T = nullptr;
    uint16_t *mask = nullptr;
    void *desc = nullptr;
    cudaEvent_t copied = nullptr, free = nullptr;
    bool used = false;
  } stg[2];
  cudaStream_t cstream = nullptr;
  unsigned long long host_calls = 0;
  size_t elem() const { return dtype == FARM_DTYPE_F32 ? 4 : 2; }
};

namespace {

__global__ void init_forest_kernel(DevMap m) {  // U: alias and union-find forest start as the identity
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < m.max_objects) m.alias[i] = i;
  if (i < m.max_objects + m.max_det) m.uf_parent[i] = i;
}

__global__ void init_objects_kernel(DevMap m) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= m.max_objects) return;
#pragma unroll
  for (int k = 0; k < 3; ++k) {
    m.aabb[i * 6 + k] = 0x7FFFFFFF;  // +NaN-side maximum of the ordered image: any finite value is smaller
    m.aabb[i * 6 + 3 + k] = (int)0x80000000;
  }
  m.leader[i] = 0xFFFFFFFFu;
}

__global__ void export_objects_kernel(DevMap m, farm_object *out, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  farm_object o;
  o.id = (int32_t)i;
  o.n_voxels = m.n_voxels[i];
  o.n_obs = m.n_obs[i];
  for (int k = 0; k < 3; ++k) {
    o.aabb_min[k] = ord2f(m.aabb[i * 6 + k]);
    o.aabb_max[k] = ord2f(m.aabb[i * 6 + 3 + k]);
    o.best_cam_pos[k] = m.best_cam[i * 3 + k];
  }
  const uint32_t bp = m.best_px[i];
  if (bp) {
    o.best_pixels = bp;
    o.best_frame = (int32_t)m.best_seq[i];  // integrate refuses frame sequence numbers beyond INT32_MAX (FARM_ERR_STATE)
    o.best_det = (int32_t)m.best_det[i];
  } else {
    o.best_pixels = 0, o.best_frame = -1, o.best_det = -1;
  }
  o.n_points = m.n_points[i];
  out[i] = o;
}

__global__ void import_objects_kernel(DevMap m, const farm_object *in, uint32_t n) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const farm_object o = in[i];
  m.n_voxels[i] = o.n_voxels;
  m.n_obs[i] = o.n_obs;
  m.n_points[i] = o.n_points;
  for (int k = 0; k < 3; ++k) {
    m.aabb[i * 6 + k] = f2ord(o.aabb_min[k]);
    m.aabb[i * 6 + 3 + k] = f2ord(o.aabb_max[k]);
    m.best_cam[i * 3 + k] = o.best_cam_pos[k];
  }
  const bool has = o.best_frame >= 0 && o.best_pixels > 0;
  m.best_px[i] = has ? o.best_pixels : 0u;
  m.best_seq[i] = has ? (unsigned long long)o.best_frame : 0ull;
  m.best_det[i] = has ? (uint32_t)o.best_det : 0u;
}

// import check: objects[i].n_voxels must equal the number of imported voxels owned by i (R10 divides by it)
__global__ void count_owner_kernel(const uint32_t *owners, long long n, uint32_t n_objects, uint32_t *cnt) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
    if (owners[i] < n_objects) atomicAdd(&cnt[owners[i]], 1u);
}
__global__ void check_owner_count_kernel(DevMap m, const uint32_t *cnt, uint32_t n_objects) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_objects && cnt[i] != m.n_voxels[i]) atomicOr(m.err, ERR_IMPORT_COUNT);
}

// R26: renormalise imported fp32 rows (fp32 arithmetic), write master, shadow and inverse shadow norm
template <typename T>
__global__ void __launch_bounds__(256) renorm_rows_kernel(DevMap m, uint32_t n) {
  __shared__ float red[8];
  __shared__ float bc;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (uint32_t r = blockIdx.x; r < n; r += gridDim.x) {
    float *row = m.desc_master + (size_t)r * m.D;
    T *sh = (T *)m.desc_shadow + (size_t)r * m.D;
    float ss = 0.f;
    for (int i = tid; i < m.D; i += 256) ss = fmaf(row[i], row[i], ss);
    for (int s = 16; s; s >>= 1) ss += __shfl_xor_sync(0xFFFFFFFFu, ss, s);
    if (lane == 0) red[warp] = ss;
    __syncthreads();
    if (tid == 0) {
      float t = 0.f;
      for (int w = 0; w < 8; ++w) t += red[w];
      bc = t;
    }
    __syncthreads();
    const float inv = bc > 0.f ? 1.0f / sqrtf(bc) : 0.f;
    float s2 = 0.f;
    for (int i = tid; i < m.D; i += 256) {
      const float v = row[i] * inv;
      row[i] = v;
      const T q = from_f32<T>(v);
      sh[i] = q;
      const float qv = to_f32<T>(q);
      s2 = fmaf(qv, qv, s2);
    }
    for (int s = 16; s; s >>= 1) s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, s);
    __syncthreads();
    if (lane == 0) red[warp] = s2;
    __syncthreads();
    if (tid == 0) {
      float t = 0.f;
      for (int w = 0; w < 8; ++w) t += red[w];
      m.inv_norm[r] = t > 0.f ? 1.0f / sqrtf(t) : 0.f;
    }
    __syncthreads();
  }
}

__global__ void import_voxels_kernel(DevMap m, const unsigned long long *keys, const uint32_t *owners, long long n,
                                     uint32_t n_objects) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const unsigned long long key = keys[i];
    const uint32_t owner = owners[i];
    if (owner >= n_objects || (key >> 63)) {
      atomicOr(m.err, ERR_IMPORT_DUPLICATE);
      continue;
    }
    const uint32_t ix = (uint32_t)(key >> 42) & 0x1FFFFFu, iy = (uint32_t)(key >> 21) & 0x1FFFFFu, iz = (uint32_t)key & 0x1FFFFFu;
    const uint32_t slot = block_find_or_insert(m, block_key(ix, iy, iz));
    if (slot == 0xFFFFFFFFu) continue;  // table full: sticky error already set
    const uint32_t old = atomicCAS(&m.blk_owner[(size_t)slot * BLK_VOXELS + block_bit(ix, iy, iz)], OWNER_INIT, owner);
    if (old != OWNER_INIT) atomicOr(m.err, ERR_IMPORT_DUPLICATE);
  }
}

// one thread per (block slot, 32-byte owner sector)
__global__ void count_voxels_kernel(DevMap m, unsigned long long *count) {
  unsigned long long c = 0;
  const unsigned long long n = ((unsigned long long)m.table_mask + 1) * 8;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    if (m.blk_key[i >> 3] == BLK_EMPTY) continue;
    const uint4 *p = reinterpret_cast<const uint4 *>(m.blk_owner + i * 8);
    const uint4 w0 = p[0], w1 = p[1];
    c += (w0.x != OWNER_INIT) + (w0.y != OWNER_INIT) + (w0.z != OWNER_INIT) + (w0.w != OWNER_INIT) + (w1.x != OWNER_INIT) +
         (w1.y != OWNER_INIT) + (w1.z != OWNER_INIT) + (w1.w != OWNER_INIT);
  }
  for (int s = 16; s; s >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, s);
  if ((threadIdx.x & 31) == 0 && c) atomicAdd(count, c);
}

__global__ void export_voxels_kernel(DevMap m, unsigned long long *keys, uint32_t *owners, unsigned long long *cursor,
                                     unsigned long long cap) {
  const unsigned long long n = ((unsigned long long)m.table_mask + 1) * 8;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    const unsigned long long bkey = m.blk_key[i >> 3];
    if (bkey == BLK_EMPTY) continue;
    const uint4 *p = reinterpret_cast<const uint4 *>(m.blk_owner + i * 8);
    const uint4 w0 = p[0], w1 = p[1];
    const uint32_t own[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
    uint32_t cnt = 0;
#pragma unroll
    for (int b = 0; b < 8; ++b) cnt += own[b] != OWNER_INIT;
    if (!cnt) continue;
    unsigned long long pos = atomicAdd(cursor, (unsigned long long)cnt);
#pragma unroll
    for (int b = 0; b < 8; ++b)
      if (own[b] != OWNER_INIT) {
        if (pos < cap) {
          keys[pos] = voxel_key_of(bkey, (uint32_t)(i & 7) * 8 + b);
          owners[pos] = m.alias ? m.alias[own[b]] : own[b];  // U4: voxels of an absorbed entity belong to its winner
        }
        ++pos;
      }
  }
}

// debug read: block key of every event of the last call
__global__ void gather_events_kernel(DevMap m, uint32_t n, unsigned long long *bkeys) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  bkeys[i] = m.blk_key[m.pl_slot[i]];
}

// G1/G2 export: mean and population covariance from sufficient statistics (zeros where the weight is 0)
__global__ void export_gaussians_kernel(const double *w, const uint32_t *w_u32, const double *g, uint32_t n, double *weight,
                                        float *mu, float *cov) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double wi = w ? w[i] : (double)w_u32[i];
  float o[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
  if (wi > 0.0) {
    const double *q = g + (size_t)i * 9;
    const double m0 = q[0] / wi, m1 = q[1] / wi, m2 = q[2] / wi;
    o[0] = (float)m0, o[1] = (float)m1, o[2] = (float)m2;
    o[3] = (float)(q[3] / wi - m0 * m0), o[4] = (float)(q[4] / wi - m0 * m1), o[5] = (float)(q[5] / wi - m0 * m2);
    o[6] = (float)(q[6] / wi - m1 * m1), o[7] = (float)(q[7] / wi - m1 * m2), o[8] = (float)(q[8] / wi - m2 * m2);
  }
  if (weight) weight[i] = wi;
  for (int k = 0; k < 3; ++k) mu[(size_t)i * 3 + k] = o[k];
  for (int k = 0; k < 6; ++k) cov[(size_t)i * 6 + k] = o[3 + k];
}

long long next_pow2(long long x) {
  long long p = 1;
  while (p < x) p <<= 1;
  return p;
}

template <typename T>
int dev_alloc(farm_map *m, T **p, size_t count, int fill_byte) {
  void *q = nullptr;
  const size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
  CU(cudaMalloc(&q, bytes));
  m->allocs.push_back(q);
  CU(cudaMemsetAsync(q, fill_byte, bytes, m->stream));
  *p = (T *)q;
  return FARM_OK;
}

int finalise_impl(farm_map *m);
int finalise(farm_map *m) {
  if (m->finalised) return FARM_OK;
  const int rc = finalise_impl(m);
  if (rc != FARM_OK) {  // leave nothing half-built behind: the next call starts from scratch
    const std::string msg = g_err;
    cudaDeviceSynchronize();
    for (void *p : m->allocs) cudaFree(p);
    m->allocs.clear();
    if (m->tc) tc_state_destroy(m->tc), m->tc = nullptr;
    if (m->side) cudaStreamDestroy(m->side), m->side = nullptr;
    if (m->ev_fork) cudaEventDestroy(m->ev_fork), m->ev_fork = nullptr;
    if (m->ev_join) cudaEventDestroy(m->ev_join), m->ev_join = nullptr;
    if (m->early) cudaStreamDestroy(m->early), m->early = nullptr;
    if (m->ev_lift) cudaEventDestroy(m->ev_lift), m->ev_lift = nullptr;
    for (int i = 0; i < 2; ++i)
      if (m->ev_end[i]) cudaEventDestroy(m->ev_end[i]), m->ev_end[i] = nullptr;
    m->dm = DevMap{};
    cudaGetLastError();
    g_err = msg;
  }
  return rc;
}
int finalise_impl(farm_map *m) {
  if (m->H <= 0 || m->W <= 0) return fail(FARM_ERR_STATE, "FARM_OPT_IMG_W / FARM_OPT_IMG_H must be set before the first call");
  if ((long long)m->H * m->W > (1ll << 31) - 1) return fail(FARM_ERR_INVALID_ARG, "IMG_W * IMG_H must be below 2^31 (pixel counts are 32-bit)");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(FARM_ERR_CUDA, "no CUDA device: the FARM mapping path has no CPU fallback");
  {
    int dev = 0, sms = 0;
    CU(cudaGetDevice(&dev));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    m->dm.num_sms = sms > 0 ? sms : 1;
  }
  // The default launch order (FARM_OPT_OVERLAP = 1 with the tensor-core similarity) needs grids of one call to be
  // co-resident: the similarity epilogue waits for prep, the decision scan for the similarity grid.  When the
  // process serialises kernel execution, fall back to the single-stream order, which has no device-side waits.
  if (const char *lb = getenv("CUDA_LAUNCH_BLOCKING"))
    if (lb[0] && lb[0] != '0') m->overlap = 0;
  if (m->max_blocks <= 0) m->max_blocks = std::max<long long>(m->max_voxels / 4, 1024);
  if (m->max_blocks > (1ll << 30)) return fail(FARM_ERR_INVALID_ARG, "voxel-block table too large (FARM_OPT_MAX_BLOCKS <= 2^30)");
  if (m->max_pairs <= 0) m->max_pairs = std::min<long long>((long long)m->H * m->W * std::min<long long>(m->max_frames, 4), 1ll << 23);
  DevMap &d = m->dm;
  d.inv_vs = 1.0f / m->voxel_size;  // R6: fp32 reciprocal, computed once
  d.w_geo = m->w_geo, d.w_sem = m->w_sem, d.tau = m->tau, d.z_min = m->z_min, d.z_max = m->z_max;
  d.D = m->D, d.dtype = m->dtype, d.H = m->H, d.W = m->W;
  d.max_objects = (uint32_t)m->max_objects;
  const size_t NO = (size_t)m->max_objects, D = (size_t)m->D;
  int rc;
#define A(ptr, count, fill)                                        \
  if ((rc = dev_alloc(m, &(ptr), (count), (fill))) != FARM_OK) return rc
  A(d.n_objects, 1, 0);
  A(d.desc_master, NO * D, 0);
  {
    uint8_t *p;
    A(p, NO * D * m->elem(), 0);
    d.desc_shadow = p;
  }
  A(d.inv_norm, NO, 0);
  A(d.n_voxels, NO, 0);
  A(d.n_obs, NO, 0);
  A(d.n_points, NO, 0);
  A(d.aabb, NO * 6, 0);
  A(d.best_px, NO, 0);
  A(d.best_seq, NO, 0);
  A(d.best_det, NO, 0);
  A(d.best_cam, NO * 3, 0);
  A(d.leader, NO, 0xFF);
  A(d.grp_cnt, NO, 0);
  const long long tcap = next_pow2(std::max<long long>(2 * m->max_blocks, 1024));
  A(d.blk_key, (size_t)tcap, 0xFF);                 // BLK_EMPTY
  A(d.blk_owner, (size_t)tcap * BLK_VOXELS, 0xFF);  // OWNER_INIT
  d.table_mask = (uint32_t)(tcap - 1);
  const long long pcap = next_pow2(2 * m->max_pairs);
  A(d.pair_set, (size_t)pcap, 0);
  A(d.pair_bits, (size_t)pcap, 0);
  d.pair_mask = (uint32_t)(pcap - 1);
  A(d.pl_bits, (size_t)m->max_pairs, 0);
  A(d.pl_slot, (size_t)m->max_pairs, 0);
  A(d.pl_j, (size_t)m->max_pairs, 0);
  A(d.pl_ps, (size_t)m->max_pairs, 0);
  d.pair_cap = (uint32_t)m->max_pairs;
  const long long ccap = std::min<long long>(std::max<long long>(m->max_pairs / 4, 16384), 1ll << 22);
  const long long ocap = next_pow2(2 * ccap);
  A(d.ov_keys, (size_t)ocap, 0);
  A(d.ov_cnt, (size_t)ocap, 0);
  d.ov_mask = (uint32_t)(ocap - 1);
  A(d.cand_slot, (size_t)ccap, 0);
  A(d.cand_key, (size_t)ccap, 0);
  A(d.cand_j, (size_t)ccap, 0);
  A(d.cand_o, (size_t)ccap, 0);
  A(d.cand_c, (size_t)ccap, 0);
  d.cand_cap = (uint32_t)ccap;
  const long long scap = std::min<long long>(2 * m->max_pairs, 1ll << 30) + (long long)d.num_sms * 8 * 512;  // + chunk padding of the lift CTAs
  A(d.surv_key, (size_t)scap, 0);
  A(d.surv_bits, (size_t)scap, 0);
  A(d.surv_j, (size_t)scap, 0);
  d.surv_cap = (uint32_t)scap;
  A(d.counters, 16, 0);
  const size_t MD = (size_t)m->max_det;
  d.max_det = (uint32_t)MD;
  A(d.det_nv, MD, 0);
  A(d.det_npx, MD, 0);
  A(d.det_box, MD * 6, 0);
  A(d.det_inv_norm, MD, 0);
  A(d.best_cand, MD, 0);
  A(d.best_dense, MD, 0);
  A(d.assoc, MD, 0);
  A(d.is_new, MD, 0);
  A(d.best_score, MD, 0);
  A(d.prep_done, 1, 0);
  if (m->inputs_ready && m->dtype != FARM_DTYPE_F32 && (m->sim_path == 0 || m->sim_path == 2) && m->overlap == 1 && !m->corr && m->geom == 0 &&
      m->D % 8 == 0) {
    A(d.scan_done, 1, 0);
    A(d.merge_done, 1, 0);
    A(d.touch_seq, NO, 0);
    A(d.n_hist, 2, 0);
    {
      uint8_t *p;
      A(p, (size_t)m->max_det * D * m->elem(), 0);
      d.delta_rows = p;
    }
    A(d.delta_id, (size_t)m->max_det, 0);
    A(d.delta_inv, (size_t)m->max_det, 0);
    A(d.delta_cnt, 2, 0);
    A(m->inv_norm2[1], MD, 0);
    A(m->best_dense2[1], MD, 0);
    m->inv_norm2[0] = d.det_inv_norm, m->best_dense2[0] = d.best_dense;
    farm_map::LiftSet &s1 = m->lset[1];
    A(s1.surv_key, (size_t)scap, 0);
    A(s1.surv_bits, (size_t)scap, 0);
    A(s1.surv_j, (size_t)scap, 0);
    A(s1.surv_cnt, 1, 0);
    A(s1.det_npx, MD, 0);
    A(s1.det_box, MD * 6, 0);
    if (m->gaussian) A(s1.det_gm, MD * 9, 0);
    A(s1.cam, (size_t)MAX_FRAMES * 16, 0);
    A(s1.stats, 1, 0);
    A(s1.counters, 16, 0);
    A(s1.det_nv, MD, 0);
    A(s1.best_cand, MD, 0);
    A(s1.assoc, MD, 0);
    A(s1.is_new, MD, 0);
    A(s1.best_score, MD, 0);
    if (m->gaussian) A(s1.hell, MD, 0);
  }
  A(d.sim_done, 2, 0);
  d.eps2 = m->voxel_size * m->voxel_size;
  if (m->covis) {
    d.covis_words = (uint32_t)((NO + 63) / 64);
    if ((size_t)d.covis_words * 8 > 96 * 1024) return fail(FARM_ERR_INVALID_ARG, "FARM_OPT_COVISIBILITY supports MAX_OBJECTS <= 786432");
    A(d.covis, NO * d.covis_words, 0);
  }
  d.dense_thr = 3.0e38f;  // the similarity epilogues emit nothing unless an option below asks for it
  d.corr = m->corr, d.geom = m->geom, d.prefilter_cos = m->prefilter_cos, d.hell_budget = m->hell_budget;
  if (m->geom == 1 && !m->gaussian) return fail(FARM_ERR_INVALID_ARG, "FARM_OPT_GEOMETRY = 1 needs FARM_OPT_GAUSSIAN = 1");
  if (m->corr && !(m->tau >= 0.f)) return fail(FARM_ERR_INVALID_ARG, "FARM_OPT_CORRESPONDENCE needs tau >= 0");
  if (m->corr || m->geom == 1) {
    // pairs the similarity epilogue must emit: H1 the prefilter; U1 with the voxel rule every pair whose semantic term alone
    // passes tau (possible only when w_sem > tau)
    if (m->geom == 1) d.dense_thr = m->prefilter_cos;
    else if (m->w_sem > m->tau && m->w_sem > 0.f) d.dense_thr = m->tau / m->w_sem * 0.9999f - 1e-6f;
    const size_t dcap = std::max<size_t>((size_t)MD * 64, 1 << 16);
    A(d.dense_d, dcap, 0);
    A(d.dense_o, dcap, 0);
    A(d.dense_c, dcap, 0);
    d.dense_cap = (uint32_t)dcap;
    const size_t ecap = dcap + (size_t)ccap;
    A(d.edge_a, ecap, 0);
    A(d.edge_b, ecap, 0);
    A(d.dd_d, ecap, 0);
    A(d.dd_e, ecap, 0);
    A(d.loser, ecap, 0);
    A(d.winner, ecap, 0);
    d.edge_cap = (uint32_t)ecap;
    A(d.det_flags, MD, 0);
    A(d.det_newid, MD, 0);
  }
  if (m->corr) {
    A(d.alias, NO, 0);
    A(d.uf_parent, NO + MD, 0);
  }
  if (m->views_k > 0) {
    d.views_k = m->views_k, d.view_cos = m->view_cos, d.view_closer = m->view_closer;
    A(d.views, NO * (size_t)m->views_k, 0);
    A(d.view_cnt, NO, 0);
  }
  if (m->edges_k > 0) {
    if (!m->gaussian) return fail(FARM_ERR_INVALID_ARG, "FARM_OPT_EDGES needs FARM_OPT_GAUSSIAN = 1");
    if (m->corr) return fail(FARM_ERR_INVALID_ARG, "FARM_OPT_EDGES is not available together with FARM_OPT_CORRESPONDENCE");
    if ((NO + 63) / 64 * 8 > 96 * 1024) return fail(FARM_ERR_INVALID_ARG, "FARM_OPT_EDGES supports MAX_OBJECTS <= 786432");
    d.edges_k = m->edges_k, d.edge_decay = m->edge_decay, d.edge_cutoff = m->edge_cutoff;
    A(d.eg_list, MD, 0);
    A(d.eg_gauss, MD * 12, 0);
    A(d.eg_f4, MD, 0);
    const long long ecap = next_pow2(std::max<long long>(8ll * m->edges_k * (long long)NO, 4096));
    A(d.ed_key, (size_t)ecap, 0xFF);
    A(d.ed_w, (size_t)ecap, 0);
    A(d.ed_t, (size_t)ecap, 0);
    A(d.ed_cnt, 1, 0);
    d.ed_mask = (uint32_t)(ecap - 1);
  }
  if (m->gaussian) {
    A(d.det_gm, MD * 9, 0);
    A(d.hell, MD, 0);
    A(d.obj_gw, NO, 0);
    A(d.obj_gm, NO * 9, 0);
  }
  A(d.cam, (size_t)MAX_FRAMES * 16, 0);
  A(d.stats, 1, 0);
  A(d.totals, 1, 0);
  A(d.err, 1, 0);
#undef A
  configure_lift_kernels();
  configure_assoc_kernels();
  configure_edge_kernels();
  init_objects_kernel<<<(unsigned)((NO + 255) / 256), 256, 0, m->stream>>>(d);
  m->launches++;
  if (m->corr) {
    init_forest_kernel<<<(unsigned)((NO + MD + 255) / 256), 256, 0, m->stream>>>(d);
    m->launches++;
  }
  CU(cudaGetLastError());
  if (m->dtype != FARM_DTYPE_F32 && m->sim_path != 1 && tc_supported(d)) m->tc = tc_state_create(d);
  if (m->tc && m->sim_path == 3) tc_state_set_pair(m->tc, 1);
  d.surv_cnt = d.counters + 2;
  m->lset[0] = {d.surv_key, d.surv_bits, d.surv_j, d.surv_cnt, d.det_npx, d.det_box, d.det_gm, d.cam, d.stats,
                d.counters, d.det_nv, d.best_cand, d.assoc, d.is_new, d.best_score, d.hell};
  if (d.touch_seq) {
    CU(cudaStreamCreateWithFlags(&m->early, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&m->ev_lift, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&m->ev_end[0], cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&m->ev_end[1], cudaEventDisableTiming));
  }
  if (m->overlap) {
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    CU(cudaStreamCreateWithPriority(&m->side, cudaStreamNonBlocking, prio_hi));  // similarity CTAs are placed first
    CU(cudaEventCreateWithFlags(&m->ev_fork, cudaEventDisableTiming));
    CU(cudaEventCreateWithFlags(&m->ev_join, cudaEventDisableTiming));
  }
  if (m->sim_path >= 2 && !m->tc) return fail(FARM_ERR_INVALID_ARG, "tensor-core similarity path not available for this dtype / D");
  m->finalised = true;
  return FARM_OK;
}

cudaEvent_t get_event(farm_map *m) {
  if (!m->ev_free.empty()) {
    cudaEvent_t e = m->ev_free.back();
    m->ev_free.pop_back();
    return e;
  }
  cudaEvent_t e;
  cudaEventCreate(&e);
  return e;
}

int device_error(farm_map *m) {
  uint32_t e = 0;
  CU(cudaMemcpyAsync(&e, m->dm.err, 4, cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  if (e == 0) return FARM_OK;
  char buf[320];
  snprintf(buf, sizeof buf, "sticky device error 0x%x:%s%s%s%s%s%s%s%s", e, (e & ERR_VOXEL_TABLE_FULL) ? " voxel table full" : "",
           (e & ERR_PAIR_TABLE_FULL) ? " per-call pair scratch full" : "",
           (e & ERR_OVERLAP_TABLE_FULL) ? " per-call overlap scratch full" : "",
           (e & ERR_OBJECT_CAPACITY) ? " object capacity" : "", (e & ERR_IMPORT_DUPLICATE) ? " import: duplicate key or bad owner" : "",
           (e & ERR_IMPORT_COUNT) ? " import: an object's n_voxels differs from the voxels listed for it" : "",
           (e & ERR_EDGE_TABLE_FULL) ? " edge dictionary full" : "",
           (e & ERR_SYNC_TIMEOUT) ? " a device-side wait between the grids of one call expired (kernels serialised? use FARM_OPT_OVERLAP = 0)" : "");
  if (e & (ERR_IMPORT_DUPLICATE | ERR_IMPORT_COUNT)) return fail(FARM_ERR_INVALID_ARG, buf);
  return fail((e & ERR_SYNC_TIMEOUT) ? FARM_ERR_STATE : FARM_ERR_CAPACITY, buf);
}

}  // namespace

extern "C" {

const char *farm_last_error(void) { return g_err.c_str(); }

int farm_map_create(float voxel_size, int D, float w_geo, float w_sem, float tau, farm_map **out) {
  if (!out) return fail(FARM_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  if (!(voxel_size > 0.f) || !std::isfinite(voxel_size)) return fail(FARM_ERR_INVALID_ARG, "voxel_size must be > 0");
  if (D < 1 || D > 8192) return fail(FARM_ERR_INVALID_ARG, "D must be in 1..8192");
  if (!(w_geo >= 0.f) || !(w_sem >= 0.f) || !std::isfinite(w_geo) || !std::isfinite(w_sem) || std::isnan(tau))
    return fail(FARM_ERR_INVALID_ARG, "w_geo and w_sem must be finite and >= 0");
  farm_map *m = new farm_map();
  m->voxel_size = voxel_size, m->D = D, m->w_geo = w_geo, m->w_sem = w_sem, m->tau = tau;
  *out = m;
  return FARM_OK;
}

int farm_map_destroy(farm_map *m) {
  if (!m) return FARM_OK;
  if (m->finalised || !m->allocs.empty()) cudaStreamSynchronize(m->stream);
  if (m->side) cudaStreamSynchronize(m->side), cudaStreamDestroy(m->side);
  if (m->early) cudaStreamSynchronize(m->early), cudaStreamDestroy(m->early);
  if (m->ev_lift) cudaEventDestroy(m->ev_lift);
  for (int i = 0; i < 2; ++i)
    if (m->ev_end[i]) cudaEventDestroy(m->ev_end[i]);
  if (m->cstream) cudaStreamSynchronize(m->cstream), cudaStreamDestroy(m->cstream);
  for (auto &g : m->stg) {
    if (g.copied) cudaEventDestroy(g.copied);
    if (g.free) cudaEventDestroy(g.free);
  }
  if (m->ev_fork) cudaEventDestroy(m->ev_fork);
  if (m->ev_join) cudaEventDestroy(m->ev_join);
  if (m->tc) tc_state_destroy(m->tc);
  for (void *p : m->allocs) cudaFree(p);
  for (auto &v : m->ev_pending)
    for (auto &p : v) cudaEventDestroy(p.first), cudaEventDestroy(p.second);
  for (cudaEvent_t e : m->ev_free) cudaEventDestroy(e);
  delete m;
  return FARM_OK;
}

int farm_map_set_option_i(farm_map *m, int key, long long v) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (m->finalised && key != FARM_OPT_TIMING) return fail(FARM_ERR_STATE, "options are frozen after the first integrate / import");
  switch (key) {
    case FARM_OPT_DESC_DTYPE:
      if (v < 0 || v > 2) return fail(FARM_ERR_INVALID_ARG, "bad dtype");
      m->dtype = (int)v;
      break;
    case FARM_OPT_MAX_OBJECTS:
      if (v < 1 || v > (1ll << 31) - 2) return fail(FARM_ERR_INVALID_ARG, "bad MAX_OBJECTS");
      m->max_objects = v;
      break;
    case FARM_OPT_MAX_VOXELS:
      if (v < 1 || v > (1ll << 30)) return fail(FARM_ERR_INVALID_ARG, "bad MAX_VOXELS");
      m->max_voxels = v;
      break;
    case FARM_OPT_IMG_W:
      if (v < 1 || v > 65536) return fail(FARM_ERR_INVALID_ARG, "bad IMG_W");
      m->W = (int)v;
      break;
    case FARM_OPT_IMG_H:
      if (v < 1 || v > 65536) return fail(FARM_ERR_INVALID_ARG, "bad IMG_H");
      m->H = (int)v;
      break;
    case FARM_OPT_MAX_DET_PER_CALL:
      if (v < 1 || v >= (1ll << DET_BITS)) return fail(FARM_ERR_INVALID_ARG, "bad MAX_DET_PER_CALL (1..65535)");
      m->max_det = v;
      break;
    case FARM_OPT_STREAM:
      m->stream = (cudaStream_t)(uintptr_t)v;
      break;
    case FARM_OPT_MAX_PAIRS_PER_CALL:
      if (v < 1024 || v > (1ll << 30)) return fail(FARM_ERR_INVALID_ARG, "bad MAX_PAIRS_PER_CALL");
      m->max_pairs = v;
      break;
    case FARM_OPT_MAX_BLOCKS:
      if (v < 1 || v > (1ll << 30)) return fail(FARM_ERR_INVALID_ARG, "bad MAX_BLOCKS");
      m->max_blocks = v;
      break;
    case FARM_OPT_MAX_FRAMES_PER_CALL:
      if (v < 1 || v > MAX_FRAMES) return fail(FARM_ERR_INVALID_ARG, "bad MAX_FRAMES_PER_CALL");
      m->max_frames = v;
      break;
    case FARM_OPT_SIM_PATH:
      if (v < 0 || v > 3) return fail(FARM_ERR_INVALID_ARG, "bad SIM_PATH");
      m->sim_path = (int)v;
      break;
    case FARM_OPT_OVERLAP:
      if (v < 0 || v > 3) return fail(FARM_ERR_INVALID_ARG, "bad OVERLAP");
      m->overlap = (int)v;
      break;
    case FARM_OPT_GAUSSIAN:
      if (v < 0 || v > 1) return fail(FARM_ERR_INVALID_ARG, "bad GAUSSIAN");
      m->gaussian = (int)v;
      break;
    case FARM_OPT_COVISIBILITY:
      if (v < 0 || v > 1) return fail(FARM_ERR_INVALID_ARG, "bad COVISIBILITY");
      m->covis = (int)v;
      break;
    case FARM_OPT_CORRESPONDENCE:
      if (v < 0 || v > 1) return fail(FARM_ERR_INVALID_ARG, "bad CORRESPONDENCE");
      m->corr = (int)v;
      break;
    case FARM_OPT_GEOMETRY:
      if (v < 0 || v > 1) return fail(FARM_ERR_INVALID_ARG, "bad GEOMETRY");
      m->geom = (int)v;
      break;
    case FARM_OPT_VIEWS:
      if (v < 0 || v > 8) return fail(FARM_ERR_INVALID_ARG, "bad VIEWS (0..8)");
      m->views_k = (int)v;
      break;
    case FARM_OPT_INPUTS_READY:
      if (v < 0 || v > 1) return fail(FARM_ERR_INVALID_ARG, "bad INPUTS_READY");
      m->inputs_ready = (int)v;
      break;
    case FARM_OPT_EDGES:
      if (v < 0 || v > 16) return fail(FARM_ERR_INVALID_ARG, "bad EDGES (0..16)");
      m->edges_k = (int)v;
      break;
    case FARM_OPT_TIMING:
      if (v < 0 || v > 2) return fail(FARM_ERR_INVALID_ARG, "bad TIMING");
      m->timing = (int)v;
      break;
    default:
      return fail(FARM_ERR_INVALID_ARG, "unknown integer option");
  }
  return FARM_OK;
}

int farm_map_set_option_f(farm_map *m, int key, float v) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (m->finalised) return fail(FARM_ERR_STATE, "options are frozen after the first integrate / import");
  if (std::isnan(v)) return fail(FARM_ERR_INVALID_ARG, "NaN option");
  if (key == FARM_OPTF_Z_MIN)
    m->z_min = v;
  else if (key == FARM_OPTF_Z_MAX)
    m->z_max = v;
  else if (key == FARM_OPTF_PREFILTER_COS)
    m->prefilter_cos = v;
  else if (key == FARM_OPTF_HELLINGER_BUDGET)
    m->hell_budget = v;
  else if (key == FARM_OPTF_VIEW_COS)
    m->view_cos = v;
  else if (key == FARM_OPTF_VIEW_CLOSER)
    m->view_closer = v;
  else if (key == FARM_OPTF_EDGE_DECAY) {
    if (!(v > 0.f && v <= 1.f)) return fail(FARM_ERR_INVALID_ARG, "EDGE_DECAY must be in (0, 1]");
    m->edge_decay = v;
  } else if (key == FARM_OPTF_EDGE_CUTOFF) {
    if (!(v >= 0.f) || !std::isfinite(v)) return fail(FARM_ERR_INVALID_ARG, "EDGE_CUTOFF must be finite and >= 0");
    m->edge_cutoff = v;
  }
  else
    return fail(FARM_ERR_INVALID_ARG, "unknown float option");
  return FARM_OK;
}

int farm_map_integrate_batch(farm_map *m, int F, const float *depth, const uint16_t *mask, const float *K,
                             const float *T, const void *desc, const int *n_det) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (F < 1 || F > m->max_frames) return fail(FARM_ERR_INVALID_ARG, "n_frames out of range (FARM_OPT_MAX_FRAMES_PER_CALL)");
  if (!depth || !mask || !K || !T || !n_det) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  CallArgs a{};
  a.F = F;
  long long M = 0;
  for (int f = 0; f < F; ++f) {
    if (n_det[f] < 0 || n_det[f] > 65535) return fail(FARM_ERR_INVALID_ARG, "n_det must be in 0..65535");
    a.base[f] = (int)M;
    M += n_det[f];
  }
  a.base[F] = (int)M;
  if (M > m->max_det) return fail(FARM_ERR_INVALID_ARG, "too many detections in one call (FARM_OPT_MAX_DET_PER_CALL)");
  if (M > 0 && !desc) return fail(FARM_ERR_INVALID_ARG, "det_descriptors is NULL");
  int rc = finalise(m);
  if (rc != FARM_OK) return rc;
  if (m->epoch == EPOCH_MAX - 1) {  // the 16-bit epoch tag wraps: clear the epoch-tagged tables once per 65534 calls
    CU(cudaMemsetAsync(m->dm.pair_set, 0, ((size_t)m->dm.pair_mask + 1) * 8, m->stream));
    CU(cudaMemsetAsync(m->dm.ov_keys, 0, ((size_t)m->dm.ov_mask + 1) * 8, m->stream));
    m->epoch = 0;
  }
  if (m->frame_seq + (unsigned long long)F > 0x7FFFFFFFull)
    return fail(FARM_ERR_STATE, "frame sequence number would exceed INT32_MAX (farm_object.best_frame is 32-bit)");
  a.M = (int)M;
  a.depth = depth, a.mask = mask, a.K = K, a.T = T, a.desc = desc;
  const DevMap &d = m->dm;
  // everything that can fail on the host is checked before the first enqueue: the map stays untouched on error
  if (m->tc && M > 0 && m->n_upper > 0 && !tc_prepare(m->tc, d, a))
    return fail(FARM_ERR_INVALID_ARG, "similarity: det_descriptors must be 16-byte aligned for the 16-bit dtypes (TMA operand)");
  a.epoch = ++m->epoch;
  const bool maintain = m->dm.touch_seq != nullptr;  // the split similarity schedule is available on this map
  if (maintain) {
    a.seq = ++m->seq;
    m->dm.det_inv_norm = m->inv_norm2[a.seq & 1], m->dm.best_dense = m->best_dense2[a.seq & 1];
    const farm_map::LiftSet &ls = m->lset[a.seq & 1];
    DevMap &w = m->dm;
    w.surv_key = ls.surv_key, w.surv_bits = ls.surv_bits, w.surv_j = ls.surv_j, w.surv_cnt = ls.surv_cnt, w.det_npx = ls.det_npx;
    w.det_box = ls.det_box, w.det_gm = ls.det_gm, w.cam = ls.cam, w.stats = ls.stats;
    w.counters = ls.counters, w.det_nv = ls.det_nv, w.best_cand = ls.best_cand, w.assoc = ls.assoc, w.is_new = ls.is_new;
    w.best_score = ls.best_score, w.hell = ls.hell;
  }
  cudaStream_t st = m->stream;
  bool launch_failed = false;
  auto stage = [&](int id, cudaStream_t st, auto &&fn) {
    // timing 1: only the similarity kernel (it has the side stream to itself, so its events do not sit between
    // the PDL-chained kernels of the main stream); timing 2: every kernel (serialises the main-stream chain)
    // Split schedule: events between two similarity kernels would undo their programmatic overlap, so with timing 1 only
    // every eighth of them is bracketed (it then runs without overlap) and farm_map_stage_times scales the sum
    bool timed = m->timing >= 2 || (m->timing == 1 && id == FARM_STAGE_SIMILARITY);
    if (timed && id == FARM_STAGE_SIMILARITY && a.split && (a.seq & 7) != 0) timed = false;
    if (id == FARM_STAGE_SIMILARITY && m->timing == 1) m->sim_timed += timed ? 1 : 0, m->sim_all += 1;
    cudaEvent_t e0 = nullptr;
    if (timed) {
      e0 = get_event(m);
      cudaEventRecord(e0, st);
    }
    int n = fn();
    if (n < 0) launch_failed = true, n = 0;
    m->launches += n;
    m->stage_launches[id] += n;
    if (timed) {
      cudaEvent_t e1 = get_event(m);
      cudaEventRecord(e1, st);
      m->ev_pending[id].push_back({e0, e1});
    }
  };
  // DAG of one call:  prep -> { similarity (side stream) || lift + probe } -> cand_score+associate -> commit+merge
  // overlap modes: 1 = similarity || (lift, probe);  2 = similarity || lift, probe after the join;
  //                3 = lift first, then similarity || probe
  const bool fork = m->overlap && m->side && a.M > 0 && m->n_upper > 0;
  cudaStream_t sim_stream = fork ? m->side : st;
  // The tensor-core similarity kernel needs prep's output (row norms, zeroed best_dense) only in its epilogue and
  // waits for it on the device (dm.prep_done), so it is forked BEFORE prep: prep leaves the critical path.
  const bool early_fork = fork && m->tc && m->overlap == 1;
  // Split schedule (FARM_OPT_INPUTS_READY, from the third call on): no fork event -- the similarity kernel follows the
  // previous call's similarity kernel on the side stream and takes what it needs of the previous call's scan and merge
  // through device counters.  Not with per-kernel timing: the events would serialise the two streams.
  a.split = (early_fork && maintain && a.seq >= 3 && m->timing < 2 && tc_can_split(m->tc)) ? 1 : 0;
  a.scan_target = m->scan_count, a.merge_target = m->merge_count;
  a.sim_fills_gpu = ((M + 127) / 128) * (((long long)m->n_upper + 255) / 256) >= d.num_sms ? 1 : 0;
  if (early_fork && !a.split) {
    cudaEventRecord(m->ev_fork, st);
    cudaStreamWaitEvent(m->side, m->ev_fork, 0);
  }
  if (a.split) {
    // the lift of this call does not depend on the map: it runs on its own stream, behind the call before the previous one
    // (the last user of this parity's buffers), while the main chain is still busy with the previous call's scan and merge.
    // Starting it later -- behind the previous call's probe -- was measured: the
    // lift then ends too close to its own probe and single-frame calls get 2-8 us longer.
    const int par = (int)(a.seq & 1);
    if (m->ev_end_set[par]) cudaStreamWaitEvent(m->early, m->ev_end[par], 0);
    stage(FARM_STAGE_PREP, m->early, [&] {
      launch_prep(d, a, m->early);  // resets this parity's buffers only: nothing the previous call still reads
      return 1;
    });
    stage(FARM_STAGE_LIFT, m->early, [&] { return launch_lift(d, a, m->early); });
    cudaEventRecord(m->ev_lift, m->early);
    cudaStreamWaitEvent(st, m->ev_lift, 0);
  }
  if (!a.split)
    stage(FARM_STAGE_PREP, st, [&] {
      m->prep_target += (uint32_t)launch_prep(d, a, st);
      return 1;
    });
  if (fork && m->overlap == 3) stage(FARM_STAGE_LIFT, st, [&] { return launch_lift(d, a, st); });
  if (fork && !early_fork) {
    cudaEventRecord(m->ev_fork, st);
    cudaStreamWaitEvent(m->side, m->ev_fork, 0);
  }
  // similarity is enqueued first so that its one-CTA-per-SM grid is resident before the other kernels fill the SMs
  stage(FARM_STAGE_SIMILARITY, sim_stream, [&] {
    if (!m->tc) return launch_similarity_fma(d, a, m->n_upper, sim_stream);
    int ctas = 0;
    uint32_t prep_after = m->prep_target;
    const int n = launch_similarity_tc(d, a, m->n_upper, sim_stream, m->tc, m->prep_target, &ctas, &prep_after);
    m->sim_target[a.seq & 1] += (uint32_t)ctas;
    m->prep_target = prep_after;
    return n;
  });
  a.prep_target = m->prep_target;
  // With the early fork the association kernel is not joined to the side stream: it is launched (PDL) right behind
  // the probe, scores the candidates while the similarity kernel finishes, and its decision scan waits for
  // dm.sim_done on the device.  The stream join moves behind the merge kernel, off the critical path.
  a.wait_sim = early_fork ? 1 : 0;
  a.sim_target = m->sim_target[a.seq & 1];
  // Split schedule: no join event.  The decision scan waits on the device for every CTA of the similarity kernel (dm.sim_done,
  // incremented after the CTA's last write), and everything the main stream does after it is ordered behind that; an event
  // between two similarity kernels would also undo their programmatic overlap.
  if (fork && !a.split) cudaEventRecord(m->ev_join, m->side);
  if (!(fork && m->overlap == 3) && !a.split) stage(FARM_STAGE_LIFT, st, [&] { return launch_lift(d, a, st); });
  if (fork && m->overlap == 2) cudaStreamWaitEvent(st, m->ev_join, 0);
  stage(FARM_STAGE_PROBE, st, [&] { return launch_probe(d, a, st) + launch_dd_overlap(d, a, st); });

  if (fork && m->overlap != 2 && !early_fork) cudaStreamWaitEvent(st, m->ev_join, 0);
  stage(FARM_STAGE_ASSOCIATE, st, [&] { return launch_cand_associate(d, a, st); });
  stage(FARM_STAGE_MERGE, st, [&] { return launch_commit_merge(d, a, m->frame_seq, st); });
  if (maintain) m->scan_count += 1, m->merge_count += (uint32_t)merge_warps_of(a);
  stage(FARM_STAGE_MERGE, st, [&] { return launch_covis_absorb(d, a, (uint32_t)std::min<long long>((long long)m->n_upper + M, m->max_objects), st); });
  stage(FARM_STAGE_MERGE, st, [&] { return launch_covisibility(d, a, st); });
  stage(FARM_STAGE_MERGE, st, [&] { return launch_alias_compress(d, a, (uint32_t)std::min<long long>((long long)m->n_upper + M, m->max_objects), st); });
  m->edge_calls++;
  stage(FARM_STAGE_MERGE, st, [&] { return launch_edges(d, a, m->edge_calls, st); });
  if (early_fork && !a.split) cudaStreamWaitEvent(st, m->ev_join, 0);
  if (maintain) {
    cudaEventRecord(m->ev_end[a.seq & 1], st);
    m->ev_end_set[a.seq & 1] = true;
  }
  m->frame_seq += F;
  m->n_upper = (uint32_t)std::min<long long>((long long)m->n_upper + M, m->max_objects);
  m->last_M = (int)M;
  m->has_last = true;
  // the host counters above describe what was enqueued, whatever the launch status says
  CU(cudaGetLastError());
  if (launch_failed) return fail(FARM_ERR_CUDA, "a kernel launch of the call failed");
  return FARM_OK;
}

int farm_map_integrate(farm_map *m, const float *depth, const uint16_t *mask, const float *K, const float *T,
                       const void *desc, int n_det) {
  return farm_map_integrate_batch(m, 1, depth, mask, K, T, desc, &n_det);
}

int farm_map_sync(farm_map *m, farm_totals *totals) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (!m->finalised) {
    if (totals) memset(totals, 0, sizeof *totals);
    return FARM_OK;
  }
  if (totals) CU(cudaMemcpyAsync(totals, m->dm.totals, sizeof(Totals), cudaMemcpyDeviceToHost, m->stream));
  uint32_t n = 0;
  CU(cudaMemcpyAsync(&n, m->dm.n_objects, 4, cudaMemcpyDeviceToHost, m->stream));
  int rc = device_error(m);
  m->n_upper = n;  // tighten the host bound
  return rc;
}

long long farm_map_kernel_launches(const farm_map *m) { return m ? m->launches : 0; }

int farm_map_get_frame_seq(farm_map *m, long long *frame_seq) {
  if (!m || !frame_seq) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  *frame_seq = (long long)m->frame_seq;
  return FARM_OK;
}

int farm_map_set_frame_seq(farm_map *m, long long frame_seq) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (frame_seq < 0 || frame_seq > 0x7FFFFFFFll) return fail(FARM_ERR_INVALID_ARG, "frame_seq must be in 0..INT32_MAX");
  if ((unsigned long long)frame_seq < m->frame_seq) return fail(FARM_ERR_STATE, "frame_seq can only move forward");
  m->frame_seq = (unsigned long long)frame_seq;
  return FARM_OK;
}

int farm_map_last_assoc(farm_map *m, int32_t *obj_id, uint8_t *is_new, float *best_score, farm_frame_stats *stats) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (!m->has_last) return fail(FARM_ERR_STATE, "no integrate call yet");
  const size_t M = (size_t)m->last_M;
  if (obj_id && M) CU(cudaMemcpyAsync(obj_id, m->dm.assoc, M * 4, cudaMemcpyDeviceToHost, m->stream));
  if (is_new && M) CU(cudaMemcpyAsync(is_new, m->dm.is_new, M, cudaMemcpyDeviceToHost, m->stream));
  if (best_score && M) CU(cudaMemcpyAsync(best_score, m->dm.best_score, M * 4, cudaMemcpyDeviceToHost, m->stream));
  static_assert(sizeof(farm_frame_stats) == sizeof(CallStats), "stats layout");
  if (stats) CU(cudaMemcpyAsync(stats, m->dm.stats, sizeof(CallStats), cudaMemcpyDeviceToHost, m->stream));
  return device_error(m);
}

int farm_map_read(farm_map *m, farm_object *objects, int *n_objects, float *descriptors, uint64_t *voxel_keys,
                  uint32_t *voxel_owner, long long *n_voxels) {
  if (!m || !n_objects) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (!m->finalised) {
    *n_objects = 0;
    if (n_voxels) *n_voxels = 0;
    return FARM_OK;
  }
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t N = 0;
  CU(cudaMemcpy(&N, m->dm.n_objects, 4, cudaMemcpyDeviceToHost));
  m->n_upper = N;
  *n_objects = (int)N;
  unsigned long long nv = 0;
  if (n_voxels || voxel_keys || voxel_owner) {
    unsigned long long *cnt;
    CU(cudaMalloc(&cnt, 8));
    CU(cudaMemsetAsync(cnt, 0, 8, m->stream));
    count_voxels_kernel<<<m->dm.num_sms * 8, 256, 0, m->stream>>>(m->dm, cnt);
    m->launches++;
    CU(cudaMemcpyAsync(&nv, cnt, 8, cudaMemcpyDeviceToHost, m->stream));
    CU(cudaStreamSynchronize(m->stream));
    if (n_voxels) *n_voxels = (long long)nv;
    if ((voxel_keys || voxel_owner) && nv) {
      unsigned long long *dk;
      uint32_t *dvo;
      CU(cudaMalloc(&dk, nv * 8));
      CU(cudaMalloc(&dvo, nv * 4));
      CU(cudaMemsetAsync(cnt, 0, 8, m->stream));
      export_voxels_kernel<<<m->dm.num_sms * 8, 256, 0, m->stream>>>(m->dm, dk, dvo, cnt, nv);
      m->launches++;
      if (voxel_keys) CU(cudaMemcpyAsync(voxel_keys, dk, nv * 8, cudaMemcpyDeviceToHost, m->stream));
      if (voxel_owner) CU(cudaMemcpyAsync(voxel_owner, dvo, nv * 4, cudaMemcpyDeviceToHost, m->stream));
      CU(cudaStreamSynchronize(m->stream));
      cudaFree(dk);
      cudaFree(dvo);
    }
    cudaFree(cnt);
  }
  if (objects && N) {
    farm_object *dobj;
    CU(cudaMalloc(&dobj, (size_t)N * sizeof(farm_object)));
    export_objects_kernel<<<(N + 255) / 256, 256, 0, m->stream>>>(m->dm, dobj, N);
    m->launches++;
    CU(cudaMemcpyAsync(objects, dobj, (size_t)N * sizeof(farm_object), cudaMemcpyDeviceToHost, m->stream));
    CU(cudaStreamSynchronize(m->stream));
    cudaFree(dobj);
  }
  if (descriptors && N) {
    CU(cudaMemcpyAsync(descriptors, m->dm.desc_master, (size_t)N * m->D * 4, cudaMemcpyDeviceToHost, m->stream));
    CU(cudaStreamSynchronize(m->stream));
  }
  return FARM_OK;
}

int farm_map_import(farm_map *m, const farm_object *objects, int n_objects, const float *descriptors,
                    const uint64_t *voxel_keys, const uint32_t *voxel_owner, long long n_voxels) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (n_objects < 0 || n_voxels < 0 || (n_objects && (!objects || !descriptors)) || (n_voxels && (!voxel_keys || !voxel_owner)))
    return fail(FARM_ERR_INVALID_ARG, "bad import arguments");
  if (m->has_last || m->n_upper) return fail(FARM_ERR_STATE, "import needs an empty map");
  if (n_objects > m->max_objects) return fail(FARM_ERR_CAPACITY, "more objects than FARM_OPT_MAX_OBJECTS");
  if (n_voxels > m->max_voxels) return fail(FARM_ERR_CAPACITY, "more voxels than FARM_OPT_MAX_VOXELS");
  for (int i = 0; i < n_objects; ++i)
    if (objects[i].id != i) return fail(FARM_ERR_INVALID_ARG, "object ids must be 0..n-1 in order");
  int rc = finalise(m);
  if (rc != FARM_OK) return rc;
  const DevMap &d = m->dm;
  if (n_objects) {
    farm_object *dobj;
    CU(cudaMalloc(&dobj, (size_t)n_objects * sizeof(farm_object)));
    CU(cudaMemcpyAsync(dobj, objects, (size_t)n_objects * sizeof(farm_object), cudaMemcpyHostToDevice, m->stream));
    import_objects_kernel<<<(n_objects + 255) / 256, 256, 0, m->stream>>>(d, dobj, (uint32_t)n_objects);
    CU(cudaMemcpyAsync(d.desc_master, descriptors, (size_t)n_objects * m->D * 4, cudaMemcpyHostToDevice, m->stream));
    const int grid = std::min(n_objects, d.num_sms * 8);
    if (m->dtype == FARM_DTYPE_F32)
      renorm_rows_kernel<float><<<grid, 256, 0, m->stream>>>(d, (uint32_t)n_objects);
    else if (m->dtype == FARM_DTYPE_F16)
      renorm_rows_kernel<__half><<<grid, 256, 0, m->stream>>>(d, (uint32_t)n_objects);
    else
      renorm_rows_kernel<__nv_bfloat16><<<grid, 256, 0, m->stream>>>(d, (uint32_t)n_objects);
    m->launches += 2;
    uint32_t n = (uint32_t)n_objects;
    CU(cudaMemcpyAsync(d.n_objects, &n, 4, cudaMemcpyHostToDevice, m->stream));
    CU(cudaStreamSynchronize(m->stream));
    cudaFree(dobj);
  }
  // voxels in chunks so that the staging buffers stay small
  const long long chunk = 1ll << 24;
  uint32_t *ocnt = nullptr;  // voxels listed per owner, checked against objects[i].n_voxels
  if (n_objects) {
    CU(cudaMalloc(&ocnt, (size_t)n_objects * 4));
    CU(cudaMemsetAsync(ocnt, 0, (size_t)n_objects * 4, m->stream));
  }
  if (n_voxels) {
    unsigned long long *dk;
    uint32_t *dow;
    CU(cudaMalloc(&dk, (size_t)std::min(chunk, n_voxels) * 8));
    CU(cudaMalloc(&dow, (size_t)std::min(chunk, n_voxels) * 4));
    for (long long off = 0; off < n_voxels; off += chunk) {
      const long long n = std::min(chunk, n_voxels - off);
      CU(cudaMemcpyAsync(dk, voxel_keys + off, (size_t)n * 8, cudaMemcpyHostToDevice, m->stream));
      CU(cudaMemcpyAsync(dow, voxel_owner + off, (size_t)n * 4, cudaMemcpyHostToDevice, m->stream));
      import_voxels_kernel<<<d.num_sms * 8, 256, 0, m->stream>>>(d, dk, dow, n, (uint32_t)n_objects);
      if (ocnt) count_owner_kernel<<<d.num_sms * 8, 256, 0, m->stream>>>(dow, n, (uint32_t)n_objects, ocnt);
      m->launches += ocnt ? 2 : 1;
      CU(cudaStreamSynchronize(m->stream));
    }
    cudaFree(dk);
    cudaFree(dow);
  }
  if (ocnt) {
    check_owner_count_kernel<<<(n_objects + 255) / 256, 256, 0, m->stream>>>(d, ocnt, (uint32_t)n_objects);
    m->launches++;
    CU(cudaStreamSynchronize(m->stream));
    cudaFree(ocnt);
  }
  CU(cudaGetLastError());
  m->n_upper = (uint32_t)n_objects;
  return device_error(m);
}

int farm_map_integrate_batch_host(farm_map *m, int F, const float *depth, const uint16_t *mask, const float *K,
                                  const float *T, const void *desc, const int *n_det) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (F < 1 || F > m->max_frames) return fail(FARM_ERR_INVALID_ARG, "n_frames out of range (FARM_OPT_MAX_FRAMES_PER_CALL)");
  if (!depth || !mask || !K || !T || !n_det) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  long long M = 0;
  for (int f = 0; f < F; ++f) {
    if (n_det[f] < 0 || n_det[f] > 65535) return fail(FARM_ERR_INVALID_ARG, "n_det must be in 0..65535");
    M += n_det[f];
  }
  if (M > m->max_det) return fail(FARM_ERR_INVALID_ARG, "too many detections in one call (FARM_OPT_MAX_DET_PER_CALL)");
  if (M > 0 && !desc) return fail(FARM_ERR_INVALID_ARG, "det_descriptors is NULL");
  int rc = finalise(m);
  if (rc != FARM_OK) return rc;
  const size_t px = (size_t)m->H * m->W;
  if (!m->cstream) {  // device staging, sized for the largest call
    CU(cudaStreamCreateWithFlags(&m->cstream, cudaStreamNonBlocking));
    for (auto &g : m->stg) {
      void *p;
      CU(cudaMalloc(&p, px * m->max_frames * 4)); m->allocs.push_back(p); g.depth = (float *)p;
      CU(cudaMalloc(&p, px * m->max_frames * 2)); m->allocs.push_back(p); g.mask = (uint16_t *)p;
      CU(cudaMalloc(&p, (size_t)m->max_frames * 9 * 4)); m->allocs.push_back(p); g.K = (float *)p;
      CU(cudaMalloc(&p, (size_t)m->max_frames * 16 * 4)); m->allocs.push_back(p); g.T = (float *)p;
      CU(cudaMalloc(&p, (size_t)m->max_det * m->D * m->elem())); m->allocs.push_back(p); g.desc = p;
      CU(cudaEventCreateWithFlags(&g.copied, cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&g.free, cudaEventDisableTiming));
    }
  }
  farm_map::Staging &g = m->stg[m->host_calls++ & 1];
  if (g.used) CU(cudaStreamWaitEvent(m->cstream, g.free, 0));  // the call that last read this set has finished
  CU(cudaMemcpyAsync(g.depth, depth, px * F * 4, cudaMemcpyHostToDevice, m->cstream));
  CU(cudaMemcpyAsync(g.mask, mask, px * F * 2, cudaMemcpyHostToDevice, m->cstream));
  CU(cudaMemcpyAsync(g.K, K, (size_t)F * 36, cudaMemcpyHostToDevice, m->cstream));
  CU(cudaMemcpyAsync(g.T, T, (size_t)F * 64, cudaMemcpyHostToDevice, m->cstream));
  if (M) CU(cudaMemcpyAsync(g.desc, desc, (size_t)M * m->D * m->elem(), cudaMemcpyHostToDevice, m->cstream));
  CU(cudaEventRecord(g.copied, m->cstream));
  CU(cudaStreamWaitEvent(m->stream, g.copied, 0));
  if (m->dm.touch_seq && m->side) CU(cudaStreamWaitEvent(m->side, g.copied, 0));  // the split similarity kernel reads the staged rows too
  if (m->dm.touch_seq && m->early) CU(cudaStreamWaitEvent(m->early, g.copied, 0));  // and so does its lift kernel
  rc = farm_map_integrate_batch(m, F, g.depth, g.mask, g.K, g.T, M ? g.desc : nullptr, n_det);
  CU(cudaEventRecord(g.free, m->stream));
  g.used = true;
  return rc;
}

int farm_map_last_assoc_async(farm_map *m, int32_t *obj_id, uint8_t *is_new, float *best_score, farm_frame_stats *stats) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (!m->has_last) return fail(FARM_ERR_STATE, "no integrate call yet");
  const size_t M = (size_t)m->last_M;
  if (obj_id && M) CU(cudaMemcpyAsync(obj_id, m->dm.assoc, M * 4, cudaMemcpyDeviceToHost, m->stream));
  if (is_new && M) CU(cudaMemcpyAsync(is_new, m->dm.is_new, M, cudaMemcpyDeviceToHost, m->stream));
  if (best_score && M) CU(cudaMemcpyAsync(best_score, m->dm.best_score, M * 4, cudaMemcpyDeviceToHost, m->stream));
  if (stats) CU(cudaMemcpyAsync(stats, m->dm.stats, sizeof(CallStats), cudaMemcpyDeviceToHost, m->stream));
  return FARM_OK;
}

static int export_gaussians(farm_map *m, const double *w, const uint32_t *w_u32, const double *g, uint32_t n, double *weight,
                            float *mu, float *cov) {
  if (!n) return FARM_OK;
  double *dw = nullptr;
  float *dmu, *dcov;
  if (weight) CU(cudaMalloc(&dw, (size_t)n * 8));
  CU(cudaMalloc(&dmu, (size_t)n * 12));
  CU(cudaMalloc(&dcov, (size_t)n * 24));
  export_gaussians_kernel<<<(n + 255) / 256, 256, 0, m->stream>>>(w, w_u32, g, n, dw, dmu, dcov);
  m->launches++;
  if (weight) CU(cudaMemcpyAsync(weight, dw, (size_t)n * 8, cudaMemcpyDeviceToHost, m->stream));
  if (mu) CU(cudaMemcpyAsync(mu, dmu, (size_t)n * 12, cudaMemcpyDeviceToHost, m->stream));
  if (cov) CU(cudaMemcpyAsync(cov, dcov, (size_t)n * 24, cudaMemcpyDeviceToHost, m->stream));
  CU(cudaStreamSynchronize(m->stream));
  cudaFree(dw), cudaFree(dmu), cudaFree(dcov);
  return FARM_OK;
}

int farm_map_last_gaussians(farm_map *m, float *mu, float *cov, float *hellinger) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (!m->gaussian) return fail(FARM_ERR_STATE, "FARM_OPT_GAUSSIAN is off");
  if (!m->has_last) return fail(FARM_ERR_STATE, "no integrate call yet");
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  const uint32_t M = (uint32_t)m->last_M;
  if (hellinger && M) CU(cudaMemcpy(hellinger, m->dm.hell, (size_t)M * 4, cudaMemcpyDeviceToHost));
  return export_gaussians(m, nullptr, m->dm.det_npx, m->dm.det_gm, M, nullptr, mu, cov);
}

int farm_map_read_gaussians(farm_map *m, double *weight, float *mu, float *cov) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (!m->gaussian) return fail(FARM_ERR_STATE, "FARM_OPT_GAUSSIAN is off");
  if (!m->finalised) return FARM_OK;
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t N = 0;
  CU(cudaMemcpy(&N, m->dm.n_objects, 4, cudaMemcpyDeviceToHost));
  return export_gaussians(m, m->dm.obj_gw, nullptr, m->dm.obj_gm, N, weight, mu, cov);
}

int farm_map_query(farm_map *m, const void *emb0, const void *emb1, const void *emb2, int d0, int d1, int d2, int emb_dtype,
                   const int32_t *cls, const float *q_target, int target_class, int n_pred, const int32_t *pred_type,
                   const float *q_landmarks, int topk, int32_t *top_ids, float *top_scores, int32_t *landmarks, float *s_sem,
                   float *gbar, float *s) {
  if (!m || !emb0 || !emb1 || !emb2 || !q_target) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (d0 < 1 || d1 < 1 || d2 < 1 || d0 > 8192 || d1 > 8192 || d2 > 8192) return fail(FARM_ERR_INVALID_ARG, "embedding sizes must be in 1..8192");
  if (emb_dtype < 0 || emb_dtype > 2) return fail(FARM_ERR_INVALID_ARG, "bad emb_dtype");
  if (n_pred < 0 || n_pred > 3 || (n_pred && (!pred_type || !q_landmarks))) return fail(FARM_ERR_INVALID_ARG, "n_pred must be in 0..3");
  for (int p = 0; p < n_pred; ++p)
    if (pred_type[p] < 0 || pred_type[p] > 3) return fail(FARM_ERR_INVALID_ARG, "unknown predicate type");
  if (topk < 0 || topk > 4096) return fail(FARM_ERR_INVALID_ARG, "topk must be in 0..4096");
  int rc = finalise(m);
  if (rc != FARM_OK) return rc;
  rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t N = 0;
  CU(cudaMemcpy(&N, m->dm.n_objects, 4, cudaMemcpyDeviceToHost));
  const void *const emb[3] = {emb0, emb1, emb2};
  const int dim[3] = {d0, d1, d2};
  std::string err;
  rc = run_query(m->dm, m->stream, N, emb, dim, emb_dtype, cls, q_target, target_class, n_pred, pred_type, q_landmarks, topk, top_ids,
                 top_scores, landmarks, s_sem, gbar, s, &m->launches, &err);
  return rc == FARM_OK ? FARM_OK : fail(rc, err);
}

int farm_map_read_alias(farm_map *m, int32_t *alias) {
  if (!m || !alias) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (!m->corr) return fail(FARM_ERR_STATE, "FARM_OPT_CORRESPONDENCE is off");
  if (!m->finalised) return FARM_OK;
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t N = 0;
  CU(cudaMemcpy(&N, m->dm.n_objects, 4, cudaMemcpyDeviceToHost));
  if (N) CU(cudaMemcpy(alias, m->dm.alias, (size_t)N * 4, cudaMemcpyDeviceToHost));
  return FARM_OK;
}

int farm_map_last_merges(farm_map *m, int32_t *loser, int32_t *winner, int *n) {
  if (!m || !n) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (!m->corr) return fail(FARM_ERR_STATE, "FARM_OPT_CORRESPONDENCE is off");
  *n = 0;
  if (!m->has_last) return FARM_OK;
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t k = 0;
  CU(cudaMemcpy(&k, m->dm.counters + 7, 4, cudaMemcpyDeviceToHost));
  *n = (int)k;
  if (k && loser) CU(cudaMemcpy(loser, m->dm.loser, (size_t)k * 4, cudaMemcpyDeviceToHost));
  if (k && winner) CU(cudaMemcpy(winner, m->dm.winner, (size_t)k * 4, cudaMemcpyDeviceToHost));
  return FARM_OK;
}

int farm_map_read_views(farm_map *m, farm_view *views, int32_t *counts) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (m->views_k <= 0) return fail(FARM_ERR_STATE, "FARM_OPT_VIEWS is off");
  if (!m->finalised) return FARM_OK;
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t N = 0;
  CU(cudaMemcpy(&N, m->dm.n_objects, 4, cudaMemcpyDeviceToHost));
  if (views && N) CU(cudaMemcpy(views, m->dm.views, (size_t)N * m->views_k * sizeof(farm_view), cudaMemcpyDeviceToHost));
  if (counts && N) CU(cudaMemcpy(counts, m->dm.view_cnt, (size_t)N * 4, cudaMemcpyDeviceToHost));
  return FARM_OK;
}

int farm_cosine_rowmax_noalloc(const void *A, int M, const void *B, int N, int D, int dtype, float *max_cos, int32_t *argmax,
                               void *stream) {
  if (M < 0 || N < 0) return fail(FARM_ERR_INVALID_ARG, "farm_cosine_rowmax_noalloc: negative size");
  if (M > FARM_NOALLOC_MAX_M)
    return fail(FARM_ERR_INVALID_ARG, "farm_cosine_rowmax_noalloc: M exceeds FARM_NOALLOC_MAX_M (4096): the scratch array is fixed-size");
  if (N > FARM_NOALLOC_MAX_N)
    return fail(FARM_ERR_INVALID_ARG, "farm_cosine_rowmax_noalloc: N exceeds FARM_NOALLOC_MAX_N (65536): the scratch array is fixed-size");
  if (D < 1 || D > 8192) return fail(FARM_ERR_INVALID_ARG, "farm_cosine_rowmax_noalloc: D must be in 1..8192");
  if (dtype != FARM_DTYPE_F32 && dtype != FARM_DTYPE_F16 && dtype != FARM_DTYPE_BF16)
    return fail(FARM_ERR_INVALID_ARG, "farm_cosine_rowmax_noalloc: bad dtype");
  if ((M > 0 && !A) || (N > 0 && !B)) return fail(FARM_ERR_INVALID_ARG, "farm_cosine_rowmax_noalloc: NULL operand");
  std::string err;
  const int rc = noalloc_cosine_rowmax(A, M, B, N, D, dtype, max_cos, argmax, (cudaStream_t)stream, &err);
  return rc == FARM_OK ? FARM_OK : fail(rc, err);
}

int farm_map_read_edges(farm_map *m, uint32_t *ea, uint32_t *eb, double *ew, uint64_t capacity, uint64_t *n_out) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (m->edges_k <= 0) return fail(FARM_ERR_STATE, "FARM_OPT_EDGES is off");
  if (n_out) *n_out = 0;
  if (!m->finalised) return FARM_OK;
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t n = 0;
  CU(cudaMemcpy(&n, m->dm.ed_cnt, 4, cudaMemcpyDeviceToHost));
  if (n_out) *n_out = n;
  if (n == 0) return FARM_OK;
  // compacted on the device, ordered on the host (an export, not part of the integrate path)
  uint32_t *da = nullptr, *db = nullptr, *dc = nullptr;
  double *dw = nullptr;
  auto release = [&] { cudaFree(da), cudaFree(db), cudaFree(dc), cudaFree(dw); };
  if (cudaMalloc(&da, (size_t)n * 4) || cudaMalloc(&db, (size_t)n * 4) || cudaMalloc(&dw, (size_t)n * 8) || cudaMalloc(&dc, 4)) {
    release();
    cudaGetLastError();
    return fail(FARM_ERR_CUDA, "farm_map_read_edges: out of device memory");
  }
  cudaMemsetAsync(dc, 0, 4, m->stream);
  m->launches += launch_edge_export(m->dm, m->edge_calls, da, db, dw, n, dc, m->stream);
  std::vector<uint32_t> ha(n), hb(n);
  std::vector<double> hw(n);
  cudaError_t e = cudaMemcpyAsync(ha.data(), da, (size_t)n * 4, cudaMemcpyDeviceToHost, m->stream);
  if (!e) e = cudaMemcpyAsync(hb.data(), db, (size_t)n * 4, cudaMemcpyDeviceToHost, m->stream);
  if (!e) e = cudaMemcpyAsync(hw.data(), dw, (size_t)n * 8, cudaMemcpyDeviceToHost, m->stream);
  if (!e) e = cudaStreamSynchronize(m->stream);
  release();
  if (e) return fail(FARM_ERR_CUDA, std::string("farm_map_read_edges: ") + cudaGetErrorString(e));
  std::vector<uint32_t> order(n);
  for (uint32_t i = 0; i < n; ++i) order[i] = i;
  std::sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) { return ha[x] != ha[y] ? ha[x] < ha[y] : hb[x] < hb[y]; });
  const uint64_t lim = std::min<uint64_t>(n, capacity);
  for (uint64_t i = 0; i < lim; ++i) {
    if (ea) ea[i] = ha[order[i]];
    if (eb) eb[i] = hb[order[i]];
    if (ew) ew[i] = hw[order[i]];
  }
  if (capacity < n && (ea || eb || ew)) return fail(FARM_ERR_CAPACITY, "farm_map_read_edges: capacity is smaller than the number of edges");
  return FARM_OK;
}

int farm_map_read_covisibility(farm_map *m, uint64_t *rows, int *words) {
  if (!m || !words) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (!m->covis) return fail(FARM_ERR_STATE, "FARM_OPT_COVISIBILITY is off");
  *words = 0;
  if (!m->finalised) return FARM_OK;
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  uint32_t N = 0;
  CU(cudaMemcpy(&N, m->dm.n_objects, 4, cudaMemcpyDeviceToHost));
  const uint32_t w = (N + 63) / 64;
  *words = (int)w;
  if (rows && N)  // strided device rows -> dense [N, w]
    CU(cudaMemcpy2D(rows, (size_t)w * 8, m->dm.covis, (size_t)m->dm.covis_words * 8, (size_t)w * 8, N, cudaMemcpyDeviceToHost));
  return FARM_OK;
}

int farm_map_stage_times(farm_map *m, float *ms, long long *launches, int reset) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (m->finalised) CU(cudaStreamSynchronize(m->stream));
  for (int s = 0; s < FARM_N_STAGES; ++s) {
    for (auto &p : m->ev_pending[s]) {
      float t = 0.f;
      if (cudaEventElapsedTime(&t, p.first, p.second) == cudaSuccess) m->stage_ms[s] += t;
      m->ev_free.push_back(p.first);
      m->ev_free.push_back(p.second);
    }
    m->ev_pending[s].clear();
    if (ms) ms[s] = (float)m->stage_ms[s];
    if (s == FARM_STAGE_SIMILARITY && ms && m->timing == 1 && m->sim_timed > 0 && m->sim_timed < m->sim_all)
      ms[s] = (float)(m->stage_ms[s] * (double)m->sim_all / (double)m->sim_timed);  // split schedule: sampled launches, scaled
    if (launches) launches[s] = m->stage_launches[s];
    if (reset) m->stage_ms[s] = 0.0, m->stage_launches[s] = 0;
  }
  if (reset) m->sim_timed = 0, m->sim_all = 0;
  return FARM_OK;
}

int farm_debug_backproject(farm_map *m, const float *depth, const uint16_t *mask, const float *K, const float *T,
                           int n_det, float *xyz, uint64_t *keys) {
  if (!m || !depth || !mask || !K || !T || !xyz || !keys) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  int rc = finalise(m);
  if (rc != FARM_OK) return rc;
  m->launches += launch_debug_backproject(m->dm, depth, mask, K, T, n_det, xyz, (unsigned long long *)keys, m->stream);
  CU(cudaGetLastError());
  return FARM_OK;
}

int farm_debug_last_voxels(farm_map *m, long long *offsets, uint64_t *keys, uint32_t *n_px, float *box) {
  if (!m || !offsets) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (!m->has_last) return fail(FARM_ERR_STATE, "no integrate call yet");
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  const int M = m->last_M;
  uint32_t n = 0;  // events (detection, block, new voxel bits) of the last call
  CU(cudaMemcpy(&n, m->dm.counters, 4, cudaMemcpyDeviceToHost));
  n = std::min(n, m->dm.pair_cap);
  std::vector<uint32_t> js(n);
  std::vector<unsigned long long> bks(n), bits(n);
  if (n) {
    unsigned long long *dk;
    CU(cudaMalloc(&dk, (size_t)n * 8));
    gather_events_kernel<<<(n + 255) / 256, 256, 0, m->stream>>>(m->dm, n, dk);
    m->launches++;
    CU(cudaMemcpyAsync(bks.data(), dk, (size_t)n * 8, cudaMemcpyDeviceToHost, m->stream));
    CU(cudaMemcpyAsync(js.data(), m->dm.pl_j, (size_t)n * 4, cudaMemcpyDeviceToHost, m->stream));
    CU(cudaMemcpyAsync(bits.data(), m->dm.pl_bits, (size_t)n * 8, cudaMemcpyDeviceToHost, m->stream));
    CU(cudaStreamSynchronize(m->stream));
    cudaFree(dk);
  }
  std::vector<long long> cnt(M + 1, 0);
  for (uint32_t i = 0; i < n; ++i) {
    js[i] &= 0x7FFFFFFFu;
    if ((int)js[i] < M) cnt[js[i] + 1] += __builtin_popcountll(bits[i]);
  }
  for (int j = 0; j < M; ++j) cnt[j + 1] += cnt[j];
  for (int j = 0; j <= M; ++j) offsets[j] = cnt[j];
  if (keys) {
    std::vector<long long> cur(cnt.begin(), cnt.end() - 1);
    for (uint32_t i = 0; i < n; ++i)
      if ((int)js[i] < M)
        for (unsigned long long w = bits[i]; w; w &= w - 1)
          keys[cur[js[i]]++] = voxel_key_of(bks[i], (uint32_t)__builtin_ctzll(w));
  }
  if (n_px && M) CU(cudaMemcpy(n_px, m->dm.det_npx, (size_t)M * 4, cudaMemcpyDeviceToHost));
  if (box && M) {
    std::vector<int> ob((size_t)M * 6);
    CU(cudaMemcpy(ob.data(), m->dm.det_box, (size_t)M * 24, cudaMemcpyDeviceToHost));
    for (size_t i = 0; i < ob.size(); ++i) {
      const int v = ob[i] ^ ((ob[i] >> 31) & 0x7FFFFFFF);
      memcpy(&box[i], &v, 4);
    }
  }
  return FARM_OK;
}

int farm_debug_last_overlaps(farm_map *m, long long *offsets, int32_t *obj_id, uint32_t *count) {
  if (!m || !offsets) return fail(FARM_ERR_INVALID_ARG, "NULL argument");
  if (!m->has_last) return fail(FARM_ERR_STATE, "no integrate call yet");
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  const int M = m->last_M;
  uint32_t n = 0;
  CU(cudaMemcpy(&n, m->dm.counters + 1, 4, cudaMemcpyDeviceToHost));
  std::vector<uint32_t> js(n), cs(n);
  std::vector<int32_t> os(n);
  if (n) {
    CU(cudaMemcpy(js.data(), m->dm.cand_j, (size_t)n * 4, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(os.data(), m->dm.cand_o, (size_t)n * 4, cudaMemcpyDeviceToHost));
    CU(cudaMemcpy(cs.data(), m->dm.cand_c, (size_t)n * 4, cudaMemcpyDeviceToHost));
  }
  std::vector<long long> cnt(M + 1, 0);
  for (uint32_t i = 0; i < n; ++i)
    if (os[i] < 0) js[i] = 0xFFFFFFFFu;  // detection-detection entries (U2) are not part of the overlap histogram
  for (uint32_t i = 0; i < n; ++i)
    if ((int)js[i] < M && (int)js[i] >= 0) cnt[js[i] + 1]++;
  for (int j = 0; j < M; ++j) cnt[j + 1] += cnt[j];
  for (int j = 0; j <= M; ++j) offsets[j] = cnt[j];
  if (obj_id || count) {
    std::vector<long long> cur(cnt.begin(), cnt.end() - 1);
    for (uint32_t i = 0; i < n; ++i)
      if ((int)js[i] < M && (int)js[i] >= 0) {
        const long long p = cur[js[i]]++;
        if (obj_id) obj_id[p] = os[i];
        if (count) count[p] = cs[i];
      }
  }
  return FARM_OK;
}

int farm_debug_last_dense(farm_map *m, float *max_cos, int32_t *argmax) {
  if (!m) return fail(FARM_ERR_INVALID_ARG, "map is NULL");
  if (!m->has_last) return fail(FARM_ERR_STATE, "no integrate call yet");
  int rc = device_error(m);
  if (rc != FARM_OK) return rc;
  const int M = m->last_M;
  std::vector<unsigned long long> bd(M);
  if (M) CU(cudaMemcpy(bd.data(), m->dm.best_dense, (size_t)M * 8, cudaMemcpyDeviceToHost));
  for (int j = 0; j < M; ++j) {
    if (bd[j]) {
      const uint32_t u = (uint32_t)(bd[j] >> 32) ^ 0x80000000u;
      const int i = (int)u;
      const int f = i ^ ((i >> 31) & 0x7FFFFFFF);
      if (max_cos) memcpy(&max_cos[j], &f, 4);
      if (argmax) argmax[j] = (int32_t)(0xFFFFFFFFu - (uint32_t)bd[j]);
    } else {
      if (max_cos) max_cos[j] = 0.f;
      if (argmax) argmax[j] = -1;
    }
  }
  return FARM_OK;
}

}  // extern "C"
