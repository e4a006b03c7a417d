// farm_edges.cu -- weighted covisibility edges (rules W1-W4; "a parallel weighted edge dictionary
// accumulates their co-occurrence, restricted to spatially proximal pairs (a k-nearest-neighbor graph in Gaussian
// Hellinger distance with a soft median cutoff) and discounted by a temporal decay").  Optional (FARM_OPT_EDGES = k);
// runs behind the merge kernel.
//   W1 S = the distinct entities that received a detection in this call and carry a Gaussian (listed by the merge
//      kernel, farm_assoc.cu: edge_member);
//   W2 N_k(a) = the k entities of S \ {a} nearest to a in Hellinger distance, ordered through the Bhattacharyya
//      distance DB (H = sqrt(1 - exp(-DB)) is increasing in it and saturates at 1 in floating point), fp32 value,
//      ties -> lower id;
//   W3 b in N_k(a) is kept iff DB(a, b) <= cutoff * (lower median of a's kNN distances), fp32;
//   W4 every unordered pair kept from either side: w <- w * decay^(calls since its last update) + 1 (fp64).
#include "farm_internal.cuh"

namespace farm {
namespace {

constexpr int KNN_WARPS = 4;
constexpr int KNN_THREADS = KNN_WARPS * 32;
constexpr unsigned long long KEY_MAX = 0xFFFFFFFFFFFFFFFFull;

__device__ __forceinline__ double det_sym3(const double c[6]) {
  return c[0] * (c[3] * c[5] - c[4] * c[4]) - c[1] * (c[1] * c[5] - c[4] * c[2]) + c[2] * (c[1] * c[4] - c[3] * c[2]);
}

// eg_gauss row (12 doubles, written by the merge kernel): mu (3), trace of S, S = Sigma + eps2 I packed (6), ln |S|, pad
constexpr int GROW = 12;

// W2: Bhattacharyya distance of two regularised Gaussians (rows of eg_gauss), fp64, returned as fp32
__device__ __forceinline__ float bhattacharyya(const double ga[GROW], const double *gb) {
  double sb[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) sb[k] = 0.5 * (ga[4 + k] + gb[4 + k]);
  const double db = det_sym3(sb);
  const double a00 = sb[3] * sb[5] - sb[4] * sb[4], a01 = sb[2] * sb[4] - sb[1] * sb[5], a02 = sb[1] * sb[4] - sb[2] * sb[3];
  const double a11 = sb[0] * sb[5] - sb[2] * sb[2], a12 = sb[1] * sb[2] - sb[0] * sb[4], a22 = sb[0] * sb[3] - sb[1] * sb[1];
  const double d0 = ga[0] - gb[0], d1 = ga[1] - gb[1], d2 = ga[2] - gb[2];
  const double q = (d0 * (a00 * d0 + a01 * d1 + a02 * d2) + d1 * (a01 * d0 + a11 * d1 + a12 * d2) + d2 * (a02 * d0 + a12 * d1 + a22 * d2)) / db;
  return (float)(0.125 * q + 0.5 * (log(db) - 0.5 * (ga[10] + gb[10])));
}

__device__ __forceinline__ unsigned long long warp_min_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long u = __shfl_xor_sync(0xFFFFFFFFu, v, o);
    v = u < v ? u : v;
  }
  return v;
}

// W4: one kept pair {x, y}.  The first thread of the call to reach the edge (atomicExch on its clock) applies the decay
// and the +1; a pair kept from both sides is counted once.
__device__ __forceinline__ void edge_touch(const DevMap &m, uint32_t x, uint32_t y, uint32_t call) {
  const uint32_t lo = min(x, y), hi = max(x, y);
  const unsigned long long key = ((unsigned long long)lo << 32) | hi;
  uint32_t h = hash32(lo, hi) & m.ed_mask;
  for (uint32_t probe = 0; probe <= m.ed_mask; ++probe) {
    unsigned long long k = __ldcg(&m.ed_key[h]);
    if (k == KEY_MAX) {
      k = atomicCAS(&m.ed_key[h], KEY_MAX, key);
      if (k == KEY_MAX) k = key, atomicAdd(m.ed_cnt, 1u);
    }
    if (k == key) {
      const uint32_t t_old = atomicExch(&m.ed_t[h], call);
      if (t_old != call) m.ed_w[h] = m.ed_w[h] * pow((double)m.edge_decay, (double)(call - t_old)) + 1.0;
      return;
    }
    h = (h + 1) & m.ed_mask;
    if (probe == 4096) break;
  }
  atomicOr(m.err, ERR_EDGE_TABLE_FULL);
}

// pops the smallest key of the warp's lane-resident sorted lists (top[0] is each lane's head)
template <int K>
__device__ __forceinline__ unsigned long long warp_pop_min(unsigned long long (&top)[K]) {
  const unsigned long long w = warp_min_u64(top[0]);
  if (top[0] == w) {  // keys are unique (they carry the id): at most one lane pops
#pragma unroll
    for (int k = 0; k + 1 < K; ++k) top[k] = top[k + 1];
    top[K - 1] = KEY_MAX;
  }
  return w;
}

// W2-W4: one warp per member a of S (S and its Gaussians come from the merge kernel: counters[8], eg_list, eg_gauss).
// Most pairs are far apart and never get near N_k(a):  DB >= |dmu|^2 / (8 lambda_max(Sbar)) >= |dmu|^2 / (4 (tr S_a + tr S_b))
// (the log term is >= 0), and the k-th smallest of any k distances already evaluated bounds the k-th nearest from above.
// The warp scans S in chunks of 32 with that ten-operation test, compacts the survivors (ballot) into a queue in shared
// memory and evaluates the exact distance -- two hundred fp64 operations -- for 32 queued candidates at a time, one per lane
// and without divergence; each lane keeps the K smallest (distance, id) keys it has evaluated in registers and the bound is
// the k-th smallest of the lanes' best keys.  k rounds of a warp minimum then pop N_k(a) in order and lane r handles the
// r-th neighbour (cutoff, dictionary update).  On configs[4] (|S| = 1600) 2-4 % of the pairs reach the exact evaluation.
template <int K>
__global__ void __launch_bounds__(KNN_THREADS) edge_knn_kernel(DevMap m, uint32_t call) {
  __shared__ uint32_t queue_all[KNN_WARPS][64];
  pdl_wait();
  const uint32_t n = min(m.counters[8], m.max_det);
  const int lane = threadIdx.x & 31;
  const int kk = min(m.edges_k, (int)n - 1);
  if (kk <= 0) return;
  uint32_t *queue = queue_all[threadIdx.x >> 5];
  const unsigned lt_mask = (1u << lane) - 1u;
  const float INF = __int_as_float(0x7F800000);
  for (uint32_t ia = blockIdx.x * KNN_WARPS + (threadIdx.x >> 5); ia < n; ia += gridDim.x * KNN_WARPS) {
    double ga[GROW];
#pragma unroll
    for (int k = 0; k < 11; ++k) ga[k] = m.eg_gauss[(size_t)ia * GROW + k];
    unsigned long long top[K];
#pragma unroll
    for (int k = 0; k < K; ++k) top[k] = KEY_MAX;
    double bound = 1.0e300;  // upper bound of the k-th smallest distance (+ slack)
    uint32_t qn = 0;
    auto evaluate = [&](uint32_t cnt) {  // exact distance of queue[0 .. cnt), one candidate per lane
      bool inserted = false;
      if ((uint32_t)lane < cnt) {
        const uint32_t ib = queue[lane];
        const float d = bhattacharyya(ga, m.eg_gauss + (size_t)ib * GROW);
        const unsigned long long key = ((unsigned long long)((uint32_t)f2ord(d) ^ 0x80000000u) << 32) | m.eg_list[ib];
        if (key < top[K - 1]) {
          inserted = true;
          top[K - 1] = key;
#pragma unroll
          for (int k = K - 1; k > 0; --k)
            if (top[k] < top[k - 1]) {
              const unsigned long long t = top[k];
              top[k] = top[k - 1], top[k - 1] = t;
            }
        }
      }
      if (__any_sync(0xFFFFFFFFu, inserted)) {  // bound <- k-th smallest of the lanes' best distances (k REDUX rounds)
        int cur = top[0] == KEY_MAX ? 0x7FFFFFFF : (int)((uint32_t)(top[0] >> 32) ^ 0x80000000u);  // order-preserving int
        int kth = 0x7FFFFFFF;
#pragma unroll
        for (int r = 0; r < K; ++r) {
          if (r < kk) {
            kth = __reduce_min_sync(0xFFFFFFFFu, cur);
            const unsigned who = __ballot_sync(0xFFFFFFFFu, cur == kth);
            if (lane == __ffs(who) - 1) cur = 0x7FFFFFFF;
          }
        }
        if (kth != 0x7FFFFFFF) bound = fmin(bound, fmax((double)ord2f(kth), 0.0) + 1.0e-6);
      }
    };
    // The scan starts at a's own chunk: S is in detection order, so a's neighbours in the list are mostly detections of
    // the same frame -- near it in space -- and the bound is tight after the first evaluation round.
    constexpr int UNR = 4;  // chunks of 32 candidates per iteration: their loads are in flight together
    const uint32_t n_chunks = (n + 31) >> 5, c0 = ia >> 5;
    const float ax = (float)ga[0], ay = (float)ga[1], az = (float)ga[2], atr = __double2float_ru(ga[3]);
    for (uint32_t c = 0; c < n_chunks; c += UNR) {
      float4 g4[UNR];
      uint32_t idx[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        uint32_t ch = c0 + c + u;
        ch = ch >= n_chunks ? ch - n_chunks : ch;
        idx[u] = c + u < n_chunks ? (ch << 5) + lane : 0xFFFFFFFFu;
        g4[u] = m.eg_f4[min(idx[u], n - 1)];
      }
      const float fb = bound < 1.0e30 ? __double2float_ru(bound) : 3.0e38f;
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        const uint32_t ib = idx[u];
        // fp32 version of the lower bound, kept conservative: each |dmu_i| is reduced by the rounding error of the two
        // coordinates (2^-24 relative each), the traces are rounded up, 0.99 covers the arithmetic
        const float d0 = fmaxf(fabsf(ax - g4[u].x) - 1.2e-7f * (fabsf(ax) + fabsf(g4[u].x)), 0.f);
        const float d1 = fmaxf(fabsf(ay - g4[u].y) - 1.2e-7f * (fabsf(ay) + fabsf(g4[u].y)), 0.f);
        const float d2 = fmaxf(fabsf(az - g4[u].z) - 1.2e-7f * (fabsf(az) + fabsf(g4[u].z)), 0.f);
        const bool pass = ib < n && ib != ia && !(0.99f * (d0 * d0 + d1 * d1 + d2 * d2) > fb * (4.0f * (atr + g4[u].w)));
        const unsigned ball = __ballot_sync(0xFFFFFFFFu, pass);
        if (pass) queue[qn + __popc(ball & lt_mask)] = ib;
        qn += __popc(ball);
        if (qn >= 32) {
          __syncwarp();
          evaluate(32);
          const uint32_t rest = qn - 32;
          const uint32_t moved = (uint32_t)lane < rest ? queue[32 + lane] : 0u;
          __syncwarp();
          if ((uint32_t)lane < rest) queue[lane] = moved;
          qn = rest;
        }
      }
    }
    __syncwarp();
    if (qn) evaluate(qn);
    __syncwarp();
    unsigned long long mine = KEY_MAX, med = KEY_MAX;
#pragma unroll
    for (int r = 0; r < K; ++r) {
      if (r < kk) {
        const unsigned long long w = warp_pop_min<K>(top);
        if (lane == r) mine = w;
        if (r == (kk - 1) / 2) med = w;
      }
    }
    if (lane < kk && mine != KEY_MAX) {
      const float d = ord2f((int)((uint32_t)(mine >> 32) ^ 0x80000000u));
      const float dm = ord2f((int)((uint32_t)(med >> 32) ^ 0x80000000u));
      if (d <= __fmul_rn(m.edge_cutoff, dm)) edge_touch(m, m.eg_list[ia], (uint32_t)mine, call);
    }
  }
}

// export: the live edges, compacted (order arbitrary; the host sorts them), weights decayed to `call`
__global__ void edge_export_kernel(DevMap m, uint32_t call, uint32_t *out_a, uint32_t *out_b, double *out_w, uint32_t cap, uint32_t *count) {
  for (uint32_t h = blockIdx.x * blockDim.x + threadIdx.x; h <= m.ed_mask; h += gridDim.x * blockDim.x) {
    const unsigned long long k = m.ed_key[h];
    if (k == KEY_MAX) continue;
    const uint32_t pos = atomicAdd(count, 1u);
    if (pos >= cap) continue;
    out_a[pos] = (uint32_t)(k >> 32), out_b[pos] = (uint32_t)k;
    out_w[pos] = m.ed_w[h] * pow((double)m.edge_decay, (double)(call - m.ed_t[h]));
  }
}

}  // namespace

void configure_edge_kernels() {  // same shared-memory carve-out as every kernel that may run beside the similarity CTAs
  const int pref = (int)cudaSharedmemCarveoutMaxShared;
  cudaFuncSetAttribute(edge_knn_kernel<4>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(edge_knn_kernel<16>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
}

int launch_edges(const DevMap &m, const CallArgs &a, uint32_t call, cudaStream_t s) {
  if (a.M == 0 || m.edges_k <= 0) return 0;
  const int grid = min((a.M + KNN_WARPS - 1) / KNN_WARPS, m.num_sms * 16);  // |S| <= M; one warp per member
  if (m.edges_k <= 4)
    launch_pdl(edge_knn_kernel<4>, dim3(grid), dim3(KNN_THREADS), 0, s, m, call);
  else
    launch_pdl(edge_knn_kernel<16>, dim3(grid), dim3(KNN_THREADS), 0, s, m, call);
  return 1;
}

int launch_edge_export(const DevMap &m, uint32_t call, uint32_t *out_a, uint32_t *out_b, double *out_w, uint32_t cap, uint32_t *count,
                       cudaStream_t s) {
  edge_export_kernel<<<m.num_sms * 4, 256, 0, s>>>(m, call, out_a, out_b, out_w, cap, count);
  return 1;
}

}  // namespace farm
