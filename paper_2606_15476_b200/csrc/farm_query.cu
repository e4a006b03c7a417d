// farm_query.cu -- retrieval-side scoring over the finished memory (rules Q1-Q5).
//   PAPER.md:366 "Candidate retrieval": the whole pool of live entities is ranked by reciprocal-rank fusion, each
//     channel contributing w / (mu + rank) with mu = 5, over four query channels in three embedding spaces
//     (w = 1.0, 0.5, 0.75, 1.0).
//   PAPER.md:367 "Predicate evaluation": closed forms over the entity centroids -- Near: Gaussian of the inter-centroid
//     distance with sigma = 0.5 m, NextTo: sigma = 1.0 m, Closest / Farthest: 1 / (|rank - r*| + 1); landmarks bound
//     greedily to their top-scoring entity.
//   PAPER.md:368 "Composite scoring": s = s_sem * ((1 - w) + w * gbar), w = 0.5, gbar = geometric mean of the predicate
//     scores, s_sem scaled by 0.3 when the entity's class differs from the parsed target class.
// The three per-entity embedding matrices, the class ids and the query vectors are INPUTS (the encoders and the parser
// are out of scope, as the detector is for the mapper).  Every step runs in the kernels below; the host code only
// orders them.
#include <cmath>
#include <string>
#include <vector>

#include "farm_internal.cuh"

namespace farm {
namespace {

constexpr int QT = 256;
constexpr double RRF_MU = 5.0;
__constant__ double c_rrf_w[4] = {1.0, 0.5, 0.75, 1.0};

// order-preserving images: a larger key is a better rank
__device__ __forceinline__ unsigned long long key_of_float_desc(float v) {
  return (unsigned long long)((uint32_t)f2ord(v) ^ 0x80000000u) << 32;
}
__device__ __forceinline__ unsigned long long key_of_double_asc(double v) {  // smaller v = larger key
  long long i = __double_as_longlong(-v);
  i ^= (i >> 63) & 0x7FFFFFFFFFFFFFFFll;
  return (unsigned long long)i ^ 0x8000000000000000ull;
}

// liveness and centroid of every entity: the Gaussian mean where the entity has one (FARM_OPT_GAUSSIAN), else the
// centre of its AABB.  An entity is live while it holds observations (absorbed entities hold none).
__global__ void query_entities_kernel(DevMap m, uint32_t N, uint8_t *alive, float *cen, uint32_t *n_live) {
  const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= N) return;
  const bool live = m.n_obs[o] > 0;
  alive[o] = live ? 1 : 0;
  float c[3] = {0.f, 0.f, 0.f};
  if (live) {
    if (m.obj_gw && m.obj_gw[o] > 0.0) {
      for (int k = 0; k < 3; ++k) c[k] = (float)(m.obj_gm[(size_t)o * 9 + k] / m.obj_gw[o]);
    } else {
      for (int k = 0; k < 3; ++k) c[k] = (float)(0.5 * ((double)ord2f(m.aabb[o * 6 + k]) + (double)ord2f(m.aabb[o * 6 + 3 + k])));
    }
    atomicAdd(n_live, 1u);
  }
  for (int k = 0; k < 3; ++k) cen[3 * (size_t)o + k] = c[k];
}

// inverse norms of the query vectors (one warp each)
__global__ void query_norms_kernel(const float *q, const int *off, const int *len, int n_vec, float *inv_norm) {
  const int w = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (w >= n_vec) return;
  float s = 0.f;
  for (int i = lane; i < len[w]; i += 32) s = fmaf(q[off[w] + i], q[off[w] + i], s);
  for (int sft = 16; sft; sft >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, sft);
  if (lane == 0) inv_norm[w] = s > 0.f ? 1.0f / sqrtf(s) : 0.f;
}

// Q1: cosine (R15 arithmetic: explicit norms, clamp) of every entity row of one embedding space with the query vectors
// that live in that space.  One warp per entity; the row is read once (128-bit loads when the layout allows) and every
// query vector is applied to it.  vec_id[k] = index of the k-th query vector of this space; out [n_vec_total, N].
constexpr int MAX_QV = 16;
template <typename T>
__global__ void __launch_bounds__(QT) query_cos_kernel(const T *__restrict__ emb, int d, uint32_t N, const uint8_t *alive,
                                                       const float *__restrict__ q, const int *__restrict__ off,
                                                       const float *__restrict__ q_inv, const int *__restrict__ vec_id, int n_vec,
                                                       float *__restrict__ out) {
  const uint32_t o = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (o >= N || !alive[o]) return;
  const T *row = emb + (size_t)o * d;
  float acc[MAX_QV], nn = 0.f;
#pragma unroll
  for (int k = 0; k < MAX_QV; ++k) acc[k] = 0.f;
  constexpr int VE = 16 / sizeof(T);
  if ((d % VE) == 0 && (((uintptr_t)emb) & 15) == 0) {
    for (int i = lane * VE; i < d; i += 32 * VE) {
      const uint4 w = __ldcs(reinterpret_cast<const uint4 *>(row + i));
      const T *e = reinterpret_cast<const T *>(&w);
      float x[VE];
#pragma unroll
      for (int t = 0; t < VE; ++t) x[t] = to_f32<T>(e[t]), nn = fmaf(x[t], x[t], nn);
#pragma unroll
      for (int k = 0; k < MAX_QV; ++k)
        if (k < n_vec) {
          const float *qv = q + off[vec_id[k]] + i;
#pragma unroll
          for (int t = 0; t < VE; ++t) acc[k] = fmaf(x[t], __ldg(qv + t), acc[k]);
        }
    }
  } else {
    for (int i = lane; i < d; i += 32) {
      const float x = to_f32<T>(row[i]);
      nn = fmaf(x, x, nn);
#pragma unroll
      for (int k = 0; k < MAX_QV; ++k)
        if (k < n_vec) acc[k] = fmaf(x, __ldg(q + off[vec_id[k]] + i), acc[k]);
    }
  }
  for (int sft = 16; sft; sft >>= 1) nn += __shfl_xor_sync(0xFFFFFFFFu, nn, sft);
  const float ib = nn > 0.f ? 1.0f / sqrtf(nn) : 0.f;
#pragma unroll
  for (int k = 0; k < MAX_QV; ++k)
    if (k < n_vec) {
      float a = acc[k];
      for (int sft = 16; sft; sft >>= 1) a += __shfl_xor_sync(0xFFFFFFFFu, a, sft);
      if (lane == 0) out[(size_t)vec_id[k] * N + o] = fminf(1.f, fmaxf(-1.f, a * q_inv[vec_id[k]] * ib));
    }
}

// keys of the cosine arrays (descending value, ties -> lower id)
__global__ void cos_keys_kernel(const float *cosv, size_t n, unsigned long long *keys) {
  const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (i < n) keys[i] = key_of_float_desc(cosv[i]);
}

// rank[a][o] = 1 + number of live entities that come before o in array a: a larger key, or an equal key and a lower id.
// One thread per entity, the array streamed through shared memory.  (Exact and deterministic; O(N^2) per array.)
__global__ void __launch_bounds__(QT) rank_kernel(const unsigned long long *keys, const uint8_t *alive, uint32_t N, uint32_t *rank) {
  __shared__ unsigned long long sk[QT];
  __shared__ uint8_t sa[QT];
  const unsigned long long *k = keys + (size_t)blockIdx.y * N;
  const uint32_t o = blockIdx.x * QT + threadIdx.x;
  const bool mine = o < N && alive[o];
  const unsigned long long kv = mine ? k[o] : 0ull;
  uint32_t cnt = 0;
  for (uint32_t base = 0; base < N; base += QT) {
    const uint32_t i = base + threadIdx.x;
    sk[threadIdx.x] = i < N ? k[i] : 0ull;
    sa[threadIdx.x] = i < N ? alive[i] : 0;
    __syncthreads();
    const uint32_t lim = min((uint32_t)QT, N - base);
    for (uint32_t t = 0; t < lim; ++t) {
      const unsigned long long ot = sk[t];
      cnt += (sa[t] && (ot > kv || (ot == kv && base + t < o))) ? 1u : 0u;
    }
    __syncthreads();
  }
  if (o < N) rank[(size_t)blockIdx.y * N + o] = mine ? cnt + 1 : 0u;
}

// Q2: fused rank score of every variable (0 = target, 1.. = landmarks): sum_c w_c / (mu + rank_c)
__global__ void fuse_kernel(const uint32_t *rank, const uint8_t *alive, uint32_t N, int n_var, double *fused) {
  const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= N) return;
  for (int v = 0; v < n_var; ++v) {
    double s = 0.0;
    if (alive[o])
      for (int c = 0; c < 4; ++c) s += c_rrf_w[c] / (RRF_MU + (double)rank[(size_t)(v * 4 + c) * N + o]);
    fused[(size_t)v * N + o] = s;
  }
}

// Q4 landmark binding: the live entity with the largest fused score of landmark variable v (ties -> lowest id); one CTA
__global__ void __launch_bounds__(1024) bind_landmark_kernel(const double *fused, const uint8_t *alive, uint32_t N, int v, int32_t *landmark) {
  __shared__ double sv[1024];
  __shared__ int si[1024];
  double best = -1.0;
  int bi = -1;
  for (uint32_t o = threadIdx.x; o < N; o += 1024)
    if (alive[o]) {
      const double s = fused[(size_t)v * N + o];
      if (bi < 0 || s > best) best = s, bi = (int)o;
    }
  sv[threadIdx.x] = best, si[threadIdx.x] = bi;
  __syncthreads();
  for (int st = 512; st; st >>= 1) {
    if ((int)threadIdx.x < st) {
      const double s2 = sv[threadIdx.x + st];
      const int i2 = si[threadIdx.x + st];
      if (i2 >= 0 && (si[threadIdx.x] < 0 || s2 > sv[threadIdx.x] || (s2 == sv[threadIdx.x] && i2 < si[threadIdx.x])))
        sv[threadIdx.x] = s2, si[threadIdx.x] = i2;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) landmark[v - 1] = si[0];
}

// inter-centroid distance of every entity to the landmark of predicate p (double, one rounded operation at a time)
__global__ void dist_kernel(const float *cen, const int32_t *landmark, int p, uint32_t N, double *dist, unsigned long long *keys) {
  const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= N) return;
  const int lm = landmark[p];
  double d2 = 0.0;
  if (lm >= 0)
    for (int k = 0; k < 3; ++k) {
      const double d = __dsub_rn((double)cen[3 * (size_t)o + k], (double)cen[3 * (size_t)lm + k]);
      d2 = __dadd_rn(d2, __dmul_rn(d, d));
    }
  const double ds = sqrt(d2);
  dist[(size_t)p * N + o] = ds;
  keys[(size_t)p * N + o] = key_of_double_asc(ds);
}

// Q4 + Q5: predicate scores, geometric mean, class factor, composite score
__global__ void score_kernel(const double *fused, const uint8_t *alive, const int32_t *cls, int target_class, uint32_t N, int P,
                             const int32_t *pred_type, const int32_t *landmark, const double *dist, const uint32_t *drank,
                             const uint32_t *n_live, float *s_sem, float *gbar, float *s, unsigned long long *skeys) {
  const uint32_t o = blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= N) return;
  double ss = 0.0, gb = 0.0, sc = 0.0;
  if (alive[o]) {
    ss = fused[o];
    if (target_class >= 0 && cls && cls[o] != target_class) ss *= 0.3;  // Q3 soft class factor
    double logsum = 0.0;
    bool zero = false;
    int used = 0;
    for (int p = 0; p < P; ++p) {
      if (landmark[p] < 0) continue;
      ++used;
      const double d = dist[(size_t)p * N + o];
      const int r = (int)drank[(size_t)p * N + o];
      double g;
      switch (pred_type[p]) {
        case 0: g = exp(-d * d / (2.0 * 0.5 * 0.5)); break;                 // Near, sigma = 0.5 m
        case 1: g = exp(-d * d / (2.0 * 1.0 * 1.0)); break;                 // NextTo, sigma = 1.0 m
        case 2: g = 1.0 / (double)(abs(r - 1) + 1); break;                  // Closest: r* = 1
        default: g = 1.0 / (double)(abs(r - (int)*n_live) + 1); break;      // Farthest: r* = number of live entities
      }
      if (g > 0.0) logsum += log(g); else zero = true;
    }
    (void)used;
    gb = P == 0 ? 1.0 : (zero ? 0.0 : exp(logsum / (double)P));
    sc = ss * ((1.0 - 0.5) + 0.5 * gb);                                     // Q5, w = 0.5
  }
  s_sem[o] = (float)ss, gbar[o] = (float)gb, s[o] = (float)sc;
  skeys[o] = key_of_float_desc((float)sc);
}

// top-K by (score descending, id ascending): K rounds of a block-wide arg-max below the previous pick; one CTA
__global__ void __launch_bounds__(1024) topk_kernel(const unsigned long long *skeys, const uint8_t *alive, uint32_t N, int K,
                                                    int32_t *top_ids) {
  __shared__ unsigned long long sk[1024];
  __shared__ unsigned long long s_last;
  if (threadIdx.x == 0) s_last = ~0ull;
  __syncthreads();
  for (int r = 0; r < K; ++r) {
    const unsigned long long last = s_last;
    unsigned long long best = 0ull;  // full key = score key | (~id): unique per entity, never 0 for a live one
    for (uint32_t o = threadIdx.x; o < N; o += 1024)
      if (alive[o]) {
        const unsigned long long k = skeys[o] | (unsigned long long)(0xFFFFFFFFu - o);
        if (k < last && k > best) best = k;
      }
    sk[threadIdx.x] = best;
    __syncthreads();
    for (int st = 512; st; st >>= 1) {
      if ((int)threadIdx.x < st && sk[threadIdx.x + st] > sk[threadIdx.x]) sk[threadIdx.x] = sk[threadIdx.x + st];
      __syncthreads();
    }
    if (threadIdx.x == 0) {
      top_ids[r] = sk[0] ? (int32_t)(0xFFFFFFFFu - (uint32_t)sk[0]) : -1;
      s_last = sk[0] ? sk[0] : 0ull;
    }
    __syncthreads();
  }
}

struct DevBuf {  // frees what a query allocated, whatever path the call leaves by
  std::vector<void *> p;
  ~DevBuf() {
    for (void *q : p) cudaFree(q);
  }
  template <typename T>
  bool get(T **out, size_t n) {
    void *q = nullptr;
    if (cudaMalloc(&q, (n ? n : 1) * sizeof(T)) != cudaSuccess) return false;
    p.push_back(q);
    *out = (T *)q;
    return true;
  }
};

}  // namespace

// returns 0 or a FARM_ERR_* code; err receives a description
int run_query(const DevMap &m, cudaStream_t st, uint32_t N, const void *const emb[3], const int dim[3], int emb_dtype, const int32_t *cls,
              const float *q_target, int target_class, int P, const int32_t *pred_type, const float *q_landmarks, int topk,
              int32_t *top_ids, float *top_scores, int32_t *landmarks, float *s_sem, float *gbar, float *s, long long *launches,
              std::string *err) {
#define QC(expr)                                                          \
  do {                                                                    \
    cudaError_t e_ = (expr);                                              \
    if (e_ != cudaSuccess) {                                              \
      *err = std::string(#expr) + ": " + cudaGetErrorString(e_);         \
      return FARM_ERR_CUDA;                                               \
    }                                                                     \
  } while (0)
  const int n_var = 1 + P, n_vec = 4 * n_var;
  const int qlen = 2 * dim[0] + dim[1] + dim[2];
  static const int space_of[4] = {0, 0, 1, 2};
  // query vectors: variable-major, channel-minor
  std::vector<float> hq((size_t)n_var * qlen);
  std::vector<int> hoff(n_vec), hlen(n_vec);
  for (int v = 0; v < n_var; ++v) {
    const float *src = v == 0 ? q_target : q_landmarks + (size_t)(v - 1) * qlen;
    std::copy(src, src + qlen, hq.begin() + (size_t)v * qlen);
    const int o4[4] = {0, dim[0], 2 * dim[0], 2 * dim[0] + dim[1]};
    for (int c = 0; c < 4; ++c) hoff[v * 4 + c] = v * qlen + o4[c], hlen[v * 4 + c] = dim[space_of[c]];
  }
  DevBuf B;
  float *dq, *dqinv, *dcos, *dcen, *dssem, *dgbar, *ds;
  int *doff, *dlen, *dvec;
  int32_t *dptype, *dlm, *dtop;
  uint8_t *dalive;
  uint32_t *dnlive, *drank, *ddrank;
  unsigned long long *dkeys, *ddkeys, *dskeys;
  double *dfused, *ddist;
  const size_t Nn = N ? N : 1;
  if (!B.get(&dq, hq.size()) || !B.get(&dqinv, n_vec) || !B.get(&dcos, (size_t)n_vec * Nn) || !B.get(&dcen, 3 * Nn) ||
      !B.get(&dssem, Nn) || !B.get(&dgbar, Nn) || !B.get(&ds, Nn) || !B.get(&doff, n_vec) || !B.get(&dlen, n_vec) ||
      !B.get(&dvec, 3 * MAX_QV) || !B.get(&dptype, P + 1) || !B.get(&dlm, P + 1) || !B.get(&dtop, topk + 1) ||
      !B.get(&dalive, Nn) || !B.get(&dnlive, 1) || !B.get(&drank, (size_t)n_vec * Nn) || !B.get(&ddrank, (size_t)(P + 1) * Nn) ||
      !B.get(&dkeys, (size_t)n_vec * Nn) || !B.get(&ddkeys, (size_t)(P + 1) * Nn) || !B.get(&dskeys, Nn) ||
      !B.get(&dfused, (size_t)n_var * Nn) || !B.get(&ddist, (size_t)(P + 1) * Nn)) {
    *err = "query: device allocation failed";
    return FARM_ERR_CUDA;
  }
  QC(cudaMemcpyAsync(dq, hq.data(), hq.size() * 4, cudaMemcpyHostToDevice, st));
  QC(cudaMemcpyAsync(doff, hoff.data(), n_vec * 4, cudaMemcpyHostToDevice, st));
  QC(cudaMemcpyAsync(dlen, hlen.data(), n_vec * 4, cudaMemcpyHostToDevice, st));
  if (P) QC(cudaMemcpyAsync(dptype, pred_type, P * 4, cudaMemcpyHostToDevice, st));
  QC(cudaMemsetAsync(dnlive, 0, 4, st));
  QC(cudaMemsetAsync(dcos, 0, (size_t)n_vec * Nn * 4, st));
  QC(cudaMemsetAsync(dlm, 0xFF, (P + 1) * 4, st));
  long long nl = 0;
  if (N) {
    const unsigned gb = (N + QT - 1) / QT;
    query_entities_kernel<<<gb, QT, 0, st>>>(m, N, dalive, dcen, dnlive), ++nl;
    query_norms_kernel<<<(n_vec * 32 + QT - 1) / QT, QT, 0, st>>>(dq, doff, dlen, n_vec, dqinv), ++nl;
    // per space: the query vectors that live in it
    std::vector<int> hvec(3 * MAX_QV, 0);
    int cnt[3] = {0, 0, 0};
    for (int v = 0; v < n_var; ++v)
      for (int c = 0; c < 4; ++c) hvec[space_of[c] * MAX_QV + cnt[space_of[c]]++] = v * 4 + c;
    QC(cudaMemcpyAsync(dvec, hvec.data(), hvec.size() * 4, cudaMemcpyHostToDevice, st));
    const unsigned gw = (unsigned)(((size_t)N * 32 + QT - 1) / QT);
    for (int sp = 0; sp < 3; ++sp) {
      if (emb_dtype == FARM_DTYPE_F32)
        query_cos_kernel<float><<<gw, QT, 0, st>>>((const float *)emb[sp], dim[sp], N, dalive, dq, doff, dqinv, dvec + sp * MAX_QV, cnt[sp], dcos);
      else if (emb_dtype == FARM_DTYPE_F16)
        query_cos_kernel<__half><<<gw, QT, 0, st>>>((const __half *)emb[sp], dim[sp], N, dalive, dq, doff, dqinv, dvec + sp * MAX_QV, cnt[sp], dcos);
      else
        query_cos_kernel<__nv_bfloat16><<<gw, QT, 0, st>>>((const __nv_bfloat16 *)emb[sp], dim[sp], N, dalive, dq, doff, dqinv, dvec + sp * MAX_QV, cnt[sp], dcos);
      ++nl;
    }
    const size_t nk = (size_t)n_vec * N;
    cos_keys_kernel<<<(unsigned)((nk + QT - 1) / QT), QT, 0, st>>>(dcos, nk, dkeys), ++nl;
    rank_kernel<<<dim3(gb, n_vec), QT, 0, st>>>(dkeys, dalive, N, drank), ++nl;
    fuse_kernel<<<gb, QT, 0, st>>>(drank, dalive, N, n_var, dfused), ++nl;
    for (int p = 0; p < P; ++p) {
      bind_landmark_kernel<<<1, 1024, 0, st>>>(dfused, dalive, N, p + 1, dlm), ++nl;
      dist_kernel<<<gb, QT, 0, st>>>(dcen, dlm, p, N, ddist, ddkeys), ++nl;
    }
    if (P) rank_kernel<<<dim3(gb, P), QT, 0, st>>>(ddkeys, dalive, N, ddrank), ++nl;
    score_kernel<<<gb, QT, 0, st>>>(dfused, dalive, cls, target_class, N, P, dptype, dlm, ddist, ddrank, dnlive, dssem, dgbar, ds, dskeys), ++nl;
    if (topk) topk_kernel<<<1, 1024, 0, st>>>(dskeys, dalive, N, topk, dtop), ++nl;
  }
  QC(cudaGetLastError());
  std::vector<int32_t> htop(topk + 1, -1);
  std::vector<float> hs(Nn, 0.f);
  if (N) {
    if (topk) QC(cudaMemcpyAsync(htop.data(), dtop, topk * 4, cudaMemcpyDeviceToHost, st));
    QC(cudaMemcpyAsync(hs.data(), ds, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
    if (s_sem) QC(cudaMemcpyAsync(s_sem, dssem, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
    if (gbar) QC(cudaMemcpyAsync(gbar, dgbar, (size_t)N * 4, cudaMemcpyDeviceToHost, st));
    if (landmarks && P) QC(cudaMemcpyAsync(landmarks, dlm, P * 4, cudaMemcpyDeviceToHost, st));
  }
  QC(cudaStreamSynchronize(st));
  for (int k = 0; k < topk; ++k) {
    if (top_ids) top_ids[k] = htop[k];
    if (top_scores) top_scores[k] = htop[k] >= 0 ? hs[htop[k]] : 0.f;
  }
  if (s)
    for (uint32_t o = 0; o < N; ++o) s[o] = hs[o];
  if (!N && landmarks)
    for (int p = 0; p < P; ++p) landmarks[p] = -1;
  if (launches) *launches += nl;
  return FARM_OK;
#undef QC
}

}  // namespace farm
