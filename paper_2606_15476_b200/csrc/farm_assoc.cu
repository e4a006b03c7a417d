// farm_assoc.cu -- step 5: candidate scoring, association (argmax / threshold / spawn) and merge.
//   R10, R17-R20 (score, strict threshold, ids in detection index order; BASELINE.json rule)
//   R12 (voxel commit, lowest detection index wins), R21 (count-weighted descriptor mean),
//   R22 (AABB), R23 (view evidence).
#include "farm_internal.cuh"

namespace farm {
FARM_TRACE_TABLE(farm_trace_assoc)  // 0 first CTA past pdl_wait, 1 scoring over (last CTA), 3 scan start (similarity done), 5 scan end, 2 merge start, 7 merge warps end
namespace {

constexpr uint32_t NONE32 = 0xFFFFFFFFu;

// ---- paper-faithful geometry (rules G1-G4): Gaussian from sufficient statistics, Hellinger distance (double)
__device__ __forceinline__ void gaussian_of(double w, const double *g, double mu[3], double c[6]) {
  mu[0] = g[0] / w, mu[1] = g[1] / w, mu[2] = g[2] / w;
  c[0] = g[3] / w - mu[0] * mu[0], c[1] = g[4] / w - mu[0] * mu[1], c[2] = g[5] / w - mu[0] * mu[2];
  c[3] = g[6] / w - mu[1] * mu[1], c[4] = g[7] / w - mu[1] * mu[2], c[5] = g[8] / w - mu[2] * mu[2];
}
__device__ __forceinline__ double det_sym3(const double c[6]) {
  return c[0] * (c[3] * c[5] - c[4] * c[4]) - c[1] * (c[1] * c[5] - c[4] * c[2]) + c[2] * (c[1] * c[4] - c[3] * c[2]);
}
// G3: H = sqrt(1 - BC), BC = |S1|^(1/4) |S2|^(1/4) / |Sb|^(1/2) * exp(-dmu^T Sb^-1 dmu / 8),
// S = Sigma + eps2 I, Sb = (S1 + S2) / 2
__device__ float hellinger_gauss(const double mu1[3], double s1[6], const double mu2[3], double s2[6], double eps2) {
  s1[0] += eps2, s1[3] += eps2, s1[5] += eps2;
  s2[0] += eps2, s2[3] += eps2, s2[5] += eps2;
  double sb[6];
#pragma unroll
  for (int k = 0; k < 6; ++k) sb[k] = 0.5 * (s1[k] + s2[k]);
  const double db = det_sym3(sb);
  const double a00 = sb[3] * sb[5] - sb[4] * sb[4], a01 = sb[2] * sb[4] - sb[1] * sb[5], a02 = sb[1] * sb[4] - sb[2] * sb[3];
  const double a11 = sb[0] * sb[5] - sb[2] * sb[2], a12 = sb[1] * sb[2] - sb[0] * sb[4], a22 = sb[0] * sb[3] - sb[1] * sb[1];
  const double d0 = mu1[0] - mu2[0], d1 = mu1[1] - mu2[1], d2 = mu1[2] - mu2[2];
  const double q = (d0 * (a00 * d0 + a01 * d1 + a02 * d2) + d1 * (a01 * d0 + a11 * d1 + a12 * d2) + d2 * (a02 * d0 + a12 * d1 + a22 * d2)) / db;
  const double bc = sqrt(sqrt(det_sym3(s1) * det_sym3(s2))) / sqrt(db) * exp(-0.125 * q);
  const double h2 = 1.0 - bc;
  return h2 > 0.0 ? (float)sqrt(h2) : 0.f;
}

// G4: Hellinger distance between detection j and the entity it was matched to, as that entity was at entry (R2).
// Out of line so that its double-precision temporaries do not inflate the association kernel's register budget
// (512 threads x <= 64 registers must fit beside the similarity CTA).
__device__ __noinline__ void match_hellinger(const double *det_gm, const double *obj_gw, const double *obj_gm, float *hell,
                                             float eps2, int j, int32_t target, uint32_t npx) {
  const double wo = obj_gw[target];
  if (!(wo > 0.0)) return;
  double gd[9], go[9], mu_d[3], c_d[6], mu_o[3], c_o[6];
#pragma unroll
  for (int k = 0; k < 9; ++k) gd[k] = __ldcg(&det_gm[(size_t)j * 9 + k]), go[k] = obj_gm[(size_t)target * 9 + k];
  gaussian_of((double)npx, gd, mu_d, c_d);
  gaussian_of(wo, go, mu_o, c_o);
  hell[j] = hellinger_gauss(mu_d, c_d, mu_o, c_o, (double)eps2);
}

// W1: entity t received a detection in this call and carries the Gaussian (w, g) after the merge: append it to S with
// its regularised Gaussian for the kNN kernel (farm_edges.cu; row of 12 doubles: mu, trace, S = Sigma + eps2 I, ln |S|).
// The order of S is arbitrary; nothing downstream depends on it.
__device__ __noinline__ void edge_member(const DevMap &m, uint32_t t, double w, const double *g) {
  const uint32_t pos = atomicAdd(&m.counters[8], 1u);
  if (pos >= m.max_det) return;  // cannot happen: one member per detection at most
  const double eps2 = (double)m.eps2;
  const double mx = g[0] / w, my = g[1] / w, mz = g[2] / w;
  double s[6] = {g[3] / w - mx * mx + eps2, g[4] / w - mx * my, g[5] / w - mx * mz,
                 g[6] / w - my * my + eps2, g[7] / w - my * mz, g[8] / w - mz * mz + eps2};
  double *o = m.eg_gauss + (size_t)pos * 12;
  o[0] = mx, o[1] = my, o[2] = mz, o[3] = s[0] + s[3] + s[5];
#pragma unroll
  for (int k = 0; k < 6; ++k) o[4 + k] = s[k];
  o[10] = log(det_sym3(s));
  m.eg_f4[pos] = make_float4((float)mx, (float)my, (float)mz, __double2float_ru(o[3]));  // the kNN scan's fp32 view (trace rounded up)
  m.eg_list[pos] = t;
}

// V1-V2: the view of one merged detection, offered to its object's retained set.  fp32, one rounded
// operation at a time: the comparisons decide which views are kept and the oracle takes them in the same precision.
__device__ __noinline__ void offer_view_record(const DevMap &m, int32_t t, const farm_view &v) {
  const float dist = v.dist;
  farm_view *set = m.views + (size_t)t * m.views_k;
  const uint32_t n = m.view_cnt[t];
  bool fresh = true;
  float closest = __int_as_float(0x7F800000);
  uint32_t far = 0;
  for (uint32_t i = 0; i < n; ++i) {
    const float dot = __fadd_rn(__fadd_rn(__fmul_rn(v.dir[0], set[i].dir[0]), __fmul_rn(v.dir[1], set[i].dir[1])), __fmul_rn(v.dir[2], set[i].dir[2]));
    if (!(dot < m.view_cos)) fresh = false;
    closest = fminf(closest, set[i].dist);
    if (set[i].dist > set[far].dist) far = i;
  }
  const bool closer = n > 0 && dist < __fmul_rn(m.view_closer, closest);
  if (n > 0 && !fresh && !closer) return;
  if (n < (uint32_t)m.views_k) {
    set[n] = v;
    m.view_cnt[t] = n + 1;
  } else if (dist < set[far].dist) {
    set[far] = v;
  }
}
__device__ __noinline__ void offer_view(const DevMap &m, int32_t t, const int *box, const float *cam, int32_t frame, int32_t det,
                                        uint32_t n_px) {
  float d[3];
#pragma unroll
  for (int k = 0; k < 3; ++k) d[k] = __fsub_rn(__fmul_rn(0.5f, __fadd_rn(ord2f(box[k]), ord2f(box[3 + k]))), cam[k]);
  const float d2 = __fadd_rn(__fadd_rn(__fmul_rn(d[0], d[0]), __fmul_rn(d[1], d[1])), __fmul_rn(d[2], d[2]));
  const float dist = __fsqrt_rn(d2);
  if (!(dist > 0.f)) return;
  farm_view v;
  v.frame = frame, v.det = det, v.n_px = n_px, v.dist = dist;
#pragma unroll
  for (int k = 0; k < 3; ++k) v.cam[k] = cam[k], v.dir[k] = __fdiv_rn(d[k], dist);
  offer_view_record(m, t, v);
}

// U4 ("Entity-level merges ... absorbing the loser's covisibility, captions, view records, and identity
// history into the winner"): the scalar state of every loser of winner t goes into t -- voxel count, points, box, best
// view (R23 order), Gaussian statistics, retained views.  Run by one lane of t's merge leader BEFORE the call's
// detections are fused; the losers' descriptors enter the R21 fold and the losers are retired after it.
__device__ __noinline__ void absorb_losers(const DevMap &m, int32_t t, uint32_t nL) {
  for (uint32_t k = 0; k < nL; ++k) {
    if (m.winner[k] != (uint32_t)t) continue;
    const uint32_t L = m.loser[k];
    atomicAdd(&m.n_voxels[t], m.n_voxels[L]);  // commit CTAs add this call's new voxels concurrently
    m.n_voxels[L] = 0;
    m.n_points[t] += m.n_points[L];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      m.aabb[t * 6 + c] = min(m.aabb[t * 6 + c], m.aabb[L * 6 + c]);
      m.aabb[t * 6 + 3 + c] = max(m.aabb[t * 6 + 3 + c], m.aabb[L * 6 + 3 + c]);
    }
    const uint32_t pl = m.best_px[L], pt = m.best_px[t];
    if (pl > pt || (pl == pt && pl > 0 &&
                    (m.best_seq[L] < m.best_seq[t] || (m.best_seq[L] == m.best_seq[t] && m.best_det[L] < m.best_det[t])))) {
      m.best_px[t] = pl, m.best_seq[t] = m.best_seq[L], m.best_det[t] = m.best_det[L];
      for (int c = 0; c < 3; ++c) m.best_cam[t * 3 + c] = m.best_cam[L * 3 + c];
    }
    if (m.obj_gw) {
      m.obj_gw[t] += m.obj_gw[L];
      for (int c = 0; c < 9; ++c) m.obj_gm[(size_t)t * 9 + c] += m.obj_gm[(size_t)L * 9 + c];
    }
    if (m.views)
      for (uint32_t i = 0; i < m.view_cnt[L]; ++i) offer_view_record(m, t, m.views[(size_t)L * m.views_k + i]);
  }
}
// the absorbed entities stay as dead ids: no observations, no voxels, zero descriptor (cosine 0 with everything)
__device__ __noinline__ void retire_loser(const DevMap &m, uint32_t L, int32_t t) {
  m.n_obs[L] = 0;
  m.n_points[L] = 0;
  m.inv_norm[L] = 0.f;
  for (int c = 0; c < 3; ++c) {
    m.aabb[L * 6 + c] = 0x7F800000;            // ordered image of +inf
    m.aabb[L * 6 + 3 + c] = (int)0x807FFFFF;   // ordered image of -inf
    m.best_cam[L * 3 + c] = 0.f;
  }
  m.best_px[L] = 0, m.best_seq[L] = 0, m.best_det[L] = 0;
  if (m.obj_gw) {
    m.obj_gw[L] = 0.0;
    for (int c = 0; c < 9; ++c) m.obj_gm[(size_t)L * 9 + c] = 0.0;
  }
  if (m.views) m.view_cnt[L] = 0;
  m.alias[L] = (uint32_t)t;
  m.leader[L] = NONE32;
}

// ---- U3: lock-free union-find over the match graph.  The root of a set is its smallest node; entities
// are numbered before detections (node of detection j = max_objects + j), so a component that holds an entity is won
// by its lowest-id entity and a component of detections only by its lowest detection.
__device__ __forceinline__ uint32_t uf_find(const uint32_t *p, uint32_t x) {
  for (;;) {
    const uint32_t q = __ldcg(&p[x]);
    if (q == x) return x;
    x = q;
  }
}
__device__ __forceinline__ void uf_union(uint32_t *p, uint32_t x, uint32_t y) {
  for (;;) {
    x = uf_find(p, x), y = uf_find(p, y);
    if (x == y) return;
    const uint32_t hi = max(x, y), lo = min(x, y);
    if (atomicCAS(&p[hi], hi, lo) == hi) return;
  }
}
__device__ __forceinline__ void add_edge(const DevMap &m, uint32_t j, uint32_t o) {  // U1: detection j retained entity o
  atomicOr(&m.det_flags[j], 1u);
  const uint32_t e = atomicAdd(&m.counters[5], 1u);
  if (e < m.edge_cap) m.edge_a[e] = m.max_objects + j, m.edge_b[e] = o; else atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
}

// H2-H3: one pair above the similarity prefilter -- Hellinger distance between the detection's and the
// entity's Gaussian, budget, g = 1 - H, score.  Out of line (double precision temporaries).
__device__ __noinline__ void hellinger_candidate(const DevMap &m, uint32_t d, uint32_t o, float cs) {
  const uint32_t npx = __ldcg(&m.det_npx[d]);
  if (npx == 0) return;  // R8: skipped detection
  float g = 0.f;
  const double wo = m.obj_gw[o];
  if (wo > 0.0) {
    double gd[9], go[9], mu_d[3], c_d[6], mu_o[3], c_o[6];
#pragma unroll
    for (int k = 0; k < 9; ++k) gd[k] = __ldcg(&m.det_gm[(size_t)d * 9 + k]), go[k] = m.obj_gm[(size_t)o * 9 + k];
    gaussian_of((double)npx, gd, mu_d, c_d);
    gaussian_of(wo, go, mu_o, c_o);
    const float hf = hellinger_gauss(mu_d, c_d, mu_o, c_o, (double)m.eps2);
    if (hf > m.hell_budget) return;  // H2: outside the budget -- not a candidate
    g = __fsub_rn(1.0f, hf);         // H3
  }
  const float score = __fadd_rn(__fmul_rn(m.w_geo, g), __fmul_rn(m.w_sem, cs));
  atomicMax(&m.best_cand[d], pack_score(score, o));
  if (m.corr && score > m.tau) add_edge(m, d, o);
}

// ---- U3 decisions (only with FARM_OPT_CORRESPONDENCE; run by the last CTA of cand_associate_kernel in place of the plain
// decision scan): union-find over the call's match graph, then per detection the component's root -- an entity (the
// detection is fused into the winner) or a detection (the component becomes one new entity, numbered in the order of
// its lowest detection, R20).  Entities that are not their component's root are recorded as (loser, winner) merges.
constexpr int CORR_THREADS = 512;
constexpr uint32_t LOSER_MARK = 0xFFFFFFFEu;
__device__ __noinline__ void correspondence_decide(const DevMap &m, const CallArgs &a, uint32_t N) {
  __shared__ uint32_t ws[32];
  __shared__ uint32_t s_running, s_matches, s_skipped;
  __shared__ unsigned long long s_uvox;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t nodeD = m.max_objects;
  uint32_t *p = m.uf_parent;
  if (tid == 0) s_running = 0, s_matches = 0, s_skipped = 0, s_uvox = 0ull;
  const uint32_t nE = min(__ldcg(&m.counters[5]), m.edge_cap), nDD = min(__ldcg(&m.counters[6]), m.edge_cap);
  for (uint32_t e = tid; e < nE; e += CORR_THREADS) uf_union(p, __ldcg(&m.edge_a[e]), __ldcg(&m.edge_b[e]));
  for (uint32_t e = tid; e < nDD; e += CORR_THREADS) {
    const uint32_t d = __ldcg(&m.dd_d[e]);
    if (!(__ldcg(&m.det_flags[d]) & 1u)) uf_union(p, nodeD + d, nodeD + __ldcg(&m.dd_e[e]));  // U2: only if d retained nothing
  }
  __threadfence();
  __syncthreads();
  // pass 1: roots; new entities for the components rooted at a detection, in index order
  uint32_t n_skipped = 0, nv_sum = 0, n_live = 0;
  for (int base = 0; base < a.M; base += CORR_THREADS) {
    const int j = base + tid;
    bool is_root = false;
    if (j < a.M) {
      nv_sum += __ldcg(&m.det_nv[j]);
      if (__ldcg(&m.det_npx[j]) == 0) {
        ++n_skipped;  // R8
      } else {
        ++n_live;
        is_root = uf_find(p, nodeD + j) == nodeD + (uint32_t)j;
      }
    }
    const unsigned b = __ballot_sync(0xFFFFFFFFu, is_root);
    if (lane == 0) ws[warp] = __popc(b);
    __syncthreads();
    uint32_t before = s_running, total = 0;
    for (int w = 0; w < CORR_THREADS / 32; ++w) {
      if (w < warp) before += ws[w];
      total += ws[w];
    }
    if (is_root) {
      const uint32_t id = N + before + __popc(b & ((1u << lane) - 1));
      if (id < m.max_objects) {
        m.det_newid[j] = id;
      } else {
        m.det_newid[j] = NONE32;
        atomicOr(m.err, ERR_OBJECT_CAPACITY);
      }
    }
    __syncthreads();
    if (tid == 0) s_running += total;
    __syncthreads();
  }
  __threadfence();
  __syncthreads();
  // pass 2: targets, scores, merge groups
  uint32_t n_new = 0;
  for (int j = tid; j < a.M; j += CORR_THREADS) {
    const uint32_t npx = __ldcg(&m.det_npx[j]);
    int32_t target = -1;
    uint32_t is_new = 0;
    float score = 0.f;
    if (npx != 0) {
      unsigned long long best = __ldcg(&m.best_cand[j]);
      const unsigned long long bd = __ldcg(&m.best_dense[j]);
      if (bd && m.geom == 0) {
        const float sd = __fadd_rn(__fmul_rn(m.w_geo, 0.f), __fmul_rn(m.w_sem, unpack_score(bd)));
        const unsigned long long pd = pack_score(sd, m.w_sem > 0.f ? unpack_id(bd) : 0u);
        best = pd > best ? pd : best;
      }
      if (best) {
        score = unpack_score(best);
        if (m.det_gm && score > m.tau) match_hellinger(m.det_gm, m.obj_gw, m.obj_gm, m.hell, m.eps2, j, (int32_t)unpack_id(best), npx);  // G4
      }
      const uint32_t r = uf_find(p, nodeD + (uint32_t)j);
      if (r < nodeD) {
        target = (int32_t)r;
      } else {
        const uint32_t id = __ldcg(&m.det_newid[r - nodeD]);
        if (id != NONE32) {
          target = (int32_t)id;
          is_new = r == nodeD + (uint32_t)j;  // the component's lowest detection creates the entity
          n_new += is_new;
        }
      }
    }
    m.assoc[j] = target;
    m.is_new[j] = (uint8_t)is_new;
    m.best_score[j] = score;
    if (target >= 0) {
      atomicMin(&m.leader[target], (uint32_t)j);
      atomicAdd(&m.grp_cnt[target], 1u);
    } else if (npx != 0) {
      ++n_skipped;  // object capacity: the detection is dropped
      --n_live;
    }
  }
  // losers: the entity end of every edge that is not its component's root
  for (uint32_t e = tid; e < nE; e += CORR_THREADS) {
    const uint32_t o = __ldcg(&m.edge_b[e]);
    const uint32_t r = uf_find(p, o);
    if (r != o && atomicCAS(&m.leader[o], NONE32, LOSER_MARK) == NONE32) {
      const uint32_t k = atomicAdd(&m.counters[7], 1u);
      m.loser[k] = o, m.winner[k] = r;  // at most one entry per entity: k < edge_cap
    }
  }
  n_skipped = __reduce_add_sync(0xFFFFFFFFu, n_skipped);
  nv_sum = __reduce_add_sync(0xFFFFFFFFu, nv_sum);
  n_live = __reduce_add_sync(0xFFFFFFFFu, n_live);
  n_new = __reduce_add_sync(0xFFFFFFFFu, n_new);
  if (lane == 0) {
    atomicAdd(&s_skipped, n_skipped);
    atomicAdd(&s_matches, n_live - n_new);
    atomicAdd(&s_uvox, (unsigned long long)nv_sum);
  }
  __threadfence();
  __syncthreads();
  // the forest returns to the identity for the next call
  for (uint32_t e = tid; e < nE; e += CORR_THREADS) p[m.edge_a[e]] = m.edge_a[e], p[m.edge_b[e]] = m.edge_b[e];
  for (uint32_t e = tid; e < nDD; e += CORR_THREADS) p[nodeD + m.dd_d[e]] = nodeD + m.dd_d[e], p[nodeD + m.dd_e[e]] = nodeD + m.dd_e[e];
  if (tid == 0) {
    uint32_t spawns = s_running;
    if (N + spawns > m.max_objects) spawns = m.max_objects - N;
    *m.n_objects = N + spawns;
    m.stats->matches = s_matches;
    m.stats->spawns = spawns;
    m.stats->skipped = s_skipped;
    m.stats->unique_voxels = s_uvox;
    atomicAdd(&m.totals->frames, (unsigned long long)a.F);
    atomicAdd(&m.totals->calls, 1ull);
    atomicAdd(&m.totals->valid_points, __ldcg(&m.stats->valid_points));
    atomicAdd(&m.totals->unique_voxels, s_uvox);
    atomicAdd(&m.totals->matches, (unsigned long long)s_matches);
    atomicAdd(&m.totals->spawns, (unsigned long long)spawns);
  }
}

// ---- candidate scoring + association, one launch.
// Phase 1 (all CTAs): one warp per non-zero overlap entry (d, o, c): cos(a_d, shadow_o) by a gather dot, g (R10),
//   score (R17), atomicMax into best_cand[d].
// Phase 2 (the last CTA to finish, found by a ticket): decisions for all detections (R18), new ids by an
//   exclusive scan in detection index order (R20), per-target leader / group size for the merge.
constexpr int CAND_THREADS = 512, CAND_WARPS = CAND_THREADS / 32, CAND_PER = 4;  // 512 x 52 registers fit beside the similarity CTA

template <typename T>
// 80 registers: 512 x 80 fits beside the similarity CTA (256 x 80) and the phase-1 dot products overlap its tail
__global__ void __maxnreg__(80) cand_associate_kernel(const __grid_constant__ DevMap m, const __grid_constant__ CallArgs a) {
  __shared__ uint32_t s_matches, s_skipped;
  __shared__ unsigned long long s_uvox;
  __shared__ bool s_last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_wait();     // launched with PDL behind the probe kernel: candidates and overlap counts are final from here on
  if (tid == 0) TRACE_MIN(farm_trace_assoc, a.seq, 0);
  if (a.split) {  // the row norms of this call come from the similarity kernel (other stream), not from prep
    if (tid == 0) spin_until(m.prep_done, a.prep_target, m.err);
    __syncthreads();
  }
  {
    const uint32_t n_cand = min(m.counters[1], m.cand_cap);
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    const int D = m.D;
    for (uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < n_cand; c += warps) {
      const uint32_t slot = m.cand_slot[c];
      const unsigned long long kv = m.cand_key[c];
      const uint32_t j = (uint32_t)(kv >> 32) & ((1u << DET_BITS) - 1);
      const uint32_t o32 = (uint32_t)kv;
      const bool dd = (o32 & DD_FLAG) != 0;  // U2: the "owner" is detection e of this call, not an entity
      const uint32_t o = o32 & ~DD_FLAG;
      const uint32_t cnt = __ldcg(&m.ov_cnt[slot]);
      __syncwarp();
      if (lane == 0) {
        m.ov_cnt[slot] = 0;  // invariant: counts are zero between calls (the tables are epoch tagged)
        m.cand_j[c] = j;
        m.cand_o[c] = (int32_t)o32;  // negative for detection-detection entries: the debug read skips them
        m.cand_c[c] = cnt;
      }
      if (m.geom == 1 && !dd) continue;  // H: entity candidates come from the similarity prefilter, not from overlap
      const T *x = (const T *)a.desc + (size_t)j * D;
      const T *y = dd ? (const T *)a.desc + (size_t)o * D : (const T *)m.desc_shadow + (size_t)o * D;
      // scalars of the score, requested together with the rows (same address in every lane: one transaction)
      const float ia = m.det_inv_norm[j], ib = dd ? m.det_inv_norm[o] : m.inv_norm[o];
      const uint32_t mn = min(__ldcg(&m.det_nv[j]), dd ? __ldcg(&m.det_nv[o]) : m.n_voxels[o]);
      float dot = 0.f;
      if (sizeof(T) == 2 && (D & 7) == 0 && (((uintptr_t)a.desc) & 15) == 0) {
        for (int i = lane * 8; i < D; i += 256) {
          const uint4 xv = *reinterpret_cast<const uint4 *>(x + i);
          const uint4 yv = *reinterpret_cast<const uint4 *>(y + i);
          const T *xe = reinterpret_cast<const T *>(&xv);
          const T *ye = reinterpret_cast<const T *>(&yv);
#pragma unroll
          for (int q = 0; q < 8; ++q) dot = fmaf(to_f32<T>(xe[q]), to_f32<T>(ye[q]), dot);
        }
      } else {
        for (int i = lane; i < D; i += 32) dot = fmaf(to_f32<T>(x[i]), to_f32<T>(y[i]), dot);
      }
#pragma unroll
      for (int sft = 16; sft; sft >>= 1) dot += __shfl_xor_sync(0xFFFFFFFFu, dot, sft);
      if (lane == 0) {
        float cs = dot * ia * ib;
        cs = fminf(1.f, fmaxf(-1.f, cs));                                  // R15
        const float g = mn ? __fdiv_rn((float)cnt, (float)mn) : 0.f;       // R10
        const float score = __fadd_rn(__fmul_rn(m.w_geo, g), __fmul_rn(m.w_sem, cs));  // R17
        if (dd) {  // U2: detection j is linked to the earlier detection o if they see the same new space and look alike
          if (score > m.tau) {
            const uint32_t e = atomicAdd(&m.counters[6], 1u);
            if (e < m.edge_cap) m.dd_d[e] = j, m.dd_e[e] = o; else atomicOr(m.err, ERR_OVERLAP_TABLE_FULL);
          }
        } else {
          atomicMax(&m.best_cand[j], pack_score(score, o));
          if (m.corr && score > m.tau) add_edge(m, j, o);  // U1
        }
      }
    }
    // pairs above the similarity threshold (emitted by the similarity epilogue): H candidates / U1 edges without overlap
    if (m.dense_d && (m.geom == 1 || m.corr)) {
      if (a.wait_sim) {  // the list is complete only when the similarity grid has finished
        if (tid == 0) spin_until(m.sim_done + (a.seq & 1), a.sim_target, m.err);
        __syncthreads();
      }
      const uint32_t n_dense = min(__ldcg(&m.counters[4]), m.dense_cap);
      for (uint32_t e = blockIdx.x * blockDim.x + threadIdx.x; e < n_dense; e += gridDim.x * blockDim.x) {
        const uint32_t d = __ldcg(&m.dense_d[e]), o = __ldcg(&m.dense_o[e]);
        const float cs = __ldcg(&m.dense_c[e]);
        if (m.geom == 1) {
          hellinger_candidate(m, d, o, cs);
        } else if (__ldcg(&m.det_npx[d]) != 0) {
          const float score = __fadd_rn(__fmul_rn(m.w_geo, 0.f), __fmul_rn(m.w_sem, cs));
          if (score > m.tau) add_edge(m, d, o);
        }
      }
    }
  }
  // ---- ticket: the last CTA to arrive runs the association
  const uint32_t N = __ldcg(m.n_objects);
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const uint32_t t = atomicAdd(&m.counters[3], 1u);
    s_last = t == gridDim.x - 1;
    if (s_last) m.counters[3] = 0;
    s_matches = 0, s_skipped = 0, s_uvox = 0ull;
  }
  __syncthreads();
  if (!s_last) return;
  if (tid == 0) TRACE_MAX(farm_trace_assoc, a.seq, 1);
  // Everything the decisions need except the dense row maxima is final once the last CTA is here (lift, probe and all
  // candidate scores are done): request it BEFORE waiting for the similarity grid, so that only best_dense is loaded after.
  unsigned long long pre_bc[CAND_PER];
  uint32_t pre_npx[CAND_PER], pre_nv[CAND_PER];
#pragma unroll
  for (int k = 0; k < CAND_PER; ++k) {
    const int j = k * CAND_THREADS + tid;
    const bool in = j < a.M;
    pre_bc[k] = in ? __ldcg(&m.best_cand[j]) : 0ull;
    pre_npx[k] = in ? __ldcg(&m.det_npx[j]) : 0u;
    pre_nv[k] = in ? __ldcg(&m.det_nv[j]) : 0u;
  }
  const unsigned long long pre_valid = tid == 0 ? __ldcg(&m.stats->valid_points) : 0ull;
  if (a.wait_sim) {  // no stream join before this kernel: wait here for the similarity grid before reading its row maxima
    if (tid == 0) spin_until(m.sim_done + (a.seq & 1), a.sim_target, m.err);  // bounded: sticky ERR_SYNC_TIMEOUT instead of a hang
    __syncthreads();
  }
  if (tid == 0) TRACE_MAX(farm_trace_assoc, a.seq, 3);
  pdl_trigger();  // the merge kernel becomes resident now, not while the similarity kernel still runs
  if (m.corr) {  // U: union-find over the match graph instead of the per-detection argmax
    correspondence_decide(m, a, N);
    return;
  }
  // Each thread decides CAND_PER detections, CAND_THREADS apart (detection base + k * CAND_THREADS + tid), so that every
  // load and store of the pass is coalesced over the warp; one pass (one barrier) per CAND_THREADS * CAND_PER detections.
  // New ids in detection index order (R20): sub-block k of the pass comes before sub-block k + 1, warps in order inside
  // a sub-block, lanes in order inside a warp.
  __shared__ uint32_t wcnt[2][CAND_PER][CAND_WARPS];  // spawns per (sub-block, warp); double buffered over the passes
  uint32_t running = 0, n_matched = 0, n_skipped = 0, nv_sum = 0;  // running: spawns of the earlier passes (every thread)
  for (int base = 0; base < a.M; base += CAND_THREADS * CAND_PER) {
    unsigned long long bc[CAND_PER], bd[CAND_PER];
    uint32_t npx[CAND_PER];
#pragma unroll
    for (int k = 0; k < CAND_PER; ++k) {  // all loads of the pass up front
      const int j = base + k * CAND_THREADS + tid;
      const bool in = j < a.M;
      bd[k] = in ? __ldcg(&m.best_dense[j]) : 0ull;
      if (base == 0) {  // the first pass was requested before the wait
        bc[k] = pre_bc[k], npx[k] = pre_npx[k], nv_sum += pre_nv[k];
      } else {
        bc[k] = in ? __ldcg(&m.best_cand[j]) : 0ull;
        npx[k] = in ? __ldcg(&m.det_npx[j]) : 0u;
        nv_sum += in ? __ldcg(&m.det_nv[j]) : 0u;
      }
    }
    uint32_t spawn_bits = 0, match_bits = 0, skip_bits = 0;
    int32_t target[CAND_PER];
    float score[CAND_PER];
    unsigned sb[CAND_PER];  // spawn ballots of the warp, per sub-block
    uint32_t(*wc)[CAND_WARPS] = wcnt[(base / (CAND_THREADS * CAND_PER)) & 1];
#pragma unroll
    for (int k = 0; k < CAND_PER; ++k) {
      target[k] = -1, score[k] = 0.f;
      bool spawn = false;
      if (base + k * CAND_THREADS + tid < a.M) {
        if (npx[k] == 0) {
          skip_bits |= 1u << k;  // R8
        } else {
          unsigned long long best = bc[k];
          if (bd[k] && m.geom == 0) {
            // objects without overlap have g = 0: score = w_geo*0 + w_sem*cos (R19)
            const float sd = __fadd_rn(__fmul_rn(m.w_geo, 0.f), __fmul_rn(m.w_sem, unpack_score(bd[k])));
            const unsigned long long pd = pack_score(sd, m.w_sem > 0.f ? unpack_id(bd[k]) : 0u);
            best = pd > best ? pd : best;
          }
          bool matched = false;
          if (best) {
            score[k] = unpack_score(best);
            if (score[k] > m.tau) {  // strict (R18)
              matched = true;
              target[k] = (int32_t)unpack_id(best);
            }
          }
          if (matched) match_bits |= 1u << k; else spawn_bits |= 1u << k, spawn = true;
        }
      }
      sb[k] = __ballot_sync(0xFFFFFFFFu, spawn);
      if (lane == 0) wc[k][warp] = __popc(sb[k]);
    }
    __syncthreads();
    uint32_t total = 0;
#pragma unroll
    for (int k = 0; k < CAND_PER; ++k) {
      // spawns before this thread's detection of sub-block k: earlier passes, earlier sub-blocks, earlier warps, earlier lanes
      uint32_t before = 0, sub_total = 0;
#pragma unroll
      for (int w = 0; w < CAND_WARPS; ++w) {
        const uint32_t c = wc[k][w];
        before += w < warp ? c : 0u;
        sub_total += c;
      }
      const int j = base + k * CAND_THREADS + tid;
      if (j < a.M) {
        uint32_t is_new = 0;
        if ((spawn_bits >> k) & 1u) {
          const uint32_t id = N + running + total + before + __popc(sb[k] & ((1u << lane) - 1));
          if (id < m.max_objects) {
            target[k] = (int32_t)id;
            is_new = 1;
          } else {
            atomicOr(m.err, ERR_OBJECT_CAPACITY);
            skip_bits |= 1u << k;
          }
        }
        if (m.det_gm && ((match_bits >> k) & 1u)) match_hellinger(m.det_gm, m.obj_gw, m.obj_gm, m.hell, m.eps2, j, target[k], npx[k]);  // G4
        m.assoc[j] = target[k];
        m.is_new[j] = (uint8_t)is_new;
        m.best_score[j] = score[k];
        if (target[k] >= 0) {
          atomicMin(&m.leader[target[k]], (uint32_t)j);
          atomicAdd(&m.grp_cnt[target[k]], 1u);
          if (m.touch_seq && !is_new) m.touch_seq[target[k]] = a.seq;  // the next call's similarity masks this row in phase 1
        }
      }
      total += sub_total;
    }
    n_matched += __popc(match_bits), n_skipped += __popc(skip_bits);
    running += total;
  }
  n_matched = __reduce_add_sync(0xFFFFFFFFu, n_matched);
  n_skipped = __reduce_add_sync(0xFFFFFFFFu, n_skipped);
  nv_sum = __reduce_add_sync(0xFFFFFFFFu, nv_sum);
  if (lane == 0) {
    if (n_matched) atomicAdd(&s_matches, n_matched);
    if (n_skipped) atomicAdd(&s_skipped, n_skipped);
    if (nv_sum) atomicAdd(&s_uvox, (unsigned long long)nv_sum);
  }
  __syncthreads();
  if (tid == 0) {
    uint32_t spawns = running;
    if (N + spawns > m.max_objects) spawns = m.max_objects - N;
    const unsigned long long pairs = s_uvox;
    *m.n_objects = N + spawns;
    m.stats->matches = s_matches;
    m.stats->spawns = spawns;
    m.stats->skipped = s_skipped;
    m.stats->unique_voxels = pairs;
    atomicAdd(&m.totals->frames, (unsigned long long)a.F);
    atomicAdd(&m.totals->calls, 1ull);
    atomicAdd(&m.totals->valid_points, pre_valid);
    atomicAdd(&m.totals->unique_voxels, pairs);
    atomicAdd(&m.totals->matches, (unsigned long long)s_matches);
    atomicAdd(&m.totals->spawns, (unsigned long long)spawns);
    TRACE_MAX(farm_trace_assoc, a.seq, 5);
    if (m.touch_seq) {  // split similarity: what the next two calls' kernels read
      m.n_hist[(a.seq + 1) & 1] = N + spawns;
      m.delta_cnt[a.seq & 1] = 0;  // this call's merge warps count their rows from here
      __threadfence();
      atomicAdd(m.scan_done, 1u);  // touch_seq, n_hist are final (every thread's stores precede the barrier above)
    }
  }
}

// ---- voxel commit + object merge, one launch.
// The last commit_blocks CTAs: R12 pass 2 -- the claim winner of every voxel inserted by this call sets the owner.
// The CTAs before them (one per detection): the lowest-index detection of every target object folds the whole group
//   (R21 count-weighted descriptor mean, R22 AABB, R23 view evidence).  No atomics on the object, deterministic
//   summation order.  Groups of one (the common case) skip the member scan.
constexpr int MERGE_THREADS = 256, MERGE_WARPS = MERGE_THREADS / 32;
constexpr int MLIST = 64;  // members of one target object kept in shared memory; larger groups are re-scanned

template <typename T>
__global__ void __launch_bounds__(MERGE_THREADS) commit_merge_kernel(const __grid_constant__ DevMap m, const __grid_constant__ CallArgs a,
                                                                     unsigned long long frame_seq0, int commit_blocks) {
  __shared__ uint32_t mlist[MERGE_WARPS][MLIST];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_trigger();  // the optional covisibility kernel may become resident behind this grid
  pdl_wait();     // launched with PDL behind cand_associate: decisions, leaders and group sizes are final from here on
  const int merge_blocks = gridDim.x - commit_blocks;
  if ((int)blockIdx.x >= merge_blocks) {  // the merge CTAs come first in launch order
    const uint32_t cb = blockIdx.x - merge_blocks;
    // 8 lanes per event (one 32-byte owner sector each), 4 events per warp and group, two groups in flight
    const uint32_t n = min(m.counters[0], m.pair_cap);
    const int sec = lane & 7;
    const uint32_t half = (uint32_t)commit_blocks * MERGE_WARPS * 4;
    for (uint32_t e0 = (cb * MERGE_WARPS + warp) * 4; e0 < n; e0 += 2 * half) {
      uint32_t e[2], jp[2], slot[2], byte[2], own[2][8];
      int32_t t[2] = {-1, -1};
      uint32_t cnt[2] = {0, 0};
      bool act[2];
#pragma unroll
      for (int u = 0; u < 2; ++u) {  // stage 1: the event records
        e[u] = e0 + u * half + (lane >> 3);
        act[u] = e[u] < n;
        jp[u] = act[u] ? m.pl_j[e[u]] : 0u;
        slot[u] = act[u] ? m.pl_slot[e[u]] : 0u;
        byte[u] = act[u] ? (uint32_t)(m.pl_bits[e[u]] >> (8 * sec)) & 0xFFu : 0u;
        if (act[u] && sec == 0) m.pair_bits[m.pl_ps[e[u]]] = 0ull;  // invariant: pair-set voxel bits are zero between calls
        act[u] = act[u] && (jp[u] >> 31) && byte[u];              // some voxel of the event was unowned at entry
      }
#pragma unroll
      for (int u = 0; u < 2; ++u)  // stage 2: target object and owner sector
        if (act[u]) {
          t[u] = m.assoc[jp[u] & 0x7FFFFFFFu];
          const uint4 *base = reinterpret_cast<const uint4 *>(m.blk_owner + (size_t)slot[u] * BLK_VOXELS + sec * 8);
          const uint4 w0 = __ldcg(base), w1 = __ldcg(base + 1);
          own[u][0] = w0.x, own[u][1] = w0.y, own[u][2] = w0.z, own[u][3] = w0.w;
          own[u][4] = w1.x, own[u][5] = w1.y, own[u][6] = w1.z, own[u][7] = w1.w;
        }
#pragma unroll
      for (int u = 0; u < 2; ++u) {  // stage 3: the claim winner sets the owner (R12)
        if (act[u] && t[u] >= 0) {
          uint32_t *base = m.blk_owner + (size_t)slot[u] * BLK_VOXELS + sec * 8;
          const uint32_t mine = OWNER_PENDING | (jp[u] & 0x7FFFFFFFu);
#pragma unroll
          for (int b = 0; b < 8; ++b)
            if (((byte[u] >> b) & 1u) && own[u][b] == mine) {
              base[b] = (uint32_t)t[u];
              cnt[u]++;
            }
        }
        const unsigned am = __ballot_sync(0xFFFFFFFFu, cnt[u] != 0);
        if (cnt[u]) {
          const unsigned same = __match_any_sync(am, t[u]);
          const uint32_t tot = __reduce_add_sync(same, cnt[u]);
          if (lane == __ffs(same) - 1) atomicAdd(&m.n_voxels[t[u]], tot);
        }
      }
    }
    return;
  }
  // ---- merge: one WARP per detection; only the lowest-index detection of a target object works (R21-R23)
  // Split similarity: every merge warp reports when it leaves (whichever return it takes); the next call's similarity kernel,
  // already running, starts its phase 2 when all of them have.
  struct Report {
    uint32_t *ctr;
    int lane;
    uint32_t seq;
    __device__ ~Report() {
      if (lane == 0) TRACE_MAX(farm_trace_assoc, seq, 7);
      if (!ctr) return;
      __syncwarp();
      if (lane == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
      }
    }
  } report{m.merge_done, lane, a.seq};
  if (lane == 0) TRACE_MIN(farm_trace_assoc, a.seq, 2);
  const int j = blockIdx.x * MERGE_WARPS + warp;
  if (j >= a.M) return;
  const int32_t t = m.assoc[j];
  if (t < 0) return;
  const uint32_t lead = __ldcg(&m.leader[t]), group = __ldcg(&m.grp_cnt[t]);
  if (lead != (uint32_t)j) return;
  const int D = m.D;
  // U4: entities absorbed by t in this call
  const uint32_t nL = m.corr ? min(__ldcg(&m.counters[7]), m.edge_cap) : 0u;
  uint32_t loser_obs = 0, n_losers = 0;
  for (uint32_t k = 0; k < nL; ++k)
    if (__ldcg(&m.winner[k]) == (uint32_t)t) loser_obs += m.n_obs[__ldcg(&m.loser[k])], ++n_losers;
  const bool has_losers = n_losers != 0;
  if (has_losers) {
    if (lane == 0) absorb_losers(m, t, nL);
    __syncwarp();
  }
  const uint32_t n_old = m.n_obs[t];
  const float nf = (float)n_old;
  float *master = m.desc_master + (size_t)t * D;
  T *shadow = (T *)m.desc_shadow + (size_t)t * D;
  const T *desc = (const T *)a.desc;
  // members in index order (deterministic summation): kept in shared memory when they fit
  uint32_t n_listed = 1;
  if (group > 1) {
    n_listed = 0;
    for (int base = j & ~31; base < a.M && n_listed < MLIST; base += 32) {
      const int jj = base + lane;
      const bool flag = jj < a.M && jj >= j && m.assoc[jj] == t;
      const unsigned b = __ballot_sync(0xFFFFFFFFu, flag);
      const uint32_t pos = n_listed + __popc(b & ((1u << lane) - 1));
      if (flag && pos < MLIST) mlist[warp][pos] = (uint32_t)jj;
      n_listed += __popc(b);
    }
    __syncwarp();
  }
  const bool listed = group <= MLIST;
  // f(jm) for every member jm of the group, ascending
  auto for_each_member = [&](auto &&f) {
    if (group <= 1) {
      f((uint32_t)j);
    } else if (listed) {
      for (uint32_t k = 0; k < group; ++k) f(mlist[warp][k]);
    } else {
      for (int jj = j; jj < a.M; ++jj)
        if (m.assoc[jj] == t) f((uint32_t)jj);
    }
  };
  // lane 0: view evidence and point box of the members (R22, R23); its loads overlap the descriptor work
  uint32_t k_members = 0;
  unsigned long long pts = 0, pts_old = 0, best_seq = 0;
  uint32_t best = 0, best_old = 0, best_det = 0;
  int bmn[3] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF}, bmx[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
  int box_old[6] = {0, 0, 0, 0, 0, 0};
  int best_frame = -1;
  double gsum[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};  // G2: sufficient statistics of the members
  if (lane == 0) {
    pts_old = m.n_points[t];
    best_old = m.best_px[t];
#pragma unroll
    for (int c = 0; c < 6; ++c) box_old[c] = m.aabb[t * 6 + c];
    for_each_member([&](uint32_t jm) {
      k_members++;
      const uint32_t npx = m.det_npx[jm];
      pts += npx;
      if (m.det_gm) {
#pragma unroll
        for (int k = 0; k < 9; ++k) gsum[k] += m.det_gm[(size_t)jm * 9 + k];
      }
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        bmn[c] = min(bmn[c], m.det_box[jm * 6 + c]);
        bmx[c] = max(bmx[c], m.det_box[jm * 6 + 3 + c]);
      }
      int f = 0;
      while (f + 1 < a.F && (int)jm >= a.base[f + 1]) ++f;
      // R23: most pixels wins, ties -> smallest (frame_seq, det): members come in ascending (frame, det) order and every
      // stored view is older than this call, so a strict > keeps the earliest
      if (npx > best) best = npx, best_frame = f, best_seq = frame_seq0 + f, best_det = jm - a.base[f];
      if (m.views) {  // V: detections offer their view in index order
        const float *Tf = a.T + 16 * f;
        const float cam[3] = {Tf[3], Tf[7], Tf[11]};
        offer_view(m, t, m.det_box + jm * 6, cam, (int32_t)(frame_seq0 + f), (int32_t)(jm - a.base[f]), npx);
      }
    });
  }
  // f_o <- normalise(n_obs * f_o + sum_m a_m / |a_m|)   (R21).  Two passes over the rows (the second one hits
  // L1/L2): pass 1 the squared norm, pass 2 the same values again, scaled and written with their shadows.
  const bool vec = sizeof(T) == 2 && group <= 1 && !has_losers && (D & 7) == 0 && (((uintptr_t)a.desc) & 15) == 0;
  auto value = [&](int i) -> float {  // generic path, one element
    float acc = 0.f;
    bool first = true;
    for_each_member([&](uint32_t jm) {
      const float x = to_f32<T>(desc[(size_t)jm * D + i]), inv = m.det_inv_norm[jm];  // zero-norm rows contribute nothing
      acc = first ? x * inv : fmaf(x, inv, acc);
      first = false;
    });
    if (n_old) acc = fmaf(nf, master[i], acc);
    if (has_losers)  // U4: the losers' descriptors, weighted by their detection counts
      for (uint32_t k = 0; k < nL; ++k)
        if (m.winner[k] == (uint32_t)t) {
          const uint32_t L = m.loser[k];
          acc = fmaf((float)m.n_obs[L], m.desc_master[(size_t)L * D + i], acc);
        }
    return acc;
  };
  const float inv_j = m.det_inv_norm[j];
  const T *row_j = desc + (size_t)j * D;
  auto value8 = [&](int i, float (&v)[8]) {  // vector path: the leader is the only member
    const uint4 w = *reinterpret_cast<const uint4 *>(row_j + i);
    const T *e = reinterpret_cast<const T *>(&w);
    float4 m0 = make_float4(0.f, 0.f, 0.f, 0.f), m1 = m0;
    if (n_old) m0 = *reinterpret_cast<const float4 *>(master + i), m1 = *reinterpret_cast<const float4 *>(master + i + 4);
    const float mv[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const float x = to_f32<T>(e[q]) * inv_j;
      v[q] = n_old ? fmaf(nf, mv[q], x) : x;
    }
  };
  float ss = 0.f;
  // vector path with D <= 1024: the row is read ONCE (all loads in flight together) and kept in registers between the
  // norm and the write-back -- one dependent round trip fewer on the critical tail of the call
  const bool keep = vec && D <= 1024;
  float kv[4][8];
  if (keep) {
#pragma unroll
    for (int it = 0; it < 4; ++it) {
      const int i = lane * 8 + it * 256;
      if (i < D) {
        value8(i, kv[it]);
#pragma unroll
        for (int q = 0; q < 8; ++q) ss = fmaf(kv[it][q], kv[it][q], ss);
      }
    }
  } else if (vec) {
    for (int i = lane * 8; i < D; i += 256) {
      float v[8];
      value8(i, v);
#pragma unroll
      for (int q = 0; q < 8; ++q) ss = fmaf(v[q], v[q], ss);
    }
  } else {
    for (int i = lane; i < D; i += 32) {
      const float v = value(i);
      ss = fmaf(v, v, ss);
    }
  }
#pragma unroll
  for (int sft = 16; sft; sft >>= 1) ss += __shfl_xor_sync(0xFFFFFFFFu, ss, sft);
  if (ss > 0.f) {  // a zero sum keeps the old value
    const float inv = 1.0f / sqrtf(ss);
    float s2 = 0.f;
    auto store8 = [&](int i, float (&v)[8]) {
      uint4 w;
      T *e = reinterpret_cast<T *>(&w);
#pragma unroll
      for (int q = 0; q < 8; ++q) {
        v[q] *= inv;
        e[q] = from_f32<T>(v[q]);  // round-to-nearest-even shadow (R1, R14)
        const float sv = to_f32<T>(e[q]);
        s2 = fmaf(sv, sv, s2);
      }
      *reinterpret_cast<float4 *>(master + i) = make_float4(v[0], v[1], v[2], v[3]);
      *reinterpret_cast<float4 *>(master + i + 4) = make_float4(v[4], v[5], v[6], v[7]);
      *reinterpret_cast<uint4 *>(shadow + i) = w;
    };
    if (keep) {
#pragma unroll
      for (int it = 0; it < 4; ++it) {
        const int i = lane * 8 + it * 256;
        if (i < D) store8(i, kv[it]);
      }
    } else if (vec) {
      for (int i = lane * 8; i < D; i += 256) {
        float v[8];
        value8(i, v);
        store8(i, v);
      }
    } else {
      for (int i = lane; i < D; i += 32) {
        const float v = value(i) * inv;
        master[i] = v;
        const T sh = from_f32<T>(v);
        shadow[i] = sh;
        const float sv = to_f32<T>(sh);
        s2 = fmaf(sv, sv, s2);
      }
    }
#pragma unroll
    for (int sft = 16; sft; sft >>= 1) s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, sft);
    if (lane == 0) m.inv_norm[t] = s2 > 0.f ? 1.0f / sqrtf(s2) : 0.f;
  }
  if (m.delta_rows) {
    // split similarity: the row as it stands now (rewritten above, or kept), its id and inverse norm also go to the delta
    // buffer -- the B operand of the next call's phase 2
    __syncwarp();
    uint32_t slot = 0;
    if (lane == 0) slot = atomicAdd(&m.delta_cnt[a.seq & 1], 1u);
    slot = __shfl_sync(0xFFFFFFFFu, slot, 0);
    if (slot < m.max_det) {
      T *drow = (T *)m.delta_rows + (size_t)slot * D;
      if (sizeof(T) == 2 && (D & 7) == 0) {
        for (int i = lane * 8; i < D; i += 256) *reinterpret_cast<uint4 *>(drow + i) = *reinterpret_cast<const uint4 *>(shadow + i);
      } else {
        for (int i = lane; i < D; i += 32) drow[i] = shadow[i];
      }
      if (lane == 0) m.delta_id[slot] = (uint32_t)t, m.delta_inv[slot] = m.inv_norm[t];
    }
  }
  if (lane == 0) {
    m.n_obs[t] = n_old + loser_obs + k_members;
    m.n_points[t] = pts_old + pts;
    if (m.det_gm) {  // G2: M1 += sum w mu, M2 += sum w (Sigma + mu mu^T), w = points
      const double gw = m.obj_gw[t] + (double)pts;
      m.obj_gw[t] = gw;
#pragma unroll
      for (int k = 0; k < 9; ++k) gsum[k] += m.obj_gm[(size_t)t * 9 + k];
#pragma unroll
      for (int k = 0; k < 9; ++k) m.obj_gm[(size_t)t * 9 + k] = gsum[k];
      if (m.edges_k > 0 && gw > 0.0) edge_member(m, (uint32_t)t, gw, gsum);  // W1
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) {  // R22
      m.aabb[t * 6 + c] = min(box_old[c], bmn[c]);
      m.aabb[t * 6 + 3 + c] = max(box_old[3 + c], bmx[c]);
    }
    if (best > best_old) {
      m.best_px[t] = best;
      m.best_seq[t] = best_seq;
      m.best_det[t] = best_det;
      const float *Tf = a.T + 16 * best_frame;
      m.best_cam[t * 3 + 0] = Tf[3];
      m.best_cam[t * 3 + 1] = Tf[7];
      m.best_cam[t * 3 + 2] = Tf[11];
    }
    m.leader[t] = NONE32;
    m.grp_cnt[t] = 0;
  }
  if (has_losers) {  // the fold above was the last reader of the losers' rows
    __syncwarp();
    for (uint32_t k = 0; k < nL; ++k)
      if (m.winner[k] == (uint32_t)t) {
        const uint32_t L = m.loser[k];
        for (int i = lane; i < D; i += 32) {
          m.desc_master[(size_t)L * D + i] = 0.f;
          ((T *)m.desc_shadow)[(size_t)L * D + i] = from_f32<T>(0.f);
        }
        if (lane == 0) retire_loser(m, L, t);
      }
  }
}

// ---- covisibility (rule C1; PAPER.md:354 step 7): every pair of distinct entities that received a detection in
// this call is marked in the N x ceil(N/64) bitset.  Each CTA builds the call's entity bitmap in shared memory
// (a few KB), lists its non-zero words (at most one per entity of the call, whatever N is) and ORs those words, minus the
// diagonal bit, into the rows of its entities, writing only the words that change.  A row is written only by the CTAs of detections that target it, and they all write the
// same words, so no atomics are needed.
constexpr int COVIS_THREADS = 256;

// U4 + C1: an absorbed entity's covisibility goes to its winner.  Pass 1 (one thread per row): every bit L of a loser
// becomes bit W of its winner.  Pass 2 (one CTA per merge): row W |= row L, row L = 0.  The diagonal bit this can leave
// in row W is cleared by covisibility_kernel, which visits every winner (a winner always received a detection).
__global__ void __launch_bounds__(COVIS_THREADS) covis_rename_kernel(DevMap m, uint32_t n_upper) {
  pdl_wait();
  const uint32_t nL = min(m.counters[7], m.edge_cap);
  if (nL == 0) return;
  const uint32_t N = min(*m.n_objects, n_upper);
  for (uint32_t r = blockIdx.x * blockDim.x + threadIdx.x; r < N; r += gridDim.x * blockDim.x) {
    unsigned long long *row = m.covis + (size_t)r * m.covis_words;
    for (uint32_t k = 0; k < nL; ++k) {
      const uint32_t L = m.loser[k], W = m.winner[k];
      if ((row[L >> 6] >> (L & 63)) & 1ull) {
        row[L >> 6] &= ~(1ull << (L & 63));
        row[W >> 6] |= 1ull << (W & 63);
      }
    }
  }
}
__global__ void __launch_bounds__(COVIS_THREADS) covis_fold_kernel(DevMap m) {
  pdl_wait();
  const uint32_t nL = min(m.counters[7], m.edge_cap);
  const uint32_t words = (*m.n_objects + 63) >> 6;
  for (uint32_t k = blockIdx.x; k < nL; k += gridDim.x) {
    unsigned long long *rl = m.covis + (size_t)m.loser[k] * m.covis_words, *rw = m.covis + (size_t)m.winner[k] * m.covis_words;
    for (uint32_t w = threadIdx.x; w < words; w += COVIS_THREADS) {
      const unsigned long long v = rl[w];
      if (v) {
        atomicOr(&rw[w], v);  // several losers may fold into one winner concurrently
        rl[w] = 0ull;
      }
    }
  }
}

__global__ void __launch_bounds__(COVIS_THREADS) covisibility_kernel(DevMap m, CallArgs a) {
  extern __shared__ unsigned long long bm[];  // [words] bitmap of the call's entities, then [n_list] uint16 word indices
  __shared__ uint32_t n_list;
  pdl_wait();
  const uint32_t N = *m.n_objects;
  const uint32_t words = (N + 63) >> 6;
  uint16_t *list = reinterpret_cast<uint16_t *>(bm + words);  // the non-zero words of bm: a row changes nowhere else
  for (uint32_t w = threadIdx.x; w < words; w += COVIS_THREADS) bm[w] = 0ull;
  if (threadIdx.x == 0) n_list = 0;
  __syncthreads();
  for (int j = threadIdx.x; j < a.M; j += COVIS_THREADS) {
    const int32_t t = m.assoc[j];
    if (t >= 0) atomicOr(&bm[(uint32_t)t >> 6], 1ull << (t & 63));
  }
  __syncthreads();
  for (uint32_t w0 = 0; w0 < words; w0 += COVIS_THREADS) {
    const uint32_t w = w0 + threadIdx.x;
    const bool nz = w < words && bm[w] != 0ull;
    const unsigned ball = __ballot_sync(0xFFFFFFFFu, nz);
    uint32_t base = 0;
    if ((threadIdx.x & 31) == 0 && ball) base = atomicAdd(&n_list, (uint32_t)__popc(ball));
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (nz) list[base + __popc(ball & ((1u << (threadIdx.x & 31)) - 1u))] = (uint16_t)w;
  }
  __syncthreads();
  const uint32_t nl = n_list;
  for (int j = blockIdx.x; j < a.M; j += gridDim.x) {
    const int32_t t = m.assoc[j];
    if (t < 0) continue;
    unsigned long long *row = m.covis + (size_t)t * m.covis_words;
    for (uint32_t i = threadIdx.x; i < nl; i += COVIS_THREADS) {
      const uint32_t w = list[i];
      unsigned long long add = bm[w], keep = ~0ull;
      if (w == ((uint32_t)t >> 6)) keep = ~(1ull << (t & 63)), add &= keep;  // no diagonal (U4: a fold may have left one)
      const unsigned long long old = row[w], now = (old | add) & keep;
      if (now != old) row[w] = now;
    }
  }
}

}  // namespace

#define FARM_DISPATCH(call)                                   \
  if (m.dtype == FARM_DTYPE_F32) { using T = float; call; }   \
  else if (m.dtype == FARM_DTYPE_F16) { using T = __half; call; } \
  else { using T = __nv_bfloat16; call; }

void configure_assoc_kernels() {
  const int pref = (int)cudaSharedmemCarveoutMaxShared;
  cudaFuncSetAttribute(cand_associate_kernel<float>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(cand_associate_kernel<__half>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(cand_associate_kernel<__nv_bfloat16>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(commit_merge_kernel<float>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(commit_merge_kernel<__half>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(commit_merge_kernel<__nv_bfloat16>, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(covisibility_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, pref);
  cudaFuncSetAttribute(covisibility_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 128 * 1024);
}

int launch_cand_associate(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  const int grid = a.M > 0 ? (m.num_sms + 1) / 2 : 1;  // half the SMs x 16 warps: one warp per candidate, ~1.2k candidates per wave
  FARM_DISPATCH((launch_pdl(cand_associate_kernel<T>, dim3(grid), dim3(CAND_THREADS), 0, s, m, a)));
  return 1;
}
int launch_covis_absorb(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s) {
  if (a.M == 0 || !m.covis || !m.corr) return 0;
  launch_pdl(covis_rename_kernel, dim3(m.num_sms), dim3(COVIS_THREADS), 0, s, m, n_upper);
  launch_pdl(covis_fold_kernel, dim3(m.num_sms), dim3(COVIS_THREADS), 0, s, m);
  return 2;
}
int launch_covisibility(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  if (a.M == 0 || !m.covis) return 0;
  // every CTA rebuilds the bitmap and its word list, so fewer, longer-lived CTAs win (measured 4 / 2 / 1 per SM: 26.5 / 22.6 / 25.0 us)
  const int grid = a.M < m.num_sms * 2 ? a.M : m.num_sms * 2;
  const size_t n_list_max = m.covis_words < (uint32_t)a.M ? m.covis_words : (uint32_t)a.M;  // non-zero words <= entities
  launch_pdl(covisibility_kernel, dim3(grid), dim3(COVIS_THREADS), (size_t)m.covis_words * 8 + n_list_max * 2, s, m, a);
  return 1;
}
int merge_warps_of(const CallArgs &a) { return a.M > 0 ? (a.M + MERGE_WARPS - 1) / MERGE_WARPS * MERGE_WARPS : 0; }

int launch_commit_merge(const DevMap &m, const CallArgs &a, unsigned long long frame_seq0, cudaStream_t s) {
  if (a.M == 0) return 0;
  const int commit_blocks = m.num_sms * 4;
  const int merge_blocks = (a.M + MERGE_WARPS - 1) / MERGE_WARPS;  // one warp per detection
  if (a.split && a.sim_fills_gpu) {
    // Split schedule with a similarity grid that takes every SM: no programmatic early launch.  CTAs of this grid that sit in pdl_wait() while the decision scan runs
    // hold their registers (256 x 119), and the next call's similarity kernel -- which starts in exactly that window -- would
    // find no room on those SMs until this grid has drained (measured: its last CTA started 22-25 us late).
    FARM_DISPATCH((commit_merge_kernel<T><<<dim3(commit_blocks + merge_blocks), dim3(MERGE_THREADS), 0, s>>>(m, a, frame_seq0, commit_blocks)));
  } else {
    FARM_DISPATCH((launch_pdl(commit_merge_kernel<T>, dim3(commit_blocks + merge_blocks), dim3(MERGE_THREADS), 0, s, m, a, frame_seq0,
                              commit_blocks)));
  }
  return 1;
}

}  // namespace farm
