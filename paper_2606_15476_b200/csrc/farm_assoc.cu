// farm_assoc.cu -- step 5: candidate scoring, association (argmax / threshold / spawn) and merge.
//   R10, R17-R20 (score, strict threshold, ids in detection index order; BASELINE.json rule)
//   R12 (voxel commit, lowest detection index wins), R21 (count-weighted descriptor mean),
//   R22 (AABB), R23 (view evidence).
#include "farm_internal.cuh"

namespace farm {
namespace {

constexpr uint32_t NONE32 = 0xFFFFFFFFu;

// ---- candidate scoring + association, one launch.
// Phase 1 (all CTAs): one warp per non-zero overlap entry (d, o, c): cos(a_d, shadow_o) by a gather dot, g (R10),
//   score (R17), atomicMax into best_cand[d].
// Phase 2 (the last CTA to finish, found by a ticket): decisions for all detections (R18), new ids by an
//   exclusive scan in detection index order (R20), per-target leader / group size for the merge.
template <typename T>
__global__ void __launch_bounds__(1024) cand_associate_kernel(DevMap m, CallArgs a) {
  __shared__ uint32_t warp_sum[32];
  __shared__ uint32_t s_running, s_matches, s_skipped;
  __shared__ unsigned long long s_uvox;
  __shared__ bool s_last;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  {
    const uint32_t n_cand = min(m.counters[1], m.cand_cap);
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    const int D = m.D;
    for (uint32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; c < n_cand; c += warps) {
      const uint32_t slot = m.cand_slot[c];
      const unsigned long long kv = m.cand_key[c];
      const uint32_t j = (uint32_t)(kv >> 32) & ((1u << DET_BITS) - 1);
      const uint32_t o = (uint32_t)kv;
      const uint32_t cnt = __ldcg(&m.ov_cnt[slot]);
      __syncwarp();
      if (lane == 0) {
        m.ov_cnt[slot] = 0;  // invariant: counts are zero between calls (the tables are epoch tagged)
        m.cand_j[c] = j;
        m.cand_o[c] = (int32_t)o;
        m.cand_c[c] = cnt;
      }
      const T *x = (const T *)a.desc + (size_t)j * D;
      const T *y = (const T *)m.desc_shadow + (size_t)o * D;
      // scalars of the score, requested together with the rows (same address in every lane: one transaction)
      const float ia = m.det_inv_norm[j], ib = m.inv_norm[o];
      const uint32_t mn = min(__ldcg(&m.det_nv[j]), m.n_voxels[o]);
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
        atomicMax(&m.best_cand[j], pack_score(score, o));
      }
    }
  }
  // ---- everything the association scan needs except best_cand is final before this kernel starts: requested here,
  // ahead of the ticket, so that the scan of the last CTA starts with its operands in registers (M <= 2048)
  const uint32_t N = __ldcg(m.n_objects);
  unsigned long long valid_points = 0;
  if (tid == 0) valid_points = __ldcg(&m.stats->valid_points);
  uint32_t pre_nv[2], pre_npx[2];
  unsigned long long pre_bd[2];
#pragma unroll
  for (int q = 0; q < 2; ++q) {
    const int j = q * 1024 + tid;
    const bool in = j < a.M;
    pre_nv[q] = in ? __ldcg(&m.det_nv[j]) : 0u;
    pre_npx[q] = in ? __ldcg(&m.det_npx[j]) : 0u;
    pre_bd[q] = in ? __ldcg(&m.best_dense[j]) : 0ull;
  }
  // ---- ticket: the last CTA to arrive runs the association
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    const uint32_t t = atomicAdd(&m.counters[3], 1u);
    s_last = t == gridDim.x - 1;
    if (s_last) m.counters[3] = 0;
    s_running = 0, s_matches = 0, s_skipped = 0, s_uvox = 0ull;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  for (int base = 0; base < a.M; base += 1024) {
    const int j = base + tid;
    const int q = base >> 10;
    uint32_t spawn = 0, matched = 0, skipped = 0;
    int32_t target = -1;
    float score = 0.f;
    const bool in = j < a.M;
    const uint32_t my_nv = q == 0 ? pre_nv[0] : q == 1 ? pre_nv[1] : (in ? __ldcg(&m.det_nv[j]) : 0u);
    const uint32_t my_npx = q == 0 ? pre_npx[0] : q == 1 ? pre_npx[1] : (in ? __ldcg(&m.det_npx[j]) : 0u);
    const unsigned long long bd = q == 0 ? pre_bd[0] : q == 1 ? pre_bd[1] : (in ? __ldcg(&m.best_dense[j]) : 0ull);
    const uint32_t nv = __reduce_add_sync(0xFFFFFFFFu, my_nv);
    if (lane == 0 && nv) atomicAdd(&s_uvox, (unsigned long long)nv);
    if (in) {
      if (my_npx == 0) {
        skipped = 1;  // R8
      } else {
        unsigned long long best = __ldcg(&m.best_cand[j]);
        if (bd) {
          // objects without overlap have g = 0: score = w_geo*0 + w_sem*cos (R19)
          const float sd = __fadd_rn(__fmul_rn(m.w_geo, 0.f), __fmul_rn(m.w_sem, unpack_score(bd)));
          const unsigned long long pd = pack_score(sd, m.w_sem > 0.f ? unpack_id(bd) : 0u);
          best = pd > best ? pd : best;
        }
        if (best) {
          score = unpack_score(best);
          if (score > m.tau) {  // strict (R18)
            matched = 1;
            target = (int32_t)unpack_id(best);
          }
        }
        spawn = matched ? 0u : 1u;
      }
    }
    // block exclusive scan of the spawn flags
    const unsigned b = __ballot_sync(0xFFFFFFFFu, spawn);
    if (lane == 0) warp_sum[warp] = __popc(b);
    __syncthreads();
    uint32_t before = 0, total = 0;
    for (int w = 0; w < 32; ++w) {
      const uint32_t c = warp_sum[w];
      before += w < warp ? c : 0;
      total += c;
    }
    const uint32_t running = s_running;
    if (spawn) {
      const uint32_t id = N + running + before + __popc(b & ((1u << lane) - 1));
      if (id < m.max_objects) {
        target = (int32_t)id;
      } else {
        atomicOr(m.err, ERR_OBJECT_CAPACITY);
        spawn = 0, skipped = 1;
      }
    }
    if (j < a.M) {
      m.assoc[j] = target;
      m.is_new[j] = (uint8_t)spawn;
      m.best_score[j] = score;
      if (target >= 0) {
        atomicMin(&m.leader[target], (uint32_t)j);
        atomicAdd(&m.grp_cnt[target], 1u);
      }
    }
    const unsigned bm = __ballot_sync(0xFFFFFFFFu, matched), bs = __ballot_sync(0xFFFFFFFFu, skipped);
    if (lane == 0) {
      if (bm) atomicAdd(&s_matches, (uint32_t)__popc(bm));
      if (bs) atomicAdd(&s_skipped, (uint32_t)__popc(bs));
    }
    __syncthreads();
    if (tid == 0) s_running = running + total;
    __syncthreads();
  }
  if (tid == 0) {
    uint32_t spawns = s_running;
    if (N + spawns > m.max_objects) spawns = m.max_objects - N;
    const unsigned long long pairs = s_uvox;
    *m.n_objects = N + spawns;
    m.stats->matches = s_matches;
    m.stats->spawns = spawns;
    m.stats->skipped = s_skipped;
    m.stats->unique_voxels = pairs;
    atomicAdd(&m.totals->frames, (unsigned long long)a.F);
    atomicAdd(&m.totals->calls, 1ull);
    atomicAdd(&m.totals->valid_points, valid_points);
    atomicAdd(&m.totals->unique_voxels, pairs);
    atomicAdd(&m.totals->matches, (unsigned long long)s_matches);
    atomicAdd(&m.totals->spawns, (unsigned long long)spawns);
  }
}

// ---- voxel commit + object merge, one launch.
// The last commit_blocks CTAs: R12 pass 2 -- the claim winner of every voxel inserted by this call sets the owner.
// The CTAs before them (one per detection): the lowest-index detection of every target object folds the whole group
//   (R21 count-weighted descriptor mean, R22 AABB, R23 view evidence).  No atomics on the object, deterministic
//   summation order.  Groups of one (the common case) skip the member scan.
constexpr int MERGE_THREADS = 128, MERGE_WARPS = MERGE_THREADS / 32;

template <typename T>
__global__ void __launch_bounds__(MERGE_THREADS) commit_merge_kernel(DevMap m, CallArgs a, unsigned long long frame_seq0,
                                                           int commit_blocks) {
  extern __shared__ float acc[];  // [D]
  __shared__ uint32_t list[MERGE_THREADS];
  __shared__ uint32_t warp_cnt[MERGE_WARPS];
  __shared__ float red[MERGE_WARPS], red2[MERGE_WARPS];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int merge_blocks = gridDim.x - commit_blocks;
  if ((int)blockIdx.x >= merge_blocks) {  // the long-running merge CTAs come first in launch order
    const uint32_t cb = blockIdx.x - merge_blocks;
    // 8 lanes per event (one 32-byte owner sector each), 4 events per warp and step
    const uint32_t n = min(m.counters[0], m.pair_cap);
    const int sec = lane & 7;
    const uint32_t step = (uint32_t)commit_blocks * MERGE_WARPS * 4;
    for (uint32_t e0 = (cb * MERGE_WARPS + warp) * 4; e0 < n; e0 += step) {
      const uint32_t e = e0 + (lane >> 3);
      int32_t t = -1;
      uint32_t cnt = 0;
      if (e < n) {
        const uint32_t jp = m.pl_j[e];
        if (sec == 0) m.pair_bits[m.pl_ps[e]] = 0ull;  // invariant: the pair set's voxel bits are zero between calls
        const uint32_t byte = (uint32_t)(m.pl_bits[e] >> (8 * sec)) & 0xFFu;
        if ((jp >> 31) && byte) {  // some voxel of the event was unowned at entry
          const uint32_t j = jp & 0x7FFFFFFFu;
          t = m.assoc[j];
          uint32_t *base = m.blk_owner + (size_t)m.pl_slot[e] * BLK_VOXELS + sec * 8;
          const uint4 w0 = __ldcg(reinterpret_cast<const uint4 *>(base));
          const uint4 w1 = __ldcg(reinterpret_cast<const uint4 *>(base) + 1);
          const uint32_t own[8] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
          if (t >= 0) {
#pragma unroll
            for (int b = 0; b < 8; ++b)
              if (((byte >> b) & 1u) && own[b] == (OWNER_PENDING | j)) {  // this detection holds the claim (R12)
                base[b] = (uint32_t)t;
                cnt++;
              }
          }
        }
      }
      const unsigned act = __ballot_sync(0xFFFFFFFFu, cnt != 0);
      if (cnt) {
        const unsigned same = __match_any_sync(act, t);
        const uint32_t tot = __reduce_add_sync(same, cnt);
        if (lane == __ffs(same) - 1) atomicAdd(&m.n_voxels[t], tot);
      }
    }
    return;
  }
  const int D = m.D;
  // 8 elements per thread and step (128-bit loads of the storage-dtype rows, 2 x 128-bit of the fp32 masters)
  const bool vec = (D & 7) == 0 && (((uintptr_t)a.desc) & 15) == 0;
  for (int j = blockIdx.x; j < a.M; j += merge_blocks) {
    const int32_t t = m.assoc[j];
    if (t < 0) continue;                                   // uniform per CTA
    const uint32_t lead = __ldcg(&m.leader[t]), group = __ldcg(&m.grp_cnt[t]);
    if (lead != (uint32_t)j) continue;
    // everything the fold needs is requested up front so that the loads overlap
    const uint32_t n_old = m.n_obs[t];
    float *master = m.desc_master + (size_t)t * D;
    T *shadow = (T *)m.desc_shadow + (size_t)t * D;
    unsigned long long pts_old = 0, best_old = 0;
    int box_old[6];
    if (tid == 0) {
      pts_old = m.n_points[t];
      best_old = m.best_view[t];
#pragma unroll
      for (int c = 0; c < 6; ++c) box_old[c] = m.aabb[t * 6 + c];
    }
    uint32_t k_members = 0;
    unsigned long long pts = 0, best = 0;
    int bmn[3] = {0x7FFFFFFF, 0x7FFFFFFF, 0x7FFFFFFF}, bmx[3] = {(int)0x80000000, (int)0x80000000, (int)0x80000000};
    int best_frame = -1;
    auto member_evidence = [&](uint32_t jm) {  // thread 0: R22 / R23 contribution of one member
      k_members++;
      const uint32_t npx = m.det_npx[jm];
      pts += npx;
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        bmn[c] = min(bmn[c], m.det_box[jm * 6 + c]);
        bmx[c] = max(bmx[c], m.det_box[jm * 6 + 3 + c]);
      }
      int f = 0;
      while (f + 1 < a.F && (int)jm >= a.base[f + 1]) ++f;
      const unsigned long long seq = frame_seq0 + f;
      const uint32_t det = jm - a.base[f];
      // R23: most pixels wins, ties -> smallest (frame_seq, det)
      const unsigned long long pv = ((unsigned long long)(npx & 0xFFFFFFu) << 40) | ((~seq & 0xFFFFFFull) << 16) |
                                    (unsigned long long)(~det & 0xFFFFu);
      if (pv > best) best = pv, best_frame = f;
    };
    auto add_row = [&](uint32_t jm, bool first) {  // acc (+)= a_jm / |a_jm|; zero-norm rows contribute nothing (R21)
      const float inv = m.det_inv_norm[jm];
      const T *row = (const T *)a.desc + (size_t)jm * D;
      if (vec && sizeof(T) == 2) {
        for (int i = tid * 8; i < D; i += MERGE_THREADS * 8) {
          const uint4 w = *reinterpret_cast<const uint4 *>(row + i);
          const T *e = reinterpret_cast<const T *>(&w);
#pragma unroll
          for (int q = 0; q < 8; ++q) acc[i + q] = first ? to_f32<T>(e[q]) * inv : fmaf(to_f32<T>(e[q]), inv, acc[i + q]);
        }
      } else {
        for (int i = tid; i < D; i += MERGE_THREADS) acc[i] = first ? to_f32<T>(row[i]) * inv : fmaf(to_f32<T>(row[i]), inv, acc[i]);
      }
    };
    __syncthreads();  // acc of the previous iteration is no longer read
    if (group <= 1) {  // the common case: the leader is the only member
      add_row((uint32_t)j, true);
      if (tid == 0) member_evidence((uint32_t)j);
    } else {
      bool first = true;
      for (int base = j & ~(MERGE_THREADS - 1); base < a.M; base += MERGE_THREADS) {  // members have index >= j
        const int jj = base + tid;
        const bool flag = jj < a.M && jj >= j && m.assoc[jj] == t;
        const unsigned b = __ballot_sync(0xFFFFFFFFu, flag);
        if (lane == 0) warp_cnt[warp] = __popc(b);
        __syncthreads();
        uint32_t before = 0, total = 0;
#pragma unroll
        for (int w = 0; w < MERGE_WARPS; ++w) {
          before += w < warp ? warp_cnt[w] : 0;
          total += warp_cnt[w];
        }
        if (flag) list[before + __popc(b & ((1u << lane) - 1))] = (uint32_t)jj;
        __syncthreads();
        for (uint32_t q = 0; q < total; ++q) {  // members in index order: deterministic summation
          add_row(list[q], first);
          first = false;
          if (tid == 0) member_evidence(list[q]);
        }
        __syncthreads();
      }
    }
    // f_o <- normalise(n_obs * f_o + sum)   (R21); each thread revisits exactly the elements it accumulated
    float ss = 0.f;
    if (vec && sizeof(T) == 2) {
      for (int i = tid * 8; i < D; i += MERGE_THREADS * 8) {
        float4 m0 = make_float4(0.f, 0.f, 0.f, 0.f), m1 = m0;
        if (n_old) m0 = *reinterpret_cast<const float4 *>(master + i), m1 = *reinterpret_cast<const float4 *>(master + i + 4);
        const float mv[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          const float v = n_old ? fmaf((float)n_old, mv[q], acc[i + q]) : acc[i + q];
          acc[i + q] = v;
          ss = fmaf(v, v, ss);
        }
      }
    } else {
      for (int i = tid; i < D; i += MERGE_THREADS) {
        const float v = n_old ? fmaf((float)n_old, master[i], acc[i]) : acc[i];
        acc[i] = v;
        ss = fmaf(v, v, ss);
      }
    }
#pragma unroll
    for (int sft = 16; sft; sft >>= 1) ss += __shfl_xor_sync(0xFFFFFFFFu, ss, sft);
    if (lane == 0) red[warp] = ss;
    __syncthreads();
    float tot = 0.f;
#pragma unroll
    for (int w = 0; w < MERGE_WARPS; ++w) tot += red[w];
    if (tot > 0.f) {  // a zero sum keeps the old value
      const float inv = 1.0f / sqrtf(tot);
      float s2 = 0.f;
      if (vec && sizeof(T) == 2) {
        for (int i = tid * 8; i < D; i += MERGE_THREADS * 8) {
          float v[8];
          uint4 w;
          T *e = reinterpret_cast<T *>(&w);
#pragma unroll
          for (int q = 0; q < 8; ++q) {
            v[q] = acc[i + q] * inv;
            e[q] = from_f32<T>(v[q]);  // round-to-nearest-even shadow (R1, R14)
            const float sv = to_f32<T>(e[q]);
            s2 = fmaf(sv, sv, s2);
          }
          *reinterpret_cast<float4 *>(master + i) = make_float4(v[0], v[1], v[2], v[3]);
          *reinterpret_cast<float4 *>(master + i + 4) = make_float4(v[4], v[5], v[6], v[7]);
          *reinterpret_cast<uint4 *>(shadow + i) = w;
        }
      } else {
        for (int i = tid; i < D; i += MERGE_THREADS) {
          const float v = acc[i] * inv;
          master[i] = v;
          const T sh = from_f32<T>(v);
          shadow[i] = sh;
          const float sv = to_f32<T>(sh);
          s2 = fmaf(sv, sv, s2);
        }
      }
#pragma unroll
      for (int sft = 16; sft; sft >>= 1) s2 += __shfl_xor_sync(0xFFFFFFFFu, s2, sft);
      if (lane == 0) red2[warp] = s2;
      __syncthreads();
      if (tid == 0) {
        float t2 = 0.f;
#pragma unroll
        for (int w = 0; w < MERGE_WARPS; ++w) t2 += red2[w];
        m.inv_norm[t] = t2 > 0.f ? 1.0f / sqrtf(t2) : 0.f;
      }
    }
    if (tid == 0) {
      m.n_obs[t] = n_old + k_members;
      m.n_points[t] = pts_old + pts;
#pragma unroll
      for (int c = 0; c < 3; ++c) {  // R22
        m.aabb[t * 6 + c] = min(box_old[c], bmn[c]);
        m.aabb[t * 6 + 3 + c] = max(box_old[3 + c], bmx[c]);
      }
      if (best > best_old) {
        m.best_view[t] = best;
        const float *Tf = a.T + 16 * best_frame;
        m.best_cam[t * 3 + 0] = Tf[3];
        m.best_cam[t * 3 + 1] = Tf[7];
        m.best_cam[t * 3 + 2] = Tf[11];
      }
      m.leader[t] = NONE32;
      m.grp_cnt[t] = 0;
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
}

int launch_cand_associate(const DevMap &m, const CallArgs &a, cudaStream_t s) {
  const int grid = a.M > 0 ? 37 : 1;  // 37 x 32 warps = one warp per candidate for ~1.2k candidates per wave
  FARM_DISPATCH((cand_associate_kernel<T><<<grid, 1024, 0, s>>>(m, a)));
  return 1;
}
int launch_commit_merge(const DevMap &m, const CallArgs &a, unsigned long long frame_seq0, cudaStream_t s) {
  if (a.M == 0) return 0;
  const int commit_blocks = 148 * 4;
  const int merge_blocks = a.M < 148 * 16 ? a.M : 148 * 16;  // one CTA per detection: a single wave
  FARM_DISPATCH((commit_merge_kernel<T><<<commit_blocks + merge_blocks, MERGE_THREADS, (size_t)m.D * sizeof(float), s>>>(
      m, a, frame_seq0, commit_blocks)));
  return 1;
}

}  // namespace farm
