// farm_sim_fma.cu -- step 4 on CUDA cores: dense detection x object cosine with a fused row max / argmax.
//   cos(a_d, b_o) for every detection d and every object o of the entry snapshot (R14-R16; PAPER.md:350
//   "a single batched detection-by-entity similarity matrix"), never materialised: the epilogue keeps
//   max_o clamp(cos) and its lowest-id argmax per detection (all the association needs, R19).
// This is the path for fp32 descriptors (config 0; TF32 tensor math would cost ~1e-4 of accuracy) and the
// fallback for the 16-bit dtypes; the tensor-core path lives in farm_sim_tc.cu.
#include "farm_internal.cuh"

namespace farm {
namespace {

constexpr int BM = 64, BN = 64, BK = 16, SIM_THREADS = 256;

template <typename T>
__global__ void __launch_bounds__(SIM_THREADS) similarity_fma_kernel(DevMap m, CallArgs a) {
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN + 4];
  const int N = (int)*m.n_objects, M = a.M, D = m.D;
  const int tiles_n = (N + BN - 1) / BN, tiles_m = (M + BM - 1) / BM;
  const T *A = (const T *)a.desc;
  const T *B = (const T *)m.desc_shadow;
  const int tid = threadIdx.x;
  const int ty = tid >> 4, tx = tid & 15;
  const int lr = tid >> 2, lk = (tid & 3) * 4;  // loader: row, first k
  for (int tile = blockIdx.x; tile < tiles_n * tiles_m; tile += gridDim.x) {
    const int tm = tile % tiles_m, tn = tile / tiles_m;
    const int m0 = tm * BM, n0 = tn * BN;
    float acc[4][4] = {};
    for (int k0 = 0; k0 < D; k0 += BK) {
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const int k = k0 + lk + q;
        As[lk + q][lr] = (m0 + lr < M && k < D) ? to_f32<T>(A[(size_t)(m0 + lr) * D + k]) : 0.f;
        Bs[lk + q][lr] = (n0 + lr < N && k < D) ? to_f32<T>(B[(size_t)(n0 + lr) * D + k]) : 0.f;
      }
      __syncthreads();
#pragma unroll
      for (int k = 0; k < BK; ++k) {
        float av[4], bv[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) av[q] = As[k][ty * 4 + q], bv[q] = Bs[k][tx * 4 + q];
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
          for (int c = 0; c < 4; ++c) acc[r][c] = fmaf(av[r], bv[c], acc[r][c]);
      }
      __syncthreads();
    }
    // fused epilogue: scale by the inverse norms (R15), clamp, row max / argmax (lowest id on ties)
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int row = m0 + ty * 4 + r;
      const float ia = row < M ? m.det_inv_norm[row] : 0.f;
      unsigned long long best = 0ull;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int col = n0 + tx * 4 + c;
        if (col < N) {
          float cs = acc[r][c] * ia * m.inv_norm[col];
          cs = fminf(1.f, fmaxf(-1.f, cs));
          if (row < M && cs > m.dense_thr) dense_emit(m, (uint32_t)row, (uint32_t)col, cs);  // H1 / U1 (off: thr = +inf)
          const unsigned long long p = pack_score(cs, (uint32_t)col);
          best = p > best ? p : best;
        }
      }
#pragma unroll
      for (int o = 8; o; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xFFFFFFFFu, best, o);
        best = other > best ? other : best;
      }
      if (tx == 0 && row < M && best) atomicMax(&m.best_dense[row], best);
    }
  }
}

}  // namespace

int launch_similarity_fma(const DevMap &m, const CallArgs &a, uint32_t n_upper, cudaStream_t s) {
  if (a.M == 0 || n_upper == 0) return 0;
  const long long tiles = (long long)((a.M + BM - 1) / BM) * ((n_upper + BN - 1) / BN);
  const int grid = (int)(tiles < m.num_sms * 4 ? tiles : m.num_sms * 4);
  if (m.dtype == FARM_DTYPE_F32)
    similarity_fma_kernel<float><<<grid, SIM_THREADS, 0, s>>>(m, a);
  else if (m.dtype == FARM_DTYPE_F16)
    similarity_fma_kernel<__half><<<grid, SIM_THREADS, 0, s>>>(m, a);
  else
    similarity_fma_kernel<__nv_bfloat16><<<grid, SIM_THREADS, 0, s>>>(m, a);
  return 1;
}

}  // namespace farm
