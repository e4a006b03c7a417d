// farm_noalloc.cu -- farm_cosine_rowmax_noalloc: step 4 (dense cosine with fused row max / argmax, R14-R16, R18;
// PAPER.md:350) for callers that cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc.  A variant of similarity_fma_kernel (farm_sim_fma.cu) whose scratch -- the inverse row norms of both
// operands and the packed (max, argmax) word per row that the epilogue's atomicMax works on -- lives in ONE file-scope
// device array instead of a map's allocations.  The entry point calls no cudaMalloc / cudaFree and no allocating library
// routine.  Every GPU that loads the library holds the array (FARM_NOALLOC_SCRATCH_BYTES = 304 KB) until the process exits.
// All calls share it and it keeps the last call's contents: each call rewrites the norms it reads and clears the packed
// words of its rows first; two calls that overlap on the GPU (different streams) race on it.
#include <mutex>
#include <string>

#include "farm_internal.cuh"

namespace farm {
namespace {

constexpr int NA_MAX_M = FARM_NOALLOC_MAX_M, NA_MAX_N = FARM_NOALLOC_MAX_N;
constexpr size_t OFF_INV_A = 0;                                   // float [NA_MAX_M]
constexpr size_t OFF_INV_B = OFF_INV_A + (size_t)NA_MAX_M * 4;    // float [NA_MAX_N]
constexpr size_t OFF_BEST = OFF_INV_B + (size_t)NA_MAX_N * 4;     // unsigned long long [NA_MAX_M]
constexpr size_t SCRATCH_BYTES = OFF_BEST + (size_t)NA_MAX_M * 8;
static_assert(SCRATCH_BYTES == FARM_NOALLOC_SCRATCH_BYTES, "farm.h states the size of the scratch array");
static_assert(OFF_INV_B % 256 == 0 && OFF_BEST % 256 == 0, "sub-arrays stay 256-byte aligned");

// In host code this name is a host-side stand-in, NOT a device address: kernels get the address that
// cudaGetSymbolAddress returns for the current device (scratch_of_current_device below).
static __device__ __align__(256) unsigned char g_noalloc_scratch[SCRATCH_BYTES];

struct Scratch {
  float *inv_a, *inv_b;
  unsigned long long *best;
};

// inverse norms of the M rows of A and the N rows of B (one warp per row; R15 explicit norms, 0 for a zero row) and the
// cleared (max, argmax) words of this call's rows
template <typename T>
__global__ void noalloc_prep_kernel(const T *A, int M, const T *B, int N, int D, Scratch sc) {
  const int row = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (row >= M + N) return;
  const T *p = row < M ? A + (size_t)row * D : B + (size_t)(row - M) * D;
  float s = 0.f;
  for (int i = lane; i < D; i += 32) {
    const float x = to_f32<T>(p[i]);
    s = fmaf(x, x, s);
  }
#pragma unroll
  for (int o = 16; o; o >>= 1) s += __shfl_xor_sync(0xFFFFFFFFu, s, o);
  if (lane == 0) {
    const float inv = s > 0.f ? 1.0f / sqrtf(s) : 0.f;
    if (row < M)
      sc.inv_a[row] = inv, sc.best[row] = 0ull;
    else
      sc.inv_b[row - M] = inv;
  }
}

constexpr int BM = 64, BN = 64, BK = 16, SIM_THREADS = 256;

// similarity_fma_kernel with plain operands: same tiling, same accumulation order, same epilogue (scale, clamp, packed
// row max with the lowest id winning ties)
template <typename T>
__global__ void __launch_bounds__(SIM_THREADS) noalloc_similarity_kernel(const T *A, int M, const T *B, int N, int D, Scratch sc) {
  __shared__ float As[BK][BM + 4];
  __shared__ float Bs[BK][BN + 4];
  const int tiles_n = (N + BN - 1) / BN, tiles_m = (M + BM - 1) / BM;
  const int tid = threadIdx.x;
  const int ty = tid >> 4, tx = tid & 15;
  const int lr = tid >> 2, lk = (tid & 3) * 4;
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
#pragma unroll
    for (int r = 0; r < 4; ++r) {
      const int row = m0 + ty * 4 + r;
      const float ia = row < M ? sc.inv_a[row] : 0.f;
      unsigned long long best = 0ull;
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        const int col = n0 + tx * 4 + c;
        if (col < N) {
          float cs = acc[r][c] * ia * sc.inv_b[col];
          cs = fminf(1.f, fmaxf(-1.f, cs));
          const unsigned long long p = pack_score(cs, (uint32_t)col);
          best = p > best ? p : best;
        }
      }
#pragma unroll
      for (int o = 8; o; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(0xFFFFFFFFu, best, o);
        best = other > best ? other : best;
      }
      if (tx == 0 && row < M && best) atomicMax(&sc.best[row], best);
    }
  }
}

__global__ void noalloc_unpack_kernel(int M, Scratch sc, float *max_cos, int32_t *argmax) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= M) return;
  const unsigned long long p = sc.best[j];
  if (max_cos) max_cos[j] = p ? unpack_score(p) : 0.f;
  if (argmax) argmax[j] = p ? (int32_t)unpack_id(p) : -1;
}

// Device address of the scratch array on the CURRENT device, looked up once per device.
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char *g_addr[MAX_DEVICES] = {};
int g_sms[MAX_DEVICES] = {};

cudaError_t scratch_of_current_device(Scratch *out, int *num_sms) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_addr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);  // with `dev` current: the address is per device
    if (e != cudaSuccess) return e;
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    g_addr[dev] = (unsigned char *)p, g_sms[dev] = sms;
  }
  unsigned char *base = g_addr[dev];
  out->inv_a = (float *)(base + OFF_INV_A);
  out->inv_b = (float *)(base + OFF_INV_B);
  out->best = (unsigned long long *)(base + OFF_BEST);
  *num_sms = g_sms[dev];
  return cudaSuccess;
}

template <typename T>
void launch_all(const void *A, int M, const void *B, int N, int D, const Scratch &sc, int num_sms, float *max_cos, int32_t *argmax,
                cudaStream_t s) {
  const long long rows = (long long)M + N;
  noalloc_prep_kernel<T><<<(unsigned)((rows * 32 + 255) / 256), 256, 0, s>>>((const T *)A, M, (const T *)B, N, D, sc);
  if (N > 0) {
    const long long tiles = (long long)((M + BM - 1) / BM) * ((N + BN - 1) / BN);
    const int grid = (int)(tiles < (long long)num_sms * 4 ? tiles : (long long)num_sms * 4);
    noalloc_similarity_kernel<T><<<grid, SIM_THREADS, 0, s>>>((const T *)A, M, (const T *)B, N, D, sc);
  }
  noalloc_unpack_kernel<<<(M + 255) / 256, 256, 0, s>>>(M, sc, max_cos, argmax);
}

}  // namespace

int noalloc_cosine_rowmax(const void *A, int M, const void *B, int N, int D, int dtype, float *max_cos, int32_t *argmax,
                          cudaStream_t s, std::string *err) {
  if (M == 0) return FARM_OK;
  Scratch sc;
  int num_sms = 0;
  cudaError_t e = scratch_of_current_device(&sc, &num_sms);
  if (e != cudaSuccess) {
    *err = std::string("farm_cosine_rowmax_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e);
    return FARM_ERR_CUDA;
  }
  if (dtype == FARM_DTYPE_F32)
    launch_all<float>(A, M, B, N, D, sc, num_sms, max_cos, argmax, s);
  else if (dtype == FARM_DTYPE_F16)
    launch_all<__half>(A, M, B, N, D, sc, num_sms, max_cos, argmax, s);
  else
    launch_all<__nv_bfloat16>(A, M, B, N, D, sc, num_sms, max_cos, argmax, s);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    *err = std::string("farm_cosine_rowmax_noalloc: launch: ") + cudaGetErrorString(e);
    return FARM_ERR_CUDA;
  }
  return FARM_OK;
}

}  // namespace farm
