// gm_boot.cuh -- kernels of the bootstrap row (Sec. 5.2; reading B1):
// the list of used pixels, the counter-based draws with replacement, the fold of the
// multiplicities into the weights of a refit, and the population variance of the refits.
// The draw follows the definition in include/gm.h; it shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace gm {

__device__ __forceinline__ unsigned long long boot_mix64(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

// used[b][k] = row-major index of the k-th pixel of galaxy b with mask != 0; n_used[b] = their
// number.  One CTA per galaxy; chunks of 1024 pixels are scanned in order, so the list is
// ascending.  mask == nullptr: every pixel is used and the list is not read.
constexpr int kUsedThreads = 1024;
__global__ void __launch_bounds__(kUsedThreads) k_used_list(int N, const uint8_t* __restrict__ mask,
                                                            int* __restrict__ used, int* __restrict__ n_used) {
  __shared__ int wsum[kUsedThreads / 32];
  __shared__ int base;
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (!mask) {
    if (tid == 0) n_used[b] = N;
    return;
  }
  const uint8_t* mk = mask + (size_t)b * N;
  int* out = used + (size_t)b * N;
  if (tid == 0) base = 0;
  __syncthreads();
  for (int p0 = 0; p0 < N; p0 += kUsedThreads) {
    const int p = p0 + tid;
    const int f = (p < N && mk[p] != 0) ? 1 : 0;
    const unsigned bal = __ballot_sync(0xffffffffu, f);
    const int in_warp = __popc(bal & ((1u << lane) - 1u));
    if (lane == 0) wsum[wid] = __popc(bal);
    __syncthreads();
    int off = base;
    for (int w = 0; w < wid; ++w) off += wsum[w];
    if (f) out[off + in_warp] = p;
    __syncthreads();
    if (tid == 0) {
      int t = 0;
      for (int w = 0; w < kUsedThreads / 32; ++w) t += wsum[w];
      base += t;
    }
    __syncthreads();
  }
  if (tid == 0) n_used[b] = base;
}

// one thread per draw d of galaxy blockIdx.y; integer atomics, so the counts do not depend on order
__global__ void k_boot_draw(int N, unsigned long long seed, unsigned long long id0, unsigned long long r,
                            const int* __restrict__ used, const int* __restrict__ n_used, int has_mask,
                            int* __restrict__ counts) {
  const int b = blockIdx.y;
  const int d = blockIdx.x * blockDim.x + threadIdx.x;
  const int nu = n_used[b];
  if (d >= nu) return;
  const unsigned long long id = id0 + (unsigned long long)b;
  const unsigned long long base = boot_mix64(boot_mix64(seed ^ (id * 0x9E3779B97F4A7C15ull)) + r);
  const unsigned long long z = boot_mix64(base + (unsigned long long)d);
  const unsigned long long k = ((z >> 32) * (unsigned long long)nu) >> 32;
  const int pix = has_mask ? used[(size_t)b * N + k] : (int)k;
  atomicAdd(counts + (size_t)b * N + pix, 1);
}

// weights of the refit: w = c / sigma^2 as sigma_r = sigma / sqrt(c) with mask_r = (c > 0)
__global__ void k_boot_fold(long long n, const int* __restrict__ counts, const float* __restrict__ sigma,
                            float* __restrict__ sigma_r, uint8_t* __restrict__ mask_r) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int c = counts[i];
  const float s = sigma[i];
  sigma_r[i] = c > 0 ? s / sqrtf((float)c) : s;
  mask_r[i] = c > 0 ? 1 : 0;
}

// sigma^2 = (1/M) sum (m_i - mean)^2, fp64, resample order
__global__ void k_boot_stats(int BP, int M, const float* __restrict__ samples, float* __restrict__ sigma_boot,
                             float* __restrict__ mean_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= BP) return;
  double s = 0.0;
  for (int r = 0; r < M; ++r) s += (double)samples[(size_t)r * BP + i];
  const double mean = s / M;
  double v = 0.0;
  for (int r = 0; r < M; ++r) {
    const double d = (double)samples[(size_t)r * BP + i] - mean;
    v += d * d;
  }
  sigma_boot[i] = (float)sqrt(v / M);
  if (mean_out) mean_out[i] = (float)mean;
}

}  // namespace gm
