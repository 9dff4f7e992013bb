// Library-side ordering of the Gaussians (BASELINE.json configs: "Gaussians placed on random
// surface points" -- PAPER.md:88-93 defines no order, so a trained asset's order is arbitrary).
//
// avatar_load sorts the Gaussians ONCE by the Morton code of their canonical position and keeps the permutation: every
// per-Gaussian table and scratch buffer of the library is stored in that spatial order (neighbouring threads then test
// neighbouring depth-map texels, agree on the shading skip tests and hit the same screen tiles), while everything the
// caller sees -- input arrays, [n_gauss] outputs and gradients, the Gaussian indices in the sorted splat lists, what
// rga_read_buffer returns -- stays in the CALLER's order.  No method arithmetic here: a permutation of independent items.
#include "rga_internal.h"

__device__ __forceinline__ unsigned f2ord(float f) { unsigned u = __float_as_uint(f); return (u & 0x80000000u) ? ~u : (u | 0x80000000u); }
__device__ __forceinline__ float ord2f(unsigned u) { return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u); }

// min / max of n points (device reduction; replaces a host loop): bb[0..2] = min as ordered uints, bb[3..5] = max
__global__ void __launch_bounds__(256) aabb_points_kernel(int n, const float* __restrict__ p, unsigned* __restrict__ bb) {
  float lo[3] = {3.4e38f, 3.4e38f, 3.4e38f}, hi[3] = {-3.4e38f, -3.4e38f, -3.4e38f};
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
#pragma unroll
    for (int c = 0; c < 3; ++c) { const float v = p[3 * (size_t)i + c]; lo[c] = fminf(lo[c], v); hi[c] = fmaxf(hi[c], v); }
#pragma unroll
  for (int c = 0; c < 3; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      lo[c] = fminf(lo[c], __shfl_xor_sync(0xffffffffu, lo[c], o)); hi[c] = fmaxf(hi[c], __shfl_xor_sync(0xffffffffu, hi[c], o));
    }
    if ((threadIdx.x & 31) == 0) { atomicMin(bb + c, f2ord(lo[c])); atomicMax(bb + 3 + c, f2ord(hi[c])); }
  }
}

__global__ void aabb_decode_kernel(const unsigned* __restrict__ bb, float* __restrict__ out) {
  if (threadIdx.x < 6) out[threadIdx.x] = ord2f(bb[threadIdx.x]);
}

cudaError_t rga_points_aabb(const float* pos, int n, unsigned* scratch6, float* out6_dev, cudaStream_t s) {
  const unsigned init[6] = {0xffffffffu, 0xffffffffu, 0xffffffffu, 0u, 0u, 0u};
  cudaError_t e = cudaMemcpyAsync(scratch6, init, sizeof init, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return e;
  int grid = (n + 255) / 256; if (grid > 1024) grid = 1024;
  aabb_points_kernel<<<grid, 256, 0, s>>>(n, pos, scratch6);
  aabb_decode_kernel<<<1, 32, 0, s>>>(scratch6, out6_dev);
  return cudaGetLastError();
}

__device__ __forceinline__ unsigned spread10(unsigned x) {
  x &= 0x3ffu;
  x = (x | (x << 16)) & 0x030000ffu; x = (x | (x << 8)) & 0x0300f00fu;
  x = (x | (x << 4)) & 0x030c30c3u; x = (x | (x << 2)) & 0x09249249u;
  return x;
}

// key = Morton code (10 bits per axis over the points' bounding box) << 32 | index; padding entries sort last
__global__ void morton_key_kernel(int n, int npad, const float* __restrict__ p, const float* __restrict__ bb,
                                  unsigned long long* __restrict__ keys) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= npad) return;
  if (i >= n) { keys[i] = ~0ull; return; }
  unsigned q[3];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float lo = bb[c], ext = bb[3 + c] - lo;
    const float t = ext > 0.f ? (p[3 * (size_t)i + c] - lo) / ext : 0.f;
    q[c] = (unsigned)fminf(fmaxf(t * 1023.0f, 0.0f), 1023.0f);
  }
  const unsigned code = spread10(q[0]) | (spread10(q[1]) << 1) | (spread10(q[2]) << 2);
  keys[i] = ((unsigned long long)code << 32) | (unsigned)i;
}

// one compare-exchange stage of an ascending bitonic network in global memory (load time only; keys are unique)
__global__ void bitonic_stage_kernel(unsigned long long* __restrict__ keys, int npad, int j, int k) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= npad / 2) return;
  const int i = 2 * t - (t & (j - 1));                      // lower index of pair t for partner distance j
  const int p = i + j;
  const bool up = (i & k) == 0;
  const unsigned long long a = keys[i], b = keys[p];
  if ((a > b) == up) { keys[i] = b; keys[p] = a; }
}

// the last stages (partner distance < 1024) of one merge step inside shared memory: 2,048 keys per CTA
__global__ void __launch_bounds__(1024) bitonic_tail_kernel(unsigned long long* __restrict__ keys, int npad, int jstart, int k, int all_k) {
  __shared__ unsigned long long s[2048];
  const int base = blockIdx.x * 2048;
  s[threadIdx.x] = keys[base + threadIdx.x]; s[threadIdx.x + 1024] = keys[base + threadIdx.x + 1024];
  __syncthreads();
  // all_k: run the whole network for k = 2 .. 2048 (the first steps of the sort); else the stages j = jstart .. 1 of step k
  for (int kk = all_k ? 2 : k; kk <= (all_k ? 2048 : k); kk <<= 1) {
    for (int j = all_k ? (kk >> 1) : jstart; j > 0; j >>= 1) {
      const int t = threadIdx.x, i = 2 * t - (t & (j - 1)), p = i + j;
      const bool up = ((base + i) & kk) == 0;
      const unsigned long long a = s[i], b = s[p];
      if ((a > b) == up) { s[i] = b; s[p] = a; }
      __syncthreads();
    }
  }
  keys[base + threadIdx.x] = s[threadIdx.x]; keys[base + threadIdx.x + 1024] = s[threadIdx.x + 1024];
}

__global__ void order_finish_kernel(int n, const unsigned long long* __restrict__ keys, int* __restrict__ order, int* __restrict__ inv) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int g = (int)(unsigned)(keys[i] & 0xffffffffull);
  order[i] = g; inv[g] = i;
}

// dst[i][:] = src[order[i]][:]   (caller order -> library order), rows of C 32-bit words
__global__ void gather_rows_kernel(int n, int C, const unsigned* __restrict__ src, const int* __restrict__ order, unsigned* __restrict__ dst) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)n * C) return;
  const int i = (int)(t / C), c = (int)(t - (long long)i * C);
  dst[t] = src[(size_t)order[i] * C + c];
}

// dst[order[i]][:] = src[i][:]   (library order -> caller order)
__global__ void scatter_rows_kernel(int n, int C, const unsigned* __restrict__ src, const int* __restrict__ order, unsigned* __restrict__ dst) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= (long long)n * C) return;
  const int i = (int)(t / C), c = (int)(t - (long long)i * C);
  dst[(size_t)order[i] * C + c] = src[t];
}

cudaError_t rga_gather_rows(int n, int words_per_row, const void* src, const int* order, void* dst, cudaStream_t s) {
  const long long tot = (long long)n * words_per_row;
  gather_rows_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(n, words_per_row, (const unsigned*)src, order, (unsigned*)dst);
  return cudaGetLastError();
}

cudaError_t rga_scatter_rows(int n, int words_per_row, const void* src, const int* order, void* dst, cudaStream_t s) {
  const long long tot = (long long)n * words_per_row;
  scatter_rows_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, s>>>(n, words_per_row, (const unsigned*)src, order, (unsigned*)dst);
  return cudaGetLastError();
}

// Spatial order of n points: order[i] = caller index of the i-th point in Morton order, inv = its inverse.
// keys: scratch of npad = max(2048, next power of two >= n) u64; bb_dev: float[6] scratch; bb_u: unsigned[6] scratch.
cudaError_t rga_build_gauss_order(const float* pos, int n, unsigned long long* keys, int npad, unsigned* bb_u, float* bb_dev,
                                  int* order, int* inv, cudaStream_t s) {
  cudaError_t e = rga_points_aabb(pos, n, bb_u, bb_dev, s);
  if (e != cudaSuccess) return e;
  morton_key_kernel<<<(npad + 255) / 256, 256, 0, s>>>(n, npad, pos, bb_dev, keys);
  bitonic_tail_kernel<<<npad / 2048, 1024, 0, s>>>(keys, npad, 0, 0, 1);              // k = 2 .. 2048
  for (int k = 4096; k <= npad; k <<= 1) {
    for (int j = k >> 1; j >= 1024; j >>= 1) bitonic_stage_kernel<<<(npad / 2 + 255) / 256, 256, 0, s>>>(keys, npad, j, k);
    bitonic_tail_kernel<<<npad / 2048, 1024, 0, s>>>(keys, npad, 512, k, 0);          // j = 512 .. 1
  }
  order_finish_kernel<<<(n + 255) / 256, 256, 0, s>>>(n, keys, order, inv);
  return cudaGetLastError();
}
