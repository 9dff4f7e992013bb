// H8 (depth digit) + H10: per-tile sort and front-to-back alpha compositing (PAPER.md:103 -> 3DGS rasteriser, DESIGN.md
// A18; black background PAPER.md:239-241 is the default of the bg parameter).
// One CTA per 16x16 tile.  The tile's bucket of (depth bits << 32 | Gaussian) keys (binned by sort_kernels.cu) is
// loaded into shared memory, sorted there with an ascending-only bitonic network (exact integer compare, so the order
// equals the stable (tile, depth) sort of the emission order), written back as the sorted key/value lists, and then
// blended front to back straight from shared memory in batches of 256; a CTA stops as soon as every pixel has saturated
// (T(1-alpha) < 1e-4).  The blend is FAST arithmetic (FMA, ex2.approx): compared with the fp64 oracle under tolerance.
#include "rga_internal.h"

#define CB 256

// ascending-only bitonic network on buf[0..n): every compare-exchange puts the minimum at the lower index, so virtual
// +inf padding above n never moves and n need not be a power of two.
__device__ __forceinline__ void bitonic_sort(unsigned long long* buf, int n) {
  for (int k = 2; (k >> 1) < n; k <<= 1) {
    for (int i = threadIdx.x; i < n; i += CB) {             // mirror step: i <-> i ^ (k-1)
      int p = i ^ (k - 1);
      if (p > i && p < n) { unsigned long long a = buf[i], b = buf[p]; if (b < a) { buf[i] = b; buf[p] = a; } }
    }
    __syncthreads();
    for (int j = k >> 2; j > 0; j >>= 1) {
      for (int i = threadIdx.x; i < n; i += CB) {
        int p = i ^ j;
        if (p > i && p < n) { unsigned long long a = buf[i], b = buf[p]; if (b < a) { buf[i] = b; buf[p] = a; } }
      }
      __syncthreads();
    }
  }
}

// Handles the tiles whose bucket length n satisfies n_lo < n <= n_hi (others return at once); buckets longer than the
// shared-memory capacity `scap` are sorted in place in global memory by the same network.
__global__ void __launch_bounds__(CB) composite_kernel(int W, int H, int TX, unsigned capacity, int scap, int n_lo, int n_hi,
    const uint2* __restrict__ ranges, unsigned long long* __restrict__ lkeys, unsigned long long* __restrict__ keys_out,
    unsigned* __restrict__ vals_out, const float2* __restrict__ mu2d, const float4* __restrict__ conic_o,
    const float4* __restrict__ color, float3 bg, float* __restrict__ image, float* __restrict__ t_final,
    unsigned* __restrict__ n_contrib) {
  extern __shared__ __align__(16) unsigned long long s_keys[];
  __shared__ float2 s_mu[CB];
  __shared__ float4 s_co[CB];
  __shared__ float4 s_col[CB];
  const int tile = blockIdx.y * TX + blockIdx.x;
  uint2 rg = ranges[tile];
  rg.x = min(rg.x, capacity); rg.y = min(rg.y, capacity);
  const int n = (int)(rg.y - rg.x);
  if (n <= n_lo || n > n_hi) return;
  unsigned long long* buf = lkeys + rg.x;
  if (n <= scap) {
    for (int i = threadIdx.x; i < n; i += CB) s_keys[i] = buf[i];
    buf = s_keys;
  }
  __syncthreads();
  bitonic_sort(buf, n);
  for (int i = threadIdx.x; i < n; i += CB) {                // the sorted (tile, depth) keys and values (H8 output)
    unsigned long long k = buf[i];
    keys_out[rg.x + i] = ((unsigned long long)(unsigned)tile << 32) | (k >> 32);
    vals_out[rg.x + i] = (unsigned)k;
  }
  const int px = blockIdx.x * RGA_TILE + (threadIdx.x & 15), py = blockIdx.y * RGA_TILE + (threadIdx.x >> 4);
  const bool inside = px < W && py < H;
  const float fx = (float)px + 0.5f, fy = (float)py + 0.5f;        // DESIGN.md A21: sample at the pixel centre
  bool done = !inside;
  float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
  unsigned last = 0;
  for (int b = 0; b < n; b += CB) {
    if (__syncthreads_count(done) == CB) break;
    const int m = min(CB, n - b);
    if ((int)threadIdx.x < m) {
      unsigned g = (unsigned)buf[b + threadIdx.x];
      s_mu[threadIdx.x] = mu2d[g]; s_co[threadIdx.x] = conic_o[g]; s_col[threadIdx.x] = color[g];
    }
    __syncthreads();
    // four entries per trip: their alphas are independent (ILP for the exp chain); only the blend is sequential
    for (int j = 0; j < m && !done; j += 4) {
      float a[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const float2 mm = s_mu[j + u]; const float4 co = s_co[j + u];
        const float dx = mm.x - fx, dy = mm.y - fy;
        const float power = -0.5f * (co.x * dx * dx + co.z * dy * dy) - co.y * dx * dy;
        const float al = fminf(0.99f, co.w * __expf(power));
        a[u] = (power > 0.f || j + u >= m) ? 0.f : al;
      }
      if (fmaxf(fmaxf(a[0], a[1]), fmaxf(a[2], a[3])) < 1.f / 255.f) continue;
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (!done && a[u] >= 1.f / 255.f) {
          const float test_T = T * (1.f - a[u]);
          if (test_T < 1e-4f) done = true;
          else {
            const float4 c = s_col[j + u];
            const float w = a[u] * T;
            C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
            T = test_T; last = (unsigned)(b + j + u + 1);
          }
        }
      }
    }
  }
  if (inside) {
    size_t p = (size_t)py * W + px;
    image[3 * p] = C0 + T * bg.x; image[3 * p + 1] = C1 + T * bg.y; image[3 * p + 2] = C2 + T * bg.z;
    t_final[p] = T; n_contrib[p] = last;
  }
}

// empty tiles: background only
__global__ void __launch_bounds__(256) clear_kernel(int npix, float3 bg, float* __restrict__ image, float* __restrict__ t_final,
                                                    unsigned* __restrict__ n_contrib) {
  int p = blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= npix) return;
  image[3 * p] = bg.x; image[3 * p + 1] = bg.y; image[3 * p + 2] = bg.z; t_final[p] = 1.f; n_contrib[p] = 0u;
}

#define SCAP_SMALL 2048
#define SCAP_LARGE 24576

int rga_composite_init_attributes() {
  return (int)cudaFuncSetAttribute(composite_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, SCAP_LARGE * 8);
}

cudaError_t rga_launch_composite(rga_avatar* av, const rga_camera* cam, float3 bg, float* out, cudaStream_t s) {
  int TX = (cam->width + RGA_TILE - 1) / RGA_TILE, TY = (cam->height + RGA_TILE - 1) / RGA_TILE;
  int npix = cam->width * cam->height;
  clear_kernel<<<(npix + 255) / 256, 256, 0, s>>>(npix, bg, out, av->t_final, av->n_contrib);
  rga_prof_mark(av, "clear", s);
#define COMP_ARGS(scap, lo, hi) cam->width, cam->height, TX, (unsigned)av->max_dup, scap, lo, hi, av->ranges, av->keys[0], av->keys[1], \
    av->vals[0], av->mu2d, av->conic_o, av->color, bg, out, av->t_final, av->n_contrib
  composite_kernel<<<dim3(TX, TY), CB, SCAP_SMALL * 8, s>>>(COMP_ARGS(SCAP_SMALL, 0, SCAP_SMALL));
  rga_prof_mark(av, "composite", s);
  composite_kernel<<<dim3(TX, TY), CB, SCAP_LARGE * 8, s>>>(COMP_ARGS(SCAP_LARGE, SCAP_SMALL, 0x7fffffff));
  rga_prof_mark(av, "composite_long", s);
  av->launches += 3;
  return cudaGetLastError();
}
