// H10 per-tile front-to-back alpha compositing (PAPER.md:103 -> 3DGS rasteriser, A18; black background
// PAPER.md:239-241 is the default of the bg parameter).  FAST file: compared with the fp64 oracle under tolerance.
// One CTA per 16x16 tile; the tile's sorted Gaussian list is staged through shared memory in batches of 256;
// a CTA stops as soon as every pixel has saturated (T(1-alpha) < 1e-4).
#include "rga_internal.h"

#define CB 256

__global__ void __launch_bounds__(CB) composite_kernel(int W, int H, int TX, const uint2* __restrict__ ranges,
    const unsigned* __restrict__ vals, const float2* __restrict__ mu2d, const float4* __restrict__ conic_o,
    const float4* __restrict__ color, float3 bg, float* __restrict__ image, float* __restrict__ t_final,
    unsigned* __restrict__ n_contrib) {
  __shared__ float2 s_mu[CB];
  __shared__ float4 s_co[CB];
  __shared__ float4 s_col[CB];
  const int tile = blockIdx.y * TX + blockIdx.x;
  const int px = blockIdx.x * RGA_TILE + (threadIdx.x & 15), py = blockIdx.y * RGA_TILE + (threadIdx.x >> 4);
  const bool inside = px < W && py < H;
  const float fx = (float)px + 0.5f, fy = (float)py + 0.5f;        // DESIGN.md A21: sample at the pixel centre
  const uint2 rg = ranges[tile];
  int todo = (int)(rg.y - rg.x);
  bool done = !inside;
  float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
  unsigned contributor = 0, last = 0;
  for (unsigned b = rg.x; todo > 0; b += CB, todo -= CB) {
    if (__syncthreads_count(done) == CB) break;
    if ((int)threadIdx.x < todo) {
      unsigned g = vals[b + threadIdx.x];
      s_mu[threadIdx.x] = mu2d[g]; s_co[threadIdx.x] = conic_o[g]; s_col[threadIdx.x] = color[g];
    }
    __syncthreads();
    int n = min(CB, todo);
    for (int j = 0; !done && j < n; ++j) {
      ++contributor;
      float2 m = s_mu[j]; float4 co = s_co[j];
      float dx = m.x - fx, dy = m.y - fy;
      float power = -0.5f * (co.x * dx * dx + co.z * dy * dy) - co.y * dx * dy;
      if (power > 0.f) continue;
      float alpha = fminf(0.99f, co.w * __expf(power));
      if (alpha < 1.f / 255.f) continue;
      float test_T = T * (1.f - alpha);
      if (test_T < 1e-4f) { done = true; continue; }
      float4 c = s_col[j];
      float w = alpha * T;
      C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
      T = test_T; last = contributor;
    }
  }
  if (inside) {
    size_t p = (size_t)py * W + px;
    image[3 * p] = C0 + T * bg.x; image[3 * p + 1] = C1 + T * bg.y; image[3 * p + 2] = C2 + T * bg.z;
    t_final[p] = T; n_contrib[p] = last;
  }
}

cudaError_t rga_launch_composite(rga_avatar* av, const rga_camera* cam, float3 bg, float* out, cudaStream_t s) {
  int TX = (cam->width + RGA_TILE - 1) / RGA_TILE, TY = (cam->height + RGA_TILE - 1) / RGA_TILE;
  composite_kernel<<<dim3(TX, TY), CB, 0, s>>>(cam->width, cam->height, TX, av->ranges, av->vals[av->sorted_buf], av->mu2d,
                                               av->conic_o, av->color, bg, out, av->t_final, av->n_contrib);
  av->launches += 1;
  rga_prof_mark(av, "composite", s);
  return cudaGetLastError();
}
