// Losses of the paper's training objective: Eq.5 image loss ("the same image loss as
// 3DGS": (1 - lambda) L1 + lambda (1 - SSIM), 11x11 Gaussian window sigma 1.5, zero padding; reading A34) with its
// gradient dL/dimage -- the input of splat_backward -- and the regularisers Eq.6-9 (:134-148) with theirs.
// FAST source: compared with the fp64 oracle under tolerance.
//
//   ssim_maps_kernel   one CTA per 16x16 pixel tile, channel by channel: the tile plus a 5-pixel halo of both images in
//                      shared memory, the five window means (I, J, I^2, J^2, I J) by a horizontal then a vertical 11-tap
//                      pass, SSIM of the pixel, and the three maps A = dS/dmu (total), B = dS/dsigma^2, C = dS/dsigma_12
//                      that the gradient needs; block sums of SSIM and |I - J| go to two double accumulators.
//   ssim_grad_kernel   same tiling over the maps: dL/dI = (1 - lambda) sign(I - J) / N - lambda / N (w*A + 2 I w*B + J w*C).
#include "rga_internal.h"

#define LT 16
#define LH 5
#define LW (LT + 2 * LH)

struct SsimWin { float w[11]; };

__device__ __forceinline__ float block_sum256(float v, float* s_red) {
#pragma unroll
  for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
  __syncthreads();
  float t = 0.f;
  if (threadIdx.x < 8) t = s_red[threadIdx.x];
  if (threadIdx.x < 32) {
#pragma unroll
    for (int o = 4; o; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
  }
  __syncthreads();
  return t;            // valid in thread 0
}

__global__ void __launch_bounds__(256) ssim_maps_kernel(int W, int H, SsimWin win, const float* __restrict__ img, const float* __restrict__ tgt,
    float* __restrict__ maps, double* __restrict__ sums) {
  __shared__ float sI[LW][LW + 1], sJ[LW][LW + 1];
  __shared__ float sH[5][LW][LT + 1];
  __shared__ float s_red[8];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int x0 = blockIdx.x * LT, y0 = blockIdx.y * LT;
  const int px = x0 + tx, py = y0 + ty;
  const bool inside = px < W && py < H;
  float ssim_acc = 0.f, l1_acc = 0.f;
  for (int c = 0; c < 3; ++c) {
    __syncthreads();
    for (int t = threadIdx.x; t < LW * LW; t += 256) {
      const int r = t / LW, q = t - r * LW;
      const int yy = y0 + r - LH, xx = x0 + q - LH;
      const bool in = yy >= 0 && yy < H && xx >= 0 && xx < W;
      sI[r][q] = in ? img[3 * ((size_t)yy * W + xx) + c] : 0.f;
      sJ[r][q] = in ? tgt[3 * ((size_t)yy * W + xx) + c] : 0.f;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < LW * LT; t += 256) {                    // horizontal pass
      const int r = t / LT, q = t - r * LT;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) {
        const float p = sI[r][q + k], s = sJ[r][q + k], w = win.w[k];
        a0 = fmaf(w, p, a0); a1 = fmaf(w, s, a1); a2 = fmaf(w, p * p, a2); a3 = fmaf(w, s * s, a3); a4 = fmaf(w, p * s, a4);
      }
      sH[0][r][q] = a0; sH[1][r][q] = a1; sH[2][r][q] = a2; sH[3][r][q] = a3; sH[4][r][q] = a4;
    }
    __syncthreads();
    float m[5] = {0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int k = 0; k < 11; ++k) {
      const float w = win.w[k];
#pragma unroll
      for (int u = 0; u < 5; ++u) m[u] = fmaf(w, sH[u][ty + k][tx], m[u]);
    }
    if (inside) {
      const float m1 = m[0], m2 = m[1], s1 = m[2] - m1 * m1, s2 = m[3] - m2 * m2, s12 = m[4] - m1 * m2;
      const float C1 = 1e-4f, C2 = 9e-4f;
      const float a1 = 2.f * m1 * m2 + C1, a2 = 2.f * s12 + C2, b1 = m1 * m1 + m2 * m2 + C1, b2 = s1 + s2 + C2;
      const float ib = 1.f / (b1 * b2);
      const float S = a1 * a2 * ib;
      const float dS_dm1 = 2.f * m2 * a2 * ib - S * 2.f * m1 / b1;       // sigma terms held fixed
      const float B = -S / b2, Cm = 2.f * a1 * ib;
      const float A = dS_dm1 - 2.f * m1 * B - m2 * Cm;                   // sigma^2 = w*I^2 - mu^2, sigma_12 = w*(I J) - mu mu^
      float* mp = maps + 9 * ((size_t)py * W + px) + 3 * c;
      mp[0] = A; mp[1] = B; mp[2] = Cm;
      ssim_acc += S;
      l1_acc += fabsf(sI[ty + LH][tx + LH] - sJ[ty + LH][tx + LH]);
    }
  }
  const float s0 = block_sum256(ssim_acc, s_red), s1 = block_sum256(l1_acc, s_red);
  if (threadIdx.x == 0) { atomicAdd(sums, (double)s0); atomicAdd(sums + 1, (double)s1); }
}

__global__ void __launch_bounds__(256) ssim_grad_kernel(int W, int H, SsimWin win, float lam, const float* __restrict__ img,
    const float* __restrict__ tgt, const float* __restrict__ maps, float* __restrict__ d_image) {
  __shared__ float sM[3][LW][LW + 1];
  __shared__ float sH[3][LW][LT + 1];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int x0 = blockIdx.x * LT, y0 = blockIdx.y * LT;
  const int px = x0 + tx, py = y0 + ty;
  const bool inside = px < W && py < H;
  const float inv_n = 1.f / (3.f * (float)W * (float)H);
  for (int c = 0; c < 3; ++c) {
    __syncthreads();
    for (int t = threadIdx.x; t < LW * LW; t += 256) {
      const int r = t / LW, q = t - r * LW;
      const int yy = y0 + r - LH, xx = x0 + q - LH;
      const bool in = yy >= 0 && yy < H && xx >= 0 && xx < W;
      const float* mp = maps + (in ? 9 * ((size_t)yy * W + xx) + 3 * c : 0);
      sM[0][r][q] = in ? mp[0] : 0.f; sM[1][r][q] = in ? mp[1] : 0.f; sM[2][r][q] = in ? mp[2] : 0.f;
    }
    __syncthreads();
    for (int t = threadIdx.x; t < LW * LT; t += 256) {
      const int r = t / LT, q = t - r * LT;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f;
#pragma unroll
      for (int k = 0; k < 11; ++k) {
        const float w = win.w[k];
        a0 = fmaf(w, sM[0][r][q + k], a0); a1 = fmaf(w, sM[1][r][q + k], a1); a2 = fmaf(w, sM[2][r][q + k], a2);
      }
      sH[0][r][q] = a0; sH[1][r][q] = a1; sH[2][r][q] = a2;
    }
    __syncthreads();
    float cA = 0.f, cB = 0.f, cC = 0.f;
#pragma unroll
    for (int k = 0; k < 11; ++k) {
      const float w = win.w[k];
      cA = fmaf(w, sH[0][ty + k][tx], cA); cB = fmaf(w, sH[1][ty + k][tx], cB); cC = fmaf(w, sH[2][ty + k][tx], cC);
    }
    if (inside) {
      const size_t i = 3 * ((size_t)py * W + px) + c;
      const float p = img[i], s = tgt[i], d = p - s;
      const float sg = d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f);
      d_image[i] = inv_n * ((1.f - lam) * sg - lam * (cA + 2.f * p * cB + s * cC));
    }
  }
}

__global__ void image_loss_finish_kernel(int W, int H, float lam, const double* __restrict__ sums, float* __restrict__ out_loss) {
  const double n = 3.0 * (double)W * (double)H;
  const double ssim = sums[0] / n, l1 = sums[1] / n;
  out_loss[0] = (float)((1.0 - (double)lam) * l1 + (double)lam * (1.0 - ssim));
  out_loss[1] = (float)l1; out_loss[2] = (float)ssim;
}

cudaError_t rga_launch_image_loss(rga_avatar* av, const float* image, const float* target, int W, int H, float lam, float* out_loss,
                                  float* out_dimage, cudaStream_t s) {
  SsimWin win; double g[11], tot = 0.0;
  for (int k = 0; k < 11; ++k) { g[k] = exp(-(double)((k - 5) * (k - 5)) / (2.0 * 1.5 * 1.5)); tot += g[k]; }
  for (int k = 0; k < 11; ++k) win.w[k] = (float)(g[k] / tot);
  cudaError_t e = cudaMemsetAsync(av->loss_sums, 0, 2 * sizeof(double), s);
  if (e != cudaSuccess) return e;
  const dim3 grid((W + LT - 1) / LT, (H + LT - 1) / LT);
  ssim_maps_kernel<<<grid, 256, 0, s>>>(W, H, win, image, target, av->loss_maps, av->loss_sums);
  rga_prof_mark(av, "ssim_maps", s);
  if (out_dimage) {
    ssim_grad_kernel<<<grid, 256, 0, s>>>(W, H, win, lam, image, target, av->loss_maps, out_dimage);
    rga_prof_mark(av, "ssim_grad", s);
  }
  if (out_loss) image_loss_finish_kernel<<<1, 1, 0, s>>>(W, H, lam, av->loss_sums, out_loss);
  av->launches += 1 + (out_dimage != nullptr) + (out_loss != nullptr);
  return cudaGetLastError();
}
