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

// ---------------------------------------------------------------------------------------------------------------
// Regularisers Eq.6-9, reading A35 (slope 0 at the kinks).  One thread per vertex does Eq.6
// (its own K_v neighbour set: the gradient of its own attributes stays in registers, the opposite sign goes to the
// neighbour by an atomic; sums of +-1 are exact in fp32, so the result does not depend on the order) and Eq.8; one thread
// per Gaussian does Eq.7 and Eq.9.  Loss sums: block reduction, then one double atomic per CTA.
__device__ __forceinline__ float sgnf(float d) { return d > 0.f ? 1.f : (d < 0.f ? -1.f : 0.f); }

__global__ void __launch_bounds__(256) reg_vertex_kernel(int nv, int Kv, const float* __restrict__ alb, const float* __restrict__ rough,
    const float* __restrict__ spec, const int* __restrict__ knn_v, const float4* __restrict__ disp4, const float* __restrict__ disp3,
    float* __restrict__ d_alb, float* __restrict__ d_rough, float* __restrict__ d_spec, float* __restrict__ d_disp, double* __restrict__ sums) {
  __shared__ float s_red[8];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  float smooth = 0.f, dl = 0.f;
  if (i < nv) {
    const float a0 = alb[3 * i], a1 = alb[3 * i + 1], a2 = alb[3 * i + 2], r = rough[i], p = spec[i];
    float g0 = 0.f, g1 = 0.f, g2 = 0.f, gr = 0.f, gp = 0.f;
    for (int j = 0; j < Kv; ++j) {
      const int k = knn_v[(size_t)i * Kv + j];
      if (k == i) continue;
      const float e0 = a0 - alb[3 * k], e1 = a1 - alb[3 * k + 1], e2 = a2 - alb[3 * k + 2], er = r - rough[k], ep = p - spec[k];
      smooth += fabsf(e0) + fabsf(e1) + fabsf(e2) + fabsf(er) + fabsf(ep);
      const float s0 = sgnf(e0), s1 = sgnf(e1), s2 = sgnf(e2), sr = sgnf(er), sp = sgnf(ep);
      g0 += s0; g1 += s1; g2 += s2; gr += sr; gp += sp;
      if (d_alb) { if (s0 != 0.f) atomicAdd(d_alb + 3 * k, -s0); if (s1 != 0.f) atomicAdd(d_alb + 3 * k + 1, -s1); if (s2 != 0.f) atomicAdd(d_alb + 3 * k + 2, -s2); }
      if (d_rough && sr != 0.f) atomicAdd(d_rough + k, -sr);
      if (d_spec && sp != 0.f) atomicAdd(d_spec + k, -sp);
    }
    if (d_alb) { atomicAdd(d_alb + 3 * i, g0); atomicAdd(d_alb + 3 * i + 1, g1); atomicAdd(d_alb + 3 * i + 2, g2); }
    if (d_rough) atomicAdd(d_rough + i, gr);
    if (d_spec) atomicAdd(d_spec + i, gp);
    float x = 0.f, y = 0.f, z = 0.f;
    if (disp4) { const float4 d = disp4[i]; x = d.x; y = d.y; z = d.z; }
    else if (disp3) { x = disp3[3 * i]; y = disp3[3 * i + 1]; z = disp3[3 * i + 2]; }
    const float n2 = x * x + y * y + z * z;
    float inv = 0.f;
    if (n2 > 0.f) { dl = sqrtf(n2); inv = 1.f / dl; }
    if (d_disp) { d_disp[3 * i] = x * inv; d_disp[3 * i + 1] = y * inv; d_disp[3 * i + 2] = z * inv; }
  }
  const float t0 = block_sum256(smooth, s_red), t1 = block_sum256(dl, s_red);
  if (threadIdx.x == 0) { atomicAdd(sums, (double)t0); atomicAdd(sums + 2, (double)t1); }
}

__global__ void __launch_bounds__(256) reg_gauss_kernel(int ng, int Kg, float s0, const float4* __restrict__ g_pos, const float* __restrict__ v_pos,
    const int* __restrict__ knn_g, const float4* __restrict__ g_scale_op, float* __restrict__ d_gpos, float* __restrict__ d_scale,
    double* __restrict__ sums, const int* __restrict__ order) {
  __shared__ float s_red[8];
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  float md = 0.f, sc = 0.f;
  if (g < ng) {
    const float4 x = g_pos[g];
    float gx = 0.f, gy = 0.f, gz = 0.f;
    for (int j = 0; j < Kg; ++j) {
      const int k = knn_g[(size_t)g * Kg + j];
      const float dx = x.x - v_pos[3 * k], dy = x.y - v_pos[3 * k + 1], dz = x.z - v_pos[3 * k + 2];
      const float n2 = dx * dx + dy * dy + dz * dz;
      if (n2 > 0.f) { const float l = sqrtf(n2), inv = 1.f / l; md += l; gx += dx * inv; gy += dy * inv; gz += dz * inv; }
    }
    const size_t gc = (size_t)order[g];        // gradients go out in the caller's order
    if (d_gpos) { d_gpos[3 * gc] = gx; d_gpos[3 * gc + 1] = gy; d_gpos[3 * gc + 2] = gz; }
    const float4 s = g_scale_op[g];
    const float e0 = s.x - s0, e1 = s.y - s0, e2 = s.z - s0;
    sc = fmaxf(e0, 0.f) + fmaxf(e1, 0.f) + fmaxf(e2, 0.f);
    if (d_scale) { d_scale[3 * gc] = e0 > 0.f ? 1.f : 0.f; d_scale[3 * gc + 1] = e1 > 0.f ? 1.f : 0.f; d_scale[3 * gc + 2] = e2 > 0.f ? 1.f : 0.f; }
  }
  const float t0 = block_sum256(md, s_red), t1 = block_sum256(sc, s_red);
  if (threadIdx.x == 0) { atomicAdd(sums + 1, (double)t0); atomicAdd(sums + 3, (double)t1); }
}

__global__ void reg_finish_kernel(const double* __restrict__ sums, float* __restrict__ out) {
  if (threadIdx.x < 4) out[threadIdx.x] = (float)sums[threadIdx.x];
}

cudaError_t rga_launch_regularisers(rga_avatar* av, float s0, float* out_losses, float* d_alb, float* d_rough, float* d_spec, float* d_gpos,
                                    float* d_disp, float* d_scale, cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(av->reg_sums, 0, 4 * sizeof(double), s);
  if (e != cudaSuccess) return e;
  const size_t nv = av->n_verts;
  if (d_alb && (e = cudaMemsetAsync(d_alb, 0, 12 * nv, s)) != cudaSuccess) return e;
  if (d_rough && (e = cudaMemsetAsync(d_rough, 0, 4 * nv, s)) != cudaSuccess) return e;
  if (d_spec && (e = cudaMemsetAsync(d_spec, 0, 4 * nv, s)) != cudaSuccess) return e;
  reg_vertex_kernel<<<(av->n_verts + 255) / 256, 256, 0, s>>>(av->n_verts, av->k_v, av->vt_albedo, av->vt_rough, av->vt_spec, av->knn_v,
      av->disp_is_mlp ? av->v_disp : nullptr, av->disp_is_mlp ? nullptr : av->vt_disp, d_alb, d_rough, d_spec, d_disp, av->reg_sums);
  rga_prof_mark(av, "reg_vertex", s);
  reg_gauss_kernel<<<(av->n_gauss + 255) / 256, 256, 0, s>>>(av->n_gauss, av->k_g, s0, av->g_pos, av->vt_pos, av->knn_g, av->g_scale_op,
      d_gpos, d_scale, av->reg_sums, av->g_order);
  rga_prof_mark(av, "reg_gauss", s);
  if (out_losses) reg_finish_kernel<<<1, 32, 0, s>>>(av->reg_sums, out_losses);
  av->launches += 2 + (out_losses != nullptr);
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------------------
// rga_image_loss_static (include/rga.h): Eq.5 and its gradient WITHOUT an avatar handle and without any allocation -- for
// callers that cannot reach cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it).
// The scratch the two kernels above need (nine floats per pixel between them, two double accumulators) lives in ONE
// file-scope device array of a fixed size: every GPU that loads librga.so holds these 9.0 MiB until the process exits.
// In HOST code the array's name is only a stand-in for the symbol, not a device address; the address is asked for once per
// device with cudaGetSymbolAddress, with that device current, and the kernels get that pointer.
// The array is shared by every call and keeps the last call's contents: the accumulators are cleared on the stream at the
// start of each call, the per-pixel maps are written for every pixel of the image before the gradient kernel reads them (it
// reads no pixel outside the image), so nothing stale is used.  Two calls that overlap on the GPU (different streams) race.
#include <mutex>

#define RGA_STATIC_LOSS_HEAD 256                      /* bytes in front of the maps: the two double accumulators */
static __device__ __align__(256) unsigned char g_static_loss_scratch[RGA_STATIC_LOSS_HEAD + (size_t)RGA_IMAGE_LOSS_STATIC_MAX_PIXELS * 9 * sizeof(float)];

static std::mutex g_static_loss_mutex;
static unsigned char* g_static_loss_ptr[RGA_STATIC_MAX_DEVICES];       // per device: the array's DEVICE address, once known

// device address of the scratch array on the CURRENT device (looked up once per device); nullptr + *err on failure
static unsigned char* static_loss_scratch(cudaError_t* err) {
  int dev = -1;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  if (dev < 0 || dev >= RGA_STATIC_MAX_DEVICES) { *err = cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> lock(g_static_loss_mutex);
  if (!g_static_loss_ptr[dev]) {
    void* p = nullptr;
    *err = cudaGetSymbolAddress(&p, g_static_loss_scratch);
    if (*err != cudaSuccess) return nullptr;
    g_static_loss_ptr[dev] = static_cast<unsigned char*>(p);
  }
  return g_static_loss_ptr[dev];
}

// W * H <= RGA_IMAGE_LOSS_STATIC_MAX_PIXELS is the caller's check (api.cu).  No cudaMalloc / cudaFree here or below.
cudaError_t rga_launch_image_loss_static(const float* image, const float* target, int W, int H, float lam, float* out_loss,
                                         float* out_dimage, cudaStream_t s) {
  cudaError_t e = cudaSuccess;
  unsigned char* base = static_loss_scratch(&e);
  if (!base) return e;
  double* sums = reinterpret_cast<double*>(base);
  float* maps = reinterpret_cast<float*>(base + RGA_STATIC_LOSS_HEAD);
  SsimWin win; double g[11], tot = 0.0;
  for (int k = 0; k < 11; ++k) { g[k] = exp(-(double)((k - 5) * (k - 5)) / (2.0 * 1.5 * 1.5)); tot += g[k]; }
  for (int k = 0; k < 11; ++k) win.w[k] = (float)(g[k] / tot);
  e = cudaMemsetAsync(sums, 0, 2 * sizeof(double), s);                 // the accumulators must start at zero
  if (e != cudaSuccess) return e;
  const dim3 grid((W + LT - 1) / LT, (H + LT - 1) / LT);
  ssim_maps_kernel<<<grid, 256, 0, s>>>(W, H, win, image, target, maps, sums);
  if (out_dimage) ssim_grad_kernel<<<grid, 256, 0, s>>>(W, H, win, lam, image, target, maps, out_dimage);
  if (out_loss) image_loss_finish_kernel<<<1, 1, 0, s>>>(W, H, lam, sums, out_loss);
  return cudaGetLastError();
}
