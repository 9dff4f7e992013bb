// Backward of the splat, H10 then H6 (SURVEY.md 8(f) item 4; PAPER.md:103 -> the 3DGS rasteriser [8], :128 "the same
// image loss as 3DGS"): given dL/dimage, the gradient of the forward image with its discrete decisions frozen (tile
// lists and order, culled Gaussians, per-pixel skips and the stopping entry) with respect to every Gaussian's splatted
// colour, opacity, posed mean and 3D covariance.  FAST source: compared with the fp64 autograd oracle under tolerance.
//
//   composite_backward_kernel   persistent CTAs over the forward's work items (one RGA_SEG-entry segment of one tile's
//                               list), one thread per pixel of the tile (the forward's 8x4-pixel warp blocks).  With
//                               F_i the colour composited up to and including entry i and I the pixel's final colour,
//                                   dL/dalpha_i = T_i <G, c_i> - <G, I - F_i> / (1 - alpha_i),
//                               so the list can be walked FRONT TO BACK like the forward, and a segment can start on
//                               its own: T and <G, F> in front of it are folded from the per-segment partials (C, T)
//                               the forward left in `part`; I is the rendered image.  (The first version walked each
//                               tile's list back to front in one CTA, recovering T by division: 383 us at config 1
//                               against 89 us, for the same reason the forward is segment-parallel.)
//                               Per entry a warp reduces nine sums over its 32 pixels with a transposed butterfly
//                               (14 shuffles instead of 45) into the segment's shared-memory accumulators; after the
//                               segment one thread per entry issues the global atomics.
//                               The nine sums: dL/dc (3) and the moments S = sum w, sum w dx, sum w dy, sum w dx^2,
//                               sum w dx dy, sum w dy^2 of w = alpha dL/dalpha (0 where alpha is clamped to 0.99: the
//                               clamp has derivative 0, reading A32) with d = mu - pixel, from which
//                               dL/do = S_0 / o, dL/dmu = -(A S_x + B S_y, C S_y + B S_x), dL/d(A,B,C) = -(S_xx / 2, S_xy, S_yy / 2).
//   project_backward_kernel     one thread per Gaussian: finishes the sums above and pulls dL/dmu, dL/dconic back through
//                               conic = (T Sigma T^T + 0.3 I)^-1, T = J(t) R_wc, mu = pi(t), t = R_wc x + t_wc, including the
//                               clamp of t_x / t_z, t_y / t_z inside J (zero slope where it is active).
#include "rga_internal.h"

#define BB 256
#define LOG2E_F 1.4426950408889634f

__device__ __forceinline__ int btile_px(unsigned t) { return (int)(((t >> 5) & 1u) * 8u + (t & 7u)); }
__device__ __forceinline__ int btile_py(unsigned t) { return (int)((t >> 6) * 4u + ((t >> 3) & 3u)); }
__device__ __forceinline__ float bex2_approx(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// sum of v[0..7] over the warp: afterwards lane 4 k holds the total of v[k]
__device__ __forceinline__ float warp_reduce8(const float (&v)[8], int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  float w[4], u[2];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const float mine = b4 ? v[k + 4] : v[k], send = b4 ? v[k] : v[k + 4];
    w[k] = mine + __shfl_xor_sync(0xffffffffu, send, 16);
  }
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    const float mine = b3 ? w[k + 2] : w[k], send = b3 ? w[k] : w[k + 2];
    u[k] = mine + __shfl_xor_sync(0xffffffffu, send, 8);
  }
  const float mine = b2 ? u[1] : u[0], send = b2 ? u[0] : u[1];
  float z = mine + __shfl_xor_sync(0xffffffffu, send, 4);
  z += __shfl_xor_sync(0xffffffffu, z, 2);
  z += __shfl_xor_sync(0xffffffffu, z, 1);
  return z;          // value index = (lane >> 2) & 7
}

// one work item = one RGA_SEG-entry segment of one tile's list (the forward's work items and its per-segment partials)
struct BwdSeg { float2 mu[RGA_SEG]; float4 co[RGA_SEG]; float4 col[RGA_SEG]; float2 ext[RGA_SEG]; unsigned id[RGA_SEG]; float acc[RGA_SEG][9]; };

__global__ void __launch_bounds__(BB) composite_backward_kernel(int W, int H, int TX, float3 bg, const unsigned* __restrict__ num_items,
    const unsigned* __restrict__ item_tab, const unsigned* __restrict__ seg_off, const uint2* __restrict__ ranges,
    const unsigned* __restrict__ vals, const float2* __restrict__ mu2d, const float4* __restrict__ conic_o,
    const float4* __restrict__ color, const float4* __restrict__ part, const unsigned* __restrict__ n_contrib,
    const float* __restrict__ image, const float* __restrict__ dL_dimage, float* __restrict__ grad) {
  __shared__ BwdSeg st;
  const unsigned n_items = *num_items;
  const int tid = threadIdx.x, lane = tid & 31;
  for (unsigned item = blockIdx.x; item < n_items; item += gridDim.x) {
    const unsigned tile = item_tab[item];
    const unsigned so = seg_off[tile];
    const int seg = (int)(item - so);
    const uint2 rg = ranges[tile];
    const int b0 = seg * RGA_SEG;
    const int m = min(RGA_SEG, (int)(rg.y - rg.x) - b0);
    const int px = (int)(tile % TX) * RGA_TILE + btile_px(tid), py = (int)(tile / TX) * RGA_TILE + btile_py(tid);
    const bool inside = px < W && py < H;
    const size_t p = (size_t)py * W + px;
    const int last = inside ? (int)n_contrib[p] : 0;                     // entries [0, last) can contribute to this pixel
    int wlast = last;
#pragma unroll
    for (int o = 16; o; o >>= 1) wlast = max(wlast, __shfl_xor_sync(0xffffffffu, wlast, o));
    if (!__syncthreads_or(b0 < wlast)) continue;                         // no pixel of the tile reaches this segment
    if (tid < m) {
      const unsigned g = vals[rg.x + b0 + tid];
      const float4 c = conic_o[g];
      st.id[tid] = g; st.mu[tid] = mu2d[g]; st.col[tid] = color[g];
      st.co[tid] = make_float4(-0.5f * LOG2E_F * c.x, -LOG2E_F * c.y, -0.5f * LOG2E_F * c.z, c.w);
      const float L2 = 2.0f * __logf(255.0f * c.w), det = c.x * c.z - c.y * c.y;
      float hx = -1.f, hy = -1.f;
      if (L2 > 0.f && det > 0.f) { hx = sqrtf(L2 * c.z / det) * 1.001f + 0.01f; hy = sqrtf(L2 * c.x / det) * 1.001f + 0.01f; }
      st.ext[tid] = make_float2(hx, hy);
    }
    for (int k = tid; k < RGA_SEG * 9; k += BB) (&st.acc[0][0])[k] = 0.f;
    __syncthreads();
    if (b0 < wlast) {
      const float fx = (float)px + 0.5f, fy = (float)py + 0.5f;
      float g0 = 0.f, g1 = 0.f, g2 = 0.f, sI = 0.f;
      if (inside) {
        g0 = dL_dimage[3 * p]; g1 = dL_dimage[3 * p + 1]; g2 = dL_dimage[3 * p + 2];
        sI = image[3 * p] * g0 + image[3 * p + 1] * g1 + image[3 * p + 2] * g2;           // <G, final colour of the pixel>
      }
      // transmittance and <G, colour composited so far> in front of this segment, from the forward's segment partials
      float T = 1.f, sF = 0.f;
      const float4* pp = part + (size_t)so * BB + tid;
      for (int s0 = 0; s0 < seg; s0 += 4) {
        float4 q[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) if (s0 + u < seg) q[u] = pp[(size_t)(s0 + u) * BB];
#pragma unroll
        for (int u = 0; u < 4; ++u)
          if (s0 + u < seg) { sF = fmaf(T, q[u].x * g0 + q[u].y * g1 + q[u].z * g2, sF); T *= q[u].w; }
      }
      const float bcx = (float)((int)(tile % TX) * RGA_TILE + btile_px(tid & ~31u)) + 4.0f;
      const float bcy = (float)((int)(tile / TX) * RGA_TILE + btile_py(tid & ~31u)) + 2.0f;
      const int jend = min(m, wlast - b0);
      for (int j = 0; j < jend; ++j) {
        const float2 mm = st.mu[j], ex = st.ext[j];
        if (fabsf(mm.x - bcx) > ex.x + 3.5f || fabsf(mm.y - bcy) > ex.y + 1.5f) continue;
        const float4 co = st.co[j];
        const float dx = mm.x - fx, dy = mm.y - fy;
        const float p2 = fmaf(dx, fmaf(co.x, dx, co.y * dy), (co.z * dy) * dy);   // log2(e) * power, rounded as in the forward's seg_alpha
        const float raw = co.w * bex2_approx(p2);
        const float a = fminf(0.99f, raw);
        const bool valid = (b0 + j < last) && !(p2 > 0.f || a < 1.f / 255.f);
        if (!__any_sync(0xffffffffu, valid)) continue;
        float v[8], s0 = 0.f;
#pragma unroll
        for (int k = 0; k < 8; ++k) v[k] = 0.f;
        if (valid) {
          const float4 c = st.col[j];
          const float wgt = a * T, sc = c.x * g0 + c.y * g1 + c.z * g2, om = 1.f - a;
          v[0] = wgt * g0; v[1] = wgt * g1; v[2] = wgt * g2;
          sF = fmaf(wgt, sc, sF);
          // dL/dalpha = T <G, c> - <G, everything behind this entry> / (1 - alpha); "behind" = final colour - prefix
          const float dLda = T * sc - __fdividef(sI - sF, om);
          T *= om;
          const float w = raw > 0.99f ? 0.f : a * dLda;
          s0 = w;
          v[3] = w * dx; v[4] = w * dy; v[5] = w * dx * dx; v[6] = w * dx * dy; v[7] = w * dy * dy;
        }
        const float z = warp_reduce8(v, lane);
#pragma unroll
        for (int o = 16; o; o >>= 1) s0 += __shfl_xor_sync(0xffffffffu, s0, o);
        if ((lane & 3) == 0) {
          const int k = lane >> 2;                                        // 0..7 -> acc slots 0,1,2 (colour) and 4..8 (moments)
          atomicAdd(&st.acc[j][k < 3 ? k : k + 1], z);
          if (lane == 0) atomicAdd(&st.acc[j][3], s0);
        }
      }
    }
    __syncthreads();
    if (tid < m) {
      float* gdst = grad + 12 * (size_t)st.id[tid];
#pragma unroll
      for (int k = 0; k < 9; ++k) { const float x = st.acc[tid][k]; if (x != 0.f) atomicAdd(gdst + k, x); }
    }
    __syncthreads();
  }
}

struct CamB { float R[9], t[3], fx, fy, limx, limy; };

__global__ void __launch_bounds__(256) project_backward_kernel(int ng, CamB cam, const float4* __restrict__ g_posed,
    const float* __restrict__ g_cov, const float4* __restrict__ conic_o, const unsigned* __restrict__ touched, float* __restrict__ grad,
    float* __restrict__ out_dcolor, float* __restrict__ out_dopacity, float* __restrict__ out_dmean, float* __restrict__ out_dcov,
    const int* __restrict__ order) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ng) return;
  const int gc = order[g];                 // the caller's index: [n_gauss] outputs are written in the caller's order
  float* gr = grad + 12 * (size_t)g;
  float dcol[3] = {gr[0], gr[1], gr[2]}, dop = 0.f, dmean[3] = {0.f, 0.f, 0.f}, dcov[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  float dmx = 0.f, dmy = 0.f, dA = 0.f, dB = 0.f, dC = 0.f;
  if (touched[g]) {
    const float4 q = conic_o[g];
    const float S0 = gr[3], Sx = gr[4], Sy = gr[5], Sxx = gr[6], Sxy = gr[7], Syy = gr[8];
    dop = q.w > 0.f ? S0 / q.w : 0.f;
    dmx = -(q.x * Sx + q.y * Sy); dmy = -(q.z * Sy + q.y * Sx);
    dA = -0.5f * Sxx; dB = -Sxy; dC = -0.5f * Syy;
    // conic Q = M^-1:  dL/dM = -Q G Q with G = [[dA, dB/2], [dB/2, dC]]
    const float h = 0.5f * dB;
    const float X00 = dA * q.x + h * q.y, X01 = dA * q.y + h * q.z, X10 = h * q.x + dC * q.y, X11 = h * q.y + dC * q.z;
    const float g00 = -(q.x * X00 + q.y * X10), g01 = -((q.x * X01 + q.y * X11) + (q.y * X00 + q.z * X10)), g11 = -(q.y * X01 + q.z * X11);
    const float4 x = g_posed[g];
    const float* R = cam.R;
    const float t0 = R[0] * x.x + R[1] * x.y + R[2] * x.z + cam.t[0];
    const float t1 = R[3] * x.x + R[4] * x.y + R[5] * x.z + cam.t[1];
    const float t2 = R[6] * x.x + R[7] * x.y + R[8] * x.z + cam.t[2];
    const float iz = 1.f / t2, iz2 = iz * iz;
    const float u = t0 * iz, v = t1 * iz;
    const bool cu = u < -cam.limx || u > cam.limx, cv = v < -cam.limy || v > cam.limy;       // the clamp is active
    const float uc = fminf(cam.limx, fmaxf(-cam.limx, u)), vc = fminf(cam.limy, fmaxf(-cam.limy, v));
    const float J00 = cam.fx * iz, J02 = -cam.fx * uc * iz, J11 = cam.fy * iz, J12 = -cam.fy * vc * iz;
    float T0[3], T1[3], V0[3], V1[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) { T0[j] = J00 * R[j] + J02 * R[6 + j]; T1[j] = J11 * R[3 + j] + J12 * R[6 + j]; }
    const float* s = g_cov + 6 * (size_t)g;
    const float S[9] = {s[0], s[1], s[2], s[1], s[3], s[4], s[2], s[4], s[5]};
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      V0[a] = T0[0] * S[a] + T0[1] * S[3 + a] + T0[2] * S[6 + a];
      V1[a] = T1[0] * S[a] + T1[1] * S[3 + a] + T1[2] * S[6 + a];
    }
    // M00 = T0^T S T0 + 0.3, M01 = T0^T S T1, M11 = T1^T S T1 + 0.3;  g01 is dL/dM01 with M01 counted once
    float GS[3][3];
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = 0; b < 3; ++b) GS[a][b] = g00 * T0[a] * T0[b] + g01 * T0[a] * T1[b] + g11 * T1[a] * T1[b];
    dcov[0] = GS[0][0]; dcov[1] = GS[0][1] + GS[1][0]; dcov[2] = GS[0][2] + GS[2][0];
    dcov[3] = GS[1][1]; dcov[4] = GS[1][2] + GS[2][1]; dcov[5] = GS[2][2];
    float gT0[3], gT1[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) { gT0[a] = 2.f * g00 * V0[a] + g01 * V1[a]; gT1[a] = 2.f * g11 * V1[a] + g01 * V0[a]; }
    const float gJ00 = gT0[0] * R[0] + gT0[1] * R[1] + gT0[2] * R[2], gJ02 = gT0[0] * R[6] + gT0[1] * R[7] + gT0[2] * R[8];
    const float gJ11 = gT1[0] * R[3] + gT1[1] * R[4] + gT1[2] * R[5], gJ12 = gT1[0] * R[6] + gT1[1] * R[7] + gT1[2] * R[8];
    const float gt0 = dmx * cam.fx * iz + (cu ? 0.f : -gJ02 * cam.fx * iz2);
    const float gt1 = dmy * cam.fy * iz + (cv ? 0.f : -gJ12 * cam.fy * iz2);
    const float gt2 = -(dmx * cam.fx * t0 + dmy * cam.fy * t1) * iz2 - (gJ00 * cam.fx + gJ11 * cam.fy) * iz2 +
                      gJ02 * (cu ? cam.fx * uc * iz2 : 2.f * cam.fx * t0 * iz2 * iz) + gJ12 * (cv ? cam.fy * vc * iz2 : 2.f * cam.fy * t1 * iz2 * iz);
#pragma unroll
    for (int j = 0; j < 3; ++j) dmean[j] = R[j] * gt0 + R[3 + j] * gt1 + R[6 + j] * gt2;
  } else {
    dcol[0] = dcol[1] = dcol[2] = 0.f;
  }
  gr[3] = dop; gr[4] = dmx; gr[5] = dmy; gr[6] = dA; gr[7] = dB; gr[8] = dC;      // the buffer now holds d_opacity, d_mu, d_conic
  if (out_dcolor) { out_dcolor[3 * (size_t)gc] = dcol[0]; out_dcolor[3 * (size_t)gc + 1] = dcol[1]; out_dcolor[3 * (size_t)gc + 2] = dcol[2]; }
  if (out_dopacity) out_dopacity[gc] = dop;
  if (out_dmean) { out_dmean[3 * (size_t)gc] = dmean[0]; out_dmean[3 * (size_t)gc + 1] = dmean[1]; out_dmean[3 * (size_t)gc + 2] = dmean[2]; }
  if (out_dcov) {
#pragma unroll
    for (int k = 0; k < 6; ++k) out_dcov[6 * (size_t)gc + k] = dcov[k];
  }
}

cudaError_t rga_launch_splat_backward(rga_avatar* av, const rga_camera* cam, float3 bg, const float* image, const float* dL_dimage,
                                      float* out_dcolor, float* out_dopacity, float* out_dmean, float* out_dcov, cudaStream_t s) {
  const int TX = (cam->width + RGA_TILE - 1) / RGA_TILE;
  cudaError_t e = cudaMemsetAsync(av->splat_grad, 0, sizeof(float) * 12 * (size_t)av->n_gauss, s);
  if (e != cudaSuccess) return e;
  composite_backward_kernel<<<av->num_sms * 4, BB, 0, s>>>(cam->width, cam->height, TX, bg, av->num_items, av->item_tab, av->seg_off,
                                                           av->ranges, av->vals[1], av->mu2d, av->conic_o, av->color, av->part,
                                                           av->n_contrib, image, dL_dimage, av->splat_grad);
  rga_prof_mark(av, "composite_backward", s);
  CamB k;
  for (int i = 0; i < 9; ++i) k.R[i] = cam->R_wc[i];
  for (int i = 0; i < 3; ++i) k.t[i] = cam->t_wc[i];
  k.fx = cam->fx; k.fy = cam->fy;
  k.limx = 1.3f * ((float)cam->width / (2.0f * cam->fx)); k.limy = 1.3f * ((float)cam->height / (2.0f * cam->fy));
  project_backward_kernel<<<(av->n_gauss + 255) / 256, 256, 0, s>>>(av->n_gauss, k, av->g_posed, av->g_cov, av->conic_o, av->touched,
                                                                    av->splat_grad, out_dcolor, out_dopacity, out_dmean, out_dcov, av->g_order);
  rga_prof_mark(av, "project_backward", s);
  av->launches += 2;
  return cudaGetLastError();
}
