// H1/H2 pose_skin: forward linear-blend skinning of mesh vertices and Gaussians, Gaussian covariance
// Sigma = A A^T with A = M3x3 R(q) diag(s) (PAPER.md:95 "rotated accordingly", :103; A3), posed AABB and the
// orthographic window of the visibility pass (A13).
// EXACT file: -fmad=false, only + - * / sqrt, operation order fixed by DESIGN.md "Arithmetic contract".
#include "rga_internal.h"

__device__ __forceinline__ unsigned f2ord(float f) { unsigned u = __float_as_uint(f); return (u & 0x80000000u) ? ~u : (u | 0x80000000u); }
__device__ __forceinline__ float ord2f(unsigned u) { return __uint_as_float((u & 0x80000000u) ? (u & 0x7fffffffu) : ~u); }

// M = sum_b w_b G_b, b ascending from +0.  Zero weights are skipped: adding w_b*G = +-0 never changes M.
__device__ __forceinline__ void blend(const float* __restrict__ w, int B, const float* sG, float* M) {
#pragma unroll
  for (int e = 0; e < 12; ++e) M[e] = 0.f;
  if ((B & 3) == 0) {
    const float4* w4 = reinterpret_cast<const float4*>(w);
    for (int b4 = 0; b4 < B / 4; ++b4) {
      float4 ww = __ldg(w4 + b4);
      float wv[4] = {ww.x, ww.y, ww.z, ww.w};
#pragma unroll
      for (int k = 0; k < 4; ++k)
        if (wv[k] != 0.f) {
          const float* G = sG + (b4 * 4 + k) * 12;
#pragma unroll
          for (int e = 0; e < 12; ++e) M[e] = M[e] + wv[k] * G[e];
        }
    }
  } else {
    for (int b = 0; b < B; ++b) {
      float wb = __ldg(w + b);
      if (wb != 0.f) {
        const float* G = sG + b * 12;
#pragma unroll
        for (int e = 0; e < 12; ++e) M[e] = M[e] + wb * G[e];
      }
    }
  }
}

// window = bounding sphere of the posed AABB, radius padded by 1/64; then re-arm the AABB for the next pose.  Run by one
// thread of the last vertex block of skin_kernel; the AABB words were written by atomics, so they are read past L1.
__device__ __forceinline__ void window_from_aabb(unsigned* aabb, float* window) {
  float mn[3], mx[3], dg[3];
  for (int c = 0; c < 3; ++c) { mn[c] = ord2f(__ldcg(aabb + c)); mx[c] = ord2f(__ldcg(aabb + 3 + c)); }
  for (int c = 0; c < 3; ++c) { window[c] = (mn[c] + mx[c]) * 0.5f; dg[c] = mx[c] - mn[c]; }
  float rr = (0.5f * sqrtf((dg[0] * dg[0] + dg[1] * dg[1]) + dg[2] * dg[2])) * 1.015625f;
  window[3] = (rr > 0.f) ? rr : 1.0f;
  for (int c = 0; c < 3; ++c) { aabb[c] = 0xffffffffu; aabb[3 + c] = 0u; }
}

#ifndef SKIN_THREADS
#define SKIN_THREADS 256
#endif
__global__ void __launch_bounds__(SKIN_THREADS) skin_kernel(int nv, int ng, int B, int vblocks, int block_base, const float* __restrict__ bone,
    const float4* __restrict__ v_xbar, const float4* __restrict__ v_n, const float* __restrict__ v_w,
    const float4* __restrict__ g_static, const float* __restrict__ g_w, const float4* __restrict__ g_quat,
    const float4* __restrict__ g_scale_op,
    float4* __restrict__ v_posed, float4* __restrict__ v_nposed, float4* __restrict__ g_posed, float4* __restrict__ g_nposed,
    float* __restrict__ g_cov, unsigned* __restrict__ aabb, float* __restrict__ window) {
  extern __shared__ float sG[];
  for (int t = threadIdx.x; t < B * 12; t += blockDim.x) sG[t] = bone[t];
  __syncthreads();
  const int blk = blockIdx.x + block_base;                 // vertex blocks first, then Gaussian blocks
  const bool is_vert = blk < vblocks;
  int i = (is_vert ? blk : blk - vblocks) * blockDim.x + threadIdx.x;
  int n = is_vert ? nv : ng;
  float M[12];
  float px = 0.f, py = 0.f, pz = 0.f;
  bool act = i < n;
  if (act) {
    float4 xb = is_vert ? v_xbar[i] : g_static[4 * (size_t)i];
    float4 nn = is_vert ? v_n[i] : g_static[4 * (size_t)i + 1];
    blend((is_vert ? v_w : g_w) + (size_t)i * B, B, sG, M);
    px = ((M[0] * xb.x + M[1] * xb.y) + M[2] * xb.z) + M[3];
    py = ((M[4] * xb.x + M[5] * xb.y) + M[6] * xb.z) + M[7];
    pz = ((M[8] * xb.x + M[9] * xb.y) + M[10] * xb.z) + M[11];
    float tx = (M[0] * nn.x + M[1] * nn.y) + M[2] * nn.z;
    float ty = (M[4] * nn.x + M[5] * nn.y) + M[6] * nn.z;
    float tz = (M[8] * nn.x + M[9] * nn.y) + M[10] * nn.z;
    float len = sqrtf((tx * tx + ty * ty) + tz * tz);
    if (len > 0.f) { tx = tx / len; ty = ty / len; tz = tz / len; }
    if (is_vert) { v_posed[i] = make_float4(px, py, pz, 0.f); v_nposed[i] = make_float4(tx, ty, tz, 0.f); }
    else {
      g_posed[i] = make_float4(px, py, pz, 0.f); g_nposed[i] = make_float4(tx, ty, tz, 0.f);
      float4 q = g_quat[i]; float4 so = g_scale_op[i];
      float ql = sqrtf(((q.x * q.x + q.y * q.y) + q.z * q.z) + q.w * q.w);
      float w = q.x / ql, x = q.y / ql, y = q.z / ql, z = q.w / ql;
      float R[9] = {1.0f - 2.0f * (y * y + z * z), 2.0f * (x * y - w * z), 2.0f * (x * z + w * y),
                    2.0f * (x * y + w * z), 1.0f - 2.0f * (x * x + z * z), 2.0f * (y * z - w * x),
                    2.0f * (x * z - w * y), 2.0f * (y * z + w * x), 1.0f - 2.0f * (x * x + y * y)};
      float s[3] = {so.x, so.y, so.z};
      float RS[9], A[9];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) RS[3 * r + c] = R[3 * r + c] * s[c];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) A[3 * r + c] = (M[4 * r] * RS[c] + M[4 * r + 1] * RS[3 + c]) + M[4 * r + 2] * RS[6 + c];
      float* o = g_cov + 6 * (size_t)i;
      o[0] = (A[0] * A[0] + A[1] * A[1]) + A[2] * A[2];
      o[1] = (A[0] * A[3] + A[1] * A[4]) + A[2] * A[5];
      o[2] = (A[0] * A[6] + A[1] * A[7]) + A[2] * A[8];
      o[3] = (A[3] * A[3] + A[4] * A[4]) + A[5] * A[5];
      o[4] = (A[3] * A[6] + A[4] * A[7]) + A[5] * A[8];
      o[5] = (A[6] * A[6] + A[7] * A[7]) + A[8] * A[8];
    }
  }
  if (is_vert) {                                   // posed AABB: warp reduce, one atomic per warp per bound
    const float INF = __int_as_float(0x7f800000);
    float mn[3] = {act ? px : INF, act ? py : INF, act ? pz : INF};
    float mx[3] = {act ? px : -INF, act ? py : -INF, act ? pz : -INF};
#pragma unroll
    for (int o = 16; o > 0; o >>= 1)
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        mn[c] = fminf(mn[c], __shfl_xor_sync(0xffffffffu, mn[c], o));
        mx[c] = fmaxf(mx[c], __shfl_xor_sync(0xffffffffu, mx[c], o));
      }
    if ((threadIdx.x & 31) == 0)
#pragma unroll
      for (int c = 0; c < 3; ++c) { atomicMin(aabb + c, f2ord(mn[c])); atomicMax(aabb + 3 + c, f2ord(mx[c])); }
    // the vertex block that finishes last turns the AABB into the rasteriser's window (c, r) and re-arms the AABB and the
    // block counter aabb[6] for the next pose (this was a one-thread kernel of its own on the frame's critical path)
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(aabb + 6, 1u) == (unsigned)(vblocks - 1);
    __syncthreads();
    if (s_last && threadIdx.x == 0) {
      __threadfence();
      window_from_aabb(aabb, window);
      aabb[6] = 0u;
    }
  }
}

// which: 0 = mesh and Gaussians (pose_skin), 1 = mesh + window only, 2 = Gaussians only.  rga_render_frame issues 1 on
// the main stream (the rasteriser needs nothing else) and 2 on the second stream.
cudaError_t rga_launch_skin(rga_avatar* av, const float* bone_mats, int which, cudaStream_t s) {
  const int vblocks = (av->n_verts + SKIN_THREADS - 1) / SKIN_THREADS, gblocks = (av->n_gauss + SKIN_THREADS - 1) / SKIN_THREADS;
  const int base = which == 2 ? vblocks : 0, nblocks = which == 0 ? vblocks + gblocks : (which == 1 ? vblocks : gblocks);
  skin_kernel<<<nblocks, SKIN_THREADS, av->n_bones * 12 * sizeof(float), s>>>(
      av->n_verts, av->n_gauss, av->n_bones, vblocks, base, bone_mats, av->v_xbar, av->v_normal, av->v_skin_w, av->g_static,
      av->g_skin_w, av->g_quat, av->g_scale_op, av->v_posed, av->v_nposed, av->g_posed, av->g_nposed, av->g_cov, av->aabb, av->window);
  rga_prof_mark(av, which == 2 ? "skin_gauss" : (which == 1 ? "skin_mesh" : "skin"), s);
  av->launches += 1;
  return cudaGetLastError();
}
