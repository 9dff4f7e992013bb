// Backward of H2 + Eq.1: pulls the posed-space gradients of a frame (dL/d xbar_gd, dL/d nbar_gd,
// dL/d Sigma from splat_backward / shade_backward, and the per-Gaussian material gradients) back to what the paper
// optimises: the canonical Gaussian position, rotation and scale, the pose (bone transforms, :155
// "we also optimize the input poses") and, through the transpose of Eq.1 (:90-93) with S_g and the weights frozen, the
// vertex attributes dx, n, a, gamma, p.  The skinning weights are not differentiated (SMPL's, :86).
// FAST source: compared with the fp64 autograd oracle under tolerance.
//
// One thread per Gaussian.  Forward (skin_kernels.cu): M = sum_b w_b G_b, xbar = M [p; 1] with p = x_g + dx_g,
// nbar = normalize(M3 n_g), n_g = normalize(Eq.1(n_v)), Sigma = A A^T with A = M3 R(q/|q|) diag(s).  The bone gradient
// sum_g w_gb dL/dM_g is accumulated per CTA in shared memory and flushed with one global atomic per entry; the vertex
// gradients are scattered with global atomics (K_g per Gaussian and component).
#include "rga_internal.h"

#define PB_MAXK 8

// sum of v[0..15] over the warp by a transposed butterfly (16 shuffles instead of 80): afterwards lane 2 k holds the total of v[k]
__device__ __forceinline__ float warp_reduce16(const float (&v)[16], int lane) {
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4, b1 = lane & 2;
  float a[8], b[4], c[2];
#pragma unroll
  for (int k = 0; k < 8; ++k) a[k] = (b4 ? v[k + 8] : v[k]) + __shfl_xor_sync(0xffffffffu, b4 ? v[k] : v[k + 8], 16);
#pragma unroll
  for (int k = 0; k < 4; ++k) b[k] = (b3 ? a[k + 4] : a[k]) + __shfl_xor_sync(0xffffffffu, b3 ? a[k] : a[k + 4], 8);
#pragma unroll
  for (int k = 0; k < 2; ++k) c[k] = (b2 ? b[k + 2] : b[k]) + __shfl_xor_sync(0xffffffffu, b2 ? b[k] : b[k + 2], 4);
  float z = (b1 ? c[1] : c[0]) + __shfl_xor_sync(0xffffffffu, b1 ? c[0] : c[1], 2);
  z += __shfl_xor_sync(0xffffffffu, z, 1);
  return z;          // value index = (lane >> 1) & 15
}

__global__ void __launch_bounds__(256) pose_backward_kernel(int ng, int B, int Kg, const float* __restrict__ bone,
    const float4* __restrict__ g_static, const float* __restrict__ g_w, const float4* __restrict__ g_quat, const float4* __restrict__ g_scale_op,
    const int* __restrict__ knn_g, const float* __restrict__ ubar_g, const float* __restrict__ vt_normal,
    const float* __restrict__ d_mean, const float* __restrict__ d_mean2, const float* __restrict__ d_normal, const float* __restrict__ d_cov, const float* __restrict__ d_alb,
    const float* __restrict__ d_rough, const float* __restrict__ d_spec,
    float* __restrict__ o_gpos, float* __restrict__ o_gquat, float* __restrict__ o_gscale, float* __restrict__ o_bones,
    float* __restrict__ o_vdisp, float* __restrict__ o_vnormal, float* __restrict__ o_valb, float* __restrict__ o_vrough, float* __restrict__ o_vspec,
    const int* __restrict__ order) {
  extern __shared__ float smem[];
  float* sG = smem;                 // [B][12] bone transforms
  float* sB = smem + 12 * B;        // [B][12] their gradient, this CTA's share
  for (int t = threadIdx.x; t < 12 * B; t += blockDim.x) { sG[t] = bone[t]; sB[t] = 0.f; }
  __syncthreads();
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  float gM[12];
#pragma unroll
  for (int e = 0; e < 12; ++e) gM[e] = 0.f;
  if (g < ng) {
    const int gc = order[g];          // the caller's index: [n_gauss] gradient arrays come and go in the caller's order
    const float* w = g_w + (size_t)g * B;
    float M[12];
#pragma unroll
    for (int e = 0; e < 12; ++e) M[e] = 0.f;
    for (int b = 0; b < B; ++b) {
      const float wb = __ldg(w + b);
      if (wb != 0.f) {
#pragma unroll
        for (int e = 0; e < 12; ++e) M[e] = fmaf(wb, sG[12 * b + e], M[e]);
      }
    }
    const float4 p4 = g_static[4 * (size_t)g], n4 = g_static[4 * (size_t)g + 1];
    const float p[3] = {p4.x, p4.y, p4.z}, n[3] = {n4.x, n4.y, n4.z};
    int kk[PB_MAXK]; float uu[PB_MAXK];
    for (int j = 0; j < Kg; ++j) { kk[j] = knn_g[(size_t)g * Kg + j]; uu[j] = ubar_g[(size_t)g * Kg + j]; }
    // ---- position: xbar = M3 p + t
    float gx[3] = {0.f, 0.f, 0.f};
    if (d_mean) { gx[0] = d_mean[3 * (size_t)gc]; gx[1] = d_mean[3 * (size_t)gc + 1]; gx[2] = d_mean[3 * (size_t)gc + 2]; }
    if (d_mean2) { gx[0] += d_mean2[3 * (size_t)gc]; gx[1] += d_mean2[3 * (size_t)gc + 1]; gx[2] += d_mean2[3 * (size_t)gc + 2]; }
    float gp[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) gp[c] = M[c] * gx[0] + M[4 + c] * gx[1] + M[8 + c] * gx[2];
#pragma unroll
    for (int r = 0; r < 3; ++r) { gM[4 * r] = gx[r] * p[0]; gM[4 * r + 1] = gx[r] * p[1]; gM[4 * r + 2] = gx[r] * p[2]; gM[4 * r + 3] = gx[r]; }
    if (o_gpos) { o_gpos[3 * (size_t)gc] = gp[0]; o_gpos[3 * (size_t)gc + 1] = gp[1]; o_gpos[3 * (size_t)gc + 2] = gp[2]; }
    if (o_vdisp && (d_mean || d_mean2))
      for (int j = 0; j < Kg; ++j)
#pragma unroll
        for (int c = 0; c < 3; ++c) { const float v = uu[j] * gp[c]; if (v != 0.f) atomicAdd(o_vdisp + 3 * (size_t)kk[j] + c, v); }
    // ---- normal: nbar = t / |t|, t = M3 n_g, n_g = nraw / |nraw|, nraw = Eq.1(n_v)
    if (d_normal) {
      const float gn[3] = {d_normal[3 * (size_t)gc], d_normal[3 * (size_t)gc + 1], d_normal[3 * (size_t)gc + 2]};
      if (gn[0] != 0.f || gn[1] != 0.f || gn[2] != 0.f) {
        float t[3];
#pragma unroll
        for (int r = 0; r < 3; ++r) t[r] = M[4 * r] * n[0] + M[4 * r + 1] * n[1] + M[4 * r + 2] * n[2];
        const float len = sqrtf(t[0] * t[0] + t[1] * t[1] + t[2] * t[2]);
        if (len > 0.f) {
          const float il = 1.f / len;
          const float nb[3] = {t[0] * il, t[1] * il, t[2] * il};
          const float dt = gn[0] * nb[0] + gn[1] * nb[1] + gn[2] * nb[2];
          const float gt[3] = {(gn[0] - dt * nb[0]) * il, (gn[1] - dt * nb[1]) * il, (gn[2] - dt * nb[2]) * il};
#pragma unroll
          for (int r = 0; r < 3; ++r) { gM[4 * r] += gt[r] * n[0]; gM[4 * r + 1] += gt[r] * n[1]; gM[4 * r + 2] += gt[r] * n[2]; }
          if (o_vnormal) {
            float gng[3], nr[3] = {0.f, 0.f, 0.f};
#pragma unroll
            for (int c = 0; c < 3; ++c) gng[c] = M[c] * gt[0] + M[4 + c] * gt[1] + M[8 + c] * gt[2];
            for (int j = 0; j < Kg; ++j)
#pragma unroll
              for (int c = 0; c < 3; ++c) nr[c] = fmaf(uu[j], vt_normal[3 * (size_t)kk[j] + c], nr[c]);
            const float ln = sqrtf(nr[0] * nr[0] + nr[1] * nr[1] + nr[2] * nr[2]);
            if (ln > 0.f) {
              const float d2 = gng[0] * n[0] + gng[1] * n[1] + gng[2] * n[2], iln = 1.f / ln;
              for (int j = 0; j < Kg; ++j)
#pragma unroll
                for (int c = 0; c < 3; ++c) { const float v = uu[j] * (gng[c] - d2 * n[c]) * iln; if (v != 0.f) atomicAdd(o_vnormal + 3 * (size_t)kk[j] + c, v); }
            }
          }
        }
      }
    }
    // ---- covariance: Sigma = A A^T, A = M3 R diag(s)
    float gq[4] = {0.f, 0.f, 0.f, 0.f}, gs[3] = {0.f, 0.f, 0.f};
    if (d_cov) {
      const float* c6 = d_cov + 6 * (size_t)gc;
      const float G[9] = {c6[0], 0.5f * c6[1], 0.5f * c6[2], 0.5f * c6[1], c6[3], 0.5f * c6[4], 0.5f * c6[2], 0.5f * c6[4], c6[5]};
      const float4 q4 = g_quat[g]; const float4 so = g_scale_op[g];
      const float ql = sqrtf(q4.x * q4.x + q4.y * q4.y + q4.z * q4.z + q4.w * q4.w), iq = 1.f / ql;
      const float qw = q4.x * iq, qx = q4.y * iq, qy = q4.z * iq, qz = q4.w * iq;
      const float R[9] = {1.f - 2.f * (qy * qy + qz * qz), 2.f * (qx * qy - qw * qz), 2.f * (qx * qz + qw * qy),
                          2.f * (qx * qy + qw * qz), 1.f - 2.f * (qx * qx + qz * qz), 2.f * (qy * qz - qw * qx),
                          2.f * (qx * qz - qw * qy), 2.f * (qy * qz + qw * qx), 1.f - 2.f * (qx * qx + qy * qy)};
      const float s[3] = {so.x, so.y, so.z};
      float RS[9], A[9], gA[9], gRS[9];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) RS[3 * r + c] = R[3 * r + c] * s[c];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) A[3 * r + c] = M[4 * r] * RS[c] + M[4 * r + 1] * RS[3 + c] + M[4 * r + 2] * RS[6 + c];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) gA[3 * r + c] = 2.f * (G[3 * r] * A[c] + G[3 * r + 1] * A[3 + c] + G[3 * r + 2] * A[6 + c]);
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          gM[4 * r + c] += gA[3 * r] * RS[3 * c] + gA[3 * r + 1] * RS[3 * c + 1] + gA[3 * r + 2] * RS[3 * c + 2];      // gA RS^T
          gRS[3 * r + c] = M[r] * gA[c] + M[4 + r] * gA[3 + c] + M[8 + r] * gA[6 + c];                               // M3^T gA
        }
      float gR[9];
#pragma unroll
      for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) { gs[c] += gRS[3 * r + c] * R[3 * r + c]; gR[3 * r + c] = gRS[3 * r + c] * s[c]; }
      const float hw = 2.f * (-qz * gR[1] + qy * gR[2] + qz * gR[3] - qx * gR[5] - qy * gR[6] + qx * gR[7]);
      const float hx = 2.f * (qy * gR[1] + qz * gR[2] + qy * gR[3] - 2.f * qx * gR[4] - qw * gR[5] + qz * gR[6] + qw * gR[7] - 2.f * qx * gR[8]);
      const float hy = 2.f * (-2.f * qy * gR[0] + qx * gR[1] + qw * gR[2] + qx * gR[3] + qz * gR[5] - qw * gR[6] + qz * gR[7] - 2.f * qy * gR[8]);
      const float hz = 2.f * (-2.f * qz * gR[0] - qw * gR[1] + qx * gR[2] + qw * gR[3] - 2.f * qz * gR[4] + qy * gR[5] + qx * gR[6] + qy * gR[7]);
      const float dq = hw * qw + hx * qx + hy * qy + hz * qz;                 // q / |q|: remove the radial part, divide by |q|
      gq[0] = (hw - dq * qw) * iq; gq[1] = (hx - dq * qx) * iq; gq[2] = (hy - dq * qy) * iq; gq[3] = (hz - dq * qz) * iq;
    }
    if (o_gquat) { o_gquat[4 * (size_t)gc] = gq[0]; o_gquat[4 * (size_t)gc + 1] = gq[1]; o_gquat[4 * (size_t)gc + 2] = gq[2]; o_gquat[4 * (size_t)gc + 3] = gq[3]; }
    if (o_gscale) { o_gscale[3 * (size_t)gc] = gs[0]; o_gscale[3 * (size_t)gc + 1] = gs[1]; o_gscale[3 * (size_t)gc + 2] = gs[2]; }
    // ---- materials: transpose of Eq.1
    for (int j = 0; j < Kg; ++j) {
      const size_t k = (size_t)kk[j];
      if (o_valb && d_alb)
#pragma unroll
        for (int c = 0; c < 3; ++c) { const float v = uu[j] * d_alb[3 * (size_t)gc + c]; if (v != 0.f) atomicAdd(o_valb + 3 * k + c, v); }
      if (o_vrough && d_rough) { const float v = uu[j] * d_rough[gc]; if (v != 0.f) atomicAdd(o_vrough + k, v); }
      if (o_vspec && d_spec) { const float v = uu[j] * d_spec[gc]; if (v != 0.f) atomicAdd(o_vspec + k, v); }
    }
  }
  // ---- pose: dL/dG_b = sum_g w_gb dL/dM_g.  Neighbouring Gaussians share their bones: per bone the warp reduces its 12
  // sums with shuffles and adds them once (one atomic per thread and entry serialised 256-fold on the same few addresses)
  if (o_bones) {
    const int lane = threadIdx.x & 31;
    bool any = false;
#pragma unroll
    for (int e = 0; e < 12; ++e) any = any || gM[e] != 0.f;
    for (int b = 0; b < B; ++b) {
      const float wb = (g < ng && any) ? __ldg(g_w + (size_t)g * B + b) : 0.f;
      if (!__any_sync(0xffffffffu, wb != 0.f)) continue;
      float v[16];
#pragma unroll
      for (int e = 0; e < 12; ++e) v[e] = wb * gM[e];
      v[12] = v[13] = v[14] = v[15] = 0.f;
      const float z = warp_reduce16(v, lane);
      const int e = lane >> 1;
      if (!(lane & 1) && e < 12 && z != 0.f) atomicAdd(sB + 12 * b + e, z);
    }
  }
  __syncthreads();
  if (o_bones)
    for (int t = threadIdx.x; t < 12 * B; t += blockDim.x) { const float v = sB[t]; if (v != 0.f) atomicAdd(o_bones + t, v); }
}

cudaError_t rga_launch_pose_backward(rga_avatar* av, const float* bone_mats, const rga_posed_grads* in, const rga_canonical_grads* out, cudaStream_t s) {
  cudaError_t e = cudaSuccess;
  const size_t nv = av->n_verts;
#define PB_ZERO(ptr, bytes) if ((ptr) && (e = cudaMemsetAsync((ptr), 0, (bytes), s)) != cudaSuccess) return e;
  PB_ZERO(out->d_bones, 48 * (size_t)av->n_bones) PB_ZERO(out->d_vert_disp, 12 * nv) PB_ZERO(out->d_vert_normal, 12 * nv)
  PB_ZERO(out->d_vert_albedo, 12 * nv) PB_ZERO(out->d_vert_rough, 4 * nv) PB_ZERO(out->d_vert_spec, 4 * nv)
#undef PB_ZERO
  const size_t smem = 2 * 12 * (size_t)av->n_bones * sizeof(float);
  pose_backward_kernel<<<(av->n_gauss + 255) / 256, 256, smem, s>>>(av->n_gauss, av->n_bones, av->k_g, bone_mats, av->g_static, av->g_skin_w,
      av->g_quat, av->g_scale_op, av->knn_g, av->ubar_g, av->vt_normal, in->d_mean, in->d_mean2, in->d_normal, in->d_cov, in->d_albedo, in->d_rough, in->d_spec,
      out->d_gauss_pos, out->d_gauss_quat, out->d_gauss_scale, out->d_bones, out->d_vert_disp, out->d_vert_normal, out->d_vert_albedo,
      out->d_vert_rough, out->d_vert_spec, av->g_order);
  rga_prof_mark(av, "pose_backward", s);
  av->launches += 1;
  return cudaGetLastError();
}
