// Backward of H5 shade_gaussians: given dL/dcolour per Gaussian, the gradient w.r.t. the albedo,
// roughness, specular, posed normal and posed position (through w_o) of every Gaussian and w.r.t. the environment map,
// i.e. the material and lighting parameters the paper trains (BRDF Appendix A :454-471).
// Visibility is a frozen input.  FAST source: compared with the fp64 autograd oracle under tolerance.
//
// Same layout as the forward (shade_kernels.cu): 4 lanes per Gaussian, each walking a strided quarter of the environment
// texels from the table staged in shared memory.  Per live (Gaussian, texel) pair, with s the specular term and
// q = dL/d(ln s):  d ln s = c_nh d(n.h) + dlnF d(w_o.h) + c_ni d(n.w_i) + c_no d(n.w_o) + (...) d(roughness), and since
// h = (w_i + w_o) / |w_i + w_o| every vector gradient is a combination of w_i, w_o and n, so a lane only accumulates two
// weighted sums of w_i and a few scalars.  The environment gradient of a texel sums over Gaussians: the 8 lanes of a warp
// that hold the same texel are reduced by shuffles, added to a per-CTA table in shared memory, and the persistent CTAs
// flush that table with global atomics once at the end.
// A Gaussian whose dL/dcolour is zero (culled, hidden, or its radiance clamped: reading A33) is skipped.
#include "rga_internal.h"

#define PI_F 3.14159265358979323846f
#define SB_THREADS 128
#define SB_LANES 4

__device__ __forceinline__ float sb_rsq(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sb_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sb_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

template <int MODE>
__global__ void __launch_bounds__(SB_THREADS) shade_backward_kernel(int ng, int ne, int K, int words, int Kg, int Kv,
    const float4* __restrict__ g_posed, const float4* __restrict__ g_nposed, const float4* __restrict__ g_static,
    const float* __restrict__ env_table, const int* __restrict__ t2d, const unsigned* __restrict__ visbits,
    const unsigned char* __restrict__ vcount, const int* __restrict__ knn_g, const float* __restrict__ ubar_g,
    float3 cam, float inv_gamma, const float4* __restrict__ radiance, const float* __restrict__ dL_dcolor,
    float* __restrict__ out_dalbedo, float* __restrict__ out_drough, float* __restrict__ out_dspec, float* __restrict__ out_dnormal,
    float* __restrict__ out_dpos, float* __restrict__ out_denv, int* __restrict__ work, const int* __restrict__ order) {
  extern __shared__ __align__(16) float smem[];
  float4* sE = reinterpret_cast<float4*>(smem);                          // [ne][2]: (w, A), (L A, 0)
  float* sG = reinterpret_cast<float*>(sE + 2 * ne);                     // [ne][3] environment gradient of this CTA
  unsigned short* sD = reinterpret_cast<unsigned short*>(sG + 3 * ne);   // [ne] texel -> direction
  for (int t = threadIdx.x; t < 2 * ne; t += blockDim.x) sE[t] = reinterpret_cast<const float4*>(env_table)[t];
  for (int t = threadIdx.x; t < 3 * ne; t += blockDim.x) sG[t] = 0.f;
  if (MODE != 2) for (int t = threadIdx.x; t < ne; t += blockDim.x) sD[t] = (unsigned short)(t2d ? t2d[t] : t);
  __syncthreads();
  const int GPB = SB_THREADS / SB_LANES;
  const int lane = threadIdx.x % SB_LANES;
  const float ip = 1.f / PI_F;
  __shared__ int s_base;
  for (;;) {
    // groups of GPB Gaussians are handed out dynamically: their cost varies with the share that faces the camera
    __syncthreads();
    if (threadIdx.x == 0) s_base = atomicAdd(work, GPB);
    __syncthreads();
    const int gbase = s_base;
    if (gbase >= ng) break;
    const int g = gbase + threadIdx.x / SB_LANES;
    bool active = g < ng;
    const int gc = active ? order[g] : 0;           // the caller's index: dL_dcolor and the [n_gauss] outputs are in the caller's order
    float4 x = make_float4(0.f, 0.f, 0.f, 0.f), n = x, ar = x;
    float gL0 = 0.f, gL1 = 0.f, gL2 = 0.f, spec = 0.f;
    if (active) {
      const float4 Lo = radiance[g];
      const float c0 = dL_dcolor[3 * (size_t)gc], c1 = dL_dcolor[3 * (size_t)gc + 1], c2 = dL_dcolor[3 * (size_t)gc + 2];
      // colour = clamp(L_o, 0, 1)^(1/gamma): slope (1/gamma) L_o^(1/gamma - 1) strictly inside the limits, 0 otherwise
      if (Lo.x > 0.f && Lo.x < 1.f) gL0 = c0 * inv_gamma * exp2f((inv_gamma - 1.f) * log2f(Lo.x));
      if (Lo.y > 0.f && Lo.y < 1.f) gL1 = c1 * inv_gamma * exp2f((inv_gamma - 1.f) * log2f(Lo.y));
      if (Lo.z > 0.f && Lo.z < 1.f) gL2 = c2 * inv_gamma * exp2f((inv_gamma - 1.f) * log2f(Lo.z));
      active = gL0 != 0.f || gL1 != 0.f || gL2 != 0.f;
    }
    float wox = 0.f, woy = 0.f, woz = 0.f, winv = 0.f;
    if (active) {
      x = g_posed[g]; n = g_nposed[g];
      ar = g_static[4 * (size_t)g + 2]; spec = g_static[4 * (size_t)g + 3].x;
      wox = cam.x - x.x; woy = cam.y - x.y; woz = cam.z - x.z;
      winv = rsqrtf(wox * wox + woy * woy + woz * woz);
      wox *= winv; woy *= winv; woz *= winv;
    }
    // accumulators: diffuse sums (albedo), specular, roughness, normal (sum a w_i, coefficient of w_o), w_o (sum c w_i, coefficients of n, w_o)
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, gp = 0.f, gr = 0.f, nx = 0.f, ny = 0.f, nz = 0.f, nwoc = 0.f, wx = 0.f, wy = 0.f, wz = 0.f, wnc = 0.f, wwoc = 0.f;
    if (__any_sync(0xffffffffu, active)) {
      const float nwo_raw = n.x * wox + n.y * woy + n.z * woz;
      const float nwo = fmaxf(nwo_raw, 0.f);
      const float rough = ar.w, al = rough * rough, al2 = al * al;
      const float kk = (rough + 1.f) * (rough + 1.f) * 0.125f, omk = 1.f - kk;
      const float go = nwo * omk + kk;
      const float tox = fmaf(-nwo_raw, n.x, wox), toy = fmaf(-nwo_raw, n.y, woy), toz = fmaf(-nwo_raw, n.z, woz);
      const float cS = al2 / (4.f * PI_F * go);
      const float c_no = nwo_raw > 0.f ? -omk / go : 0.f;
      const float a0g = ar.x * ip * gL0, a1g = ar.y * ip * gL1, a2g = ar.z * ip * gL2;
      float u0 = 0.f, u1 = 0.f, u2 = 0.f; int j0 = 0, j1 = 0, j2 = 0;
      if (MODE == 1 && active) {
        const float ikv = 1.0f / (float)Kv;
        j0 = knn_g[(size_t)g * Kg]; u0 = ubar_g[(size_t)g * Kg] * ikv;
        if (Kg > 1) { j1 = knn_g[(size_t)g * Kg + 1]; u1 = ubar_g[(size_t)g * Kg + 1] * ikv; }
        if (Kg > 2) { j2 = knn_g[(size_t)g * Kg + 2]; u2 = ubar_g[(size_t)g * Kg + 2] * ikv; }
      }
      const unsigned* vb = visbits + (size_t)(active ? g : 0) * words;
      int cur_wd = -1; unsigned cur_bits = 0u;
      for (int kb = 0; kb < ne; kb += SB_LANES) {
        const int k = kb + lane;
        float e0 = 0.f, e1 = 0.f, e2 = 0.f;                               // this pair's environment gradient
        bool live = active && k < ne;
        float4 wi = make_float4(0.f, 0.f, 0.f, 0.f);
        float cs = 0.f, v = 1.f;
        if (live) {
          wi = sE[2 * k];
          cs = n.x * wi.x + n.y * wi.y + n.z * wi.z;
          live = cs > 0.f;
        }
        if (live) {
          if (MODE == 0) {
            const int d = sD[k];
            if ((d >> 5) != cur_wd) { cur_wd = d >> 5; cur_bits = __ldg(vb + cur_wd); }
            live = (cur_bits >> (d & 31)) & 1u;
          } else if (MODE == 1) {
            const int d = sD[k];
            v = u0 * (float)__ldg(vcount + (size_t)j0 * K + d);
            if (Kg > 1) v += u1 * (float)__ldg(vcount + (size_t)j1 * K + d);
            if (Kg > 2) v += u2 * (float)__ldg(vcount + (size_t)j2 * K + d);
            live = v != 0.f;
          }
        }
        if (live) {
          const float4 LA = sE[2 * k + 1];
          // |w_i + w_o|^2 from the summed components: 2 + 2 w_o.w_i cancels to a few fp32 ulps of 2 when the light stands almost
          // opposite the viewer (|w_i + w_o| = 0.004: 1.5 % error in the half vector, 6e-3 in the radiance; found by the random sweep)
          const float hsx = wi.x + wox, hsy = wi.y + woy, hsz = wi.z + woz;
          const float hl2 = fmaxf(hsx * hsx + hsy * hsy + hsz * hsz, 1e-12f);
          const float hinv = sb_rsq(hl2);
          const float nh = (cs + nwo_raw) * hinv;
          const float oh = (0.5f * hl2) * hinv;
          const float tx = fmaf(-cs, n.x, wi.x) + tox, ty = fmaf(-cs, n.y, wi.y) + toy, tz = fmaf(-cs, n.z, wi.z) + toz;
          const float den = fmaf(al2 * nh, nh, (tx * tx + ty * ty + tz * tz) * (hinv * hinv));
          const float E = sb_ex2((-5.55473f * oh - 6.98316f) * oh);
          const float F = fmaf(0.96f, E, 0.04f);
          const float gi = fmaf(cs, omk, kk);
          const float rden = sb_rcp(den), rgi = sb_rcp(gi);
          const float sp = cS * F * rden * rden * rgi;
          const float w = v * cs;
          const float Lg = gL0 * LA.x + gL1 * LA.y + gL2 * LA.z;          // <dL/dL_o, L_k A_k>
          const float Ld = a0g * LA.x + a1g * LA.y + a2g * LA.z;          // the same through a / pi
          d0 = fmaf(LA.x, w, d0); d1 = fmaf(LA.y, w, d1); d2 = fmaf(LA.z, w, d2);
          gp = fmaf(Lg * w, sp, gp);
          // environment: d/dL_kc = A_k w (a_c / pi + p s) dL/dL_o,c
          const float Aw = wi.w * w, ps = spec * sp;
          e0 = Aw * fmaf(ar.x, ip, ps) * gL0; e1 = Aw * fmaf(ar.y, ip, ps) * gL1; e2 = Aw * fmaf(ar.z, ip, ps) * gL2;
          const float dLdcs = v * fmaf(ps, Lg, Ld);                       // through the explicit cosine factor
          const float q = w * ps * Lg;                                    // dL / d(ln s)
          const float c_nh = -4.f * nh * (al2 - 1.f) * rden, c_ni = -omk * rgi;
          const float dlnF = 0.96f * E * 0.6931471805599453f * (-11.10946f * oh - 6.98316f) * sb_rcp(F);
          // normal:  dLdcs w_i + q (c_nh h + c_ni w_i + c_no w_o),  h = (w_i + w_o) hinv
          const float an = dLdcs + q * (c_ni + c_nh * hinv);
          nx = fmaf(an, wi.x, nx); ny = fmaf(an, wi.y, ny); nz = fmaf(an, wi.z, nz);
          nwoc += q * (c_nh * hinv + c_no);
          // roughness: d ln s / d gamma = 4/gamma - 8 nh^2 gamma^3 / den - ((1 - n.w_i)/g_i + (1 - n.w_o)/g_o) (gamma + 1)/4
          gr += q * (4.f / rough - 8.f * nh * nh * rough * al * rden - ((1.f - cs) * rgi + (1.f - nwo) / go) * (rough + 1.f) * 0.25f);
          // w_o:  q [ c_nh (n - nh h) hinv + dlnF (h + (w_o - oh h) hinv) + c_no n ]
          const float cw = q * hinv * (dlnF - hinv * (c_nh * nh + dlnF * oh));
          wx = fmaf(cw, wi.x, wx); wy = fmaf(cw, wi.y, wy); wz = fmaf(cw, wi.z, wz);
          wwoc += cw + q * dlnF * hinv;
          wnc += q * (c_nh * hinv + c_no);
        }
        // the 8 lanes of the warp with this lane's texel
        if (__any_sync(0xffffffffu, live)) {
#pragma unroll
          for (int o = SB_LANES; o < 32; o <<= 1) {
            e0 += __shfl_xor_sync(0xffffffffu, e0, o); e1 += __shfl_xor_sync(0xffffffffu, e1, o); e2 += __shfl_xor_sync(0xffffffffu, e2, o);
          }
          if ((threadIdx.x & 31) < SB_LANES && k < ne) {
            if (e0 != 0.f) atomicAdd(sG + 3 * k, e0);
            if (e1 != 0.f) atomicAdd(sG + 3 * k + 1, e1);
            if (e2 != 0.f) atomicAdd(sG + 3 * k + 2, e2);
          }
        }
      }
      // the 4 lanes of a Gaussian
#pragma unroll
      for (int o = SB_LANES / 2; o > 0; o >>= 1) {
        d0 += __shfl_xor_sync(0xffffffffu, d0, o); d1 += __shfl_xor_sync(0xffffffffu, d1, o); d2 += __shfl_xor_sync(0xffffffffu, d2, o);
        gp += __shfl_xor_sync(0xffffffffu, gp, o); gr += __shfl_xor_sync(0xffffffffu, gr, o);
        nx += __shfl_xor_sync(0xffffffffu, nx, o); ny += __shfl_xor_sync(0xffffffffu, ny, o); nz += __shfl_xor_sync(0xffffffffu, nz, o);
        nwoc += __shfl_xor_sync(0xffffffffu, nwoc, o);
        wx += __shfl_xor_sync(0xffffffffu, wx, o); wy += __shfl_xor_sync(0xffffffffu, wy, o); wz += __shfl_xor_sync(0xffffffffu, wz, o);
        wnc += __shfl_xor_sync(0xffffffffu, wnc, o); wwoc += __shfl_xor_sync(0xffffffffu, wwoc, o);
      }
    }
    if (g < ng && lane == 0) {
      float o_n[3] = {0.f, 0.f, 0.f}, o_x[3] = {0.f, 0.f, 0.f};
      if (active) {
        o_n[0] = nx + nwoc * wox; o_n[1] = ny + nwoc * woy; o_n[2] = nz + nwoc * woz;
        const float gwx = wx + wnc * n.x + wwoc * wox, gwy = wy + wnc * n.y + wwoc * woy, gwz = wz + wnc * n.z + wwoc * woz;
        const float dt = gwx * wox + gwy * woy + gwz * woz;               // w_o = (cam - x) / |cam - x|
        o_x[0] = -(gwx - dt * wox) * winv; o_x[1] = -(gwy - dt * woy) * winv; o_x[2] = -(gwz - dt * woz) * winv;
      }
      if (out_dalbedo) { out_dalbedo[3 * (size_t)gc] = gL0 * d0 * ip; out_dalbedo[3 * (size_t)gc + 1] = gL1 * d1 * ip; out_dalbedo[3 * (size_t)gc + 2] = gL2 * d2 * ip; }
      if (out_dspec) out_dspec[gc] = gp;
      if (out_drough) out_drough[gc] = gr;
      if (out_dnormal) { out_dnormal[3 * (size_t)gc] = o_n[0]; out_dnormal[3 * (size_t)gc + 1] = o_n[1]; out_dnormal[3 * (size_t)gc + 2] = o_n[2]; }
      if (out_dpos) { out_dpos[3 * (size_t)gc] = o_x[0]; out_dpos[3 * (size_t)gc + 1] = o_x[1]; out_dpos[3 * (size_t)gc + 2] = o_x[2]; }
    }
  }
  __syncthreads();
  if (out_denv)
    for (int t = threadIdx.x; t < 3 * ne; t += blockDim.x) { const float e = sG[t]; if (e != 0.f) atomicAdd(out_denv + t, e); }
}

cudaError_t rga_launch_shade_backward(rga_avatar* av, const rga_env* env, float3 cam, int vis_mode, const float* dL_dcolor, float* out_dalbedo,
                                      float* out_drough, float* out_dspec, float* out_dnormal, float* out_dpos, float* out_denv, cudaStream_t s) {
  const int ne = env->rows * env->cols;
  const size_t smem = (size_t)ne * 32 + (size_t)ne * 12 + (size_t)ne * 2;
  const float ig = 1.0f / env->gamma;
  cudaError_t e = cudaSuccess;
  if (out_denv && (e = cudaMemsetAsync(out_denv, 0, sizeof(float) * 3 * (size_t)ne, s)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(av->work_counter, 0, sizeof(int), s)) != cudaSuccess) return e;
  const int gpb = SB_THREADS / SB_LANES;
  const int grid = min((av->n_gauss + gpb - 1) / gpb, av->num_sms * 8);
#define SB_ARGS av->n_gauss, ne, av->vis_dirs, av->vis_words, av->k_g, av->k_v, av->g_posed, av->g_nposed, av->g_static, av->env_table, \
    env->texel_to_dir, av->visbits, av->vcount, av->knn_g, av->ubar_g, cam, ig, av->radiance, dL_dcolor, out_dalbedo, out_drough, out_dspec, \
    out_dnormal, out_dpos, out_denv, av->work_counter, av->g_order
  if (vis_mode == 0) shade_backward_kernel<0><<<grid, SB_THREADS, smem, s>>>(SB_ARGS);
  else if (vis_mode == 1) shade_backward_kernel<1><<<grid, SB_THREADS, smem, s>>>(SB_ARGS);
  else shade_backward_kernel<2><<<grid, SB_THREADS, smem, s>>>(SB_ARGS);
  av->launches += 1;
  rga_prof_mark(av, "shade_backward", s);
  return cudaGetLastError();
}

// the backward kernels stage 46 bytes per environment texel: fewer texels fit than in the forward kernels (34 bytes)
int rga_shade_backward_max_texels() { return (int)((227 * 1024 - 1024) / 46); }

int rga_shade_backward_init_attributes(int max_env) {
  if (max_env > rga_shade_backward_max_texels()) max_env = rga_shade_backward_max_texels();   // larger maps: forward only (shade_backward refuses them)
  const size_t smem = (size_t)max_env * 46;
  cudaError_t e = cudaSuccess;
  if (smem > 48 * 1024) {
    e = cudaFuncSetAttribute(shade_backward_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(shade_backward_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(shade_backward_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  return (int)e;
}
