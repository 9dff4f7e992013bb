// H5 shade_gaussians: Eq.2 with the Appendix-A BRDF (Eq.12-15), then gamma.
// FAST file (default FMA contraction, MUFU intrinsics): the result is compared with the fp64 oracle under the
// north_star tolerance (2e-3 max-abs on colour), not bit-exactly.
//
// Layout: persistent CTAs draw groups of consecutive Gaussians from a ticket counter; one Gaussian per lane, the texel
// warp-uniform (see the comment above shade_kernel).  The env table (w_k, L_k A_k) is staged in shared memory once per
// CTA; visibility comes as bits (mode 0) or is 1 (mode 2).  Paper mode (mode 1: vertex counts gathered through S_g) runs
// shade_paper_kernel below, with several lanes per Gaussian.
#include "rga_internal.h"

#define PI_F 3.14159265358979323846f

// Reading A6: equirectangular z-up grid; A = exact solid angle of the texel = 2 sin(theta_c) sin(pi/(2R)) 2pi/C
// (the product form of cos(i pi/R) - cos((i+1) pi/R), free of cancellation in fp32).
__global__ void env_table_kernel(int rows, int cols, const float* __restrict__ radiance, float* __restrict__ table) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= rows * cols) return;
  int i = k / cols, j = k - i * cols;
  float st, ct, sp, cp;
  sincospif(((float)i + 0.5f) / (float)rows, &st, &ct);
  sincospif(2.0f * ((float)j + 0.5f) / (float)cols, &sp, &cp);
  float A = 2.0f * st * sinpif(0.5f / (float)rows) * (2.0f * PI_F / (float)cols);
  float4* t = reinterpret_cast<float4*>(table) + 2 * (size_t)k;
  t[0] = make_float4(st * cp, st * sp, ct, A);                       // .w = A_k: read by the backward pass only
  t[1] = make_float4(radiance[3 * k] * A, radiance[3 * k + 1] * A, radiance[3 * k + 2] * A, 0.f);
}

cudaError_t rga_launch_env_table(rga_avatar* av, const rga_env* env, cudaStream_t s) {
  int n = env->rows * env->cols;
  env_table_kernel<<<(n + 127) / 128, 128, 0, s>>>(env->rows, env->cols, env->radiance, av->env_table);
  av->launches += 1;
  rga_prof_mark(av, "env_table", s);
  return cudaGetLastError();
}

// MUFU approximations (relative error ~1e-6; the result is compared under the 2e-3 tolerance)
__device__ __forceinline__ float rsq_approx(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rcp_approx(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float ex2_approx(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// Work decomposition: persistent CTAs of SH_WARPS warps draw groups of SH_GROUP consecutive Gaussians from a ticket counter.
// The group's camera-facing Gaussians are compacted (the others only get zeros: PAPER.md:101), then every warp walks ITS
// 32-texel blocks of the environment map (block w, w + SH_WARPS, ...) with one Gaussian per lane.  The texel is warp-uniform, so its table row is a broadcast
// read and -- Gaussians being stored in spatial order, with similar normals and shadows -- the two skip tests
// (w_i.n <= 0, visibility bit clear) mostly agree across the warp: a texel that no lane needs costs the test only
// (the first version gave four lanes to a Gaussian and every lane its own texel, so a warp ran the BRDF block in nearly
// every trip with half of its lanes idle: 67 us at config 1).  Slice partials are folded in slice order in shared memory.
#ifndef SH_UNROLL
#define SH_UNROLL 8
#endif
#define RGA_STR(x) #x
#define RGA_UNROLL(n) _Pragma(RGA_STR(unroll n))
#ifndef SH_THREADS
#define SH_THREADS 256
#endif
#define SH_WARPS (SH_THREADS / 32)
#ifndef SH_MINB
#define SH_MINB 1             // minimum resident CTAs per SM asked of the compiler (register cap)
#endif
#ifndef SH_GROUP
#define SH_GROUP 32
#endif

template <int MODE>
__global__ void __launch_bounds__(SH_THREADS, SH_MINB) shade_kernel(int ng, int ne, int K, int words, int Kg, int Kv,
    const float4* __restrict__ g_posed, const float4* __restrict__ g_nposed, const float4* __restrict__ g_static,
    const float* __restrict__ env_table, const int* __restrict__ t2d, const unsigned* __restrict__ visbits,
    const unsigned char* __restrict__ vcount, const int* __restrict__ knn_g, const float* __restrict__ ubar_g,
    float3 cam, float inv_gamma, float4* __restrict__ radiance, float4* __restrict__ color, unsigned* __restrict__ counter) {
  extern __shared__ __align__(16) float smem[];
  float4* sE = reinterpret_cast<float4*>(smem);                          // [ne][2]
  float* sPart = reinterpret_cast<float*>(sE + 2 * ne);                  // [SH_WARPS][6][SH_GROUP] slice partials
  unsigned short* sD = reinterpret_cast<unsigned short*>(sPart + SH_WARPS * 6 * SH_GROUP);   // [ne] texel -> direction
  __shared__ int s_list[SH_GROUP];
  __shared__ int s_cnt[SH_GROUP / 32];
  __shared__ unsigned s_ticket;
  for (int t = threadIdx.x; t < 2 * ne; t += blockDim.x) sE[t] = reinterpret_cast<const float4*>(env_table)[t];
  int ident_local = 1;                                                   // texel k -> direction k: a block of 32 texels is one word
  if (MODE != 2) for (int t = threadIdx.x; t < ne; t += blockDim.x) { const int d = t2d ? t2d[t] : t; sD[t] = (unsigned short)d; ident_local &= (d == t); }
  const bool ident = __syncthreads_and(ident_local) != 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const unsigned ngroups = (unsigned)((ng + SH_GROUP - 1) / SH_GROUP);
  const int nblk = (ne + 31) >> 5;                                       // warp w walks the 32-texel blocks w, w + SH_WARPS, ...
  for (;;) {
    __syncthreads();                                                     // s_ticket, s_list and sPart are reused
    if (threadIdx.x == 0) s_ticket = atomicAdd(counter, 1u);
    __syncthreads();
    const unsigned ticket = s_ticket;
    if (ticket >= ngroups) {
      // every CTA draws exactly one ticket beyond the groups: the last of them re-arms the counter for the next launch
      if (threadIdx.x == 0 && ticket == ngroups + gridDim.x - 1u) *counter = 0u;
      break;
    }
    // a Gaussian facing away from the camera gets opacity 0, so its colour is never used.  Skip it only
    // when the sign is certain (the exact test lives in the projection kernel).
    bool keep = false; unsigned bal = 0u;
    const int gl = (int)ticket * SH_GROUP + (int)threadIdx.x;
    if (threadIdx.x < SH_GROUP) {
      if (gl < ng) {
        const float4 x = g_posed[gl], n = g_nposed[gl];
        const float wx = cam.x - x.x, wy = cam.y - x.y, wz = cam.z - x.z;
        keep = !(n.x * wx + n.y * wy + n.z * wz < -1e-4f * sqrtf(wx * wx + wy * wy + wz * wz));
        if (!keep) { radiance[gl] = make_float4(0.f, 0.f, 0.f, 0.f); color[gl] = make_float4(0.f, 0.f, 0.f, 0.f); }
      }
      bal = __ballot_sync(0xffffffffu, keep);
      if (lane == 0) s_cnt[warp] = __popc(bal);
    }
    __syncthreads();
    int m = 0;
#pragma unroll
    for (int w = 0; w < SH_GROUP / 32; ++w) { const int c = s_cnt[w]; if (keep && w == warp) s_list[m + __popc(bal & ((1u << lane) - 1u))] = gl; m += c; }
    __syncthreads();
    for (int c0 = 0; c0 < m; c0 += 32) {
      const int li = c0 + lane;
      const bool valid = li < m;
      const int g = s_list[valid ? li : c0];                             // idle lanes shadow the chunk's first Gaussian
      const float4 x = g_posed[g], n = g_nposed[g];
      float wox = cam.x - x.x, woy = cam.y - x.y, woz = cam.z - x.z;
      const float winv = rsqrtf(wox * wox + woy * woy + woz * woz);
      wox *= winv; woy *= winv; woz *= winv;
      const float rough = g_static[4 * (size_t)g + 2].w;
      const float nwo_raw = n.x * wox + n.y * woy + n.z * woz;
      const float nwo = fmaxf(nwo_raw, 0.f);
      const float al = rough * rough, al2 = al * al;                     // Eq.13: alpha = gamma^2
      const float kk = (rough + 1.f) * (rough + 1.f) * 0.125f, omk = 1.f - kk;   // Eq.15
      const float go = nwo * omk + kk;
      // 1 - (n.h)^2 = |t|^2 / |w_i + w_o|^2 with t the part of w_i + w_o tangent to n, summed from the two tangent parts
      // (the direct form 1 - nh^2 cancels badly for alpha^2 ~ 1e-4); this is w_o's
      const float tox = fmaf(-nwo_raw, n.x, wox), toy = fmaf(-nwo_raw, n.y, woy), toz = fmaf(-nwo_raw, n.z, woz);
      const float cS = al2 / (4.f * PI_F * go);                          // D F G /(4 ni no) = cS F / (den^2 gi)
      const unsigned* vb = visbits + (size_t)g * words;
      float d0 = 0.f, d1 = 0.f, d2 = 0.f, s0 = 0.f, s1 = 0.f, s2 = 0.f;
      for (int blk = warp; blk < nblk; blk += SH_WARPS) {
        const int kb = blk << 5, kn = min(32, ne - kb);
        // visibility of the block's texels as one mask per lane (bit j = texel kb + j)
        unsigned vm = 0xffffffffu;
        if (MODE == 0) {
          if (ident) vm = __ldg(vb + blk);
          else {
            int cur_wd = -1; unsigned cur_bits = 0u; vm = 0u;
            for (int j = 0; j < kn; ++j) {
              const int d = sD[kb + j];
              if ((d >> 5) != cur_wd) { cur_wd = d >> 5; cur_bits = __ldg(vb + cur_wd); }       // warp-uniform branch
              vm |= ((cur_bits >> (d & 31)) & 1u) << j;
            }
          }
        }
        if (!valid) vm = 0u;
        if (!__any_sync(0xffffffffu, vm != 0u)) continue;
        const float4* sEk = sE + 2 * kb;
        RGA_UNROLL(SH_UNROLL)
        for (int j = 0; j < kn; ++j) {
          const float4 wi = sEk[2 * j];
          const float cs = n.x * wi.x + n.y * wi.y + n.z * wi.z;
          bool live = (cs > 0.f) && ((vm >> j) & 1u);                    // max(0, w_i . n) and the visibility bit
          if (!__any_sync(0xffffffffu, live)) continue;
          if (live) {
            const float4 LA = sEk[2 * j + 1];
            // |w_i + w_o|^2 from the summed components: 2 + 2 w_o.w_i cancels to a few fp32 ulps of 2 when the light stands almost
            // opposite the viewer (|w_i + w_o| = 0.004: 1.5 % error in the half vector, 6e-3 in the radiance; found by the random sweep)
            const float hsx = wi.x + wox, hsy = wi.y + woy, hsz = wi.z + woz;
            const float hl2 = fmaxf(hsx * hsx + hsy * hsy + hsz * hsz, 1e-12f);
            const float hinv = rsq_approx(hl2);
            const float nh = (cs + nwo_raw) * hinv;
            const float oh = (0.5f * hl2) * hinv;                        // w_o . h = (1 + w_o.w_i) / |w_i + w_o|
            const float tx = fmaf(-cs, n.x, wi.x) + tox, ty = fmaf(-cs, n.y, wi.y) + toy, tz = fmaf(-cs, n.z, wi.z) + toz;
            const float den = fmaf(al2 * nh, nh, (tx * tx + ty * ty + tz * tz) * (hinv * hinv));   // (n.h)^2 (a^2 - 1) + 1, Eq.13
            const float F = fmaf(0.96f, ex2_approx((-5.55473f * oh - 6.98316f) * oh), 0.04f);     // Eq.14
            const float gi = fmaf(cs, omk, kk);
            const float sp = cS * F * rcp_approx(den * den * gi);
            const float w = cs;                                          // visibility is the mask (modes 0, 2)
            const float ws = w * sp;
            d0 = fmaf(LA.x, w, d0); d1 = fmaf(LA.y, w, d1); d2 = fmaf(LA.z, w, d2);
            s0 = fmaf(LA.x, ws, s0); s1 = fmaf(LA.y, ws, s1); s2 = fmaf(LA.z, ws, s2);
          }
        }
      }
      if (valid) {
        float* o = sPart + (size_t)warp * 6 * SH_GROUP + li;
        o[0] = d0; o[SH_GROUP] = d1; o[2 * SH_GROUP] = d2; o[3 * SH_GROUP] = s0; o[4 * SH_GROUP] = s1; o[5 * SH_GROUP] = s2;
      }
    }
    __syncthreads();
    if ((int)threadIdx.x < m) {
      const int g = s_list[threadIdx.x];
      float a[6];
#pragma unroll
      for (int q = 0; q < 6; ++q) {
        float acc = 0.f;
#pragma unroll
        for (int w = 0; w < SH_WARPS; ++w) acc += sPart[((size_t)w * 6 + q) * SH_GROUP + threadIdx.x];
        a[q] = acc;
      }
      const float4 ar = g_static[4 * (size_t)g + 2];                     // albedo rgb, roughness
      const float spec = g_static[4 * (size_t)g + 3].x;
      const float ip = 1.f / PI_F;
      float L0 = ar.x * ip * a[0] + spec * a[3], L1 = ar.y * ip * a[1] + spec * a[4], L2 = ar.z * ip * a[2] + spec * a[5];   // Eq.12
      radiance[g] = make_float4(L0, L1, L2, 0.f);
      float c0 = exp2f(inv_gamma * log2f(fminf(fmaxf(L0, 0.f), 1.f)));
      float c1 = exp2f(inv_gamma * log2f(fminf(fmaxf(L1, 0.f), 1.f)));
      float c2 = exp2f(inv_gamma * log2f(fminf(fmaxf(L2, 0.f), 1.f)));
      color[g] = make_float4(c0, c1, c2, 0.f);
    }
  }
}

// Paper-mode shading (vis_mode 1: visibility = Eq.1 over the K_g neighbour vertices' filtered counts).
// LANES threads cooperate on one Gaussian and every lane walks its own texels: the lanes of a Gaussian then read
// neighbouring bytes of the same three vcount rows (with one Gaussian per lane, as in shade_kernel, the 3 x 512 byte
// gathers of a warp go to 96 different rows: 105 us against 89 us at config 1).
template <int LANES>
__global__ void __launch_bounds__(128) shade_paper_kernel(int ng, int ne, int K, int words, int Kg, int Kv,
    const float4* __restrict__ g_posed, const float4* __restrict__ g_nposed, const float4* __restrict__ g_static,
    const float* __restrict__ env_table, const int* __restrict__ t2d, const unsigned* __restrict__ visbits,
    const unsigned char* __restrict__ vcount, const int* __restrict__ knn_g, const float* __restrict__ ubar_g,
    float3 cam, float inv_gamma, float4* __restrict__ radiance, float4* __restrict__ color) {
  extern __shared__ __align__(16) float smem[];
  float4* sE = reinterpret_cast<float4*>(smem);                          // [ne][2]
  unsigned short* sD = reinterpret_cast<unsigned short*>(sE + 2 * ne);   // [ne] texel -> direction
  for (int t = threadIdx.x; t < 2 * ne; t += blockDim.x) sE[t] = reinterpret_cast<const float4*>(env_table)[t];
  for (int t = threadIdx.x; t < ne; t += blockDim.x) sD[t] = (unsigned short)(t2d ? t2d[t] : t);
  __syncthreads();
  const int GPB = 128 / LANES;                                           // Gaussians per block
  const int lane = threadIdx.x % LANES;
  const int g = blockIdx.x * GPB + threadIdx.x / LANES;
  if (g >= ng) return;                                                   // whole LANES-group exits together
  const float4 x = g_posed[g], n = g_nposed[g];
  float wox = cam.x - x.x, woy = cam.y - x.y, woz = cam.z - x.z;
  const float wl2 = wox * wox + woy * woy + woz * woz;
  const float facing = n.x * wox + n.y * woy + n.z * woz;
  // a Gaussian facing away from the camera gets opacity 0, so its colour is never used.  Skip it only
  // when the sign is certain (the exact test lives in the projection kernel).
  if (facing < -1e-4f * sqrtf(wl2)) {
    if (lane == 0) { radiance[g] = make_float4(0.f, 0.f, 0.f, 0.f); color[g] = make_float4(0.f, 0.f, 0.f, 0.f); }
    return;
  }
  const float winv = rsqrtf(wl2);
  wox *= winv; woy *= winv; woz *= winv;
  const float4 ar = g_static[4 * (size_t)g + 2];                         // albedo rgb, roughness
  const float spec = g_static[4 * (size_t)g + 3].x;
  const float nwo_raw = n.x * wox + n.y * woy + n.z * woz;
  const float nwo = fmaxf(nwo_raw, 0.f);
  const float rough = ar.w, al = rough * rough, al2 = al * al;           // Eq.13: alpha = gamma^2
  const float kk = (rough + 1.f) * (rough + 1.f) * 0.125f, omk = 1.f - kk;   // Eq.15
  const float go = nwo * omk + kk;
  // 1 - (n.h)^2 = |t|^2 / |w_i + w_o|^2 with t the part of w_i + w_o tangent to n, summed from the two tangent parts
  // (the direct form 1 - nh^2 cancels badly for alpha^2 ~ 1e-4); this is w_o's
  const float tox = fmaf(-nwo_raw, n.x, wox), toy = fmaf(-nwo_raw, n.y, woy), toz = fmaf(-nwo_raw, n.z, woz);
  const float cS = al2 / (4.f * PI_F * go);                              // D F G /(4 ni no) = cS F / (den^2 gi)
  float u0 = 0.f, u1 = 0.f, u2 = 0.f; int j0 = 0, j1 = 0, j2 = 0;
  {
    const float ikv = 1.0f / (float)Kv;
    j0 = knn_g[(size_t)g * Kg]; u0 = ubar_g[(size_t)g * Kg] * ikv;
    if (Kg > 1) { j1 = knn_g[(size_t)g * Kg + 1]; u1 = ubar_g[(size_t)g * Kg + 1] * ikv; }
    if (Kg > 2) { j2 = knn_g[(size_t)g * Kg + 2]; u2 = ubar_g[(size_t)g * Kg + 2] * ikv; }
  }
  float d0 = 0.f, d1 = 0.f, d2 = 0.f, s0 = 0.f, s1 = 0.f, s2 = 0.f;
  for (int k = lane; k < ne; k += LANES) {
    const float4 wi = sE[2 * k];
    const float cs = n.x * wi.x + n.y * wi.y + n.z * wi.z;
    if (cs <= 0.f) continue;                                             // max(0, w_i . n)
    float v = 1.f;
    {
      const int d = sD[k];
      v = u0 * (float)__ldg(vcount + (size_t)j0 * K + d);
      if (Kg > 1) v += u1 * (float)__ldg(vcount + (size_t)j1 * K + d);
      if (Kg > 2) v += u2 * (float)__ldg(vcount + (size_t)j2 * K + d);
      if (v == 0.f) continue;
    }
    const float4 LA = sE[2 * k + 1];
    // |w_i + w_o|^2 from the summed components: 2 + 2 w_o.w_i cancels to a few fp32 ulps of 2 when the light stands almost
    // opposite the viewer (|w_i + w_o| = 0.004: 1.5 % error in the half vector, 6e-3 in the radiance; found by the random sweep)
    const float hsx = wi.x + wox, hsy = wi.y + woy, hsz = wi.z + woz;
    const float hl2 = fmaxf(hsx * hsx + hsy * hsy + hsz * hsz, 1e-12f);
    const float hinv = rsq_approx(hl2);
    const float nh = (cs + nwo_raw) * hinv;
    const float oh = (0.5f * hl2) * hinv;                                // w_o . h = (1 + w_o.w_i) / |w_i + w_o|
    const float tx = fmaf(-cs, n.x, wi.x) + tox, ty = fmaf(-cs, n.y, wi.y) + toy, tz = fmaf(-cs, n.z, wi.z) + toz;
    const float den = fmaf(al2 * nh, nh, (tx * tx + ty * ty + tz * tz) * (hinv * hinv));   // (n.h)^2 (a^2 - 1) + 1, Eq.13
    const float F = fmaf(0.96f, ex2_approx((-5.55473f * oh - 6.98316f) * oh), 0.04f);     // Eq.14
    const float gi = fmaf(cs, omk, kk);
    const float sp = cS * F * rcp_approx(den * den * gi);
    const float w = v * cs;
    const float ws = w * sp;
    d0 = fmaf(LA.x, w, d0); d1 = fmaf(LA.y, w, d1); d2 = fmaf(LA.z, w, d2);
    s0 = fmaf(LA.x, ws, s0); s1 = fmaf(LA.y, ws, s1); s2 = fmaf(LA.z, ws, s2);
  }
  // the LANES-group always exits together, so its own lane mask is the legal one for the shuffles
  const unsigned gmask = (LANES == 32) ? 0xffffffffu : (((1u << LANES) - 1u) << (((threadIdx.x & 31) / LANES) * LANES));
#pragma unroll
  for (int o = LANES / 2; o > 0; o >>= 1) {
    d0 += __shfl_xor_sync(gmask, d0, o, LANES); d1 += __shfl_xor_sync(gmask, d1, o, LANES);
    d2 += __shfl_xor_sync(gmask, d2, o, LANES); s0 += __shfl_xor_sync(gmask, s0, o, LANES);
    s1 += __shfl_xor_sync(gmask, s1, o, LANES); s2 += __shfl_xor_sync(gmask, s2, o, LANES);
  }
  if (lane == 0) {
    const float ip = 1.f / PI_F;
    float L0 = ar.x * ip * d0 + spec * s0, L1 = ar.y * ip * d1 + spec * s1, L2 = ar.z * ip * d2 + spec * s2;   // Eq.12
    radiance[g] = make_float4(L0, L1, L2, 0.f);
    float c0 = exp2f(inv_gamma * log2f(fminf(fmaxf(L0, 0.f), 1.f)));
    float c1 = exp2f(inv_gamma * log2f(fminf(fmaxf(L1, 0.f), 1.f)));
    float c2 = exp2f(inv_gamma * log2f(fminf(fmaxf(L2, 0.f), 1.f)));
    color[g] = make_float4(c0, c1, c2, 0.f);
  }
}

#define SHADE_PAPER_LANES 4

static size_t shade_smem(int ne) { return (size_t)ne * 32 + (size_t)SH_WARPS * 6 * SH_GROUP * 4 + (size_t)ne * 2; }

cudaError_t rga_launch_shade(rga_avatar* av, const rga_env* env, float3 cam, int vis_mode, cudaStream_t s) {
  const int ne = env->rows * env->cols;
  const size_t smem = shade_smem(ne);
  const float ig = 1.0f / env->gamma;
  // persistent grid: as many CTAs as are resident at once (cached per mode and table size)
  static int occ_cache[3] = {0, 0, 0}; static size_t occ_smem[3] = {0, 0, 0};
  const int md = vis_mode == 0 ? 0 : (vis_mode == 1 ? 1 : 2);
  if (!occ_cache[md] || occ_smem[md] != smem) {
    int occ = 0; cudaError_t e;
    if (md == 0) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, shade_kernel<0>, SH_THREADS, smem);
    else if (md == 1) { e = cudaSuccess; occ = 1; }                     // paper mode runs shade_paper_kernel (plain grid)
    else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, shade_kernel<2>, SH_THREADS, smem);
    if (e != cudaSuccess) return e;
    occ_cache[md] = occ > 0 ? occ : 1; occ_smem[md] = smem;
  }
  const int ngroups = (av->n_gauss + SH_GROUP - 1) / SH_GROUP;
  int grid = av->num_sms * occ_cache[md];
  if (grid > ngroups) grid = ngroups;
  if (grid < 1) grid = 1;
#define SHADE_ARGS av->n_gauss, ne, av->vis_dirs, av->vis_words, av->k_g, av->k_v, av->g_posed, av->g_nposed, av->g_static, \
    av->env_table, env->texel_to_dir, av->visbits, av->vcount, av->knn_g, av->ubar_g, cam, ig, av->radiance, av->color, av->shade_counter
  if (vis_mode == 0) shade_kernel<0><<<grid, SH_THREADS, smem, s>>>(SHADE_ARGS);
  else if (vis_mode == 1) {
    const int gpb = 128 / SHADE_PAPER_LANES;
    shade_paper_kernel<SHADE_PAPER_LANES><<<(av->n_gauss + gpb - 1) / gpb, 128, (size_t)ne * 34, s>>>(
        av->n_gauss, ne, av->vis_dirs, av->vis_words, av->k_g, av->k_v, av->g_posed, av->g_nposed, av->g_static, av->env_table,
        env->texel_to_dir, av->visbits, av->vcount, av->knn_g, av->ubar_g, cam, ig, av->radiance, av->color);
  }
  else shade_kernel<2><<<grid, SH_THREADS, smem, s>>>(SHADE_ARGS);
  av->launches += 1;
  rga_prof_mark(av, "shade", s);
  return cudaGetLastError();
}

int rga_shade_init_attributes(int max_env) {
  const size_t smem = shade_smem(max_env);
  cudaError_t e = cudaSuccess;
  if (smem > 48 * 1024) {
    e = cudaFuncSetAttribute(shade_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(shade_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(shade_paper_kernel<SHADE_PAPER_LANES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  }
  return (int)e;
}
