// H4a + H5 fused for rga_render_frame (depth-test visibility, PAPER.md:124 / BASELINE.json north_star (b); Eq.2 with the
// Appendix-A BRDF).
//
// Inside one frame the camera, the environment map and its texel -> direction map are all known when visibility is tested,
// so a (Gaussian, direction) depth test whose result Eq.2 can never read is not made:
//   * a Gaussian facing away from the camera has opacity 0: front_compact_kernel lists the others once, and
//     the fused kernel walks that list -- every lane of every warp holds a Gaussian that is shaded;
//   * Eq.2 weighs v_g[k] by max(0, w_i^k . n): a direction none of whose texels can have w_i . n > 0 is skipped (per
//     direction d the bound eps_d = largest chord between w_d and the texels that read it, + 1e-3);
//   * the 32 visibility bits of a direction word stay in a register and drive the BRDF loop over that word's texels
//     directly; the word is also written to RGA_BUF_VISBITS (untested directions as 0) for parity checks.
// A team of 8 warps owns 32 consecutive listed Gaussians (one per lane) and splits the direction words; tables (light
// frames, environment rows, texels by direction) are staged in shared memory once per CTA.
//
// Arithmetic: the depth test is the EXACT chain of DESIGN.md "Arithmetic contract" -- written with explicit
// __fmaf_rn / __fadd_rn / __fmul_rn / __fdiv_rn / __fsqrt_rn so that this FAST file's contraction cannot touch it; its
// constants and the pre-scaled light frames come from light_frames_kernel in the EXACT file vis_kernels.cu.  The BRDF
// part is FAST arithmetic, compared with the fp64 oracle under the north_star tolerance.
#include "rga_internal.h"

#define PI_F 3.14159265358979323846f
#ifndef VS_TEAM_WARPS
#define VS_TEAM_WARPS 8        /* measured: teams of 4 / 16 warps give 177 / 151 us at config 1 against 118 us */
#endif
#define VS_CTAS_PER_SM(T) (32 / (VS_TEAM_WARPS * (T)) > 0 ? 32 / (VS_TEAM_WARPS * (T)) : 1)
#define VS_TEAM_THREADS (VS_TEAM_WARPS * 32)

__device__ __forceinline__ float vs_rsq(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float vs_rcp(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float vs_ex2(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float vs_sqrt(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ void team_sync(int team) { asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "r"(VS_TEAM_THREADS) : "memory"); }

// ---------------------------------------------------------------------------------------------------------------------
// camera-facing Gaussians, in library order; the others get zero radiance / colour / visibility words.
// Same test as shade_kernel and vis_depth_test_kernel (skip only when the sign is certain; the exact rule is H6's).
__global__ void __launch_bounds__(256) front_compact_kernel(int ng, int words, float3 cam, const float4* __restrict__ g_posed,
    const float4* __restrict__ g_nposed, int* __restrict__ front_list, unsigned* __restrict__ n_front, float4* __restrict__ radiance,
    float4* __restrict__ color, unsigned* __restrict__ visbits) {
  __shared__ int s_w[8];
  __shared__ unsigned s_base;
  const int g = blockIdx.x * blockDim.x + threadIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  bool keep = false;
  if (g < ng) {
    const float4 x = g_posed[g], n = g_nposed[g];
    const float wx = cam.x - x.x, wy = cam.y - x.y, wz = cam.z - x.z;
    keep = !(n.x * wx + n.y * wy + n.z * wz < -1e-4f * sqrtf(wx * wx + wy * wy + wz * wz));
    if (!keep) { radiance[g] = make_float4(0.f, 0.f, 0.f, 0.f); color[g] = make_float4(0.f, 0.f, 0.f, 0.f); }
  }
  const unsigned bal = __ballot_sync(0xffffffffu, keep);
  if (lane == 0) s_w[warp] = __popc(bal);
  __syncthreads();
  int before = 0, total = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) { const int c = s_w[w]; if (w < warp) before += c; total += c; }
  if (threadIdx.x == 0) s_base = total ? atomicAdd(n_front, (unsigned)total) : 0u;
  __syncthreads();
  if (keep) front_list[s_base + before + __popc(bal & ((1u << lane) - 1u))] = g;
}

// ---------------------------------------------------------------------------------------------------------------------
// texels grouped by the direction they read (texel_to_dir; NULL = identity): dir_start[K+1], tex_list[ne] (ascending
// texel index inside a direction) and eps[d] = largest chord |w_k - w_d| over its texels + 1e-3 (a direction without
// texels gets eps = -4: never needed).  One CTA; ne <= 4096, K <= 2048.
__global__ void __launch_bounds__(1024) texel_csr_kernel(int ne, int K, const int* __restrict__ t2d, const float* __restrict__ env_table,
    const float* __restrict__ dirs, unsigned short* __restrict__ dir_start, unsigned short* __restrict__ tex_list, unsigned short* __restrict__ tex_dir, float* __restrict__ dir_eps,
    float* __restrict__ env_pairs) {
  __shared__ unsigned s_cnt[2048 + 1];
  __shared__ unsigned s_eps[2048];
  __shared__ unsigned short s_d[4096];
  for (int d = threadIdx.x; d <= K; d += blockDim.x) { s_cnt[d] = 0u; if (d < K) s_eps[d] = 0u; }
  __syncthreads();
  for (int k = threadIdx.x; k < ne; k += blockDim.x) {
    int d = t2d ? t2d[k] : k;
    d = d < 0 ? 0 : (d >= K ? K - 1 : d);
    s_d[k] = (unsigned short)d;
    atomicAdd(&s_cnt[d + 1], 1u);
    const float4 w = reinterpret_cast<const float4*>(env_table)[2 * (size_t)k];
    const float ex = w.x - dirs[3 * d], ey = w.y - dirs[3 * d + 1], ez = w.z - dirs[3 * d + 2];
    atomicMax(&s_eps[d], __float_as_uint(sqrtf(ex * ex + ey * ey + ez * ez)));     // non-negative floats order like their bits
  }
  __syncthreads();
  if (threadIdx.x == 0) for (int d = 0; d < K; ++d) s_cnt[d + 1] += s_cnt[d];       // K <= 2048: a few microseconds, off the critical path
  __syncthreads();
  for (int d = threadIdx.x; d <= K; d += blockDim.x) {
    dir_start[d] = (unsigned short)s_cnt[d];
    if (d < K) dir_eps[d] = (s_cnt[d + 1] > s_cnt[d]) ? __uint_as_float(s_eps[d]) + 1e-3f : -4.0f;
  }
  // fill in any order (shared-memory cursors), then every direction puts its few texels into ascending order
  __shared__ unsigned short s_list[4096];
  __syncthreads();
  for (int d = threadIdx.x; d < K; d += blockDim.x) s_eps[d] = s_cnt[d];            // s_eps reused as the fill cursors
  __syncthreads();
  for (int k = threadIdx.x; k < ne; k += blockDim.x) s_list[atomicAdd(&s_eps[s_d[k]], 1u)] = (unsigned short)k;
  __syncthreads();
  for (int d = threadIdx.x; d < K; d += blockDim.x) {
    const int b = (int)s_cnt[d], e = (int)s_cnt[d + 1];
    for (int i = b + 1; i < e; ++i) {                                               // insertion sort of a handful of entries
      const unsigned short v = s_list[i]; int j = i - 1;
      while (j >= b && s_list[j] > v) { s_list[j + 1] = s_list[j]; --j; }
      s_list[j + 1] = v;
    }
    for (int i = b; i < e; ++i) { tex_list[i] = s_list[i]; tex_dir[i] = (unsigned short)d; }
  }
  // the environment rows in LIST order, two list positions side by side (12 floats per pair: wi.x0 wi.x1 wi.y0 wi.y1 wi.z0 wi.z1
  // LA.r0 LA.r1 LA.g0 LA.g1 LA.b0 LA.b1): the image of the fused kernel's shared-memory table, staged there by one bulk copy
  __syncthreads();
  for (int t = threadIdx.x; t < ((ne + 1) & ~1); t += blockDim.x) {
    float4 wi = make_float4(0.f, 0.f, 1.f, 0.f), LA = make_float4(0.f, 0.f, 0.f, 0.f);       // padding of an odd list: adds nothing
    if (t < ne) {
      const int k = (int)s_list[t];
      wi = reinterpret_cast<const float4*>(env_table)[2 * k]; LA = reinterpret_cast<const float4*>(env_table)[2 * k + 1];
    }
    float* e = env_pairs + 12 * (size_t)(t >> 1) + (t & 1);
    e[0] = wi.x; e[2] = wi.y; e[4] = wi.z; e[6] = LA.x; e[8] = LA.y; e[10] = LA.z;
  }
}

// ---------------------------------------------------------------------------------------------------------------------
struct VsArgs {
  int K, R, ne, words;
  const float4* frames;              // [2 + 3K]: (cx,cy,cz,hR) (bt,bw,slope_max,R) then per direction (us,w.x) (vs,w.y) (wn,w.z)
  const float* env_table;            // [ne][8]
  const float* env_pairs;            // [ceil(ne / 2)][12]: the rows in list order, pairs side by side (texel_csr_kernel)
  const unsigned short* dir_start; const unsigned short* tex_list; const unsigned short* tex_dir; const float* dir_eps;
  const unsigned* zmap;
  const int* front_list; const unsigned* n_front;
  const float4* g_posed; const float4* g_nposed; const float4* g_static;
  float3 cam; float inv_gamma;
  float4* radiance; float4* color; unsigned* visbits; unsigned* counter;
};

static size_t vs_smem_bytes(int K, int ne, int teams) {
  return (size_t)K * 48 + (size_t)((ne + 1) / 2) * 48 + (size_t)K * 4 + (size_t)(K + 2) * 2 + (size_t)(ne + 4) * 4 + 16 +
         (size_t)2 * teams * VS_TEAM_WARPS * 6 * 32 * 4;
}

// One BRDF term of Eq.2 (Eq.12-15) for the lanes whose weight c = max(0, w_i . n) v is positive; accumulates diffuse (d) and
// specular (s) sums per channel.
struct VsBrdf { float wox, woy, woz, nwo_raw, al2, omk, kk, cS, tox, toy, toz; };

// Packed fp32 (sm_100 FFMA2 / FMUL2 / FADD2: one issue slot, two IEEE operations): the BRDF loop takes the texels of a
// direction unit TWO at a time, the pair's values side by side in 64-bit registers.  The kernel is bound by issue slots, not
// by the FMA pipe (profiles/r02_vis_shade.md), so halving the count of its fp32 instructions is what pays.
__device__ __forceinline__ float2 vs_bc(float a) { return make_float2(a, a); }
#define VS_FMA2 __ffma2_rn
#define VS_MUL2 __fmul2_rn
#define VS_ADD2 __fadd2_rn

// The rare middle case of a depth test: z lies between the two ends of the bias beta(tau).  An approximate tau decides unless z
// is within `margin` of the threshold; only then the exact IEEE sqrt and divide of the contract are evaluated -- the bit is the
// same.  Out of line: inlined into every one of the sixteen unrolled tests it made the loop larger than the instruction cache.
__device__ __noinline__ bool vs_slope_test(float z, float zm, float c, float bt, float bw, float slope_max, float margin) {
  float tau = slope_max;
  if (c > 0.0f) {
    const float s2 = fmaxf(__fmaf_rn(-c, c, 1.0f), 0.0f);
    tau = fminf(fmaxf(__fmul_rn(vs_sqrt(s2), vs_rcp(c)), 1.0f), slope_max);
  }
  const float dlt = __fadd_rn(z, -__fadd_rn(zm, __fmaf_rn(bt, tau, bw)));
  if (fabsf(dlt) > margin) return dlt < 0.0f;
  float te = slope_max;
  if (c > 0.0f) {
    const float s2 = fmaxf(__fsub_rn(1.0f, __fmul_rn(c, c)), 0.0f);
    te = fminf(fmaxf(__fdiv_rn(__fsqrt_rn(s2), c), 1.0f), slope_max);
  }
  return z <= __fadd_rn(zm, __fadd_rn(__fmul_rn(bt, te), bw));
}

template <int TEAMS, bool IDENT>
__global__ void __launch_bounds__(VS_TEAM_THREADS * TEAMS, VS_CTAS_PER_SM(TEAMS)) vis_shade_kernel(const VsArgs a) {
  extern __shared__ __align__(16) unsigned char vs_raw[];
  const int K = a.K, ne = a.ne, R = a.R, words = a.words;
  // per direction three float4: A = (us.xyz, vs.x)  B = (vs.yz, wn.xy)  C = (wn.z, w.xyz)
  float4* sF = reinterpret_cast<float4*>(vs_raw);                                  // [3K]
  // environment rows in LIST order (texels sorted by the direction they read), two texels side by side: per pair three float4
  // (wi.x0 wi.x1 wi.y0 wi.y1) (wi.z0 wi.z1 LA.r0 LA.r1) (LA.g0 LA.g1 LA.b0 LA.b1)
  float4* sE = sF + 3 * K;                                                        // [3 ceil(ne / 2)]
  float* sPart = reinterpret_cast<float*>(sE + 3 * ((ne + 1) >> 1));              // [2][TEAMS][8][6][32] (two groups in flight)
  float* sEps = sPart + 2 * TEAMS * VS_TEAM_WARPS * 6 * 32;                       // [K]
  unsigned short* sStart = reinterpret_cast<unsigned short*>(sEps + K);           // [K + 1]
  unsigned short* sTexD = sStart + ((K + 2) & ~1);                                // [ne + 2] direction of the texel at each list position
  __shared__ unsigned s_ticket[2][TEAMS];
  // The two large tables arrive by bulk copies (cp.async.bulk, the TMA's linear form) that one thread issues and that signal an
  // mbarrier with their byte count; both lie in global memory exactly as they lie here (light frames: written by the
  // rasteriser; environment pairs: by texel_csr_kernel).  The small tables are staged by the threads meanwhile.
  __shared__ __align__(8) unsigned long long s_bar;
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&s_bar);
  const uint32_t bytesF = (uint32_t)K * 48u, bytesE = (uint32_t)((ne + 1) >> 1) * 48u;
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(1u) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytesF + bytesE) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"((uint32_t)__cvta_generic_to_shared(sF)), "l"(a.frames + 2), "r"(bytesF), "r"(bar) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"((uint32_t)__cvta_generic_to_shared(sE)), "l"(a.env_pairs), "r"(bytesE), "r"(bar) : "memory");
  }
  for (int t = threadIdx.x; t < K; t += blockDim.x) sEps[t] = a.dir_eps[t];
  if (!IDENT) {
    for (int t = threadIdx.x; t <= K; t += blockDim.x) sStart[t] = a.dir_start[t];
    for (int t = threadIdx.x; t < ne + 2; t += blockDim.x) sTexD[t] = t < ne ? a.tex_dir[t] : (unsigned short)0;
  }
  const float4 h0 = a.frames[0], h1 = a.frames[1];
  if ((threadIdx.x & (VS_TEAM_THREADS - 1)) == 0) s_ticket[0][threadIdx.x / VS_TEAM_THREADS] = atomicAdd(a.counter, 1u);   // the team's first group
  __syncthreads();                                                                // s_bar initialised, small tables staged
  {
    uint32_t done = 0;
    while (!done)
      asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                   : "=r"(done) : "r"(bar), "r"(0u) : "memory");
  }
  const float cx = h0.x, cy = h0.y, cz = h0.z, hR = h0.w, bt = h1.x, bw = h1.y, slope_max = h1.z;
  const int lane = threadIdx.x & 31, team = threadIdx.x / VS_TEAM_THREADS, tw = (threadIdx.x >> 5) & (VS_TEAM_WARPS - 1);
  const bool team_lead = (threadIdx.x & (VS_TEAM_THREADS - 1)) == 0;
  const unsigned nfront = *a.n_front, ngroups = (nfront + 31u) >> 5;
  // beta(tau) is monotone in tau on [1, slope_max]: most tests are decided by its two ends without evaluating tau
  const float beta_lo = __fadd_rn(__fmul_rn(bt, 1.0f), bw), beta_hi = __fadd_rn(__fmul_rn(bt, slope_max), bw);
  const bool bounds_ok = bt >= 0.f && slope_max >= 1.0f;
  const float INF = __int_as_float(0x7f800000);
  const float blo = bounds_ok ? beta_lo : -INF, bhi = bounds_ok ? beta_hi : INF;
  const float margin = 1e-6f + 1e-5f * fabsf(bt) * fmaxf(slope_max, 1.0f);
  const float Rm1 = (float)(R - 1), Rf = (float)R;
  const size_t RR = (size_t)R * R;
  const int nunits = 2 * words;                                                   // a unit = 16 directions (half a visibility word)
  // ONE barrier per group: the team's lead draws the NEXT ticket while the group is computed (the atomic's round trip hides
  // behind the work) and publishes it, with the warps' partial sums, at the barrier that ends the group; tickets and partial
  // sums are double-buffered, so the first warp folds group i while the others are already in group i + 1.
  const unsigned beyond_last = ngroups + gridDim.x * TEAMS - 1u;
  unsigned short* vis16 = reinterpret_cast<unsigned short*>(a.visbits);
  for (int it = 0;; ++it) {
    const unsigned group = s_ticket[it & 1][team];
    if (group >= ngroups) {
      // every team draws exactly one ticket beyond the groups: the last of them re-arms the counter for the next launch
      if (team_lead && group == beyond_last) *a.counter = 0u;
      break;
    }
    unsigned next_ticket = 0u;
    if (team_lead) next_ticket = atomicAdd(a.counter, 1u);
    float* myPart = sPart + (((size_t)(it & 1) * TEAMS + team) * VS_TEAM_WARPS + tw) * 6 * 32;
    const unsigned li = group * 32u + (unsigned)lane;
    const bool valid = li < nfront;
    const int g = a.front_list[valid ? li : group * 32u];                         // idle lanes shadow the group's first Gaussian
    const float4 x = a.g_posed[g], n = a.g_nposed[g];
    VsBrdf q;
    {
      float wox = a.cam.x - x.x, woy = a.cam.y - x.y, woz = a.cam.z - x.z;
      const float winv = rsqrtf(wox * wox + woy * woy + woz * woz);
      q.wox = wox * winv; q.woy = woy * winv; q.woz = woz * winv;
      const float rough = a.g_static[4 * (size_t)g + 2].w;
      q.nwo_raw = n.x * q.wox + n.y * q.woy + n.z * q.woz;
      const float al = rough * rough; q.al2 = al * al;                              // Eq.13: alpha = gamma^2
      q.kk = (rough + 1.f) * (rough + 1.f) * 0.125f; q.omk = 1.f - q.kk;            // Eq.15
      // 1 - (n.h)^2 = |t|^2 / |w_i + w_o|^2 with t the tangential part of w_i + w_o (the direct form cancels for small alpha)
      q.tox = fmaf(-q.nwo_raw, n.x, q.wox); q.toy = fmaf(-q.nwo_raw, n.y, q.woy); q.toz = fmaf(-q.nwo_raw, n.z, q.woz);
      q.cS = q.al2 / (4.f * PI_F * (fmaxf(q.nwo_raw, 0.f) * q.omk + q.kk));         // D F G /(4 ni no) = cS F / (den^2 gi)
    }
    const float dx = __fsub_rn(x.x, cx), dy = __fsub_rn(x.y, cy), dz = __fsub_rn(x.z, cz);
    // the pair's constants: the same value in both halves
    const float2 nx2 = vs_bc(n.x), ny2 = vs_bc(n.y), nz2 = vs_bc(n.z), mnx2 = vs_bc(-n.x), mny2 = vs_bc(-n.y), mnz2 = vs_bc(-n.z);
    const float2 wox2 = vs_bc(q.wox), woy2 = vs_bc(q.woy), woz2 = vs_bc(q.woz), nwo2 = vs_bc(q.nwo_raw), al22 = vs_bc(q.al2),
                 omk2 = vs_bc(q.omk), kk2 = vs_bc(q.kk), cS2 = vs_bc(q.cS);
    float2 d0 = vs_bc(0.f), d1 = vs_bc(0.f), d2 = vs_bc(0.f), s0 = vs_bc(0.f), s1 = vs_bc(0.f), s2 = vs_bc(0.f);   // (even, odd) list positions
    // units are dealt to the team's warps round robin (static, so that every sum has one fixed order): warp w takes the
    // half-words w, w + 8, ... -- the rows of a lat-long direction grid are spread evenly over the warps
    for (int unit = tw; unit < nunits; unit += VS_TEAM_WARPS) {
      const int k0 = unit << 4, kend = min(16, K - k0);
      if (kend <= 0) continue;
      // ---- which of the unit's directions can Eq.2 read for my Gaussian: n . w_d > -eps_d (a conservative test; any rounding)
      unsigned needm = 0u;
#pragma unroll
      for (int b = 0; b < 16; ++b) {
        if (b < kend) {
          const float4 C = sF[3 * (k0 + b) + 2];
          const float c = fmaf(n.z, C.w, fmaf(n.y, C.z, fmaf(n.x, C.y, sEps[k0 + b])));
          needm |= (c > 0.f ? 1u : 0u) << b;
        }
      }
      if (!valid) needm = 0u;
      const unsigned wneed = __reduce_or_sync(0xffffffffu, needm);
      // ---- depth tests, four directions (four gathers) at a time; a chunk no lane needs is skipped
      unsigned bits = 0u;
      const unsigned* zk = a.zmap + (size_t)k0 * RR;
#pragma unroll
      for (int b0 = 0; b0 < 16; b0 += 4) {
        if (((wneed >> b0) & 0xfu) == 0u) continue;
        float z[4], zm[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int b = min(b0 + u, kend - 1);
          const float4 A = sF[3 * (k0 + b)], B = sF[3 * (k0 + b) + 1], C = sF[3 * (k0 + b) + 2];
          const float px = __fmaf_rn(A.z, dz, __fmaf_rn(A.y, dy, __fmaf_rn(A.x, dx, hR)));
          const float py = __fmaf_rn(B.y, dz, __fmaf_rn(B.x, dy, __fmaf_rn(A.w, dx, hR)));
          z[u] = __fmaf_rn(C.x, dz, __fmaf_rn(B.w, dy, __fmaf_rn(B.z, dx, 0.5f)));
          // floor-then-clamp == clamp-then-floor for finite px; floor via +2^23 rounded DOWN (exact for 0 <= x < 2^23)
          const float fxm = __fadd_rd(fminf(fmaxf(px, 0.0f), Rm1), 8388608.0f);
          const float fym = __fadd_rd(fminf(fmaxf(py, 0.0f), Rm1), 8388608.0f);
          const int idx = __float_as_int(__fmaf_rn(__fadd_rn(fym, -8388608.0f), Rf, fxm)) & 0x7fffff;
          zm[u] = __uint_as_float(__ldg(zk + (size_t)b * RR + idx));              // empty texel = 0xffffffff = NaN
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          // visible iff z <= zm + beta(tau); NaN compares false, so "not (z > ...)" also covers the empty texel
          bool vis = !(z[u] > __fadd_rn(zm[u], blo));
          if (!vis && !(z[u] > __fadd_rn(zm[u], bhi))) {
            const float4 C = sF[3 * (k0 + min(b0 + u, kend - 1)) + 2];
            const float c = __fadd_rn(__fadd_rn(__fmul_rn(n.x, C.y), __fmul_rn(n.y, C.z)), __fmul_rn(n.z, C.w));   // dot3(n_gd, w)
            vis = vs_slope_test(z[u], zm[u], c, bt, bw, slope_max, margin);
          }
          bits |= (vis ? 1u : 0u) << (b0 + u);
        }
      }
      bits &= needm;
      if (valid) vis16[((size_t)g * words) * 2 + unit] = (unsigned short)bits;     // little-endian halves of the u32 visibility word
      // ---- Eq.2 over the texels that read the unit's directions; a texel no lane needs costs the test only
      const unsigned anyb = __reduce_or_sync(0xffffffffu, bits);
      if (anyb == 0u) continue;
      const int t0 = IDENT ? k0 : sStart[k0], t1 = IDENT ? k0 + kend : sStart[k0 + kend];
#pragma unroll 2
      for (int t = t0 & ~1; t < t1; t += 2) {                                     // list positions t (even) and t + 1
        const float4* ep = sE + 3 * (t >> 1);
        const float4 Wa = ep[0], Wb = ep[1];
        const float2 wix = make_float2(Wa.x, Wa.y), wiy = make_float2(Wa.z, Wa.w), wiz = make_float2(Wb.x, Wb.y), LAx = make_float2(Wb.z, Wb.w);
        const float2 c = VS_FMA2(nz2, wiz, VS_FMA2(ny2, wiy, VS_MUL2(nx2, wix)));      // w_i . n
        const int j0 = ((IDENT ? t : (int)sTexD[t]) - k0) & 31, j1 = ((IDENT ? t + 1 : (int)sTexD[t + 1]) - k0) & 31;
        const bool live0 = t >= t0 && ((bits >> j0) & 1u) && c.x > 0.f;             // max(0, w_i . n) and the visibility bit
        const bool live1 = t + 1 < t1 && ((bits >> j1) & 1u) && c.y > 0.f;
        if (!__any_sync(0xffffffffu, live0 || live1)) continue;
        const float4 Wc = ep[2];
        const float2 LAy = make_float2(Wc.x, Wc.y), LAz = make_float2(Wc.z, Wc.w);
        const float2 sx = VS_ADD2(wix, wox2), sy = VS_ADD2(wiy, woy2), sz = VS_ADD2(wiz, woz2);     // w_i + w_o
        float2 hl2 = VS_FMA2(sz, sz, VS_FMA2(sy, sy, VS_MUL2(sx, sx)));                  // |w_i + w_o|^2
        hl2.x = fmaxf(hl2.x, 1e-12f); hl2.y = fmaxf(hl2.y, 1e-12f);
        const float2 hinv = make_float2(vs_rsq(hl2.x), vs_rsq(hl2.y));
        const float2 ns = VS_ADD2(c, nwo2);                                              // n . (w_i + w_o)
        const float2 nh = VS_MUL2(ns, hinv);
        const float2 oh = VS_MUL2(VS_MUL2(vs_bc(0.5f), hl2), hinv);                      // w_o . h
        // 1 - (n.h)^2 = |t|^2 / |w_i + w_o|^2 with t the tangential part of w_i + w_o (the direct form cancels for small alpha)
        const float2 tx = VS_FMA2(ns, mnx2, sx), ty = VS_FMA2(ns, mny2, sy), tz = VS_FMA2(ns, mnz2, sz);
        const float2 tt = VS_FMA2(tz, tz, VS_FMA2(ty, ty, VS_MUL2(tx, tx)));
        const float2 den = VS_FMA2(VS_MUL2(al22, nh), nh, VS_MUL2(tt, VS_MUL2(hinv, hinv)));   // (n.h)^2 (a^2 - 1) + 1, Eq.13
        const float2 u = VS_MUL2(VS_FMA2(vs_bc(-5.55473f), oh, vs_bc(-6.98316f)), oh);
        const float2 F = VS_FMA2(vs_bc(0.96f), make_float2(vs_ex2(u.x), vs_ex2(u.y)), vs_bc(0.04f));        // Eq.14
        const float2 gi = VS_FMA2(c, omk2, kk2);
        const float2 qd = VS_MUL2(VS_MUL2(den, den), gi);
        const float2 sp = VS_MUL2(VS_MUL2(cS2, F), make_float2(vs_rcp(qd.x), vs_rcp(qd.y)));
        const float2 w = make_float2(live0 ? c.x : 0.f, live1 ? c.y : 0.f);               // branch-free: dead entries add zero
        const float2 ws = VS_MUL2(w, sp);
        d0 = VS_FMA2(LAx, w, d0); d1 = VS_FMA2(LAy, w, d1); d2 = VS_FMA2(LAz, w, d2);
        s0 = VS_FMA2(LAx, ws, s0); s1 = VS_FMA2(LAy, ws, s1); s2 = VS_FMA2(LAz, ws, s2);
      }
    }
    // ---- the warps' partial sums are folded in warp order by one warp of the team (the duty rotates), which finishes Eq.12 and the gamma curve
    myPart[lane] = d0.x + d0.y; myPart[32 + lane] = d1.x + d1.y; myPart[64 + lane] = d2.x + d2.y;
    myPart[96 + lane] = s0.x + s0.y; myPart[128 + lane] = s1.x + s1.y; myPart[160 + lane] = s2.x + s2.y;
    if (team_lead) s_ticket[(it + 1) & 1][team] = next_ticket;
    team_sync(team);
    if (tw != (it & (VS_TEAM_WARPS - 1))) continue;                               // the fold duty goes round the team's warps
    float acc[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      float sum = 0.f;
#pragma unroll
      for (int w = 0; w < VS_TEAM_WARPS; ++w) sum += sPart[((((size_t)(it & 1) * TEAMS + team) * VS_TEAM_WARPS + w) * 6 + c) * 32 + lane];
      acc[c] = sum;
    }
    if (valid) {
      const float4 ar = a.g_static[4 * (size_t)g + 2];                             // albedo rgb, roughness
      const float spec = a.g_static[4 * (size_t)g + 3].x;
      const float ip = 1.f / PI_F;
      const float L0 = ar.x * ip * acc[0] + spec * acc[3], L1 = ar.y * ip * acc[1] + spec * acc[4], L2 = ar.z * ip * acc[2] + spec * acc[5];   // Eq.12
      a.radiance[g] = make_float4(L0, L1, L2, 0.f);
      a.color[g] = make_float4(exp2f(a.inv_gamma * log2f(fminf(fmaxf(L0, 0.f), 1.f))), exp2f(a.inv_gamma * log2f(fminf(fmaxf(L1, 0.f), 1.f))),
                               exp2f(a.inv_gamma * log2f(fminf(fmaxf(L2, 0.f), 1.f))), 0.f);
    }
  }
}

// can the fused path take this frame?  (tables must fit shared memory; index types are 16 bit)
int rga_vis_shade_teams(int K, int ne) {
  if (K < 1 || K > 2048 || ne < 1 || ne > 4096) return 0;
  const size_t lim = 227 * 1024 - 1024;
  // as many CTAs per SM as fill its 32 warp slots at 64 registers; more teams per CTA when the tables are too large for that
  for (int t = 1; t * VS_TEAM_WARPS <= 32; t *= 2)
    if (vs_smem_bytes(K, ne, t) <= lim / (size_t)VS_CTAS_PER_SM(t) - 1024) return t;
  return 0;
}

int rga_vis_shade_init_attributes() {
  const int mx = 227 * 1024 - 1024;
  cudaError_t e = cudaFuncSetAttribute(vis_shade_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
#if VS_TEAM_WARPS * 4 <= 32
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
#endif
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  return (int)e;
}

// side stream: list of camera-facing Gaussians (needs the Gaussian skinning)
cudaError_t rga_launch_front_compact(rga_avatar* av, int words, float3 cam, cudaStream_t s) {
  cudaError_t e = cudaMemsetAsync(av->n_front, 0, sizeof(unsigned), s);
  if (e != cudaSuccess) return e;
  // visibility words of the Gaussians that are not listed stay 0 (one bulk clear instead of strided per-thread stores)
  if ((e = cudaMemsetAsync(av->visbits, 0, (size_t)av->n_gauss * words * sizeof(unsigned), s)) != cudaSuccess) return e;
  front_compact_kernel<<<(av->n_gauss + 255) / 256, 256, 0, s>>>(av->n_gauss, words, cam, av->g_posed, av->g_nposed, av->front_list, av->n_front,
                                                                av->radiance, av->color, av->visbits);
  rga_prof_mark(av, "front_compact", s);
  av->launches += 1;
  return cudaGetLastError();
}

// side stream: texels by direction (needs the environment table)
cudaError_t rga_launch_texel_csr(rga_avatar* av, const rga_env* env, const rga_vis_params* vis, cudaStream_t s) {
  texel_csr_kernel<<<1, 1024, 0, s>>>(env->rows * env->cols, vis->n_dirs, env->texel_to_dir, av->env_table, vis->dirs, av->dir_start, av->tex_list,
                                      av->tex_dir, av->dir_eps, av->env_pairs);
  rga_prof_mark(av, "texel_csr", s);
  av->launches += 1;
  return cudaGetLastError();
}

cudaError_t rga_launch_vis_shade(rga_avatar* av, const rga_vis_params* vis, const rga_env* env, float3 cam, cudaStream_t s) {
  const int K = vis->n_dirs, ne = env->rows * env->cols, teams = rga_vis_shade_teams(K, ne);
  if (teams == 0) return cudaErrorInvalidConfiguration;
  VsArgs a;
  a.K = K; a.R = vis->res; a.ne = ne; a.words = (K + 31) / 32;
  a.frames = reinterpret_cast<const float4*>(av->frames); a.env_table = av->env_table; a.env_pairs = av->env_pairs;
  a.dir_start = av->dir_start; a.tex_list = av->tex_list; a.tex_dir = av->tex_dir; a.dir_eps = av->dir_eps; a.zmap = av->zmap;
  a.front_list = av->front_list; a.n_front = av->n_front;
  a.g_posed = av->g_posed; a.g_nposed = av->g_nposed; a.g_static = av->g_static;
  a.cam = cam; a.inv_gamma = 1.0f / env->gamma;
  a.radiance = av->radiance; a.color = av->color; a.visbits = av->visbits; a.counter = av->vs_counter;
  const size_t smem = vs_smem_bytes(K, ne, teams);
  const int per_sm = VS_CTAS_PER_SM(teams);
  int grid = av->num_sms * per_sm;
  const int max_groups = (av->n_gauss + 31) / 32;
  if (grid * teams > max_groups) grid = (max_groups + teams - 1) / teams;
  if (grid < 1) grid = 1;
  const bool ident = env->texel_to_dir == nullptr && ne == K;              // texel k reads direction k: no texel lists
  if (teams == 1) { if (ident) vis_shade_kernel<1, true><<<grid, VS_TEAM_THREADS, smem, s>>>(a); else vis_shade_kernel<1, false><<<grid, VS_TEAM_THREADS, smem, s>>>(a); }
  else if (teams == 2) { if (ident) vis_shade_kernel<2, true><<<grid, 2 * VS_TEAM_THREADS, smem, s>>>(a); else vis_shade_kernel<2, false><<<grid, 2 * VS_TEAM_THREADS, smem, s>>>(a); }
#if VS_TEAM_WARPS * 4 <= 32
  else { if (ident) vis_shade_kernel<4, true><<<grid, 4 * VS_TEAM_THREADS, smem, s>>>(a); else vis_shade_kernel<4, false><<<grid, 4 * VS_TEAM_THREADS, smem, s>>>(a); }
#else
  else return cudaErrorInvalidConfiguration;
#endif
  rga_prof_mark(av, "vis_shade", s);
  av->launches += 1;
  return cudaGetLastError();
}
