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
#define VS_TEAM_WARPS 8
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
    const float* __restrict__ dirs, unsigned short* __restrict__ dir_start, unsigned short* __restrict__ tex_list, unsigned short* __restrict__ tex_dir, float* __restrict__ dir_eps) {
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
}

// ---------------------------------------------------------------------------------------------------------------------
struct VsArgs {
  int K, R, ne, words;
  const float4* frames;              // [2 + 3K]: (cx,cy,cz,hR) (bt,bw,slope_max,R) then per direction (us,w.x) (vs,w.y) (wn,w.z)
  const float* env_table;            // [ne][8]
  const unsigned short* dir_start; const unsigned short* tex_list; const unsigned short* tex_dir; const float* dir_eps;
  const unsigned* zmap;
  const int* front_list; const unsigned* n_front;
  const float4* g_posed; const float4* g_nposed; const float4* g_static;
  float3 cam; float inv_gamma;
  float4* radiance; float4* color; unsigned* visbits; unsigned* counter;
};

static size_t vs_smem_bytes(int K, int ne, int teams) {
  return (size_t)K * 48 + (size_t)ne * 32 + (size_t)K * 4 + (size_t)(K + 2) * 2 + (size_t)(ne + 2) * 4 + 16 +
         (size_t)teams * VS_TEAM_WARPS * 6 * 32 * 4;
}

// One BRDF term of Eq.2 (Eq.12-15) for the lanes whose weight c = max(0, w_i . n) v is positive; accumulates diffuse (d) and
// specular (s) sums per channel.
struct VsBrdf { float wox, woy, woz, nwo_raw, al2, omk, kk, cS, tox, toy, toz; };

template <int TEAMS, bool IDENT>
__global__ void __launch_bounds__(VS_TEAM_THREADS * TEAMS, (TEAMS == 1 ? 4 : (TEAMS == 2 ? 2 : 1))) vis_shade_kernel(const VsArgs a) {
  extern __shared__ __align__(16) unsigned char vs_raw[];
  const int K = a.K, ne = a.ne, R = a.R, words = a.words;
  // per direction three float4: A = (us.xyz, vs.x)  B = (vs.yz, wn.xy)  C = (wn.z, w.xyz)
  float4* sF = reinterpret_cast<float4*>(vs_raw);                                  // [3K]
  float4* sE = sF + 3 * K;                                                        // [2 ne]
  float* sPart = reinterpret_cast<float*>(sE + 2 * ne);                           // [TEAMS][8][6][32]
  float* sEps = sPart + TEAMS * VS_TEAM_WARPS * 6 * 32;                           // [K]
  unsigned short* sStart = reinterpret_cast<unsigned short*>(sEps + K);           // [K + 1]
  unsigned short* sTex = sStart + ((K + 2) & ~1);                                 // [ne] texels sorted by direction
  unsigned short* sTexD = sTex + ((ne + 1) & ~1);                                 // [ne] their directions
  __shared__ unsigned s_ticket[TEAMS];
  for (int t = threadIdx.x; t < K; t += blockDim.x) {
    const float4 u = a.frames[2 + 3 * t], v = a.frames[3 + 3 * t], w = a.frames[4 + 3 * t];
    sF[3 * t] = make_float4(u.x, u.y, u.z, v.x); sF[3 * t + 1] = make_float4(v.y, v.z, w.x, w.y); sF[3 * t + 2] = make_float4(w.z, u.w, v.w, w.w);
    sEps[t] = a.dir_eps[t];
  }
  for (int t = threadIdx.x; t < 2 * ne; t += blockDim.x) sE[t] = reinterpret_cast<const float4*>(a.env_table)[t];
  if (!IDENT) {
    for (int t = threadIdx.x; t <= K; t += blockDim.x) sStart[t] = a.dir_start[t];
    for (int t = threadIdx.x; t < ne; t += blockDim.x) { sTex[t] = a.tex_list[t]; sTexD[t] = a.tex_dir[t]; }
  }
  const float4 h0 = a.frames[0], h1 = a.frames[1];
  __syncthreads();
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
  float* myPart = sPart + ((size_t)team * VS_TEAM_WARPS + tw) * 6 * 32;
  unsigned short* vis16 = reinterpret_cast<unsigned short*>(a.visbits);
  for (;;) {
    team_sync(team);                                                              // s_ticket and sPart are reused
    if (team_lead) s_ticket[team] = atomicAdd(a.counter, 1u);
    team_sync(team);
    const unsigned group = s_ticket[team];
    if (group >= ngroups) {
      // every team draws exactly one ticket beyond the groups: the last of them re-arms the counter for the next launch
      if (team_lead && group == ngroups + gridDim.x * TEAMS - 1u) *a.counter = 0u;
      break;
    }
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
    float d0 = 0.f, d1 = 0.f, d2 = 0.f, s0 = 0.f, s1 = 0.f, s2 = 0.f;
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
            // in between: an approximate tau decides unless z is within `margin` of the threshold; only then the exact
            // IEEE sqrt and divide of the contract are evaluated -- the bit is the same
            const float4 C = sF[3 * (k0 + min(b0 + u, kend - 1)) + 2];
            const float c = __fadd_rn(__fadd_rn(__fmul_rn(n.x, C.y), __fmul_rn(n.y, C.z)), __fmul_rn(n.z, C.w));   // dot3(n_gd, w)
            float tau = slope_max;
            if (c > 0.0f) {
              const float s2 = fmaxf(__fmaf_rn(-c, c, 1.0f), 0.0f);
              tau = fminf(fmaxf(__fmul_rn(vs_sqrt(s2), vs_rcp(c)), 1.0f), slope_max);
            }
            const float dlt = __fadd_rn(z[u], -__fadd_rn(zm[u], __fmaf_rn(bt, tau, bw)));
            if (fabsf(dlt) > margin) vis = dlt < 0.0f;
            else {
              float te = slope_max;
              if (c > 0.0f) {
                const float s2 = fmaxf(__fsub_rn(1.0f, __fmul_rn(c, c)), 0.0f);
                te = fminf(fmaxf(__fdiv_rn(__fsqrt_rn(s2), c), 1.0f), slope_max);
              }
              vis = z[u] <= __fadd_rn(zm[u], __fadd_rn(__fmul_rn(bt, te), bw));
            }
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
#pragma unroll 4
      for (int t = t0; t < t1; ++t) {
        const int k = IDENT ? t : sTex[t];
        const int j = (IDENT ? t : (int)sTexD[t]) - k0;
        const float4 wi = sE[2 * k];
        const float c = n.x * wi.x + n.y * wi.y + n.z * wi.z;
        const bool live = ((bits >> j) & 1u) && (c > 0.f);                       // max(0, w_i . n) and the visibility bit
        if (!__any_sync(0xffffffffu, live)) continue;
        const float4 LA = sE[2 * k + 1];
        const float ow = q.wox * wi.x + q.woy * wi.y + q.woz * wi.z;
        const float hl2 = fmaxf(2.f + 2.f * ow, 1e-12f);                         // |w_i + w_o|^2
        const float hinv = vs_rsq(hl2);
        const float nh = (c + q.nwo_raw) * hinv;
        const float oh = (0.5f * hl2) * hinv;                                    // w_o . h
        const float tx = fmaf(-c, n.x, wi.x) + q.tox, ty = fmaf(-c, n.y, wi.y) + q.toy, tz = fmaf(-c, n.z, wi.z) + q.toz;
        const float den = fmaf(q.al2 * nh, nh, (tx * tx + ty * ty + tz * tz) * (hinv * hinv));   // (n.h)^2 (a^2 - 1) + 1, Eq.13
        const float F = fmaf(0.96f, vs_ex2((-5.55473f * oh - 6.98316f) * oh), 0.04f);           // Eq.14
        const float gi = fmaf(c, q.omk, q.kk);
        const float sp = q.cS * F * vs_rcp(den * den * gi);
        const float w = live ? c : 0.f;                                          // branch-free: dead lanes add zero
        const float ws = w * sp;
        d0 = fmaf(LA.x, w, d0); d1 = fmaf(LA.y, w, d1); d2 = fmaf(LA.z, w, d2);
        s0 = fmaf(LA.x, ws, s0); s1 = fmaf(LA.y, ws, s1); s2 = fmaf(LA.z, ws, s2);
      }
    }
    // ---- the warps' partial sums are folded in warp order by the team's first warp, which finishes Eq.12 and the gamma curve
    myPart[lane] = d0; myPart[32 + lane] = d1; myPart[64 + lane] = d2; myPart[96 + lane] = s0; myPart[128 + lane] = s1; myPart[160 + lane] = s2;
    team_sync(team);
    if (tw != 0) continue;
    float acc[6];
#pragma unroll
    for (int c = 0; c < 6; ++c) {
      float sum = 0.f;
#pragma unroll
      for (int w = 0; w < VS_TEAM_WARPS; ++w) sum += sPart[(((size_t)team * VS_TEAM_WARPS + w) * 6 + c) * 32 + lane];
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
  if (vs_smem_bytes(K, ne, 1) <= 56 * 1024) return 1;                              // four CTAs of one team per SM
  if (vs_smem_bytes(K, ne, 2) <= 113 * 1024) return 2;
  if (vs_smem_bytes(K, ne, 4) <= lim) return 4;
  return 0;
}

int rga_vis_shade_init_attributes() {
  const int mx = 227 * 1024 - 1024;
  cudaError_t e = cudaFuncSetAttribute(vis_shade_kernel<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<2, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<2, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_shade_kernel<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx);
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
                                      av->tex_dir, av->dir_eps);
  rga_prof_mark(av, "texel_csr", s);
  av->launches += 1;
  return cudaGetLastError();
}

cudaError_t rga_launch_vis_shade(rga_avatar* av, const rga_vis_params* vis, const rga_env* env, float3 cam, cudaStream_t s) {
  const int K = vis->n_dirs, ne = env->rows * env->cols, teams = rga_vis_shade_teams(K, ne);
  if (teams == 0) return cudaErrorInvalidConfiguration;
  VsArgs a;
  a.K = K; a.R = vis->res; a.ne = ne; a.words = (K + 31) / 32;
  a.frames = reinterpret_cast<const float4*>(av->frames); a.env_table = av->env_table;
  a.dir_start = av->dir_start; a.tex_list = av->tex_list; a.tex_dir = av->tex_dir; a.dir_eps = av->dir_eps; a.zmap = av->zmap;
  a.front_list = av->front_list; a.n_front = av->n_front;
  a.g_posed = av->g_posed; a.g_nposed = av->g_nposed; a.g_static = av->g_static;
  a.cam = cam; a.inv_gamma = 1.0f / env->gamma;
  a.radiance = av->radiance; a.color = av->color; a.visbits = av->visbits; a.counter = av->vs_counter;
  const size_t smem = vs_smem_bytes(K, ne, teams);
  const int per_sm = teams == 1 ? 4 : (teams == 2 ? 2 : 1);
  int grid = av->num_sms * per_sm;
  const int max_groups = (av->n_gauss + 31) / 32;
  if (grid * teams > max_groups) grid = (max_groups + teams - 1) / teams;
  if (grid < 1) grid = 1;
  const bool ident = env->texel_to_dir == nullptr && ne == K;              // texel k reads direction k: no texel lists
  if (teams == 1) { if (ident) vis_shade_kernel<1, true><<<grid, VS_TEAM_THREADS, smem, s>>>(a); else vis_shade_kernel<1, false><<<grid, VS_TEAM_THREADS, smem, s>>>(a); }
  else if (teams == 2) { if (ident) vis_shade_kernel<2, true><<<grid, 2 * VS_TEAM_THREADS, smem, s>>>(a); else vis_shade_kernel<2, false><<<grid, 2 * VS_TEAM_THREADS, smem, s>>>(a); }
  else { if (ident) vis_shade_kernel<4, true><<<grid, 4 * VS_TEAM_THREADS, smem, s>>>(a); else vis_shade_kernel<4, false><<<grid, 4 * VS_TEAM_THREADS, smem, s>>>(a); }
  rga_prof_mark(av, "vis_shade", s);
  av->launches += 1;
  return cudaGetLastError();
}
