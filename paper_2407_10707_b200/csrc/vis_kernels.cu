// H3/H4 visibility_raster: orthographic rasterisation of the posed mesh from every light direction
// into a shared-memory depth map (atomicMin on packed depth), then either the per-Gaussian shadow-map depth test
// (mode 0; BASELINE.json north_star (b)) or the paper's triangle-ID visibility with the
// median/median/mean vertex filters (mode 1; Eq.3-4).
// EXACT file: -fmad=false; + - * / sqrt and integer arithmetic only.
#include "rga_internal.h"

// DESIGN.md A13: w = direction toward the light; u = normalize(e x w), e = z unless |w_z| > 0.999 then x; v = w x u.
// The frame is pre-scaled once per direction: us = u sR, vs = v sR, wn = -w inv2r (see "Arithmetic contract").
struct LightFrame { float us[3], vs[3], wn[3], w[3]; };
struct WinConst { float cx, cy, cz, r, sR, hR, inv2r; };

__device__ __forceinline__ WinConst make_win(const float* __restrict__ window, int R) {
  WinConst W;
  W.cx = window[0]; W.cy = window[1]; W.cz = window[2]; W.r = window[3];
  W.hR = 0.5f * (float)R; W.sR = W.hR / W.r; W.inv2r = 1.0f / (2.0f * W.r);
  return W;
}

__device__ __forceinline__ LightFrame make_frame(const float* __restrict__ dir, const WinConst& W) {
  LightFrame f;
  f.w[0] = dir[0]; f.w[1] = dir[1]; f.w[2] = dir[2];
  float e0 = 0.f, e1 = 0.f, e2 = 1.f;
  if (fabsf(f.w[2]) > 0.999f) { e0 = 1.f; e2 = 0.f; }
  float c0 = e1 * f.w[2] - e2 * f.w[1], c1 = e2 * f.w[0] - e0 * f.w[2], c2 = e0 * f.w[1] - e1 * f.w[0];
  float len = sqrtf((c0 * c0 + c1 * c1) + c2 * c2);
  float u0 = c0 / len, u1 = c1 / len, u2 = c2 / len;
  float v0 = f.w[1] * u2 - f.w[2] * u1, v1 = f.w[2] * u0 - f.w[0] * u2, v2 = f.w[0] * u1 - f.w[1] * u0;
  f.us[0] = u0 * W.sR; f.us[1] = u1 * W.sR; f.us[2] = u2 * W.sR;
  f.vs[0] = v0 * W.sR; f.vs[1] = v1 * W.sR; f.vs[2] = v2 * W.sR;
  f.wn[0] = -(f.w[0] * W.inv2r); f.wn[1] = -(f.w[1] * W.inv2r); f.wn[2] = -(f.w[2] * W.inv2r);
  return f;
}

// px = (u.d) sR + R/2, py likewise, z = (r - w.d)/(2r): three explicit fused chains (bit-identical to std::fma)
__device__ __forceinline__ void light_project_xy(float dx, float dy, float dz, const WinConst& W, const LightFrame& f,
                                                 float& px, float& py) {
  px = __fmaf_rn(f.us[2], dz, __fmaf_rn(f.us[1], dy, __fmaf_rn(f.us[0], dx, W.hR)));
  py = __fmaf_rn(f.vs[2], dz, __fmaf_rn(f.vs[1], dy, __fmaf_rn(f.vs[0], dx, W.hR)));
}
__device__ __forceinline__ float light_project_z(float dx, float dy, float dz, const LightFrame& f) {
  return __fmaf_rn(f.wn[2], dz, __fmaf_rn(f.wn[1], dy, __fmaf_rn(f.wn[0], dx, 0.5f)));
}

// ------------------------------------------------------------------------------------------------------------- H3
// One CTA per (direction, band of rows).  The band's depth map lives in shared memory: u32 depth (mode 0) or
// u64 depth<<32|triangle (WITH_ID).  Each warp walks triangles with a block stride, one per lane.  A triangle whose
// clipped pixel box is small is rasterised by its own lane with incremental int32 edge functions; the rare large ones
// (slivers, close-ups) go to the warp's queue in shared memory and are rasterised by the whole warp, one lane per
// pixel, so a long triangle never stalls the 31 other lanes (ncu on the first version: 7 of 32 lanes active).  There
// is no block barrier inside the triangle loop.
// Coverage and depth follow DESIGN.md "Arithmetic contract" exactly: vertices snapped to 1/256 pixel, integer edge
// functions (inclusive, two-sided), z = (z0 + (e1/area)(z1-z0)) + (e2/area)(z2-z0) in fp32, clamped at 0.
#define RAST_THREADS 512
#define RAST_QW 96             // per-warp queue slots (drained when fewer than 32 remain)
#define RAST_SMALL 12          // pixel-box size up to which a lane rasterises its own triangle

struct TriSetup {
  int x0, y0, x1, y1, x2, y2;          // 1/256-pixel coordinates
  float d0[3], d1[3], d2[3];           // vertex - window centre (depth is projected only when needed)
  int ia, ib, ja, jb;                  // pixel box clipped to the map and the band
  bool ok;                             // pixel box not empty
  bool narrow;                         // unclipped box below 2^14 sub-pixels in x and y: edge functions fit int32
};

__device__ __forceinline__ TriSetup tri_setup(int t, const int* __restrict__ faces, const float4* __restrict__ v_posed,
                                              const WinConst& W, const LightFrame& F, int R, int row0, int rows) {
  TriSetup s;
  int i0 = __ldg(faces + 3 * t), i1 = __ldg(faces + 3 * t + 1), i2 = __ldg(faces + 3 * t + 2);
  float4 a = __ldg(v_posed + i0), b = __ldg(v_posed + i1), c = __ldg(v_posed + i2);
  s.d0[0] = a.x - W.cx; s.d0[1] = a.y - W.cy; s.d0[2] = a.z - W.cz;
  s.d1[0] = b.x - W.cx; s.d1[1] = b.y - W.cy; s.d1[2] = b.z - W.cz;
  s.d2[0] = c.x - W.cx; s.d2[1] = c.y - W.cy; s.d2[2] = c.z - W.cz;
  float px, py;
  light_project_xy(s.d0[0], s.d0[1], s.d0[2], W, F, px, py);
  s.x0 = __float2int_rn(px * 256.0f); s.y0 = __float2int_rn(py * 256.0f);
  light_project_xy(s.d1[0], s.d1[1], s.d1[2], W, F, px, py);
  s.x1 = __float2int_rn(px * 256.0f); s.y1 = __float2int_rn(py * 256.0f);
  light_project_xy(s.d2[0], s.d2[1], s.d2[2], W, F, px, py);
  s.x2 = __float2int_rn(px * 256.0f); s.y2 = __float2int_rn(py * 256.0f);
  int mnx = min(s.x0, min(s.x1, s.x2)), mxx = max(s.x0, max(s.x1, s.x2));
  int mny = min(s.y0, min(s.y1, s.y2)), mxy = max(s.y0, max(s.y1, s.y2));
  // pixel i has its centre at 256 i + 128: first centre >= mn, last centre <= mx
  s.ia = max((mnx + 127) >> 8, 0); s.ib = min((mxx - 128) >> 8, R - 1);
  s.ja = max((mny + 127) >> 8, row0); s.jb = min((mxy - 128) >> 8, row0 + rows - 1);
  s.narrow = (mxx - mnx) < 16384 && (mxy - mny) < 16384;
  s.ok = s.ia <= s.ib && s.ja <= s.jb;
  return s;
}

template <bool WITH_ID>
__device__ __forceinline__ void put_sample(unsigned* sz32, unsigned long long* sz64, int p, float z, int t) {
  z = fmaxf(z, 0.0f);
  if (WITH_ID) atomicMin(sz64 + p, ((unsigned long long)__float_as_uint(z) << 32) | (unsigned)t);
  else atomicMin(sz32 + p, __float_as_uint(z));
}

// whole warp, one lane per pixel of the triangle's box; int64 edge functions (any size)
template <bool WITH_ID>
__device__ __forceinline__ void raster_big(int tq, int lane, const int* __restrict__ faces, const float4* __restrict__ v_posed,
    const WinConst& W, const LightFrame& F, int R, int row0, int rows, unsigned* sz32, unsigned long long* sz64) {
  const TriSetup s = tri_setup(tq, faces, v_posed, W, F, R, row0, rows);
  const long long x0 = s.x0, y0 = s.y0, x1 = s.x1, y1 = s.y1, x2 = s.x2, y2 = s.y2;
  const long long area = (x1 - x0) * (y2 - y0) - (y1 - y0) * (x2 - x0);
  if (area == 0) return;
  const float z0 = light_project_z(s.d0[0], s.d0[1], s.d0[2], F), z1 = light_project_z(s.d1[0], s.d1[1], s.d1[2], F),
              z2 = light_project_z(s.d2[0], s.d2[1], s.d2[2], F);
  const int bw = s.ib - s.ia + 1, cnt = bw * (s.jb - s.ja + 1);
  const float fa = (float)area, d1 = z1 - z0, d2 = z2 - z0;
  for (int q = lane; q < cnt; q += 32) {
    const int j = s.ja + q / bw, i = s.ia + q % bw;
    const long long qx = 256ll * i + 128, qy = 256ll * j + 128;
    const long long e0 = (x2 - x1) * (qy - y1) - (y2 - y1) * (qx - x1);
    const long long e1 = (x0 - x2) * (qy - y2) - (y0 - y2) * (qx - x2);
    const long long e2 = (x1 - x0) * (qy - y0) - (y1 - y0) * (qx - x0);
    if ((e0 >= 0 && e1 >= 0 && e2 >= 0) || (e0 <= 0 && e1 <= 0 && e2 <= 0)) {
      float t1 = (float)e1 / fa, t2 = (float)e2 / fa;
      put_sample<WITH_ID>(sz32, sz64, (j - row0) * R + i, (z0 + t1 * d1) + t2 * d2, tq);
    }
  }
}

template <bool WITH_ID>
__global__ void __launch_bounds__(RAST_THREADS) vis_raster_kernel(int nf, int R, int band_rows, int n_bands, int nv_words,
    const float4* __restrict__ v_posed, const int* __restrict__ faces, const float* __restrict__ dirs,
    const float* __restrict__ window, unsigned* __restrict__ zmap, int* __restrict__ idmap,
    unsigned* __restrict__ vbits_raw, int words, int n_verts) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int s_queue[RAST_THREADS / 32][RAST_QW];
  const int k = blockIdx.x / n_bands, band = blockIdx.x % n_bands;
  const int row0 = band * band_rows, rows = min(band_rows, R - row0);
  const int npix = rows * R;
  unsigned* sz32 = reinterpret_cast<unsigned*>(smem_raw);
  unsigned long long* sz64 = reinterpret_cast<unsigned long long*>(smem_raw);
  unsigned* svert = reinterpret_cast<unsigned*>(smem_raw + (size_t)band_rows * R * 8);     // WITH_ID only: vertex bitset
  if (WITH_ID) {
    for (int p = threadIdx.x; p < npix; p += blockDim.x) sz64[p] = ~0ull;
    for (int p = threadIdx.x; p < nv_words; p += blockDim.x) svert[p] = 0u;
  } else {
    for (int p = threadIdx.x; p < npix; p += blockDim.x) sz32[p] = 0xffffffffu;
  }
  const WinConst W = make_win(window, R);
  const LightFrame F = make_frame(dirs + 3 * k, W);
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int* myq = s_queue[warp];
  int qn = 0;                                             // warp-uniform

  for (int base = warp * 32; base < nf; base += blockDim.x) {
    const int t = base + lane;
    bool big = false;
    if (t < nf) {
      const TriSetup s = tri_setup(t, faces, v_posed, W, F, R, row0, rows);
      if (s.ok) {
        const int bw = s.ib - s.ia + 1, bh = s.jb - s.ja + 1;
        if (s.narrow && bw * bh <= RAST_SMALL) {
          // int32 edge functions, orientation normalised so that "inside" is e0,e1,e2 >= 0
          const int area = (s.x1 - s.x0) * (s.y2 - s.y0) - (s.y1 - s.y0) * (s.x2 - s.x0);
          if (area != 0) {
            const int sg = area > 0 ? 1 : -1;
            const int qx = 256 * s.ia + 128, qy = 256 * s.ja + 128;
            int r0 = sg * ((s.x2 - s.x1) * (qy - s.y1) - (s.y2 - s.y1) * (qx - s.x1));
            int r1 = sg * ((s.x0 - s.x2) * (qy - s.y2) - (s.y0 - s.y2) * (qx - s.x2));
            int r2 = sg * ((s.x1 - s.x0) * (qy - s.y0) - (s.y1 - s.y0) * (qx - s.x0));
            const int ax0 = -sg * 256 * (s.y2 - s.y1), ax1 = -sg * 256 * (s.y0 - s.y2), ax2 = -sg * 256 * (s.y1 - s.y0);
            const int ay0 = sg * 256 * (s.x2 - s.x1), ay1 = sg * 256 * (s.x0 - s.x2), ay2 = sg * 256 * (s.x1 - s.x0);
            float z0 = 0.f, d1 = 0.f, d2 = 0.f;
            const float fa = (float)(sg * area);
            bool have_z = false;
            for (int j = s.ja; j <= s.jb; ++j) {
              int e0 = r0, e1 = r1, e2 = r2;
              for (int i = s.ia; i <= s.ib; ++i) {
                if ((e0 | e1 | e2) >= 0) {
                  if (!have_z) {                                      // most sub-pixel triangles never get here
                    z0 = light_project_z(s.d0[0], s.d0[1], s.d0[2], F);
                    d1 = light_project_z(s.d1[0], s.d1[1], s.d1[2], F) - z0;
                    d2 = light_project_z(s.d2[0], s.d2[1], s.d2[2], F) - z0;
                    have_z = true;
                  }
                  float t1 = (float)e1 / fa, t2 = (float)e2 / fa;
                  put_sample<WITH_ID>(sz32, sz64, (j - row0) * R + i, (z0 + t1 * d1) + t2 * d2, t);
                }
                e0 += ax0; e1 += ax1; e2 += ax2;
              }
              r0 += ay0; r1 += ay1; r2 += ay2;
            }
          }
        } else big = true;
      }
    }
    const unsigned bm = __ballot_sync(0xffffffffu, big);
    if (bm) {
      if (big) myq[qn + __popc(bm & ((1u << lane) - 1u))] = t;
      qn += __popc(bm);
      __syncwarp();
      if (qn > RAST_QW - 32) {
        for (int e = 0; e < qn; ++e) raster_big<WITH_ID>(myq[e], lane, faces, v_posed, W, F, R, row0, rows, sz32, sz64);
        qn = 0;
        __syncwarp();
      }
    }
  }
  for (int e = 0; e < qn; ++e) raster_big<WITH_ID>(myq[e], lane, faces, v_posed, W, F, R, row0, rows, sz32, sz64);
  __syncthreads();

  size_t gbase = ((size_t)k * R + row0) * R;
  if (WITH_ID) {
    for (int p = threadIdx.x; p < npix; p += blockDim.x) {
      unsigned long long key = sz64[p];
      zmap[gbase + p] = (unsigned)(key >> 32);
      int tri = (key == ~0ull) ? -1 : (int)(unsigned)(key & 0xffffffffu);
      idmap[gbase + p] = tri;
      if (vbits_raw && tri >= 0) {                      // a triangle that appears marks its 3 vertices
        int v0 = __ldg(faces + 3 * tri), v1 = __ldg(faces + 3 * tri + 1), v2 = __ldg(faces + 3 * tri + 2);
        atomicOr(svert + (v0 >> 5), 1u << (v0 & 31));
        atomicOr(svert + (v1 >> 5), 1u << (v1 & 31));
        atomicOr(svert + (v2 >> 5), 1u << (v2 & 31));
      }
    }
    if (vbits_raw) {
      __syncthreads();
      const unsigned bit = 1u << (k & 31);
      for (int wd = threadIdx.x; wd < nv_words; wd += blockDim.x) {
        unsigned m = svert[wd];
        while (m) {
          int b = __ffs(m) - 1; m &= m - 1;
          int vtx = wd * 32 + b;
          if (vtx < n_verts) atomicOr(vbits_raw + (size_t)vtx * words + (k >> 5), bit);
        }
      }
    }
  } else {
    for (int p = threadIdx.x; p < npix; p += blockDim.x) zmap[gbase + p] = sz32[p];
  }
}

size_t rga_vis_raster_smem(int res, int with_id, int n_verts, int* band_rows) {
  const size_t budget = 200 * 1024;
  size_t per_row = (size_t)res * (with_id ? 8 : 4);
  size_t extra = with_id ? (size_t)((n_verts + 31) / 32) * 4 : 0;
  int rows = (int)((budget - extra) / per_row);
  if (rows > res) rows = res;
  if (rows < 1) rows = 1;
  int bands = (res + rows - 1) / rows;
  rows = (res + bands - 1) / bands;                       // even bands
  *band_rows = rows;
  return per_row * rows + extra;
}

cudaError_t rga_launch_vis_raster(rga_avatar* av, const rga_vis_params* p, cudaStream_t s) {
  const bool with_id = p->mode == 1 || p->keep_maps;
  int band_rows = 0;
  size_t smem = rga_vis_raster_smem(p->res, with_id, av->n_verts, &band_rows);
  int n_bands = (p->res + band_rows - 1) / band_rows;
  int words = (p->n_dirs + 31) / 32, nv_words = (av->n_verts + 31) / 32;
  dim3 grid(p->n_dirs * n_bands);
  if (with_id) {
    unsigned* raw = (p->mode == 1) ? av->vbits_raw : nullptr;
    if (raw) cudaMemsetAsync(raw, 0, (size_t)av->n_verts * words * 4, s);
    vis_raster_kernel<true><<<grid, RAST_THREADS, smem, s>>>(av->n_faces, p->res, band_rows, n_bands, nv_words, av->v_posed, av->faces,
                                                   p->dirs, av->window, av->zmap, av->idmap, raw, words, av->n_verts);
  } else {
    vis_raster_kernel<false><<<grid, RAST_THREADS, smem, s>>>(av->n_faces, p->res, band_rows, n_bands, nv_words, av->v_posed, av->faces,
                                                    p->dirs, av->window, av->zmap, av->idmap, nullptr, words, av->n_verts);
  }
  av->launches += 1;
  rga_prof_mark(av, "vis_raster", s);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------ H4a
// Shadow-map test, Gaussian-major: one thread per Gaussian keeps its position/normal in registers and walks all
// directions; neighbouring (Morton-ordered) Gaussians hit neighbouring texels, so the depth-map gathers stay in
// L1/L2.  32 directions are packed into one output word.  The slope factor tau (sqrt and divide) is only evaluated when
// the two monotone bounds beta(1) <= beta(tau) <= beta(slope_max) do not already decide the comparison.
#define DT_THREADS 128
__global__ void __launch_bounds__(DT_THREADS) vis_depth_test_kernel(int ng, int K, int R, const float4* __restrict__ g_posed,
    const float4* __restrict__ g_nposed, const float* __restrict__ dirs, const float* __restrict__ window,
    const unsigned* __restrict__ zmap, float bias_texels, float bias_world, float slope_max, int words_per_part,
    unsigned* __restrict__ visbits) {
  extern __shared__ __align__(16) float4 sF4[];                   // 3 float4 per direction: (us, w.x) (vs, w.y) (wn, w.z)
  const int words = (K + 31) >> 5;
  const int wd0 = blockIdx.y * words_per_part, wd1 = min(words, wd0 + words_per_part);
  const int k0 = wd0 * 32, k1 = min(K, wd1 * 32);
  const WinConst W = make_win(window, R);
  for (int k = k0 + threadIdx.x; k < k1; k += blockDim.x) {
    LightFrame f = make_frame(dirs + 3 * k, W);
    float4* o = sF4 + 3 * (k - k0);
    o[0] = make_float4(f.us[0], f.us[1], f.us[2], f.w[0]);
    o[1] = make_float4(f.vs[0], f.vs[1], f.vs[2], f.w[1]);
    o[2] = make_float4(f.wn[0], f.wn[1], f.wn[2], f.w[2]);
  }
  __syncthreads();
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ng) return;
  const float bt = bias_texels / (float)R, bw = bias_world * W.inv2r;
  const float beta_lo = bt * 1.0f + bw, beta_hi = bt * slope_max + bw;
  const bool bounds_ok = bt >= 0.f && slope_max >= 1.0f;
  const float Rm1 = (float)(R - 1);
  const float4 x = g_posed[g], n = g_nposed[g];
  const float dx = x.x - W.cx, dy = x.y - W.cy, dz = x.z - W.cz;
  const size_t RR = (size_t)R * R;
  for (int wd = wd0; wd < wd1; ++wd) {
    unsigned bits = 0;
    const int kend = min(32, K - wd * 32);
    const unsigned* zk = zmap + (size_t)wd * 32 * RR;
    const float4* fk = sF4 + 3 * (wd * 32 - k0);
#pragma unroll 4
    for (int b = 0; b < kend; ++b) {
      const float4 fu = fk[3 * b], fv = fk[3 * b + 1], fw = fk[3 * b + 2];
      const float px = __fmaf_rn(fu.z, dz, __fmaf_rn(fu.y, dy, __fmaf_rn(fu.x, dx, W.hR)));
      const float py = __fmaf_rn(fv.z, dz, __fmaf_rn(fv.y, dy, __fmaf_rn(fv.x, dx, W.hR)));
      const float z = __fmaf_rn(fw.z, dz, __fmaf_rn(fw.y, dy, __fmaf_rn(fw.x, dx, 0.5f)));
      // floor-then-clamp of the contract == clamp-then-truncate for every finite px
      const int ix = __float2int_rz(fminf(fmaxf(px, 0.0f), Rm1)), iy = __float2int_rz(fminf(fmaxf(py, 0.0f), Rm1));
      const unsigned zb = __ldg(zk + (size_t)b * RR + iy * R + ix);
      bool vis;
      if (zb == 0xffffffffu) vis = true;
      else {
        const float zm = __uint_as_float(zb);
        if (bounds_ok && z <= zm + beta_lo) vis = true;
        else if (bounds_ok && !(z <= zm + beta_hi)) vis = false;
        else {
          const float cs = (n.x * fu.w + n.y * fv.w) + n.z * fw.w;
          float tau;
          if (cs > 0.0f) {
            float s2 = fmaxf(1.0f - cs * cs, 0.0f);
            tau = sqrtf(s2) / cs;
            tau = fminf(fmaxf(tau, 1.0f), slope_max);
          } else tau = slope_max;
          vis = z <= zm + (bt * tau + bw);
        }
      }
      bits |= (vis ? 1u : 0u) << b;
    }
    visbits[(size_t)g * words + wd] = bits;
  }
}

cudaError_t rga_launch_vis_depth_test(rga_avatar* av, const rga_vis_params* p, cudaStream_t s) {
  // directions are split over blockIdx.y so that small avatars still fill the machine (100k Gaussians alone give
  // 676 threads per SM); neighbouring threads stay neighbouring Gaussians, whose texel gathers coalesce in L1
  int words = (p->n_dirs + 31) / 32;
  int parts = words < 4 ? words : 4;
  int wpp = (words + parts - 1) / parts;
  parts = (words + wpp - 1) / wpp;
  dim3 grid((av->n_gauss + DT_THREADS - 1) / DT_THREADS, parts);
  vis_depth_test_kernel<<<grid, DT_THREADS, (size_t)wpp * 32 * 3 * sizeof(float4), s>>>(
      av->n_gauss, p->n_dirs, p->res, av->g_posed, av->g_nposed, p->dirs, av->window, av->zmap, p->depth_bias_texels,
      p->depth_bias_world, p->slope_max, wpp, av->visbits);
  av->launches += 1;
  rga_prof_mark(av, "vis_depth_test", s);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------ H4b
// Eq.3-4 on bit-packed maps: thread = (vertex, word of 32 directions).  The K_v neighbour words are
// summed with a bit-sliced (carry-save) counter, so 32 directions are filtered at once.
__device__ __forceinline__ void sliced_count(const int* __restrict__ nb, int Kv, const unsigned* __restrict__ bits, int words,
                                             int wd, unsigned c[5]) {
#pragma unroll
  for (int s = 0; s < 5; ++s) c[s] = 0u;
  for (int q = 0; q < Kv; ++q) {
    unsigned carry = __ldg(bits + (size_t)__ldg(nb + q) * words + wd);
#pragma unroll
    for (int s = 0; s < 5; ++s) { unsigned t = c[s] & carry; c[s] ^= carry; carry = t; }
  }
}

__global__ void __launch_bounds__(256) vis_median_kernel(int nv, int words, int Kv, const int* __restrict__ knn_v,
                                                         const unsigned* __restrict__ in, unsigned* __restrict__ out) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nv * words) return;
  int j = t / words, wd = t - j * words;
  unsigned c[5];
  sliced_count(knn_v + (size_t)j * Kv, Kv, in, words, wd, c);
  const int T = (Kv + 1) / 2;                                      // median of Kv (odd) bits = count >= T
  unsigned gt = 0u, eq = ~0u;
#pragma unroll
  for (int s = 4; s >= 0; --s) {
    unsigned tb = ((T >> s) & 1) ? ~0u : 0u;
    gt |= eq & c[s] & ~tb;
    eq &= ~(c[s] ^ tb);
  }
  out[t] = gt | eq;
}

__global__ void __launch_bounds__(256) vis_mean_kernel(int nv, int words, int K, int Kv, const int* __restrict__ knn_v,
                                                       const unsigned* __restrict__ in, unsigned char* __restrict__ vcount) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nv * words) return;
  int j = t / words, wd = t - j * words;
  unsigned c[5];
  sliced_count(knn_v + (size_t)j * Kv, Kv, in, words, wd, c);
  unsigned char* dst = vcount + (size_t)j * K + wd * 32;
  int kend = min(32, K - wd * 32);
  if (kend == 32 && (K & 15) == 0) {
    unsigned out[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      unsigned v = 0;
#pragma unroll
      for (int b = 0; b < 4; ++b) {
        int bit = q * 4 + b;
        unsigned cnt = ((c[0] >> bit) & 1) | (((c[1] >> bit) & 1) << 1) | (((c[2] >> bit) & 1) << 2) |
                       (((c[3] >> bit) & 1) << 3) | (((c[4] >> bit) & 1) << 4);
        v |= cnt << (8 * b);
      }
      out[q] = v;
    }
    uint4* d4 = reinterpret_cast<uint4*>(dst);
    d4[0] = make_uint4(out[0], out[1], out[2], out[3]);
    d4[1] = make_uint4(out[4], out[5], out[6], out[7]);
  } else {
    for (int bit = 0; bit < kend; ++bit)
      dst[bit] = (unsigned char)(((c[0] >> bit) & 1) | (((c[1] >> bit) & 1) << 1) | (((c[2] >> bit) & 1) << 2) |
                                 (((c[3] >> bit) & 1) << 3) | (((c[4] >> bit) & 1) << 4));
  }
}

cudaError_t rga_launch_vis_paper(rga_avatar* av, const rga_vis_params* p, cudaStream_t s) {
  int words = (p->n_dirs + 31) / 32;
  int n = av->n_verts * words, grid = (n + 255) / 256;
  vis_median_kernel<<<grid, 256, 0, s>>>(av->n_verts, words, av->k_v, av->knn_v, av->vbits_raw, av->vbits_a);
  rga_prof_mark(av, "vis_median1", s);
  vis_median_kernel<<<grid, 256, 0, s>>>(av->n_verts, words, av->k_v, av->knn_v, av->vbits_a, av->vbits_b);
  rga_prof_mark(av, "vis_median2", s);
  vis_mean_kernel<<<grid, 256, 0, s>>>(av->n_verts, words, p->n_dirs, av->k_v, av->knn_v, av->vbits_b, av->vcount);
  rga_prof_mark(av, "vis_mean", s);
  av->launches += 3;
  return cudaGetLastError();
}

int rga_vis_init_attributes() {
  cudaError_t e = cudaFuncSetAttribute(vis_raster_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 210 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_raster_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 210 * 1024);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_depth_test_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
  return (int)e;
}
