// H3/H4 visibility_raster: orthographic rasterisation of the posed mesh from every light direction
// into a shared-memory depth map (atomicMin on packed depth), then either the per-Gaussian shadow-map depth test
// (mode 0; BASELINE.json north_star (b)) or the paper's triangle-ID visibility with the
// median/median/mean vertex filters (mode 1; Eq.3-4).
// EXACT file: -fmad=false; + - * / sqrt and integer arithmetic only.
#include <cstdlib>
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
// Persistent CTAs (one per SM) walk the (direction, band of rows) units.  Per unit:
//   A.  every vertex is projected ONCE into shared memory: snapped (X,Y) packed in 32 bits (X,Y < 2^16 because the
//       window contains every posed vertex and R <= 256);
//   B1. warps fetch 32 triangles at a time (dynamic counter), one per lane: one 8-byte packed face, three shared-memory
//       gathers, pixel box; triangles whose box holds no pixel centre (53 % at config 1) end there, the others are
//       compacted into the warp's queue;
//   B2. whenever 32 are queued, each lane writes its triangle's edge-function coefficients to the warp's table; every
//       box row is cut into runs of up to 4 pixel centres and the runs of all 32 boxes are dealt out over all lanes
//       (warp scan + head bitmask), so a sliver never idles the other lanes; a lane steps three int32 edge functions
//       along its run (3 IADD per sample); runs with a covered sample (most have none) are compacted again;
//   C.  whenever 32 such runs are queued, the triangle's vertex depths are projected on demand and the covered samples
//       are interpolated and atomicMin'ed into the shared-memory map (u32 depth, or u64 depth<<32|tri).
// The finished band is written to HBM once, coalesced.  ncu on the first version (one projection per triangle corner,
// per-lane pixel loops): 693 warp instructions per 32 triangles at 17.9 active lanes (profiles/r01a_ncu_full.md).
// Coverage and depth follow DESIGN.md "Arithmetic contract" exactly: vertices snapped to 1/256 pixel, integer edge
// functions (inclusive, two-sided; int32 when the triangle spans < 64 pixels, else int64), area = e0+e1+e2 (exact
// identity), z = (z0 + (e1/area)(z1-z0)) + (e2/area)(z2-z0) in fp32, clamped at 0.
#define RAST_MAX_RES 256       // snapped coordinates must fit 16 bits
#define RAST_MAX_BANDS 64      // bands of a map that does not fit shared memory whole

__device__ __forceinline__ void face_unpack(unsigned long long f, int& i0, int& i1, int& i2) {
  i0 = (int)(f & 0x1fffffull); i1 = (int)((f >> 21) & 0x1fffffull); i2 = (int)((f >> 42) & 0x1fffffull);
}

__global__ void pack_faces_kernel(int nf, const int* __restrict__ faces, unsigned long long* __restrict__ packed) {
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nf) return;
  unsigned long long a = (unsigned)faces[3 * t], b = (unsigned)faces[3 * t + 1], c = (unsigned)faces[3 * t + 2];
  packed[t] = a | (b << 21) | (c << 42);
}

cudaError_t rga_launch_pack_faces(rga_avatar* av, cudaStream_t s) {
  pack_faces_kernel<<<(av->n_faces + 255) / 256, 256, 0, s>>>(av->n_faces, av->faces, av->faces_packed);
  return cudaGetLastError();
}

// Per-warp working set in shared memory
#define RAST_Q 64              // queue entries: < 32 left over + <= 32 pushed
#ifndef RAST_SEGW
#define RAST_SEGW 4            // a sampling unit is a run of up to 4 pixel centres of one box row
#endif
struct RasterWarp {
  uint4 tab[4][32];            // round table (component-major: lanes read neighbouring owners without bank conflicts):
                               // edge-function coefficients and box of the 32 triangles being sampled
  uint4 q2[RAST_Q];            // runs with covered samples: {triangle | mask << 24 | tall << 28 | wide << 31, first pixel, e1, e2}
  int q1[RAST_Q];              // triangles whose pixel box is not empty
  int q1s[RAST_Q];             // ... of which the box is ONE run (one line of up to RAST_SEGW pixel centres, int32 edge functions)
};

struct RasterCtx {
  int R, row0, rows;
  const unsigned* sXY;
  const float4* v_posed; const unsigned long long* faces_packed;
  unsigned* sz32; unsigned long long* sz64;
  const float* zf;             // shared memory: window centre (3) and the depth row of the light frame wn (3)
  const float* sZ;             // shared memory: depth of every vertex for this direction (with the table in shared memory), or NULL
};

// pixel box of a triangle given its packed corners, clipped to the map and the band; returns the sample count
__device__ __forceinline__ int tri_box(unsigned P0, unsigned P1, unsigned P2, const int R, const int row0, const int rows,
                                       int& ia, int& ja, int& bw, int& bh, bool& narrow) {
  const int x0 = P0 & 0xffff, y0 = P0 >> 16, x1 = P1 & 0xffff, y1 = P1 >> 16, x2 = P2 & 0xffff, y2 = P2 >> 16;
  const int mnx = min(x0, min(x1, x2)), mxx = max(x0, max(x1, x2));
  const int mny = min(y0, min(y1, y2)), mxy = max(y0, max(y1, y2));
  // pixel i has its centre at 256 i + 128: first centre >= mn, last centre <= mx
  ia = max((mnx + 127) >> 8, 0); const int ib = min((mxx - 128) >> 8, R - 1);
  ja = max((mny + 127) >> 8, row0); const int jb = min((mxy - 128) >> 8, row0 + rows - 1);
  narrow = (mxx - mnx) < 16384 && (mxy - mny) < 16384;
  bw = ib - ia + 1;
  bh = jb - ja + 1;
  return (bw > 0 && bh > 0) ? bw * bh : 0;
}

template <bool WITH_ID>
__device__ __forceinline__ void put_depth(const RasterCtx& c, int p, unsigned t, float f1, float f2, float fa, float z0, float z1,
                                          float z2) {
  const float t1 = f1 / fa, t2 = f2 / fa;
  float z = (z0 + t1 * (z1 - z0)) + t2 * (z2 - z0);
  z = fmaxf(z, 0.0f);
  if (WITH_ID) atomicMin(c.sz64 + p, ((unsigned long long)__float_as_uint(z) << 32) | t);
  else atomicMin(c.sz32 + p, __float_as_uint(z));
}

// C. depth of the covered samples of up to 32 row segments (one per lane) and the atomicMin on the map.  The vertex
// depths are projected here, once per segment; e1, e2 step along the row by their x-coefficients.
template <bool WITH_ID>
__device__ __forceinline__ void raster_depth(const RasterCtx& c, const RasterWarp* w, int base, int n, int lane) {
  if (lane >= n) return;
  const uint4 q = w->q2[base + lane];
  const unsigned t = q.x & 0xffffffu, mask = (q.x >> 24) & 0xfu;
  int i0, i1, i2;
  face_unpack(__ldg(c.faces_packed + t), i0, i1, i2);
  // a tall run (down a column) was sampled with x and y exchanged: exchange them here too (a 16-bit rotation of the packed
  // corner); edge functions and area both change sign under the exchange, so e1 / area and e2 / area are unchanged
  const bool tall = (q.x >> 28) & 1u;
  const int rot = tall ? 16 : 0;
  const unsigned P0 = __funnelshift_l(c.sXY[i0], c.sXY[i0], rot), P1 = __funnelshift_l(c.sXY[i1], c.sXY[i1], rot),
                 P2 = __funnelshift_l(c.sXY[i2], c.sXY[i2], rot);
  const int x0 = P0 & 0xffff, y0 = P0 >> 16, x1 = P1 & 0xffff, y1 = P1 >> 16, x2 = P2 & 0xffff, y2 = P2 >> 16;
  // z = fma(wn.z, d.z, fma(wn.y, d.y, fma(wn.x, d.x, 0.5))): the frame is read from shared memory (kept in registers it
  // cost the sampling loop 20 registers it never uses)
  float z0, z1, z2;
  if (c.sZ) { z0 = c.sZ[i0]; z1 = c.sZ[i1]; z2 = c.sZ[i2]; }          // projected once per vertex in phase A (same chain)
  else {
    const float4 a = __ldg(c.v_posed + i0), b = __ldg(c.v_posed + i1), e = __ldg(c.v_posed + i2);
    const float cx = c.zf[0], cy = c.zf[1], cz = c.zf[2], wnx = c.zf[3], wny = c.zf[4], wnz = c.zf[5];
    z0 = __fmaf_rn(wnz, a.z - cz, __fmaf_rn(wny, a.y - cy, __fmaf_rn(wnx, a.x - cx, 0.5f)));
    z1 = __fmaf_rn(wnz, b.z - cz, __fmaf_rn(wny, b.y - cy, __fmaf_rn(wnx, b.x - cx, 0.5f)));
    z2 = __fmaf_rn(wnz, e.z - cz, __fmaf_rn(wny, e.y - cy, __fmaf_rn(wnx, e.x - cx, 0.5f)));
  }
  const int pstep = tall ? c.R : 1;                                 // the run goes down a column (pixel stride R) or along a row
  if (!(q.x >> 31)) {
    const int area = (x1 - x0) * (y2 - y0) - (y1 - y0) * (x2 - x0);
    const int ax1 = -256 * (y0 - y2), ax2 = -256 * (y1 - y0);
    const float fa = (float)area;
    for (unsigned m = mask; m; m &= m - 1u) {                         // usually one covered sample per run
      const int u = __ffs(m) - 1;
      put_depth<WITH_ID>(c, (int)q.y + u * pstep, t, (float)((int)q.z + u * ax1), (float)((int)q.w + u * ax2), fa, z0, z1, z2);
    }
  } else {                                                          // triangle spanning >= 64 pixels: int64 edge functions
    const int prow = (int)q.y / c.R + c.row0, pcol = (int)q.y % c.R;
    const long long X0 = x0, Y0 = y0, X1 = x1, Y1 = y1, X2 = x2, Y2 = y2;
    const long long area = (X1 - X0) * (Y2 - Y0) - (Y1 - Y0) * (X2 - X0);
    for (int u = 0; u < RAST_SEGW; ++u) {
      if ((mask >> u) & 1u) {
        // sample (column, row) of the map; in the exchanged space of a tall run its coordinates are (row, column)
        const int sc = pcol + (tall ? 0 : u), sr = prow + (tall ? u : 0);
        const long long qx = 256ll * (tall ? sr : sc) + 128, qy = 256ll * (tall ? sc : sr) + 128;
        const long long e1 = (X0 - X2) * (qy - Y2) - (Y0 - Y2) * (qx - X2);
        const long long e2 = (X1 - X0) * (qy - Y0) - (Y1 - Y0) * (qx - X0);
        put_depth<WITH_ID>(c, (int)q.y + u * pstep, t, (float)e1, (float)e2, (float)area, z0, z1, z2);
      }
    }
  }
}

// B2. one round: lane l owns queued triangle l (l < n).  Every box row is cut into segments of up to RAST_SEGW pixel
// centres; the segments of all n boxes are dealt out 32 at a time, one per lane, and a lane steps its edge functions
// along the row.  Returns the new fill of the covered-segment queue.
template <bool WITH_ID>
__device__ __forceinline__ int raster_round(const RasterCtx& c, RasterWarp* w, int qbase, int n, int lane, int q2n) {
  int cnt = 0;
  unsigned boxw = 0u, ay2u = 0u; float inv = 1.0f;
  if (lane < n) {
    const int t = w->q1[qbase + lane];
    int i0, i1, i2;
    face_unpack(__ldg(c.faces_packed + t), i0, i1, i2);
    unsigned P0 = c.sXY[i0], P1 = c.sXY[i1], P2 = c.sXY[i2];
    int ia, ja, bw, bh; bool narrow;
    tri_box(P0, P1, P2, c.R, c.row0, c.rows, ia, ja, bw, bh, narrow);
    // runs go along the LONGER side of the box (the body's limbs make most boxes taller than wide: with runs along x only a
    // 1 x 3 box was three runs of one sample).  A tall box is sampled with x and y EXCHANGED -- a 16-bit rotation of the
    // packed corners and a swap of the box -- so the code below only knows runs along x; all three edge functions change sign
    // together under the exchange, which the two-sided inside test does not see.
    const bool tall = bh > bw;
    const unsigned origin = (unsigned)((ja - c.row0) * c.R + ia);
    if (tall) {
      P0 = __funnelshift_l(P0, P0, 16); P1 = __funnelshift_l(P1, P1, 16); P2 = __funnelshift_l(P2, P2, 16);
      int tmp = ia; ia = ja; ja = tmp; tmp = bw; bw = bh; bh = tmp;
    }
    const int nsr = (bw + RAST_SEGW - 1) / RAST_SEGW;                 // runs per line
    cnt = bh * nsr;
    const int x0 = P0 & 0xffff, y0 = P0 >> 16, x1 = P1 & 0xffff, y1 = P1 >> 16, x2 = P2 & 0xffff, y2 = P2 >> 16;
    const int qx = 256 * ia + 128, qy = 256 * ja + 128;
    int C0 = -1, C1 = 1, C2 = 0, ax0 = 0, ax1 = 0, ax2 = 0, ay0 = 0, ay1 = 0, ay2 = 0;      // "never covered"
    if (narrow) {
      // e_k at sample (ia + col, ja + row) = C_k + ax_k col + ay_k row  (all int32: the box spans < 2^14 sub-pixels)
      const int e0 = (x2 - x1) * (qy - y1) - (y2 - y1) * (qx - x1);
      const int e1 = (x0 - x2) * (qy - y2) - (y0 - y2) * (qx - x2);
      const int e2 = (x1 - x0) * (qy - y0) - (y1 - y0) * (qx - x0);
      if (e0 + e1 + e2 != 0) {                                        // area == 0: skipped (contract)
        C0 = e0; C1 = e1; C2 = e2;
        ax0 = -256 * (y2 - y1); ax1 = -256 * (y0 - y2); ax2 = -256 * (y1 - y0);
        ay0 = 256 * (x2 - x1); ay1 = 256 * (x0 - x2); ay2 = 256 * (x1 - x0);
      }
    }
    boxw = origin | ((unsigned)(bw - 1) << 16) | (narrow ? (1u << 24) : 0u) | (tall ? (1u << 25) : 0u);
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"((float)nsr));       // only splits an index (error analysis below)
    ay2u = (unsigned)ay2;
    w->tab[0][lane] = make_uint4((unsigned)C0, (unsigned)ax0, (unsigned)ay0, (unsigned)C1);
    w->tab[1][lane] = make_uint4((unsigned)ax1, (unsigned)ay1, (unsigned)C2, (unsigned)ax2);
    w->tab[3][lane] = make_uint4((unsigned)t, (unsigned)ia | ((unsigned)ja << 16), 0u, 0u);
  }
  int inc = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
  const int exc = inc - cnt;
  const int total = __shfl_sync(0xffffffffu, inc, 31);
  if (lane < n) w->tab[2][lane] = make_uint4(ay2u, (unsigned)exc, boxw, __float_as_uint(inv));
  __syncwarp();
  int headbase = 0;
  for (int c0 = 0; c0 < total; c0 += 32) {
    const unsigned rel = (unsigned)(exc - c0);
    const unsigned bit = (rel < 32u && cnt > 0) ? (1u << rel) : 0u;
    const unsigned H = __reduce_or_sync(0xffffffffu, bit);
    // queued triangles all have samples, so the index among the heads is the owning lane
    const int owner = max(headbase + __popc(H & (0xffffffffu >> (31 - lane))) - 1, 0);
    headbase += __popc(H);
    const int s = c0 + lane;
    unsigned mask = 0u;
    uint4 out = make_uint4(0u, 0u, 0u, 0u);
    if (s < total) {
      const uint4 a = w->tab[0][owner], b = w->tab[1][owner], d = w->tab[2][owner];
      const int li = s - (int)d.y, obw = (int)((d.z >> 16) & 0xffu) + 1, nsr = (obw + RAST_SEGW - 1) / RAST_SEGW;
      // li / nsr: (li + 0.5) / nsr is >= 1/128 away from an integer, the approximate reciprocal is within 2^-22
      const int row = (int)(((float)li + 0.5f) * __uint_as_float(d.w));
      const int col0 = (li - row * nsr) * RAST_SEGW, ncol = min(RAST_SEGW, obw - col0);      // row = line, col0 = offset along the run
      const bool tall = d.z & (1u << 25);
      out.y = (d.z & 0xffffu) + (unsigned)(tall ? col0 * c.R + row : row * c.R + col0);
      if (tall) out.x = 1u << 28;
      if (d.z & (1u << 24)) {
        int e0 = (int)a.x + (int)a.y * col0 + (int)a.z * row;
        int e1 = (int)a.w + (int)b.x * col0 + (int)b.y * row;
        int e2 = (int)b.z + (int)b.w * col0 + (int)d.x * row;
        out.z = (unsigned)e1; out.w = (unsigned)e2;
#pragma unroll
        for (int u = 0; u < RAST_SEGW; ++u) {
          if (u < ncol && (min(e0, min(e1, e2)) >= 0 || max(e0, max(e1, e2)) <= 0)) mask |= 1u << u;
          e0 += (int)a.y; e1 += (int)b.x; e2 += (int)b.w;
        }
      } else {                                                        // triangle spanning >= 64 pixels: int64 edge functions
        const uint4 e = w->tab[3][owner];
        int i0, i1, i2;
        face_unpack(__ldg(c.faces_packed + e.x), i0, i1, i2);
        const int rot = tall ? 16 : 0;                              // the same exchanged space as the setup
        const unsigned P0 = __funnelshift_l(c.sXY[i0], c.sXY[i0], rot), P1 = __funnelshift_l(c.sXY[i1], c.sXY[i1], rot),
                       P2 = __funnelshift_l(c.sXY[i2], c.sXY[i2], rot);
        const long long x0 = P0 & 0xffff, y0 = P0 >> 16, x1 = P1 & 0xffff, y1 = P1 >> 16, x2 = P2 & 0xffff, y2 = P2 >> 16;
        const long long area = (x1 - x0) * (y2 - y0) - (y1 - y0) * (x2 - x0);
        const long long qy = 256ll * ((int)(e.y >> 16) + row) + 128;
        for (int u = 0; u < ncol; ++u) {
          const long long qx = 256ll * ((int)(e.y & 0xffffu) + col0 + u) + 128;
          const long long e0 = (x2 - x1) * (qy - y1) - (y2 - y1) * (qx - x1);
          const long long e1 = (x0 - x2) * (qy - y2) - (y0 - y2) * (qx - x2);
          const long long e2 = (x1 - x0) * (qy - y0) - (y1 - y0) * (qx - x0);
          if (((e0 >= 0 && e1 >= 0 && e2 >= 0) || (e0 <= 0 && e1 <= 0 && e2 <= 0)) && area != 0) mask |= 1u << u;
        }
        out.x |= 1u << 31;
      }
      if (mask) out.x |= w->tab[3][owner].x | (mask << 24);
    }
    const unsigned cm = __ballot_sync(0xffffffffu, mask != 0u);
    if (cm) {
      if (mask) w->q2[q2n + __popc(cm & ((1u << lane) - 1u))] = out;
      q2n += __popc(cm);
      __syncwarp();
      if (q2n >= 32) { q2n -= 32; raster_depth<WITH_ID>(c, w, q2n, 32, lane); __syncwarp(); }
    }
  }
  return q2n;
}

// B2s. a round of SINGLE-RUN triangles (three quarters of the non-empty boxes at config 1: 1 x 1 .. 1 x 4 and their transposes):
// lane l samples its own triangle's one run -- no scan over run counts, no round table, no owner search.  It builds exactly
// the q2 entry raster_round would build for that run (same exchanged space for a tall run, same e1 / e2 at the first sample,
// same mask), so the depth stage and the result are the same.
template <bool WITH_ID>
__device__ __forceinline__ int raster_single(const RasterCtx& c, RasterWarp* w, int qbase, int n, int lane, int q2n) {
  unsigned mask = 0u;
  uint4 out = make_uint4(0u, 0u, 0u, 0u);
  if (lane < n) {
    const int t = w->q1s[qbase + lane];
    int i0, i1, i2;
    face_unpack(__ldg(c.faces_packed + t), i0, i1, i2);
    unsigned P0 = c.sXY[i0], P1 = c.sXY[i1], P2 = c.sXY[i2];
    int ia, ja, bw, bh; bool narrow;
    tri_box(P0, P1, P2, c.R, c.row0, c.rows, ia, ja, bw, bh, narrow);
    const bool tall = bh > bw;
    out.y = (unsigned)((ja - c.row0) * c.R + ia);
    if (tall) {
      P0 = __funnelshift_l(P0, P0, 16); P1 = __funnelshift_l(P1, P1, 16); P2 = __funnelshift_l(P2, P2, 16);
      int tmp = ia; ia = ja; ja = tmp; bw = bh;
      out.x = 1u << 28;
    }
    const int x0 = P0 & 0xffff, y0 = P0 >> 16, x1 = P1 & 0xffff, y1 = P1 >> 16, x2 = P2 & 0xffff, y2 = P2 >> 16;
    const int qx = 256 * ia + 128, qy = 256 * ja + 128;
    int e0 = (x2 - x1) * (qy - y1) - (y2 - y1) * (qx - x1);
    int e1 = (x0 - x2) * (qy - y2) - (y0 - y2) * (qx - x2);
    int e2 = (x1 - x0) * (qy - y0) - (y1 - y0) * (qx - x0);
    if (e0 + e1 + e2 != 0) {                                            // area == 0: skipped (contract)
      const int ax0 = -256 * (y2 - y1), ax1 = -256 * (y0 - y2), ax2 = -256 * (y1 - y0);
      out.z = (unsigned)e1; out.w = (unsigned)e2;
#pragma unroll
      for (int u = 0; u < RAST_SEGW; ++u) {
        if (u < bw && (min(e0, min(e1, e2)) >= 0 || max(e0, max(e1, e2)) <= 0)) mask |= 1u << u;
        e0 += ax0; e1 += ax1; e2 += ax2;
      }
    }
    if (mask) out.x |= (unsigned)t | (mask << 24);
  }
  const unsigned cm = __ballot_sync(0xffffffffu, mask != 0u);
  if (cm) {
    if (mask) w->q2[q2n + __popc(cm & ((1u << lane) - 1u))] = out;
    q2n += __popc(cm);
    __syncwarp();
    if (q2n >= 32) { q2n -= 32; raster_depth<WITH_ID>(c, w, q2n, 32, lane); __syncwarp(); }
  }
  return q2n;
}

template <bool WITH_ID, bool BINNED, bool GTAB>
__global__ void __launch_bounds__(896, 1) vis_raster_kernel(int nf, int nv, int R, int band_rows, int n_bands, int n_units,
    int tail_first, int split,
    const float4* __restrict__ v_posed, const unsigned long long* __restrict__ faces_packed, const float* __restrict__ dirs,
    const float* __restrict__ window, unsigned* __restrict__ zmap, int* __restrict__ idmap,
    unsigned* __restrict__ vbits_raw, int words, int cull, float4* __restrict__ frames_out, float bias_texels, float bias_world,
    float slope_max, unsigned* __restrict__ bins, int band_magic, unsigned* __restrict__ sxy_scratch) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  __shared__ int s_next;
  __shared__ unsigned s_bin_cnt[RAST_MAX_BANDS];
  __shared__ float s_zf[8];
  // layout: [RasterWarp x warps][map band_rows*R*(4|8)][sXY nv*4][sZ nv*4][svert (WITH_ID)]
  const int nthreads = blockDim.x, nwarps = nthreads >> 5;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  RasterWarp* w = reinterpret_cast<RasterWarp*>(smem_raw) + warp;
  unsigned char* mp = smem_raw + (size_t)nwarps * sizeof(RasterWarp);
  unsigned* sz32 = reinterpret_cast<unsigned*>(mp);
  unsigned long long* sz64 = reinterpret_cast<unsigned long long*>(mp);
  const size_t map_bytes = (((size_t)band_rows * R * (WITH_ID ? 8 : 4)) + 15) & ~(size_t)15;
  // snapped vertex coordinates: shared memory, or (large meshes) this CTA's slice of an L2-resident scratch buffer
  // (a compile-time choice: with a run-time one every gather of the common shared-memory case becomes a generic load)
  unsigned* sXY = GTAB ? sxy_scratch + (size_t)blockIdx.x * nv : reinterpret_cast<unsigned*>(mp + map_bytes);
  float* sZ = GTAB ? nullptr : reinterpret_cast<float*>(mp + map_bytes) + nv;      // vertex depths, beside the table in shared memory
  unsigned* svert = reinterpret_cast<unsigned*>(mp + map_bytes) + (GTAB ? 0 : 2 * nv);
  const int nv_words = (nv + 31) >> 5;
  constexpr bool FUSED_CLEAR = !WITH_ID && !BINNED;   // a depth-only whole map is cleared by the pass that writes it out

  // Work slots: units [0, tail_first) one CTA each; the units of the last, partial round of the persistent grid are cut
  // into `split` triangle ranges so that every SM works in that round too; their CTAs merge into the (pre-cleared)
  // global map with atomicMin.
  const int n_slots = tail_first + (n_units - tail_first) * split;
  for (int slot = blockIdx.x; slot < n_slots; slot += gridDim.x) {
    int unit = slot, t_begin = 0, t_end = nf;
    const bool shared_unit = slot >= tail_first && split > 1;
    if (shared_unit) {
      const int q = slot - tail_first, part = q % split;
      unit = tail_first + q / split;
      t_begin = (int)((long long)nf * part / split); t_end = (int)((long long)nf * (part + 1) / split);
    }
    // Maps that fit shared memory whole: a unit is a direction.  Larger maps (256^2) are cut into bands of rows, and a
    // unit is still ONE direction: its triangles are walked and boxed once and BINNED by band (triangle ids in an
    // L2-resident scratch list per band), then the bands are rasterised one after the other from their lists -- the
    // fetch / gather / box work is not repeated per band (it was: 7x the time for 4x the work at config 2).
    const bool binned = BINNED;
    const int k = binned ? unit : unit / n_bands;
    int band = binned ? 0 : unit - k * n_bands;
    int row0 = band * band_rows, rows = binned ? R : min(band_rows, R - row0);
    int npix = min(band_rows, R - row0) * R;
    {                                                       // frame and window live only through phase A
    const WinConst W = make_win(window, R);
    const LightFrame F = make_frame(dirs + 3 * k, W);
    if (binned && threadIdx.x < n_bands) s_bin_cnt[threadIdx.x] = 0u;
    if (threadIdx.x == 0) {
      s_next = t_begin;
      s_zf[0] = W.cx; s_zf[1] = W.cy; s_zf[2] = W.cz; s_zf[3] = F.wn[0]; s_zf[4] = F.wn[1]; s_zf[5] = F.wn[2];
      // the pre-scaled frame and the depth-test constants for the fused depth-test + shading kernel (vis_shade_kernels.cu,
      // a FAST file): written HERE, by the EXACT file's make_win / make_frame -- layout as light_frames_kernel below
      if (frames_out && band == 0 && t_begin == 0) {
        // A = (us.xyz, vs.x)  B = (vs.yz, wn.xy)  C = (wn.z, w.xyz): the layout the fused kernel keeps in shared memory, so that
        // its CTAs stage the table with one bulk copy
        frames_out[2 + 3 * k] = make_float4(F.us[0], F.us[1], F.us[2], F.vs[0]);
        frames_out[2 + 3 * k + 1] = make_float4(F.vs[1], F.vs[2], F.wn[0], F.wn[1]);
        frames_out[2 + 3 * k + 2] = make_float4(F.wn[2], F.w[0], F.w[1], F.w[2]);
        if (k == 0) {
          frames_out[0] = make_float4(W.cx, W.cy, W.cz, W.hR);
          frames_out[1] = make_float4(bias_texels / (float)R, bias_world * W.inv2r, slope_max, (float)R);
        }
      }
    }
    // clear the band (FUSED_CLEAR: only before the CTA's first unit -- the write-out below leaves the map cleared)
    if (WITH_ID) { for (int p = threadIdx.x; p < npix; p += nthreads) sz64[p] = ~0ull; }
    else if (!FUSED_CLEAR || slot == (int)blockIdx.x) {
      uint4* m4 = reinterpret_cast<uint4*>(sz32);
      const uint4 ones = make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu);
      for (int p = threadIdx.x; p < (npix + 3) >> 2; p += nthreads) m4[p] = ones;
    }
    if (WITH_ID && vbits_raw) for (int p = threadIdx.x; p < nv_words; p += nthreads) svert[p] = 0u;
    // A. project every vertex once
    for (int v = threadIdx.x; v < nv; v += nthreads) {
      const float4 a = __ldg(v_posed + v);
      float px, py;
      light_project_xy(a.x - W.cx, a.y - W.cy, a.z - W.cz, W, F, px, py);
      const int X = min(max(__float2int_rn(px * 256.0f), 0), 65535), Y = min(max(__float2int_rn(py * 256.0f), 0), 65535);
      sXY[v] = (unsigned)X | ((unsigned)Y << 16);
      if (!GTAB) sZ[v] = __fmaf_rn(F.wn[2], a.z - W.cz, __fmaf_rn(F.wn[1], a.y - W.cy, __fmaf_rn(F.wn[0], a.x - W.cx, 0.5f)));
    }
    }
    __syncthreads();

    RasterCtx c;
    c.R = R; c.row0 = row0; c.rows = rows; c.sXY = sXY; c.v_posed = v_posed; c.faces_packed = faces_packed;
    c.sz32 = sz32; c.sz64 = sz64; c.zf = s_zf; c.sZ = sZ;
    // B1. triangles: one per lane, 32 per warp fetched dynamically; non-empty boxes queued
    int qn = 0, qsn = 0, q2n = 0;                           // warp-uniform queue fills
    // Binned maps (B1 only fills the band lists): the NEXT batch is drawn from the counter and its faces are requested before the
    // current batch is worked on, so the counter's and the L2's round trips run beside the box tests (config 2: 626 -> 604 us).
    // Where B1 feeds the sampling rounds directly the two extra live registers spill (config 1: 133 -> 137 us): not there.
    int base_nxt = 0;
    unsigned long long face_nxt = 0ull;
    if (BINNED) {
      if (lane == 0) base_nxt = atomicAdd(&s_next, 32);
      base_nxt = __shfl_sync(0xffffffffu, base_nxt, 0);
      face_nxt = (base_nxt + lane < t_end) ? __ldg(faces_packed + base_nxt + lane) : 0ull;
    }
    for (;;) {
      int base = 0;
      unsigned long long face_cur = 0ull;
      if (BINNED) {
        base = base_nxt;
        if (base >= t_end) break;
        face_cur = face_nxt;
        if (lane == 0) base_nxt = atomicAdd(&s_next, 32);
        base_nxt = __shfl_sync(0xffffffffu, base_nxt, 0);
        face_nxt = (base_nxt + lane < t_end) ? __ldg(faces_packed + base_nxt + lane) : 0ull;
      } else {
        if (lane == 0) base = atomicAdd(&s_next, 32);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base >= t_end) break;
        if (base + lane < t_end) face_cur = __ldg(faces_packed + base + lane);
      }
      {
        const int t = base + lane;
        bool ne = false, narrow = false;
        int ia = 0, ja = 0, bw = 0, bh = 0;
        if (t < t_end) {
          int i0, i1, i2;
          face_unpack(face_cur, i0, i1, i2);
          const unsigned Q0 = sXY[i0], Q1 = sXY[i1], Q2 = sXY[i2];
          ne = tri_box(Q0, Q1, Q2, R, row0, rows, ia, ja, bw, bh, narrow) > 0;
          if (cull && ne) {                               // reading A36: negative snapped area = facing away from the light
            const long long ax = (int)(Q1 & 0xffff) - (int)(Q0 & 0xffff), ay = (int)(Q1 >> 16) - (int)(Q0 >> 16);
            const long long bx = (int)(Q2 & 0xffff) - (int)(Q0 & 0xffff), by = (int)(Q2 >> 16) - (int)(Q0 >> 16);
            ne = ax * by - ay * bx > 0;
          }
        }
        if (binned) {                                     // push the triangle into the list of every band its box touches
          if (ne) {
            const int jb2 = ja + bh - 1;
            const int blo = (ja * band_magic) >> 16, bhi = (jb2 * band_magic) >> 16;
            // bit 31: the whole box is one run (then so is its part in any band)
            const unsigned entry = (unsigned)t | ((narrow && min(bw, bh) == 1 && max(bw, bh) <= RAST_SEGW) ? 0x80000000u : 0u);
            for (int b = blo; b <= bhi; ++b) bins[((size_t)blockIdx.x * n_bands + b) * (size_t)nf + atomicAdd(&s_bin_cnt[b], 1u)] = entry;
          }
          continue;
        }
        // two queues: boxes that are one run (sampled by their own lane, raster_single) and the rest (runs dealt out, raster_round)
        const bool single = ne && narrow && min(bw, bh) == 1 && max(bw, bh) <= RAST_SEGW;
        const unsigned ms = __ballot_sync(0xffffffffu, single), m = __ballot_sync(0xffffffffu, ne && !single);
        if (ms) {
          if (single) w->q1s[qsn + __popc(ms & ((1u << lane) - 1u))] = t;
          qsn += __popc(ms);
          __syncwarp();
          if (qsn >= 32) {
            qsn -= 32;
            q2n = raster_single<WITH_ID>(c, w, qsn, 32, lane, q2n);
            __syncwarp();
          }
        }
        if (m) {
          if (ne && !single) w->q1[qn + __popc(m & ((1u << lane) - 1u))] = t;
          qn += __popc(m);
          __syncwarp();
          if (qn >= 32) {
            qn -= 32;
            q2n = raster_round<WITH_ID>(c, w, qn, 32, lane, q2n);
            __syncwarp();
          }
        }
      }
    }
    // leftovers: when both queues fit one round, the single-run boxes go through the run dealing too (raster_round builds the
    // same entry for them) -- one partial round instead of two (the leftovers are a tenth of a unit's time, profiles/r02_raster.md)
    if (qsn && qn && qsn + qn <= 32) { if (lane < qsn) w->q1[qn + lane] = w->q1s[lane]; qn += qsn; qsn = 0; __syncwarp(); }
    if (qsn) { q2n = raster_single<WITH_ID>(c, w, 0, qsn, lane, q2n); __syncwarp(); }
    if (qn) { q2n = raster_round<WITH_ID>(c, w, 0, qn, lane, q2n); __syncwarp(); }
    if (q2n) raster_depth<WITH_ID>(c, w, 0, q2n, lane);
    __syncthreads();

    for (band = 0; band < (binned ? n_bands : 1); ++band) {
    if (binned) {
      // rasterise band `band` from its triangle list: 32 listed triangles per round, every lane busy from the start
      row0 = band * band_rows; rows = min(band_rows, R - row0); npix = rows * R;
      c.row0 = row0; c.rows = rows;
      if (band > 0) {                                        // band 0 was cleared before phase A
        if (WITH_ID) { for (int p = threadIdx.x; p < npix; p += nthreads) sz64[p] = ~0ull; }
        else {
          uint4* m4 = reinterpret_cast<uint4*>(sz32);
          const uint4 ones = make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu);
          for (int p = threadIdx.x; p < (npix + 3) >> 2; p += nthreads) m4[p] = ones;
        }
      }
      if (threadIdx.x == 0) s_next = 0;
      __syncthreads();
      const int nlist = (int)s_bin_cnt[band];
      const unsigned* list = bins + ((size_t)blockIdx.x * n_bands + band) * (size_t)nf;
      int q2b = 0, qb = 0, qsb = 0;
      for (;;) {
        int base = 0;
        if (lane == 0) base = atomicAdd(&s_next, 32);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base >= nlist) break;
        const int cnt = min(32, nlist - base);
        const unsigned entry = lane < cnt ? __ldcg(list + base + lane) : 0u;
        const bool single = lane < cnt && (entry >> 31), multi = lane < cnt && !(entry >> 31);
        const unsigned ms = __ballot_sync(0xffffffffu, single), mm = __ballot_sync(0xffffffffu, multi);
        if (single) w->q1s[qsb + __popc(ms & ((1u << lane) - 1u))] = (int)(entry & 0xffffffu);
        if (multi) w->q1[qb + __popc(mm & ((1u << lane) - 1u))] = (int)(entry & 0xffffffu);
        qsb += __popc(ms); qb += __popc(mm);
        __syncwarp();
        if (qsb >= 32) { qsb -= 32; q2b = raster_single<WITH_ID>(c, w, qsb, 32, lane, q2b); __syncwarp(); }
        if (qb >= 32) { qb -= 32; q2b = raster_round<WITH_ID>(c, w, qb, 32, lane, q2b); __syncwarp(); }
      }
      if (qsb && qb && qsb + qb <= 32) { if (lane < qsb) w->q1[qb + lane] = w->q1s[lane]; qb += qsb; qsb = 0; __syncwarp(); }
      if (qsb) { q2b = raster_single<WITH_ID>(c, w, 0, qsb, lane, q2b); __syncwarp(); }
      if (qb) { q2b = raster_round<WITH_ID>(c, w, 0, qb, lane, q2b); __syncwarp(); }
      if (q2b) raster_depth<WITH_ID>(c, w, 0, q2b, lane);
      __syncthreads();
    }

    // write the band out
    const size_t gbase = ((size_t)k * R + row0) * R;
    if (WITH_ID) {
      for (int p = threadIdx.x; p < npix; p += nthreads) {
        const unsigned long long key = sz64[p];
        zmap[gbase + p] = (unsigned)(key >> 32);
        const int tri = (key == ~0ull) ? -1 : (int)(unsigned)(key & 0xffffffffu);
        idmap[gbase + p] = tri;
        if (vbits_raw && tri >= 0) {                      // a triangle that appears marks its 3 vertices
          int v0, v1, v2;
          face_unpack(__ldg(faces_packed + tri), v0, v1, v2);
          atomicOr(svert + (v0 >> 5), 1u << (v0 & 31));
          atomicOr(svert + (v1 >> 5), 1u << (v1 & 31));
          atomicOr(svert + (v2 >> 5), 1u << (v2 & 31));
        }
      }
      if (vbits_raw && (!binned || band == n_bands - 1)) {
        __syncthreads();
        const unsigned bit = 1u << (k & 31);
        for (int wd = threadIdx.x; wd < nv_words; wd += nthreads) {
          unsigned m = svert[wd];
          while (m) {
            const int b = __ffs(m) - 1; m &= m - 1;
            const int vtx = wd * 32 + b;
            if (vtx < nv) atomicOr(vbits_raw + (size_t)vtx * words + (k >> 5), bit);
          }
        }
      }
    } else if (shared_unit) {
      for (int p = threadIdx.x; p < npix; p += nthreads) {
        const unsigned v = sz32[p];
        if (v != 0xffffffffu) { atomicMin(zmap + gbase + p, v); if (FUSED_CLEAR) sz32[p] = 0xffffffffu; }
      }
    } else if ((R & 3) == 0) {
      uint4* m4 = reinterpret_cast<uint4*>(sz32);
      uint4* g4 = reinterpret_cast<uint4*>(zmap + gbase);
      const uint4 ones = make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu);
      for (int p = threadIdx.x; p < npix >> 2; p += nthreads) { g4[p] = m4[p]; if (FUSED_CLEAR) m4[p] = ones; }
    } else {
      for (int p = threadIdx.x; p < npix; p += nthreads) { zmap[gbase + p] = sz32[p]; if (FUSED_CLEAR) sz32[p] = 0xffffffffu; }
    }
    // The map and the vertex table are reused by the next band / unit.  FUSED_CLEAR: every thread has just cleared the texels it
    // wrote out, and the next unit's head and phase A touch nothing this pass reads (every warp is past the barrier that ends
    // phase B); the barrier after phase A orders the clearing before the next atomicMin -- one barrier and one pass fewer per unit
    if (!FUSED_CLEAR) __syncthreads();
    }
  }
}

// shared-memory plan: picks the CTA size (896 / 448 / 224 threads) that minimises bands / warps; returns bytes.
// 896 threads = 28 warps at 72 registers: the kernel needs 72 without spilling, and 1,024 threads cap it at 64 (measured at
// config 1 / 2 / 4: 1,024 threads 133.4 / 603 / 1,141 us, 896: 131.7 / 597 / 1,132 us, 768 at 80 registers: 135 / 630 / 1,184 us,
// 640 at 90: 145 / 652 / 1,221 us).
// *sxy_global = 1: the 4-byte-per-vertex table of snapped coordinates does not fit beside a useful band of the map (meshes
// beyond about 45k vertices) and lives in an L2-resident scratch buffer instead -- same kernel, slower gathers.
static size_t raster_plan(int res, int with_id, int n_verts, bool table_in_smem, int* band_rows, int* threads) {
  const size_t budget = 227 * 1024 - 512;               // static shared memory (counters, band list sizes) counts against the 227 KB
  const size_t per_row = (size_t)res * (with_id ? 8 : 4);
  size_t best = 0; double best_score = 1e30;
  *band_rows = 0; *threads = 0;
  for (int th = 896; th >= 224; th >>= 1) {
    const size_t fixed = (size_t)(th / 32) * sizeof(RasterWarp) + (table_in_smem ? (size_t)n_verts * 8 : 0) +
                         (with_id ? (size_t)((n_verts + 31) / 32) * 4 : 0) + 32;
    if (fixed + per_row > budget) continue;
    int rows = (int)((budget - fixed) / per_row);
    if (rows > res) rows = res;
    int bands = (res + rows - 1) / rows;
    rows = (res + bands - 1) / bands;                                 // even bands
    const double score = (double)bands / (double)(th / 32);
    if (score < best_score) {
      best_score = score; *band_rows = rows; *threads = th;
      best = fixed + ((per_row * rows + 15) & ~(size_t)15);
    }
  }
  return best;
}

size_t rga_vis_raster_plan(int res, int with_id, int n_verts, int* band_rows, int* threads, int* sxy_global) {
  // Two places for the table of snapped vertex coordinates: shared memory (fast gathers, but it competes with the map and the
  // warps' working sets) or an L2-resident scratch slice per CTA.  More warps win: at config 2 (27.5k vertices, 110 KB table)
  // the shared-memory plan leaves room for 16 warps only and the rasteriser idles on latency -- 860 us; with the table in L2
  // and 32 warps 615 us (profiles/r02_raster.md).  Equal warps: shared memory.
  int rows_s = 0, th_s = 0, rows_g = 0, th_g = 0;
  const size_t b_s = raster_plan(res, with_id, n_verts, true, &rows_s, &th_s);
  const size_t b_g = raster_plan(res, with_id, n_verts, false, &rows_g, &th_g);
  const int bands_s = rows_s > 0 ? (res + rows_s - 1) / rows_s : 1 << 30;
  const bool use_global = b_s == 0 || bands_s > 16 || th_g > th_s;
  *sxy_global = use_global ? 1 : 0;
  *band_rows = use_global ? rows_g : rows_s; *threads = use_global ? th_g : th_s;
  return use_global ? b_g : b_s;
}

size_t rga_vis_raster_smem(int res, int with_id, int n_verts, int* band_rows, int* threads) {
  int g = 0;
  return rga_vis_raster_plan(res, with_id, n_verts, band_rows, threads, &g);
}

cudaError_t rga_launch_vis_raster(rga_avatar* av, const rga_vis_params* p, cudaStream_t s) {
  const bool with_id = p->mode == 1 || p->keep_maps;
  int band_rows = 0, threads = 0, sxy_global = 0;
  const size_t smem = rga_vis_raster_plan(p->res, with_id, av->n_verts, &band_rows, &threads, &sxy_global);
  if (band_rows < 1 || (sxy_global && !av->rast_sxy)) return cudaErrorInvalidConfiguration;
  const int n_bands = (p->res + band_rows - 1) / band_rows;
  const int words = (p->n_dirs + 31) / 32;
  // a map cut into bands: one unit per direction, triangles binned by band (needs the scratch lists sized at load)
  const bool binned = n_bands > 1;
  if (binned && (n_bands > RAST_MAX_BANDS || !av->rast_bins || n_bands > av->rast_bins_bands)) return cudaErrorInvalidConfiguration;
  const int n_units = binned ? p->n_dirs : p->n_dirs * n_bands;
  // persistent grid, one CTA per SM.  (One CTA per work slot instead, so that SMs are handed back between directions and the
  // second stream's kernels get in earlier, was measured: the splat preparation then finishes 110 us earlier, the frame is
  // not faster -- 2,934 against 2,966 frames/s: the streams share the same SMs either way.)
  const int grid_sm = n_units < av->num_sms ? n_units : av->num_sms;
  unsigned* raw = (with_id && p->mode == 1) ? av->vbits_raw : nullptr;
  if (raw) { const cudaError_t e = cudaMemsetAsync(raw, 0, (size_t)av->n_verts * words * 4, s); if (e != cudaSuccess) return e; }
  // last, partial round of the persistent grid: cut its units into triangle ranges (depth-only maps merge with atomicMin)
  int tail_first = n_units, split = 1;
  const int rem = n_units > grid_sm ? n_units % grid_sm : 0;
  int best_split = 1;
  {
    // the split (1..4) that leaves the shortest last round: ceil(rem * s / grid) / s
    double best = 1.0;
    for (int sp = 2; sp <= 4; ++sp) {
      const double t = (double)((rem * sp + grid_sm - 1) / grid_sm) / sp;
      if (t < best - 1e-9) { best = t; best_split = sp; }
    }
  }
  if (rem > 0 && !with_id && best_split >= 2) {
    split = best_split;
    tail_first = n_units - rem;
    const size_t unit_px = (size_t)band_rows * p->res;       // bands are even; the last may be shorter (covered anyway)
    const size_t first_px = binned ? (size_t)tail_first * p->res * p->res      // a binned unit is a whole direction
                                   : (size_t)(tail_first / n_bands) * p->res * p->res + (size_t)(tail_first % n_bands) * unit_px;
    const cudaError_t e = cudaMemsetAsync(av->zmap + first_px, 0xff, ((size_t)p->n_dirs * p->res * p->res - first_px) * 4, s);
    if (e != cudaSuccess) return e;
  }
  const int grid = grid_sm;
  const int band_magic = (65536 + band_rows - 1) / band_rows;   // (row * magic) >> 16 == row / band_rows for row < 256
#define RAST_ARGS av->n_faces, av->n_verts, p->res, band_rows, n_bands, n_units, tail_first, split, av->v_posed, av->faces_packed, p->dirs, av->window, \
    av->zmap, av->idmap, raw, words, p->cull_backfaces != 0, reinterpret_cast<float4*>(av->frames), p->depth_bias_texels, p->depth_bias_world, \
    p->slope_max, binned ? av->rast_bins : nullptr, band_magic, sxy_global ? av->rast_sxy : nullptr
#define RAST_LAUNCH(ID, BIN, GT) vis_raster_kernel<ID, BIN, GT><<<grid, threads, smem, s>>>(RAST_ARGS)
  if (sxy_global) {
    if (with_id) { if (binned) RAST_LAUNCH(true, true, true); else RAST_LAUNCH(true, false, true); }
    else { if (binned) RAST_LAUNCH(false, true, true); else RAST_LAUNCH(false, false, true); }
  } else {
    if (with_id) { if (binned) RAST_LAUNCH(true, true, false); else RAST_LAUNCH(true, false, false); }
    else { if (binned) RAST_LAUNCH(false, true, false); else RAST_LAUNCH(false, false, false); }
  }
  av->launches += 1;
  rga_prof_mark(av, "vis_raster", s);
  return cudaGetLastError();
}

// scratch for the triangle lists of banded maps: bands needed at the declared maximum resolution (0: the map fits whole)
int rga_vis_raster_max_bands(int max_res, int n_verts) {
  int rows = 0, th = 0, worst = 1;
  for (int with_id = 0; with_id < 2; ++with_id)
    for (int res = 1; res <= max_res; ++res) {               // the planner is cheap; band counts are not monotone in res
      rga_vis_raster_smem(res, with_id, n_verts, &rows, &th);
      if (rows < 1) continue;
      const int b = (res + rows - 1) / rows;
      if (b > worst) worst = b;
    }
  return worst > 1 ? worst : 0;
}

// does any map size up to max_res need the vertex table in global memory?
int rga_vis_raster_needs_global_table(int max_res, int n_verts) {
  int rows = 0, th = 0, g = 0;
  for (int with_id = 0; with_id < 2; ++with_id)
    for (int res = 1; res <= max_res; ++res) { rga_vis_raster_plan(res, with_id, n_verts, &rows, &th, &g); if (g) return 1; }
  return 0;
}

// Pre-scaled light frames and depth-test constants for the fused depth-test + shading kernel (vis_shade_kernels.cu, a FAST
// file): computed HERE, in the EXACT file, by the same make_win / make_frame as every other visibility kernel.
// out: float4[2 + 3K]: (cx, cy, cz, hR) (bias_texels / R, bias_world * inv2r, slope_max, R) then per direction
// (us.xyz, vs.x) (vs.yz, wn.xy) (wn.z, w.xyz).
__global__ void light_frames_kernel(int K, int R, const float* __restrict__ dirs, const float* __restrict__ window, float bias_texels,
                                    float bias_world, float slope_max, float4* __restrict__ out) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const WinConst W = make_win(window, R);
  if (k == 0) {
    out[0] = make_float4(W.cx, W.cy, W.cz, W.hR);
    out[1] = make_float4(bias_texels / (float)R, bias_world * W.inv2r, slope_max, (float)R);
  }
  if (k >= K) return;
  const LightFrame f = make_frame(dirs + 3 * k, W);
  out[2 + 3 * k] = make_float4(f.us[0], f.us[1], f.us[2], f.vs[0]);
  out[2 + 3 * k + 1] = make_float4(f.vs[1], f.vs[2], f.wn[0], f.wn[1]);
  out[2 + 3 * k + 2] = make_float4(f.wn[2], f.w[0], f.w[1], f.w[2]);
}

cudaError_t rga_launch_light_frames(rga_avatar* av, const rga_vis_params* p, cudaStream_t s) {
  light_frames_kernel<<<(p->n_dirs + 127) / 128, 128, 0, s>>>(p->n_dirs, p->res, p->dirs, av->window, p->depth_bias_texels, p->depth_bias_world,
                                                             p->slope_max, reinterpret_cast<float4*>(av->frames));
  rga_prof_mark(av, "light_frames", s);
  av->launches += 1;
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------ H4a
// Shadow-map test, Gaussian-major: one thread per Gaussian keeps its position/normal in registers and walks all
// directions; neighbouring (Morton-ordered) Gaussians hit neighbouring texels, so the depth-map gathers stay in
// L1/L2.  32 directions are packed into one output word.  The slope factor tau (sqrt and divide) is only evaluated when
// the two monotone bounds beta(1) <= beta(tau) <= beta(slope_max) do not already decide the comparison.
#ifndef DT_THREADS
#define DT_THREADS 128
#endif
#ifndef DT_UNROLL
#define DT_UNROLL 4
#endif
#define RGA_STR(x) #x
#define RGA_UNROLL(n) _Pragma(RGA_STR(unroll n))
#ifndef DT_MAXPARTS
#define DT_MAXPARTS 16
#endif
__global__ void __launch_bounds__(DT_THREADS) vis_depth_test_kernel(int ng, int K, int R, const float4* __restrict__ g_posed,
    const float4* __restrict__ g_nposed, const float* __restrict__ dirs, const float* __restrict__ window,
    const unsigned* __restrict__ zmap, float bias_texels, float bias_world, float slope_max, int words_per_part,
    unsigned* __restrict__ visbits, int cull, float3 cam) {
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
  if (cull) {
    // rga_render_frame knows the camera: a Gaussian that faces away from it gets opacity 0, its colour is
    // never splatted and shade_gaussians skips it by this same test, so its visibility is never read -- its words are
    // written as zeros and the CTA's remaining Gaussians are compacted onto its first threads (whole warps retire)
    __shared__ int s_list[DT_THREADS];
    __shared__ int s_wcnt[DT_THREADS / 32];
    bool keep = false;
    if (g < ng) {
      const float4 x = g_posed[g], n = g_nposed[g];
      const float wx = cam.x - x.x, wy = cam.y - x.y, wz = cam.z - x.z;
      keep = !(n.x * wx + n.y * wy + n.z * wz < -1e-4f * sqrtf(wx * wx + wy * wy + wz * wz));
      if (!keep) for (int wd = wd0; wd < wd1; ++wd) visbits[(size_t)g * words + wd] = 0u;
    }
    const unsigned bal = __ballot_sync(0xffffffffu, keep);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) s_wcnt[warp] = __popc(bal);
    __syncthreads();
    int base = 0, total = 0;
    for (int w = 0; w < DT_THREADS / 32; ++w) { const int c = s_wcnt[w]; if (w < warp) base += c; total += c; }
    if (keep) s_list[base + __popc(bal & ((1u << lane) - 1u))] = g;
    __syncthreads();
    if ((int)threadIdx.x >= total) return;
    g = s_list[threadIdx.x];
  }
  if (g >= ng) return;
  const float bt = bias_texels / (float)R, bw = bias_world * W.inv2r;
  const float beta_lo = bt * 1.0f + bw, beta_hi = bt * slope_max + bw;
  const bool bounds_ok = bt >= 0.f && slope_max >= 1.0f;
  const float INF = __int_as_float(0x7f800000);
  const float blo = bounds_ok ? beta_lo : -INF, bhi = bounds_ok ? beta_hi : INF;      // no shortcut unless beta is monotone
  const float margin = 1e-6f + 1e-5f * fabsf(bt) * fmaxf(slope_max, 1.0f);             // >> error of the approximate threshold
  const float Rm1 = (float)(R - 1), Rf = (float)R;
  const float4 x = g_posed[g], n = g_nposed[g];
  const float dx = x.x - W.cx, dy = x.y - W.cy, dz = x.z - W.cz;
  const size_t RR = (size_t)R * R;
  for (int wd = wd0; wd < wd1; ++wd) {
    unsigned bits = 0;
    const int kend = min(32, K - wd * 32);
    const unsigned* zk = zmap + (size_t)wd * 32 * RR;
    const float4* fk = sF4 + 3 * (wd * 32 - k0);
    RGA_UNROLL(DT_UNROLL)
    for (int b = 0; b < kend; ++b) {
      const float4 fu = fk[3 * b], fv = fk[3 * b + 1], fw = fk[3 * b + 2];
      const float px = __fmaf_rn(fu.z, dz, __fmaf_rn(fu.y, dy, __fmaf_rn(fu.x, dx, W.hR)));
      const float py = __fmaf_rn(fv.z, dz, __fmaf_rn(fv.y, dy, __fmaf_rn(fv.x, dx, W.hR)));
      const float z = __fmaf_rn(fw.z, dz, __fmaf_rn(fw.y, dy, __fmaf_rn(fw.x, dx, 0.5f)));
      // floor-then-clamp of the contract == clamp-then-floor for every finite px.  floor without the XU pipe: adding
      // 2^23 rounding DOWN leaves floor(x) in the mantissa (0 <= x < 2^23); iy R + ix is then formed exactly in fp32
      const float fxm = __fadd_rd(fminf(fmaxf(px, 0.0f), Rm1), 8388608.0f);
      const float fym = __fadd_rd(fminf(fmaxf(py, 0.0f), Rm1), 8388608.0f);
      const int idx = __float_as_int(__fmaf_rn(__fadd_rn(fym, -8388608.0f), Rf, fxm)) & 0x7fffff;
      const float zm = __uint_as_float(__ldg(zk + (size_t)b * RR + idx));      // empty texel = 0xffffffff = NaN
      // visible iff z <= zm + beta(tau); NaN compares false, so "not (z > ...)" also covers the empty texel.
      // beta is monotone in tau in [1, slope_max]: most tests are decided by the two ends without evaluating tau.
      bool vis = !(z > __fadd_rn(zm, blo));
      if (!vis && !(z > __fadd_rn(zm, bhi))) {
        // in between: an approximate tau (MUFU sqrt / rcp, ~1e-6 relative) decides unless z is within `margin` of the
        // threshold; only then the exact IEEE sqrt and divide of the contract are evaluated -- the bit is the same
        const float cs = __fadd_rn(__fadd_rn(__fmul_rn(n.x, fu.w), __fmul_rn(n.y, fv.w)), __fmul_rn(n.z, fw.w));
        float tau = slope_max;
        if (cs > 0.0f) {
          float sq, rc; const float s2 = fmaxf(__fmaf_rn(-cs, cs, 1.0f), 0.0f);
          asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(sq) : "f"(s2));
          asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rc) : "f"(cs));
          tau = fminf(fmaxf(__fmul_rn(sq, rc), 1.0f), slope_max);
        }
        const float dlt = __fadd_rn(z, -__fadd_rn(zm, __fmaf_rn(bt, tau, bw)));
        if (fabsf(dlt) > margin) vis = dlt < 0.0f;
        else {
          float te = slope_max;
          if (cs > 0.0f) {
            const float s2 = fmaxf(1.0f - cs * cs, 0.0f);
            te = sqrtf(s2) / cs;
            te = fminf(fmaxf(te, 1.0f), slope_max);
          }
          vis = z <= zm + (bt * te + bw);
        }
      }
      bits |= (vis ? 1u : 0u) << b;
    }
    visbits[(size_t)g * words + wd] = bits;
  }
}

cudaError_t rga_launch_vis_depth_test(rga_avatar* av, const rga_vis_params* p, const float* cull_cam, cudaStream_t s) {
  // directions are split over blockIdx.y so that small avatars still fill the machine (100k Gaussians alone give
  // 676 threads per SM); neighbouring threads stay neighbouring Gaussians, whose texel gathers coalesce in L1
  int words = (p->n_dirs + 31) / 32;
  // (16 parts keep enough warps in flight for the texel gathers: with rga_render_frame's camera cull, where about half of
  // the Gaussians retire at once, 88 us with 4 parts and 73 us with 16 at config 1; without the cull 118 -> 108 us)
  const int maxparts = DT_MAXPARTS;
  int parts = words < maxparts ? words : maxparts;
  int wpp = (words + parts - 1) / parts;
  parts = (words + wpp - 1) / wpp;
  dim3 grid((av->n_gauss + DT_THREADS - 1) / DT_THREADS, parts);
  vis_depth_test_kernel<<<grid, DT_THREADS, (size_t)wpp * 32 * 3 * sizeof(float4), s>>>(
      av->n_gauss, p->n_dirs, p->res, av->g_posed, av->g_nposed, p->dirs, av->window, av->zmap, p->depth_bias_texels,
      p->depth_bias_world, p->slope_max, wpp, av->visbits, cull_cam != nullptr,
      cull_cam ? make_float3(cull_cam[0], cull_cam[1], cull_cam[2]) : make_float3(0.f, 0.f, 0.f));
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
  const int mx = 227 * 1024 - 512;            // the static counters count against the 227 KB block limit
  cudaError_t e = cudaSuccess;
#define RAST_ATTR(ID, BIN, GT) if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_raster_kernel<ID, BIN, GT>, cudaFuncAttributeMaxDynamicSharedMemorySize, mx)
  RAST_ATTR(true, false, false); RAST_ATTR(false, false, false); RAST_ATTR(true, true, false); RAST_ATTR(false, true, false);
  RAST_ATTR(true, false, true); RAST_ATTR(false, false, true); RAST_ATTR(true, true, true); RAST_ATTR(false, true, true);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(vis_depth_test_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
  return (int)e;
}
