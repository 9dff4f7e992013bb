// H6 projection + culling (PAPER.md:101 back-face rule; "the Gaussian rasterizer of 3DGS" -> ref [8];
// DESIGN.md readings A8, A18, A21).  EXACT file (-fmad=false): tile rects and sort keys are integer outputs of this
// arithmetic, so the operation order is the one fixed in DESIGN.md "Arithmetic contract".
// Also accumulates the per-tile histogram (the tile digit of the H8 sort).
#include "rga_internal.h"
#include "tile_scan.cuh"

struct CamK {
  float R[9], t[3], fx, fy, cx, cy, znear, limx, limy, C[3];
  int TX, TY;
};

__global__ void __launch_bounds__(256) project_kernel(int ng, CamK cam, const float4* __restrict__ g_posed,
    const float4* __restrict__ g_nposed, const float* __restrict__ g_cov, const float4* __restrict__ g_scale_op,
    float2* __restrict__ mu2d, float* __restrict__ depth, float4* __restrict__ conic_o, int4* __restrict__ rect,
    unsigned* __restrict__ touched, unsigned* tile_count, unsigned* __restrict__ done_counter, int ntiles, long long capacity,
    uint2* __restrict__ ranges, unsigned* __restrict__ cursor, unsigned* __restrict__ num_dup, unsigned* __restrict__ seg_off,
    unsigned* __restrict__ num_items, int* __restrict__ status) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned cnt = 0;
  if (g < ng) {
    float4 x = g_posed[g], n = g_nposed[g];
    float2 mu = make_float2(0.f, 0.f); float dep = 0.f; float4 co = make_float4(0.f, 0.f, 0.f, 0.f); int4 rc = make_int4(0, 0, 0, 0);
    const float* R = cam.R;
    float t0 = ((R[0] * x.x + R[1] * x.y) + R[2] * x.z) + cam.t[0];
    float t1 = ((R[3] * x.x + R[4] * x.y) + R[5] * x.z) + cam.t[1];
    float t2 = ((R[6] * x.x + R[7] * x.y) + R[8] * x.z) + cam.t[2];
    bool ok = t2 > cam.znear;
    if (ok) {
      float wx = cam.C[0] - x.x, wy = cam.C[1] - x.y, wz = cam.C[2] - x.z;
      ok = !(((n.x * wx + n.y * wy) + n.z * wz) < 0.0f);               // facing away -> opacity 0
    }
    if (ok) {
      float txz = fminf(cam.limx, fmaxf(-cam.limx, t0 / t2)) * t2;
      float tyz = fminf(cam.limy, fmaxf(-cam.limy, t1 / t2)) * t2;
      float J00 = cam.fx / t2, J02 = -(cam.fx * txz) / (t2 * t2), J11 = cam.fy / t2, J12 = -(cam.fy * tyz) / (t2 * t2);
      float T0[3], T1[3];
#pragma unroll
      for (int j = 0; j < 3; ++j) { T0[j] = J00 * R[j] + J02 * R[6 + j]; T1[j] = J11 * R[3 + j] + J12 * R[6 + j]; }
      const float* s = g_cov + 6 * (size_t)g;
      float S[9] = {s[0], s[1], s[2], s[1], s[3], s[4], s[2], s[4], s[5]};
      float V0[3], V1[3];
#pragma unroll
      for (int a = 0; a < 3; ++a) {
        V0[a] = (T0[0] * S[a] + T0[1] * S[3 + a]) + T0[2] * S[6 + a];
        V1[a] = (T1[0] * S[a] + T1[1] * S[3 + a]) + T1[2] * S[6 + a];
      }
      float c00 = ((V0[0] * T0[0] + V0[1] * T0[1]) + V0[2] * T0[2]) + 0.3f;
      float c01 = (V0[0] * T1[0] + V0[1] * T1[1]) + V0[2] * T1[2];
      float c11 = ((V1[0] * T1[0] + V1[1] * T1[1]) + V1[2] * T1[2]) + 0.3f;
      float det = c00 * c11 - c01 * c01;
      if (det > 0.0f) {
        float mid = 0.5f * (c00 + c11);
        float lam = mid + sqrtf(fmaxf(0.1f, mid * mid - det));
        float rad = ceilf(3.0f * sqrtf(lam));
        float mx = (cam.fx * t0) / t2 + cam.cx, my = (cam.fy * t1) / t2 + cam.cy;
        float fTX = (float)cam.TX, fTY = (float)cam.TY;
        int x0 = (int)fminf(fmaxf(floorf((mx - rad) / 16.0f), 0.0f), fTX);
        int x1 = (int)fminf(fmaxf(floorf(((mx + rad) + 15.0f) / 16.0f), 0.0f), fTX);
        int y0 = (int)fminf(fmaxf(floorf((my - rad) / 16.0f), 0.0f), fTY);
        int y1 = (int)fminf(fmaxf(floorf(((my + rad) + 15.0f) / 16.0f), 0.0f), fTY);
        int c = (x1 - x0) * (y1 - y0);
        if (c > 0) {
          cnt = (unsigned)c;
          mu = make_float2(mx, my); dep = t2;
          co = make_float4(c11 / det, -c01 / det, c00 / det, g_scale_op[g].w);
          rc = make_int4(x0, y0, x1, y1);
        }
      }
    }
    mu2d[g] = mu; depth[g] = dep; conic_o[g] = co; rect[g] = rc; touched[g] = cnt;
    // histogram of the tile digit (first pass of the (tile, depth) sort, sort_kernels.cu).  Gaussians are stored in
    // spatial order, so the lanes of a warp mostly hit the same few tiles: lanes with equal tile ids elect a leader
    // that adds their count once (the per-address serialisation of 1,300 single atomics on a hot tile was the cost)
    for (int y = rc.y; y < rc.w; ++y)
      for (int x = rc.x; x < rc.z; ++x) {
        const int tile = y * cam.TX + x;
        // (whatever subset of the warp happens to be converged here forms the peer sets: the histogram is the same for any grouping)
        const unsigned peers = __match_any_sync(__activemask(), tile);
        if ((int)(__ffs(peers) - 1) == (int)(threadIdx.x & 31)) atomicAdd(tile_count + tile, (unsigned)__popc(peers));
      }
  }
  // The CTA that finishes the histogram LAST scans it (tile_scan.cuh): ranges, cursors, D, segment offsets.  Every thread's
  // atomics precede its CTA's arrival (fence, barrier, one atomic on the arrival counter); the last arriver re-arms the counter.
  __shared__ bool s_last;
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) {
    s_last = atomicAdd(done_counter, 1u) == gridDim.x - 1u;
    if (s_last) *done_counter = 0u;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  rga_tile_scan<256>(ntiles, capacity, tile_count, ranges, cursor, num_dup, seg_off, num_items, status);
}

cudaError_t rga_launch_project(rga_avatar* av, const rga_camera* cam, cudaStream_t s) {
  CamK k;
  for (int i = 0; i < 9; ++i) k.R[i] = cam->R_wc[i];
  for (int i = 0; i < 3; ++i) k.t[i] = cam->t_wc[i];
  k.fx = cam->fx; k.fy = cam->fy; k.cx = cam->cx; k.cy = cam->cy; k.znear = cam->z_near;
  k.TX = (cam->width + RGA_TILE - 1) / RGA_TILE; k.TY = (cam->height + RGA_TILE - 1) / RGA_TILE;
  // host fp32 arithmetic below is plain IEEE single precision (no contraction: one operation per statement)
  volatile float w2 = 2.0f * cam->fx, h2 = 2.0f * cam->fy;
  volatile float tfx = (float)cam->width / w2, tfy = (float)cam->height / h2;
  volatile float lx = 1.3f * tfx, ly = 1.3f * tfy;
  k.limx = lx; k.limy = ly;
  for (int r = 0; r < 3; ++r) {                                           // camera centre C = -R^T t
    volatile float a = cam->R_wc[r] * cam->t_wc[0];
    volatile float b = cam->R_wc[3 + r] * cam->t_wc[1];
    volatile float c = cam->R_wc[6 + r] * cam->t_wc[2];
    volatile float ab = a + b;
    volatile float abc = ab + c;
    k.C[r] = -abc;
  }
  int grid = (av->n_gauss + 255) / 256;
  const cudaError_t em = cudaMemsetAsync(av->tile_count, 0, (size_t)k.TX * k.TY * sizeof(unsigned), s);
  if (em != cudaSuccess) return em;
  project_kernel<<<grid, 256, 0, s>>>(av->n_gauss, k, av->g_posed, av->g_nposed, av->g_cov, av->g_scale_op, av->mu2d,
                                      av->depth, av->conic_o, av->rect, av->touched, av->tile_count, av->proj_counter, k.TX * k.TY,
                                      av->max_dup, av->ranges, av->cursor, av->num_dup, av->seg_off, av->num_items, av->status);
  av->launches += 1;
  rga_prof_mark(av, "project", s);
  return cudaGetLastError();
}
