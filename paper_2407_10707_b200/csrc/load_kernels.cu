// L0 avatar_load kernels: brute-force KNN and Eq.1 interpolation of the
// pose-independent attributes.  EXACT file: compiled with -fmad=false; only + - * / sqrt so results are bit-identical
// to any IEEE-754 implementation that follows the same operation order.
#include "rga_internal.h"

#define KNN_TILE 1024
#define KNN_MAXK 32

// One thread per query; vertices staged through shared memory in tiles; K best kept sorted ascending.
// Scanning j upward with a strict '<' keeps the lower index on equal distances.
template <int KT>
__global__ void __launch_bounds__(256) knn_kernel(const float* __restrict__ q, int nq, const float* __restrict__ v, int nv,
                                                  int Krt, int* __restrict__ idx, float* __restrict__ d2out) {
  __shared__ float sv[KNN_TILE * 3];
  const int K = KT > 0 ? KT : Krt;
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  float qx = 0.f, qy = 0.f, qz = 0.f;
  if (i < nq) { qx = q[3 * (size_t)i]; qy = q[3 * (size_t)i + 1]; qz = q[3 * (size_t)i + 2]; }
  float bd[KT > 0 ? KT : KNN_MAXK];
  int bi[KT > 0 ? KT : KNN_MAXK];
#pragma unroll
  for (int k = 0; k < (KT > 0 ? KT : KNN_MAXK); ++k) { bd[k] = __int_as_float(0x7f800000); bi[k] = -1; }
  for (int base = 0; base < nv; base += KNN_TILE) {
    int cnt = min(KNN_TILE, nv - base);
    __syncthreads();
    for (int t = threadIdx.x; t < cnt * 3; t += blockDim.x) sv[t] = v[(size_t)base * 3 + t];
    __syncthreads();
    if (i < nq) {
      for (int j = 0; j < cnt; ++j) {
        float dx = qx - sv[3 * j], dy = qy - sv[3 * j + 1], dz = qz - sv[3 * j + 2];
        float d = (dx * dx + dy * dy) + dz * dz;
        if (d < bd[K - 1]) {
          if (KT > 0) {
#pragma unroll
            for (int p = (KT > 0 ? KT : 1) - 1; p >= 0; --p) {        // static indices: the list stays in registers
              if (p > 0 && d < bd[p - 1]) { bd[p] = bd[p - 1]; bi[p] = bi[p - 1]; }
              else { bd[p] = d; bi[p] = base + j; break; }
            }
          } else {
            int p = K - 1;
            while (p > 0 && d < bd[p - 1]) { bd[p] = bd[p - 1]; bi[p] = bi[p - 1]; --p; }
            bd[p] = d; bi[p] = base + j;
          }
        }
      }
    }
  }
  if (i < nq)
    for (int k = 0; k < K; ++k) { idx[(size_t)i * K + k] = bi[k]; d2out[(size_t)i * K + k] = bd[k]; }
}

cudaError_t rga_launch_knn(const float* q, int nq, const float* v, int nv, int K, int* idx, float* d2, cudaStream_t s) {
  int grid = (nq + 255) / 256;
  if (K == 3) knn_kernel<3><<<grid, 256, 0, s>>>(q, nq, v, nv, K, idx, d2);
  else if (K == 19) knn_kernel<19><<<grid, 256, 0, s>>>(q, nq, v, nv, K, idx, d2);
  else knn_kernel<0><<<grid, 256, 0, s>>>(q, nq, v, nv, K, idx, d2);
  return cudaGetLastError();
}

__global__ void load_verts_kernel(int n, const float* __restrict__ pos, const float* __restrict__ disp,
                                  const float* __restrict__ nrm, float4* __restrict__ xbar, float4* __restrict__ nout,
                                  float4* __restrict__ vpos) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  float dx = disp ? disp[3 * i] : 0.f, dy = disp ? disp[3 * i + 1] : 0.f, dz = disp ? disp[3 * i + 2] : 0.f;
  xbar[i] = make_float4(pos[3 * i] + dx, pos[3 * i + 1] + dy, pos[3 * i + 2] + dz, 0.f);
  vpos[i] = make_float4(pos[3 * i], pos[3 * i + 1], pos[3 * i + 2], 0.f);
  nout[i] = make_float4(nrm[3 * i], nrm[3 * i + 1], nrm[3 * i + 2], 0.f);
}

cudaError_t rga_launch_load_verts(rga_avatar* av, const float* pos, const float* disp, const float* nrm, cudaStream_t s) {
  load_verts_kernel<<<(av->n_verts + 255) / 256, 256, 0, s>>>(av->n_verts, pos, disp, nrm, av->v_xbar, av->v_normal, av->v_pos);
  return cudaGetLastError();
}

// Eq.1 for one Gaussian: weights from the K_g squared distances, then every static attribute.
__global__ void __launch_bounds__(128) load_gauss_kernel(int n, int K, int B, const int* __restrict__ knn, const float* __restrict__ d2,
                                  const float* __restrict__ gpos, const float* __restrict__ vdisp,
                                  const float* __restrict__ vnrm, const float* __restrict__ valb,
                                  const float* __restrict__ vrough, const float* __restrict__ vspec,
                                  const float* __restrict__ vw, const float* __restrict__ gquat,
                                  const float* __restrict__ gscale, const float* __restrict__ gop,
                                  float* __restrict__ ubar, float4* __restrict__ gst, float* __restrict__ gw,
                                  float4* __restrict__ quat, float4* __restrict__ scale_op, float4* __restrict__ gpos4,
                                  const float* __restrict__ vquat, const float* __restrict__ vscale, int set_opacity) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= n) return;
  float u[4]; int id[4];
  float U = 0.f;
  for (int k = 0; k < K; ++k) {
    id[k] = knn[(size_t)g * K + k];
    float dist = sqrtf(d2[(size_t)g * K + k]);
    u[k] = 1.0f / fmaxf(dist, 1e-12f);
    U = (k == 0) ? u[0] : U + u[k];
  }
  for (int k = 0; k < K; ++k) { u[k] = u[k] / U; ubar[(size_t)g * K + k] = u[k]; }
  auto interp = [&](const float* a, int C, int c) {
    float acc = u[0] * a[(size_t)id[0] * C + c];
    for (int k = 1; k < K; ++k) acc = acc + u[k] * a[(size_t)id[k] * C + c];
    return acc;
  };
  float d0 = vdisp ? interp(vdisp, 3, 0) : 0.f, d1 = vdisp ? interp(vdisp, 3, 1) : 0.f, d2v = vdisp ? interp(vdisp, 3, 2) : 0.f;
  gst[4 * (size_t)g + 0] = make_float4(gpos[3 * (size_t)g] + d0, gpos[3 * (size_t)g + 1] + d1, gpos[3 * (size_t)g + 2] + d2v, 0.f);
  gpos4[g] = make_float4(gpos[3 * (size_t)g], gpos[3 * (size_t)g + 1], gpos[3 * (size_t)g + 2], 0.f);
  float nx = interp(vnrm, 3, 0), ny = interp(vnrm, 3, 1), nz = interp(vnrm, 3, 2);
  float len = sqrtf((nx * nx + ny * ny) + nz * nz);
  if (len > 0.f) { nx = nx / len; ny = ny / len; nz = nz / len; }
  gst[4 * (size_t)g + 1] = make_float4(nx, ny, nz, 0.f);
  gst[4 * (size_t)g + 2] = make_float4(interp(valb, 3, 0), interp(valb, 3, 1), interp(valb, 3, 2), interp(vrough, 1, 0));
  gst[4 * (size_t)g + 3] = make_float4(interp(vspec, 1, 0), 0.f, 0.f, 0.f);
  for (int b = 0; b < B; ++b) gw[(size_t)g * B + b] = interp(vw, B, b);
  // rotation and scale: the caller's per-Gaussian arrays, or (the paper's layout; reading A2) Eq.1 of the
  // vertex attributes -- neighbour quaternions take the sign of neighbour 0's first (dot4 < 0 -> negated), then the
  // weighted sum in neighbour order; it is normalised where it is used (H2).  Both NULL (gaussians_update with per-Gaussian
  // rotations): kept as they are.
  if (gquat) quat[g] = make_float4(gquat[4 * (size_t)g], gquat[4 * (size_t)g + 1], gquat[4 * (size_t)g + 2], gquat[4 * (size_t)g + 3]);
  else if (vquat) {
    const float* q0 = vquat + 4 * (size_t)id[0];
    float acc[4] = {u[0] * q0[0], u[0] * q0[1], u[0] * q0[2], u[0] * q0[3]};
    for (int k = 1; k < K; ++k) {
      const float* qk = vquat + 4 * (size_t)id[k];
      const float dt = ((qk[0] * q0[0] + qk[1] * q0[1]) + qk[2] * q0[2]) + qk[3] * q0[3];
      const float sg = dt < 0.f ? -1.0f : 1.0f;
      for (int c = 0; c < 4; ++c) acc[c] = acc[c] + u[k] * (sg * qk[c]);
    }
    quat[g] = make_float4(acc[0], acc[1], acc[2], acc[3]);
  }
  if (gscale || vscale || set_opacity) {
    float4 so = scale_op[g];
    if (gscale) { so.x = gscale[3 * (size_t)g]; so.y = gscale[3 * (size_t)g + 1]; so.z = gscale[3 * (size_t)g + 2]; }
    else if (vscale) { so.x = interp(vscale, 3, 0); so.y = interp(vscale, 3, 1); so.z = interp(vscale, 3, 2); }
    if (set_opacity) so.w = gop ? gop[g] : 1.0f;
    scale_op[g] = so;
  }
}

// Eq.1 of every static attribute from the library's own copies of the vertex tables (so that gaussians_update can run
// after the caller's arrays are gone); gauss_quat == NULL keeps rotation / scale / opacity.
cudaError_t rga_launch_load_gauss(rga_avatar* av, const float* gauss_pos, const float* gauss_quat, const float* gauss_scale,
                                  const float* gauss_opacity, const float* d2, cudaStream_t s, const float* vert_quat, const float* vert_scale,
                                  int set_opacity) {
  load_gauss_kernel<<<(av->n_gauss + 127) / 128, 128, 0, s>>>(
      av->n_gauss, av->k_g, av->n_bones, av->knn_g, d2, gauss_pos, av->vt_disp, av->vt_normal, av->vt_albedo,
      av->vt_rough, av->vt_spec, av->v_skin_w, gauss_quat, gauss_scale, gauss_opacity, av->ubar_g,
      av->g_static, av->g_skin_w, av->g_quat, av->g_scale_op, av->g_pos, vert_quat, vert_scale, set_opacity);
  return cudaGetLastError();
}

// Applies a per-pose vertex displacement (displacement_mlp): x + dx for the mesh, and Eq.1 of dx over S_g
// for the Gaussians, in the operation order of load_gauss_kernel / DESIGN.md "Arithmetic contract".
__global__ void __launch_bounds__(256) disp_apply_kernel(int nv, int ng, int K, const float4* __restrict__ v_pos,
    const float4* __restrict__ v_disp, float4* __restrict__ v_xbar, const float4* __restrict__ g_pos,
    const int* __restrict__ knn_g, const float* __restrict__ ubar_g, float4* __restrict__ g_static) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nv) {
    const float4 p = v_pos[i], d = v_disp[i];
    v_xbar[i] = make_float4(p.x + d.x, p.y + d.y, p.z + d.z, 0.f);
  } else if (i - nv < ng) {
    const int g = i - nv;
    float ax = 0.f, ay = 0.f, az = 0.f;
    for (int k = 0; k < K; ++k) {
      const float u = ubar_g[(size_t)g * K + k];
      const float4 d = v_disp[knn_g[(size_t)g * K + k]];
      if (k == 0) { ax = u * d.x; ay = u * d.y; az = u * d.z; }
      else { ax = ax + u * d.x; ay = ay + u * d.y; az = az + u * d.z; }
    }
    const float4 p = g_pos[g];
    g_static[4 * (size_t)g] = make_float4(p.x + ax, p.y + ay, p.z + az, 0.f);
  }
}

// the static per-vertex displacement table of avatar_load (or zero) back into the per-pose displacement buffer
__global__ void disp_static_kernel(int nv, const float* __restrict__ vt_disp, float4* __restrict__ v_disp) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  v_disp[i] = vt_disp ? make_float4(vt_disp[3 * (size_t)i], vt_disp[3 * (size_t)i + 1], vt_disp[3 * (size_t)i + 2], 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
}

cudaError_t rga_launch_disp_static(rga_avatar* av, cudaStream_t s) {
  disp_static_kernel<<<(av->n_verts + 255) / 256, 256, 0, s>>>(av->n_verts, av->vt_disp, av->v_disp);
  av->launches += 1;
  return cudaGetLastError();
}

cudaError_t rga_launch_disp_apply(rga_avatar* av, cudaStream_t s) {
  const int n = av->n_verts + av->n_gauss;
  disp_apply_kernel<<<(n + 255) / 256, 256, 0, s>>>(av->n_verts, av->n_gauss, av->k_g, av->v_pos, av->v_disp, av->v_xbar, av->g_pos,
                                                    av->knn_g, av->ubar_g, av->g_static);
  av->launches += 1;
  rga_prof_mark(av, "disp_apply", s);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------- uniform-grid KNN (exact)
// The canonical vertices are binned once into a uniform grid (counting sort: count, scan, fill).  A query walks the cells
// ring by ring (Chebyshev distance r from its own cell) and keeps the K best by (d2, index) -- the same order the brute
// force produces by scanning indices upward with a strict '<' -- and stops once the K-th distance is below ((r-1) h)^2, the
// least any vertex of a cell of ring r or beyond can have (with a 1e-4 relative guard against the fp32 rounding of the cell
// assignment).  d2 is computed with the brute force's operation order, so indices AND distances are bit-identical.
struct KnnGrid { float ox, oy, oz, h, inv_h; int G; };

__device__ __forceinline__ int grid_coord(float x, float o, float inv_h, int G) {
  int c = (int)floorf((x - o) * inv_h);
  return c < 0 ? 0 : (c >= G ? G - 1 : c);
}

__global__ void grid_count_kernel(int nv, KnnGrid g, const float* __restrict__ v, unsigned* __restrict__ cell_count,
                                  int* __restrict__ cell_of) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  int cx = grid_coord(v[3 * i], g.ox, g.inv_h, g.G), cy = grid_coord(v[3 * i + 1], g.oy, g.inv_h, g.G),
      cz = grid_coord(v[3 * i + 2], g.oz, g.inv_h, g.G);
  int c = (cz * g.G + cy) * g.G + cx;
  cell_of[i] = c;
  atomicAdd(cell_count + c, 1u);
}

// exclusive scan of the cell counts by one block (load time only); cell_start has ncell + 1 entries
__global__ void __launch_bounds__(1024) grid_scan_kernel(int ncell, const unsigned* __restrict__ cell_count, unsigned* __restrict__ cell_start,
                                                         unsigned* __restrict__ cursor) {
  __shared__ unsigned part[1024];
  const int per = (ncell + 1023) / 1024, lo = threadIdx.x * per, hi = min(ncell, lo + per);
  unsigned s = 0;
  for (int i = lo; i < hi; ++i) s += cell_count[i];
  part[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) { unsigned acc = 0; for (int t = 0; t < 1024; ++t) { unsigned v = part[t]; part[t] = acc; acc += v; } cell_start[ncell] = acc; }
  __syncthreads();
  unsigned acc = part[threadIdx.x];
  for (int i = lo; i < hi; ++i) { cell_start[i] = acc; cursor[i] = acc; acc += cell_count[i]; }
}

__global__ void grid_fill_kernel(int nv, const int* __restrict__ cell_of, unsigned* __restrict__ cursor, int* __restrict__ cell_verts) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nv) return;
  cell_verts[atomicAdd(cursor + cell_of[i], 1u)] = i;
}

template <int KT>
__global__ void __launch_bounds__(128) knn_grid_kernel(const float* __restrict__ q, int nq, const float* __restrict__ v, KnnGrid g,
    const unsigned* __restrict__ cell_start, const int* __restrict__ cell_verts, int* __restrict__ idx, float* __restrict__ d2out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nq) return;
  const float qx = q[3 * (size_t)i], qy = q[3 * (size_t)i + 1], qz = q[3 * (size_t)i + 2];
  float bd[KT]; int bi[KT];
#pragma unroll
  for (int k = 0; k < KT; ++k) { bd[k] = __int_as_float(0x7f800000); bi[k] = 0x7fffffff; }
  const int cx = grid_coord(qx, g.ox, g.inv_h, g.G), cy = grid_coord(qy, g.oy, g.inv_h, g.G), cz = grid_coord(qz, g.oz, g.inv_h, g.G);
  for (int r = 0; r <= g.G; ++r) {
    if (r > 1) {                              // rings < r are done: every unvisited vertex is at least (r - 1) h away (see header)
      const float reach = (float)(r - 1) * g.h;
      if (bd[KT - 1] < reach * reach * 0.9999f) break;
    }
    const int z0 = max(cz - r, 0), z1 = min(cz + r, g.G - 1), y0 = max(cy - r, 0), y1 = min(cy + r, g.G - 1);
    const int x0 = max(cx - r, 0), x1 = min(cx + r, g.G - 1);
    for (int z = z0; z <= z1; ++z)
      for (int y = y0; y <= y1; ++y) {
        const bool shell_zy = abs(z - cz) == r || abs(y - cy) == r;
        for (int x = x0; x <= x1; ++x) {
          if (!shell_zy && abs(x - cx) != r) continue;          // inside the cube: visited in an earlier ring
          const int c = (z * g.G + y) * g.G + x;
          for (unsigned e = cell_start[c]; e < cell_start[c + 1]; ++e) {
            const int j = cell_verts[e];
            const float dx = qx - v[3 * (size_t)j], dy = qy - v[3 * (size_t)j + 1], dz = qz - v[3 * (size_t)j + 2];
            const float d = (dx * dx + dy * dy) + dz * dz;
            if (d < bd[KT - 1] || (d == bd[KT - 1] && j < bi[KT - 1])) {
#pragma unroll
              for (int p = KT - 1; p >= 0; --p) {
                if (p > 0 && (d < bd[p - 1] || (d == bd[p - 1] && j < bi[p - 1]))) { bd[p] = bd[p - 1]; bi[p] = bi[p - 1]; }
                else { bd[p] = d; bi[p] = j; break; }
              }
            }
          }
        }
      }
  }
  for (int k = 0; k < KT; ++k) { idx[(size_t)i * KT + k] = bi[k]; d2out[(size_t)i * KT + k] = bd[k]; }
}

// builds the grid over av->vt_pos; returns cudaSuccess with av->grid_G == 0 when no grid is used (degenerate extent)
cudaError_t rga_build_knn_grid(rga_avatar* av, const float* aabb_host, cudaStream_t s) {
  av->grid_G = 0;
  const float ex = aabb_host[3] - aabb_host[0], ey = aabb_host[4] - aabb_host[1], ez = aabb_host[5] - aabb_host[2];
  const float ext = fmaxf(ex, fmaxf(ey, ez));
  if (!(ext > 0.f) || av->n_verts < 64) return cudaSuccess;
  int G = (int)(2.5f * cbrtf((float)av->n_verts) + 0.5f);
  G = G < 4 ? 4 : (G > 128 ? 128 : G);
  av->grid_G = G; av->grid_h = ext * 1.0001f / (float)G;
  av->grid_o[0] = aabb_host[0]; av->grid_o[1] = aabb_host[1]; av->grid_o[2] = aabb_host[2];
  const int ncell = G * G * G;
  cudaError_t e;
  if ((e = cudaMalloc((void**)&av->grid_start, (size_t)(ncell + 1) * 4)) != cudaSuccess) return e;
  if ((e = cudaMalloc((void**)&av->grid_verts, (size_t)av->n_verts * 4)) != cudaSuccess) return e;
  unsigned *count = nullptr, *cursor = nullptr; int* cell_of = nullptr;
  if ((e = cudaMalloc((void**)&count, (size_t)ncell * 4)) != cudaSuccess) return e;
  if ((e = cudaMalloc((void**)&cursor, (size_t)ncell * 4)) != cudaSuccess) return e;
  if ((e = cudaMalloc((void**)&cell_of, (size_t)av->n_verts * 4)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(count, 0, (size_t)ncell * 4, s)) != cudaSuccess) return e;
  KnnGrid g = {av->grid_o[0], av->grid_o[1], av->grid_o[2], av->grid_h, 1.0f / av->grid_h, G};
  grid_count_kernel<<<(av->n_verts + 255) / 256, 256, 0, s>>>(av->n_verts, g, av->vt_pos, count, cell_of);
  grid_scan_kernel<<<1, 1024, 0, s>>>(ncell, count, av->grid_start, cursor);
  grid_fill_kernel<<<(av->n_verts + 255) / 256, 256, 0, s>>>(av->n_verts, cell_of, cursor, av->grid_verts);
  e = cudaStreamSynchronize(s);
  cudaFree(count); cudaFree(cursor); cudaFree(cell_of);
  av->launches += 3;
  return e != cudaSuccess ? e : cudaGetLastError();
}

// S_v: K_v nearest vertices of every vertex (self included) through the grid when K_v is the paper's 19
cudaError_t rga_launch_knn_verts(rga_avatar* av, float* d2, cudaStream_t s) {
  if (av->grid_G == 0 || av->k_v != 19) return rga_launch_knn(av->vt_pos, av->n_verts, av->vt_pos, av->n_verts, av->k_v, av->knn_v, d2, s);
  KnnGrid g = {av->grid_o[0], av->grid_o[1], av->grid_o[2], av->grid_h, 1.0f / av->grid_h, av->grid_G};
  knn_grid_kernel<19><<<(av->n_verts + 127) / 128, 128, 0, s>>>(av->vt_pos, av->n_verts, av->vt_pos, g, av->grid_start, av->grid_verts,
                                                                 av->knn_v, d2);
  return cudaGetLastError();
}

// K_g nearest canonical vertices of the queries through the grid (brute force when there is no grid or K_g is not 3)
cudaError_t rga_launch_knn_gauss(rga_avatar* av, const float* q, cudaStream_t s) {
  if (av->grid_G == 0 || av->k_g != 3) return rga_launch_knn(q, av->n_gauss, av->vt_pos, av->n_verts, av->k_g, av->knn_g, av->knn_d2, s);
  KnnGrid g = {av->grid_o[0], av->grid_o[1], av->grid_o[2], av->grid_h, 1.0f / av->grid_h, av->grid_G};
  knn_grid_kernel<3><<<(av->n_gauss + 127) / 128, 128, 0, s>>>(q, av->n_gauss, av->vt_pos, g, av->grid_start, av->grid_verts, av->knn_g,
                                                                av->knn_d2);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------------
// vert_normal == NULL (include/rga.h; reading A40): area-weighted vertex normals of the canonical mesh,
// n_v = normalize(sum over the faces that touch v, in ASCENDING face order, of (x_b - x_a) x (x_c - x_a)), one fp32 rounding per
// operation (this file is compiled with -fmad=false).  The order is fixed because the normal feeds the bit-exact chain
// (front-facing tests, visibility bits): a vertex -> face adjacency is built with atomics (any order) and each vertex then walks
// its list by repeated selection of the next larger face index.  Load time only.
__global__ void vn_count_kernel(int n3, const int* __restrict__ faces, unsigned* __restrict__ deg) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n3) atomicAdd(deg + faces[i], 1u);
}

__global__ void vn_fill_kernel(int n3, const int* __restrict__ faces, unsigned* __restrict__ cursor, int* __restrict__ adj) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n3) adj[atomicAdd(cursor + faces[i], 1u)] = i / 3;
}

__global__ void __launch_bounds__(128) vn_accum_kernel(int nv, const float* __restrict__ x, const int* __restrict__ faces,
                                                       const unsigned* __restrict__ start, const int* __restrict__ adj,
                                                       float* __restrict__ out) {
  int v = blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= nv) return;
  const unsigned lo = start[v], hi = start[v + 1];
  float sx = 0.f, sy = 0.f, sz = 0.f;
  int last = -1;
  for (;;) {
    int m = 0x7fffffff, cnt = 0;
    for (unsigned j = lo; j < hi; ++j) {
      int e = adj[j];
      if (e > last && e < m) { m = e; cnt = 1; }
      else if (e == m) ++cnt;                                    // a face that names v twice adds twice, as the plain loop does
    }
    if (cnt == 0) break;
    const int a = faces[3 * m], b = faces[3 * m + 1], c = faces[3 * m + 2];
    const float e1x = x[3 * b] - x[3 * a], e1y = x[3 * b + 1] - x[3 * a + 1], e1z = x[3 * b + 2] - x[3 * a + 2];
    const float e2x = x[3 * c] - x[3 * a], e2y = x[3 * c + 1] - x[3 * a + 1], e2z = x[3 * c + 2] - x[3 * a + 2];
    const float cx = e1y * e2z - e1z * e2y, cy = e1z * e2x - e1x * e2z, cz = e1x * e2y - e1y * e2x;
    for (int r = 0; r < cnt; ++r) { sx = sx + cx; sy = sy + cy; sz = sz + cz; }
    last = m;
  }
  const float len = sqrtf((sx * sx + sy * sy) + sz * sz);
  if (len > 0.f) { sx = sx / len; sy = sy / len; sz = sz / len; }
  out[3 * v] = sx; out[3 * v + 1] = sy; out[3 * v + 2] = sz;
}

// faces: device [n_faces][3] (indices already checked by the caller's contract), x: device [n_verts][3]; out: device [n_verts][3]
cudaError_t rga_launch_vertex_normals(const float* x, const int* faces, int nv, int nf, float* out, cudaStream_t s) {
  unsigned *deg = nullptr, *start = nullptr, *cursor = nullptr; int* adj = nullptr;
  const int n3 = 3 * nf;
  cudaError_t e = cudaMalloc(&deg, sizeof(unsigned) * ((size_t)nv + 1));
  if (e == cudaSuccess) e = cudaMalloc(&start, sizeof(unsigned) * ((size_t)nv + 1));
  if (e == cudaSuccess) e = cudaMalloc(&cursor, sizeof(unsigned) * ((size_t)nv + 1));
  if (e == cudaSuccess) e = cudaMalloc(&adj, sizeof(int) * (size_t)n3);
  if (e == cudaSuccess) e = cudaMemsetAsync(deg, 0, sizeof(unsigned) * ((size_t)nv + 1), s);
  if (e == cudaSuccess) {
    vn_count_kernel<<<(n3 + 255) / 256, 256, 0, s>>>(n3, faces, deg);
    grid_scan_kernel<<<1, 1024, 0, s>>>(nv, deg, start, cursor);
    vn_fill_kernel<<<(n3 + 255) / 256, 256, 0, s>>>(n3, faces, cursor, adj);
    vn_accum_kernel<<<(nv + 127) / 128, 128, 0, s>>>(nv, x, faces, start, adj, out);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  }
  cudaFree(deg); cudaFree(start); cudaFree(cursor); cudaFree(adj);
  return e;
}
