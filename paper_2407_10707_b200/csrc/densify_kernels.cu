// Algorithm 1, "Gaussian densification based on density" (PAPER.md:481-510; text :475-479, :173).  EXACT source
// (-fmad=false): every output is either an integer or an fp32 value formed in the contract's operation order, so the
// whole result is compared bit for bit (readings A29-A31).
//
//   D_v[k]  = number of (Gaussian, neighbour) pairs of S_g that name vertex k           dens_count_kernel
//   d_f[i]  = (D_v[f0] + D_v[f1] + D_v[f2]) / (6 K_g),  P[i] = max(0, d_0 - d_f[i])      dens_tri_kernel
//   N'      = floor(sum(P) p_0)                                                        dens_scan_blocks_kernel
//   n_g     = MultinomialSample(P / sum(P), N'):  N' draws by inverse CDF               dens_cdf_kernel, dens_sample_kernel
//   place every drawn Gaussian uniformly on its triangle                               dens_sample_kernel
//
// P is held in fixed point (P * 2^16 rounded to nearest) so that its prefix sums are exact integers whatever the order
// of summation; a draw is one binary search in the 64-bit running sum.
#include "rga_internal.h"

#define DENS_BLOCK 256
#define DENS_PER_THREAD 8
#define DENS_TILE (DENS_BLOCK * DENS_PER_THREAD)

__global__ void __launch_bounds__(256) dens_count_kernel(int n, const int* __restrict__ knn_g, int* __restrict__ D_v) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) atomicAdd(&D_v[knn_g[i]], 1);
}

// sum of a 64-bit value over the CTA; every thread gets the inclusive prefix, *total the CTA's sum
__device__ __forceinline__ unsigned long long block_scan_incl(unsigned long long v, unsigned long long* s_warp, unsigned long long* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned long long u = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += u;
  }
  if (lane == 31) s_warp[warp] = v;
  __syncthreads();
  unsigned long long base = 0, tot = 0;
  for (int w = 0; w < nw; ++w) { const unsigned long long x = s_warp[w]; if (w < warp) base += x; tot += x; }
  __syncthreads();
  *total = tot;
  return v + base;
}

__global__ void __launch_bounds__(DENS_BLOCK) dens_tri_kernel(int nf, int K_g, float d0, const int* __restrict__ faces,
    const int* __restrict__ D_v, unsigned* __restrict__ P_fix, unsigned long long* __restrict__ block_sum) {
  __shared__ unsigned long long s_warp[DENS_BLOCK / 32];
  const int base = blockIdx.x * DENS_TILE + threadIdx.x * DENS_PER_THREAD;
  const float den = (float)(6 * K_g);
  unsigned long long sum = 0;
#pragma unroll
  for (int u = 0; u < DENS_PER_THREAD; ++u) {
    const int i = base + u;
    if (i < nf) {
      const int c = D_v[faces[3 * i]] + D_v[faces[3 * i + 1]] + D_v[faces[3 * i + 2]];
      const float d_f = __fdiv_rn((float)c, den);
      const float P = fmaxf(0.0f, __fsub_rn(d0, d_f));
      const unsigned q = (unsigned)__float2uint_rn(__fmul_rn(P, 65536.0f));
      P_fix[i] = q;
      sum += q;
    }
  }
  unsigned long long tot;
  block_scan_incl(sum, s_warp, &tot);
  if (threadIdx.x == 0) block_sum[blockIdx.x] = tot;
}

// one CTA: exclusive scan of the per-tile sums in place; hdr[0] = sum(P) in fixed point, hdr[1] = N'
__global__ void __launch_bounds__(1024) dens_scan_blocks_kernel(int nblocks, float p0, int max_out, unsigned long long* __restrict__ block_sum,
    unsigned long long* __restrict__ hdr, int* __restrict__ out_count) {
  __shared__ unsigned long long s_warp[32];
  unsigned long long carry = 0;
  for (int b0 = 0; b0 < nblocks; b0 += 1024) {
    const int b = b0 + threadIdx.x;
    const unsigned long long v = b < nblocks ? block_sum[b] : 0ull;
    unsigned long long tot;
    const unsigned long long inc = block_scan_incl(v, s_warp, &tot);
    if (b < nblocks) block_sum[b] = carry + inc - v;
    carry += tot;
  }
  if (threadIdx.x == 0) {
    const double want = floor((double)carry * (double)p0 / 65536.0);
    const unsigned long long n_add = want < 0.0 ? 0ull : (want > 9.0e18 ? 9000000000000000000ull : (unsigned long long)want);
    hdr[0] = carry; hdr[1] = n_add;
    if (out_count) *out_count = n_add > 2147483647ull ? 2147483647 : (int)n_add;
  }
}

__global__ void __launch_bounds__(DENS_BLOCK) dens_cdf_kernel(int nf, const unsigned* __restrict__ P_fix,
    const unsigned long long* __restrict__ block_off, unsigned long long* __restrict__ cdf) {
  __shared__ unsigned long long s_warp[DENS_BLOCK / 32];
  const int base = blockIdx.x * DENS_TILE + threadIdx.x * DENS_PER_THREAD;
  unsigned q[DENS_PER_THREAD];
  unsigned long long sum = 0;
#pragma unroll
  for (int u = 0; u < DENS_PER_THREAD; ++u) { q[u] = base + u < nf ? P_fix[base + u] : 0u; sum += q[u]; }
  unsigned long long tot;
  unsigned long long run = block_off[blockIdx.x] + block_scan_incl(sum, s_warp, &tot) - sum;
#pragma unroll
  for (int u = 0; u < DENS_PER_THREAD; ++u) { run += q[u]; if (base + u < nf) cdf[base + u] = run; }
}

// thread j = draw j: triangle by inverse CDF from rnd[3j], barycentric coordinates from rnd[3j+1], rnd[3j+2]
__global__ void __launch_bounds__(256) dens_sample_kernel(int nf, int max_out, const unsigned long long* __restrict__ hdr,
    const unsigned long long* __restrict__ cdf, const unsigned* __restrict__ rnd, const int* __restrict__ faces,
    const float4* __restrict__ v_pos, float* __restrict__ out_pos, int* __restrict__ out_tri, int* __restrict__ n_g) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned long long S = hdr[0], n_add = hdr[1];
  if (j >= max_out || (unsigned long long)j >= n_add) return;
  const unsigned long long target = __umul64hi((unsigned long long)rnd[3 * j] << 32, S);     // floor(rnd / 2^32 * S)
  int lo = 0, hi = nf - 1;                                // first i with cdf[i] > target (cdf[nf-1] = S > target)
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (cdf[mid] > target) hi = mid; else lo = mid + 1;
  }
  const int t = lo;
  atomicAdd(&n_g[t], 1);
  if (out_tri) out_tri[j] = t;
  const float r1 = __fmul_rn((float)(rnd[3 * j + 1] >> 8), 5.9604644775390625e-8f);        // 2^-24
  const float r2 = __fmul_rn((float)(rnd[3 * j + 2] >> 8), 5.9604644775390625e-8f);
  const float sq = __fsqrt_rn(r1);
  const float b0 = __fsub_rn(1.0f, sq), b1 = __fmul_rn(sq, __fsub_rn(1.0f, r2)), b2 = __fmul_rn(sq, r2);
  const float4 x0 = v_pos[faces[3 * t]], x1 = v_pos[faces[3 * t + 1]], x2 = v_pos[faces[3 * t + 2]];
  out_pos[3 * j + 0] = __fadd_rn(__fadd_rn(__fmul_rn(b0, x0.x), __fmul_rn(b1, x1.x)), __fmul_rn(b2, x2.x));
  out_pos[3 * j + 1] = __fadd_rn(__fadd_rn(__fmul_rn(b0, x0.y), __fmul_rn(b1, x1.y)), __fmul_rn(b2, x2.y));
  out_pos[3 * j + 2] = __fadd_rn(__fadd_rn(__fmul_rn(b0, x0.z), __fmul_rn(b1, x1.z)), __fmul_rn(b2, x2.z));
}

cudaError_t rga_launch_densify(rga_avatar* av, float d0, float p0, const unsigned* rnd, int max_out, float* out_pos, int* out_tri,
                               int* out_count, cudaStream_t s) {
  const int nf = av->n_faces, nblocks = (nf + DENS_TILE - 1) / DENS_TILE, npairs = av->n_gauss * av->k_g;
  cudaError_t e;
  if ((e = cudaMemsetAsync(av->dens_dv, 0, sizeof(int) * (size_t)av->n_verts, s)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(av->dens_ng, 0, sizeof(int) * (size_t)nf, s)) != cudaSuccess) return e;
  if (npairs > 0) dens_count_kernel<<<(npairs + 255) / 256, 256, 0, s>>>(npairs, av->knn_g, av->dens_dv);
  rga_prof_mark(av, "dens_count", s);
  dens_tri_kernel<<<nblocks, DENS_BLOCK, 0, s>>>(nf, av->k_g, d0, av->faces, av->dens_dv, av->dens_pfix, av->dens_block);
  rga_prof_mark(av, "dens_tri", s);
  dens_scan_blocks_kernel<<<1, 1024, 0, s>>>(nblocks, p0, max_out, av->dens_block, av->dens_hdr, out_count);
  rga_prof_mark(av, "dens_scan", s);
  dens_cdf_kernel<<<nblocks, DENS_BLOCK, 0, s>>>(nf, av->dens_pfix, av->dens_block, av->dens_cdf);
  rga_prof_mark(av, "dens_cdf", s);
  if (max_out > 0) {
    dens_sample_kernel<<<(max_out + 255) / 256, 256, 0, s>>>(nf, max_out, av->dens_hdr, av->dens_cdf, rnd, av->faces, av->v_pos, out_pos,
                                                             out_tri, av->dens_ng);
    rga_prof_mark(av, "dens_sample", s);
  }
  av->launches += 4 + (npairs > 0) + (max_out > 0);
  return cudaGetLastError();
}
