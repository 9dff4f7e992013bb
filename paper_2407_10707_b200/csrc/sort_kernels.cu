// H7 scan + emit, H8 radix sort, H9 tile ranges (PAPER.md:103 -> 3DGS tile binning; BASELINE.json north_star (d)
// "a device radix sort on (tile, depth) keys").  Integer-only; D (the number of duplicates) never leaves the device.
#include "rga_internal.h"

// ------------------------------------------------------------------------------------------------------------- H7
// Block b's base offset = sum of the block sums before it (written by the projection kernel); inside the block an
// exclusive warp/block scan of tiles_touched.  Each Gaussian then writes its keys tile-row-major, so equal keys end
// up ordered by Gaussian index after a stable sort (A22).
__global__ void __launch_bounds__(256) emit_kernel(int ng, int nblocks, int TX, long long capacity,
    const unsigned* __restrict__ block_sums, const unsigned* __restrict__ touched, const int4* __restrict__ rect,
    const float* __restrict__ depth, unsigned long long* __restrict__ keys, unsigned* __restrict__ vals,
    unsigned* __restrict__ num_dup, int* __restrict__ status) {
  __shared__ unsigned red[8];
  __shared__ unsigned wbase[8];
  __shared__ unsigned sbase;
  unsigned part = 0;
  for (int b = threadIdx.x; b < (int)blockIdx.x; b += blockDim.x) part += block_sums[b];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned c = (g < ng) ? touched[g] : 0u;
  unsigned incl = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, incl, o); if ((threadIdx.x & 31) >= o) incl += t; }
  __syncthreads();
  if (threadIdx.x == 0) { unsigned s = 0; for (int w = 0; w < 8; ++w) s += red[w]; sbase = s; }
  __syncthreads();
  if ((threadIdx.x & 31) == 31) red[threadIdx.x >> 5] = incl;       // warp totals (red reused after the barrier)
  __syncthreads();
  if (threadIdx.x == 0) { unsigned s = 0; for (int w = 0; w < 8; ++w) { wbase[w] = s; s += red[w]; }
    if ((int)blockIdx.x == nblocks - 1) {
      unsigned long long D = (unsigned long long)sbase + s;
      if ((long long)D > capacity) { atomicExch(status, RGA_ERR_CAPACITY); D = (unsigned long long)capacity; }
      *num_dup = (unsigned)D;
    }
  }
  __syncthreads();
  if (c == 0) return;
  unsigned long long off = (unsigned long long)sbase + wbase[threadIdx.x >> 5] + (incl - c);
  int4 r = rect[g];
  unsigned db = __float_as_uint(depth[g]);
  for (int y = r.y; y < r.w; ++y)
    for (int x = r.x; x < r.z; ++x) {
      if ((long long)off < capacity) {
        keys[off] = ((unsigned long long)(unsigned)(y * TX + x) << 32) | db;
        vals[off] = (unsigned)g;
      }
      ++off;
    }
}

cudaError_t rga_launch_scan_emit(rga_avatar* av, int tiles_x, cudaStream_t s) {
  int nblocks = (av->n_gauss + 255) / 256;
  emit_kernel<<<nblocks, 256, 0, s>>>(av->n_gauss, nblocks, tiles_x, av->max_dup, av->offsets, av->touched, av->rect, av->depth,
                                      av->keys[0], av->vals[0], av->num_dup, av->status);
  av->launches += 1;
  rga_prof_mark(av, "scan_emit", s);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------- H8
// Stable LSD radix sort, 8-bit digits.  Per pass: (1) per-block digit histograms over the block's contiguous chunk,
// (2) one-block exclusive scan over [digit][block], (3) stable scatter: each block re-walks its chunk tile by tile,
// ranking keys inside a warp with match_any and across warps through shared counters.
#define SORT_THREADS 256
#define SORT_ITEMS 8                       // keys per thread per tile
#define SORT_TILE (SORT_THREADS * SORT_ITEMS)
#define RADIX 256

__device__ __forceinline__ void chunk_of(unsigned D, int nblk, int b, unsigned& lo, unsigned& hi) {
  unsigned tiles = (D + SORT_TILE - 1) / SORT_TILE;
  unsigned per = (tiles + nblk - 1) / nblk;
  unsigned long long l = (unsigned long long)b * per * SORT_TILE, h = l + (unsigned long long)per * SORT_TILE;
  lo = (unsigned)min(l, (unsigned long long)D); hi = (unsigned)min(h, (unsigned long long)D);
}

__global__ void __launch_bounds__(SORT_THREADS) sort_hist_kernel(const unsigned long long* __restrict__ keys,
    const unsigned* __restrict__ num_dup, int shift, unsigned* __restrict__ hist /*[RADIX][nblk]*/) {
  __shared__ unsigned h[RADIX];
  h[threadIdx.x] = 0;
  __syncthreads();
  unsigned lo, hi; chunk_of(*num_dup, gridDim.x, blockIdx.x, lo, hi);
  for (unsigned i = lo + threadIdx.x; i < hi; i += SORT_THREADS) atomicAdd(&h[(unsigned)(keys[i] >> shift) & (RADIX - 1)], 1u);
  __syncthreads();
  hist[threadIdx.x * gridDim.x + blockIdx.x] = h[threadIdx.x];
}

// exclusive scan over RADIX*nblk counters in digit-major order (one block, 1024 threads)
__global__ void __launch_bounds__(1024) sort_scan_kernel(unsigned* __restrict__ hist, int n) {
  __shared__ unsigned wsum[32];
  __shared__ unsigned carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  for (int base = 0; base < n; base += 1024) {
    int i = base + threadIdx.x;
    unsigned v = (i < n) ? hist[i] : 0u, incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, incl, o); if ((threadIdx.x & 31) >= o) incl += t; }
    if ((threadIdx.x & 31) == 31) wsum[threadIdx.x >> 5] = incl;
    __syncthreads();
    if (threadIdx.x < 32) {
      unsigned w = wsum[threadIdx.x], wi = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { unsigned t = __shfl_up_sync(0xffffffffu, wi, o); if (threadIdx.x >= o) wi += t; }
      wsum[threadIdx.x] = wi - w;
    }
    __syncthreads();
    unsigned excl = carry + wsum[threadIdx.x >> 5] + (incl - v);
    if (i < n) hist[i] = excl;
    __syncthreads();
    if (threadIdx.x == 1023) carry = excl + v;
    __syncthreads();
  }
}

__global__ void __launch_bounds__(SORT_THREADS) sort_scatter_kernel(const unsigned long long* __restrict__ kin,
    const unsigned* __restrict__ vin, unsigned long long* __restrict__ kout, unsigned* __restrict__ vout,
    const unsigned* __restrict__ num_dup, int shift, const unsigned* __restrict__ hist) {
  __shared__ unsigned base[RADIX];                 // running global offset of each digit for this block
  __shared__ unsigned wcnt[SORT_THREADS / 32][RADIX];
  base[threadIdx.x] = hist[threadIdx.x * gridDim.x + blockIdx.x];
  unsigned lo, hi; chunk_of(*num_dup, gridDim.x, blockIdx.x, lo, hi);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  // element order inside a tile: item-major so that consecutive lanes read consecutive keys:
  //   index = tile_lo + it * SORT_THREADS + threadIdx.x ; stability needs ranks to follow that same order.
  for (unsigned tl = lo; tl < hi; tl += SORT_TILE) {
    for (int it = 0; it < SORT_ITEMS; ++it) {
      __syncthreads();
      for (int w = 0; w < SORT_THREADS / 32; ++w) wcnt[w][threadIdx.x] = 0;     // RADIX == SORT_THREADS
      __syncthreads();
      unsigned i = tl + it * SORT_THREADS + threadIdx.x;
      bool act = i < hi;
      unsigned long long key = act ? kin[i] : 0ull;
      unsigned d = (unsigned)(key >> shift) & (RADIX - 1);
      unsigned m = __match_any_sync(0xffffffffu, act ? d : 0xffffffffu);
      unsigned rank_in_warp = __popc(m & lt);
      if (act && rank_in_warp == 0) wcnt[warp][d] = __popc(m);
      __syncthreads();
      unsigned before = 0;
      if (act) for (int w = 0; w < warp; ++w) before += wcnt[w][d];
      unsigned pos = act ? base[d] + before + rank_in_warp : 0u;
      __syncthreads();
      {                                                    // advance the digit bases by this slab's totals
        unsigned tot = 0;
        for (int w = 0; w < SORT_THREADS / 32; ++w) tot += wcnt[w][threadIdx.x];
        base[threadIdx.x] += tot;
      }
      if (act) { kout[pos] = key; vout[pos] = vin[i]; }
    }
  }
}

cudaError_t rga_launch_sort(rga_avatar* av, int key_bits, cudaStream_t s) {
  int nblk = av->num_sms * 2;
  int passes = (key_bits + 7) / 8, cur = 0;
  for (int p = 0; p < passes; ++p) {
    int shift = 8 * p;
    sort_hist_kernel<<<nblk, SORT_THREADS, 0, s>>>(av->keys[cur], av->num_dup, shift, av->sort_hist);
    sort_scan_kernel<<<1, 1024, 0, s>>>(av->sort_hist, RADIX * nblk);
    sort_scatter_kernel<<<nblk, SORT_THREADS, 0, s>>>(av->keys[cur], av->vals[cur], av->keys[cur ^ 1], av->vals[cur ^ 1],
                                                     av->num_dup, shift, av->sort_hist);
    cur ^= 1;
  }
  av->sorted_buf = cur;
  av->launches += 3 * passes;
  rga_prof_mark(av, "radix_sort", s);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------- H9
__global__ void ranges_kernel(const unsigned long long* __restrict__ keys, const unsigned* __restrict__ num_dup,
                              uint2* __restrict__ ranges) {
  unsigned D = *num_dup;
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < D; i += gridDim.x * blockDim.x) {
    unsigned t = (unsigned)(keys[i] >> 32);
    if (i == 0 || (unsigned)(keys[i - 1] >> 32) != t) ranges[t].x = i;
    if (i == D - 1 || (unsigned)(keys[i + 1] >> 32) != t) ranges[t].y = i + 1;
  }
}

cudaError_t rga_launch_ranges(rga_avatar* av, int ntiles, cudaStream_t s) {
  cudaMemsetAsync(av->ranges, 0, (size_t)ntiles * sizeof(uint2), s);
  ranges_kernel<<<av->num_sms * 4, 256, 0, s>>>(av->keys[av->sorted_buf], av->num_dup, av->ranges);
  av->launches += 1;
  rga_prof_mark(av, "tile_ranges", s);
  return cudaGetLastError();
}
