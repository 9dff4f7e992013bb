// H7 tile binning + H9 tile ranges, and the first (tile) digit of the H8 sort (PAPER.md:103 -> 3DGS tile binning;
// BASELINE.json north_star (d) "a device radix sort on (tile, depth) keys").
//
// The (tile << 32 | depth) key sort is done most-significant-digit first: the tile id is one radix digit with
// TX*TY buckets -- a counting sort (histogram in the projection kernel, exclusive scan here, scatter below) whose bucket
// boundaries ARE the tile ranges of H9 -- and every bucket is then sorted on (depth bits, Gaussian index) in shared
// memory by the CTA that composites that tile (composite_kernels.cu).  Sorting a bucket on (depth, index) equals the
// stable sort of the emission order of DESIGN.md A22 (Gaussians ascending), so the result is bit-identical to one
// global stable sort, with 3 launches instead of 18 and no key ever re-read from HBM.
// Integer-only; D (the number of duplicates) never leaves the device.
#include "rga_internal.h"

// exclusive scans of the per-tile counts n_t and of the per-tile segment counts ceil(n_t / RGA_SEG) (one CTA, 1024
// threads): ranges, scatter cursors, D, capacity check; segment offsets and the number of compositing work items
__global__ void __launch_bounds__(1024) tile_scan_kernel(int ntiles, long long capacity, const unsigned* __restrict__ tile_count,
    uint2* __restrict__ ranges, unsigned* __restrict__ cursor, unsigned* __restrict__ num_dup, unsigned* __restrict__ seg_off,
    unsigned* __restrict__ num_items,
    int* __restrict__ status) {
  __shared__ unsigned wsum[32], wseg[32];
  __shared__ unsigned carry, carry_seg;
  __shared__ unsigned long long total64;                  // D in 64 bits: the 32-bit running sum may wrap before the capacity check
  if (threadIdx.x == 0) { carry = 0; carry_seg = 0; total64 = 0ull; }
  __syncthreads();
  for (int base = 0; base < ntiles; base += 1024) {
    int i = base + threadIdx.x;
    unsigned v = (i < ntiles) ? tile_count[i] : 0u, incl = v;
    unsigned g = (v + RGA_SEG - 1) / RGA_SEG, gincl = g;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned t = __shfl_up_sync(0xffffffffu, incl, o), tg = __shfl_up_sync(0xffffffffu, gincl, o);
      if ((threadIdx.x & 31) >= o) { incl += t; gincl += tg; }
    }
    {
      unsigned long long v64 = v;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v64 += __shfl_xor_sync(0xffffffffu, v64, o);
      if ((threadIdx.x & 31) == 0 && v64) atomicAdd(&total64, v64);
    }
    if ((threadIdx.x & 31) == 31) { wsum[threadIdx.x >> 5] = incl; wseg[threadIdx.x >> 5] = gincl; }
    __syncthreads();
    if (threadIdx.x < 32) {
      unsigned w = wsum[threadIdx.x], wi = w, q = wseg[threadIdx.x], qi = q;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        unsigned t = __shfl_up_sync(0xffffffffu, wi, o), tq = __shfl_up_sync(0xffffffffu, qi, o);
        if (threadIdx.x >= o) { wi += t; qi += tq; }
      }
      wsum[threadIdx.x] = wi - w; wseg[threadIdx.x] = qi - q;
    }
    __syncthreads();
    unsigned excl = carry + wsum[threadIdx.x >> 5] + (incl - v);
    unsigned gexcl = carry_seg + wseg[threadIdx.x >> 5] + (gincl - g);
    if (i < ntiles) {
      ranges[i] = v ? make_uint2(excl, excl + v) : make_uint2(0u, 0u);     // empty tiles report (0,0)
      cursor[i] = excl;
      seg_off[i] = gexcl;
    }
    __syncthreads();
    if (threadIdx.x == 1023) { carry = excl + v; carry_seg = gexcl + g; }
    __syncthreads();
  }
  __syncthreads();
  const bool overflow = total64 > (unsigned long long)capacity;
  if (overflow)                       // the key buffers cannot hold this frame: report it, render the background only
    for (int i = threadIdx.x; i < ntiles; i += 1024) { ranges[i] = make_uint2(0u, 0u); seg_off[i] = 0u; }
  if (threadIdx.x == 0) {
    if (overflow) atomicExch(status, RGA_ERR_CAPACITY);
    *num_dup = total64 > 0xffffffffull ? 0xffffffffu : carry;
    seg_off[ntiles] = overflow ? 0u : carry_seg;
    *num_items = overflow ? 0u : carry_seg;
  }
}

// scatter: every (Gaussian, tile) duplicate takes the next slot of its tile's bucket; the order inside a bucket is
// arbitrary here and fixed by the per-tile sort.  local key = depth bits << 32 | Gaussian index (the caller's).
__global__ void __launch_bounds__(256) tile_scatter_kernel(int ng, int TX, long long capacity, const unsigned* __restrict__ touched,
    const int4* __restrict__ rect, const float* __restrict__ depth, const int* __restrict__ order, unsigned* __restrict__ cursor,
    unsigned long long* __restrict__ lkeys) {
  int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ng || touched[g] == 0) return;
  int4 r = rect[g];
  // the low word is the CALLER's index of the Gaussian: equal (tile, depth) keys order by it (A22)
  unsigned long long key = ((unsigned long long)__float_as_uint(depth[g]) << 32) | (unsigned)order[g];
  const unsigned lane = threadIdx.x & 31;
  for (int y = r.y; y < r.w; ++y)
    for (int x = r.x; x < r.z; ++x) {
      // lanes of the warp that hit the same tile take consecutive slots from ONE atomic (spatially ordered Gaussians)
      const int tile = y * TX + x;
      // (correct for ANY converged subset of the warp: each peer set takes its own consecutive slots, and the order inside a bucket
      // is fixed by the per-tile sort, not here)
      const unsigned peers = __match_any_sync(__activemask(), tile);
      const int leader = __ffs(peers) - 1;
      unsigned base = 0;
      if ((int)lane == leader) base = atomicAdd(cursor + tile, (unsigned)__popc(peers));
      base = __shfl_sync(peers, base, leader);
      const unsigned pos = base + __popc(peers & ((1u << lane) - 1u));
      if ((long long)pos < capacity) lkeys[pos] = key;
    }
}

cudaError_t rga_launch_bin(rga_avatar* av, int TX, int ntiles, cudaStream_t s) {
  tile_scan_kernel<<<1, 1024, 0, s>>>(ntiles, av->max_dup, av->tile_count, av->ranges, av->cursor, av->num_dup, av->seg_off,
                                      av->num_items, av->status);
  rga_prof_mark(av, "tile_scan", s);
  tile_scatter_kernel<<<(av->n_gauss + 255) / 256, 256, 0, s>>>(av->n_gauss, TX, av->max_dup, av->touched, av->rect, av->depth,
                                                               av->g_order, av->cursor, av->keys[0]);
  rga_prof_mark(av, "tile_scatter", s);
  av->launches += 2;
  return cudaGetLastError();
}
