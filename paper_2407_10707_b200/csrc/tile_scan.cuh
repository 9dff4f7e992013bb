// The tile digit's exclusive scan (H7 / H9; see sort_kernels.cu): per-tile counts n_t -> ranges, scatter cursors, D and the capacity
// check; per-tile segment counts ceil(n_t / RGA_SEG) -> segment offsets and the number of compositing work items.  Run by ONE
// CTA of THREADS threads: the CTA of project_kernel that finishes the histogram last (as a launch of its own -- one CTA of 1,024
// threads -- it had to wait until an SM had drained all four of its fused-kernel CTAs, and the blend waited for the chain behind it).
// Integer-only.  tile_count is read through L2 (written by other CTAs' atomics in the same launch).
#pragma once
#include "rga_internal.h"

template <int THREADS>
__device__ __forceinline__ void rga_tile_scan(int ntiles, long long capacity, const unsigned* tile_count, uint2* __restrict__ ranges,
    unsigned* __restrict__ cursor, unsigned* __restrict__ num_dup, unsigned* __restrict__ seg_off, unsigned* __restrict__ num_items,
    int* __restrict__ status) {
  constexpr int NW = THREADS / 32;
  __shared__ unsigned wsum[32], wseg[32];
  __shared__ unsigned carry, carry_seg;
  __shared__ unsigned long long total64;                  // D in 64 bits: the 32-bit running sum may wrap before the capacity check
  if (threadIdx.x == 0) { carry = 0; carry_seg = 0; total64 = 0ull; }
  __syncthreads();
  constexpr int IPT = 4;                                  // consecutive tiles per thread and trip (1,024 tiles per trip of 256 threads)
  for (int base = 0; base < ntiles; base += THREADS * IPT) {
    const int i0 = base + threadIdx.x * IPT;
    unsigned v[IPT], g[IPT], vsum = 0u, gsum = 0u;
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
      v[k] = (i0 + k < ntiles) ? __ldcg(tile_count + i0 + k) : 0u;
      g[k] = (v[k] + RGA_SEG - 1) / RGA_SEG;
      vsum += v[k]; gsum += g[k];
    }
    unsigned incl = vsum, gincl = gsum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      unsigned t = __shfl_up_sync(0xffffffffu, incl, o), tg = __shfl_up_sync(0xffffffffu, gincl, o);
      if ((threadIdx.x & 31) >= o) { incl += t; gincl += tg; }
    }
    {
      unsigned long long v64 = 0ull;
#pragma unroll
      for (int k = 0; k < IPT; ++k) v64 += v[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v64 += __shfl_xor_sync(0xffffffffu, v64, o);
      if ((threadIdx.x & 31) == 0 && v64) atomicAdd(&total64, v64);
    }
    if ((threadIdx.x & 31) == 31) { wsum[threadIdx.x >> 5] = incl; wseg[threadIdx.x >> 5] = gincl; }
    __syncthreads();
    if (threadIdx.x < 32) {
      unsigned w = threadIdx.x < NW ? wsum[threadIdx.x] : 0u, wi = w, q = threadIdx.x < NW ? wseg[threadIdx.x] : 0u, qi = q;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        unsigned t = __shfl_up_sync(0xffffffffu, wi, o), tq = __shfl_up_sync(0xffffffffu, qi, o);
        if (threadIdx.x >= o) { wi += t; qi += tq; }
      }
      wsum[threadIdx.x] = wi - w; wseg[threadIdx.x] = qi - q;
    }
    __syncthreads();
    unsigned excl = carry + wsum[threadIdx.x >> 5] + (incl - vsum);
    unsigned gexcl = carry_seg + wseg[threadIdx.x >> 5] + (gincl - gsum);
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
      if (i0 + k < ntiles) {
        ranges[i0 + k] = v[k] ? make_uint2(excl, excl + v[k]) : make_uint2(0u, 0u);     // empty tiles report (0,0)
        cursor[i0 + k] = excl;
        seg_off[i0 + k] = gexcl;
      }
      excl += v[k]; gexcl += g[k];
    }
    __syncthreads();
    if (threadIdx.x == THREADS - 1) { carry = excl; carry_seg = gexcl; }
    __syncthreads();
  }
  __syncthreads();
  const bool overflow = total64 > (unsigned long long)capacity;
  if (overflow)                       // the key buffers cannot hold this frame: report it, render the background only
    for (int i = threadIdx.x; i < ntiles; i += THREADS) { ranges[i] = make_uint2(0u, 0u); seg_off[i] = 0u; }
  if (threadIdx.x == 0) {
    if (overflow) atomicExch(status, RGA_ERR_CAPACITY);
    *num_dup = total64 > 0xffffffffull ? 0xffffffffu : carry;
    seg_off[ntiles] = overflow ? 0u : carry_seg;
    *num_items = overflow ? 0u : carry_seg;
  }
}
