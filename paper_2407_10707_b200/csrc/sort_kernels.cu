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

// (the exclusive scans of the per-tile counts and segment counts: tile_scan.cuh, run by the last CTA of project_kernel)

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
  tile_scatter_kernel<<<(av->n_gauss + 255) / 256, 256, 0, s>>>(av->n_gauss, TX, av->max_dup, av->touched, av->rect, av->depth,
                                                               av->g_order, av->cursor, av->keys[0]);
  rga_prof_mark(av, "tile_scatter", s);
  av->launches += 1;
  return cudaGetLastError();
}
