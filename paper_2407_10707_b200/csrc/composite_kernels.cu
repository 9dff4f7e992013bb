// H8 (depth digit) + H10: per-tile sort and front-to-back alpha compositing (PAPER.md:103 -> 3DGS rasteriser, DESIGN.md
// A18; black background PAPER.md:239-241 is the default of the bg parameter).
//
// The kernels (the first version did all of this in one CTA per tile and left the SMs 63 % idle: 208 active tiles on
// 148 SMs, each walking up to 1,304 entries serially -- profiles/r01a_ncu_full.md):
//   tile_sort_kernel        one CTA per tile: the tile's bucket of (depth bits << 32 | Gaussian) keys (binned by
//                           sort_kernels.cu) is sorted in shared memory by an ascending-only bitonic network (exact
//                           integer compare, so the order equals the stable (tile, depth) sort of the emission order)
//                           and written out as the sorted key/value lists; it also lists the tile's work items.
//                           Buckets beyond 2,048 entries: a per-tile LSD radix sort in L2 (radix_sort_tile), same launch.
//   composite_segment_kernel  front-to-back "over" is associative: (C,T) o (C',T') = (C + T C', T T').  A work item is
//                           one segment of RGA_SEG consecutive list entries of one tile; persistent CTAs blend every
//                           segment from T = 1 for the tile's 256 pixels, in parallel over all segments of all tiles.
//   composite_resolve_kernel  folds the segment partials of each pixel in order.  The 3DGS stopping rule (stop before
//                           the Gaussian that would take T below 1e-4) is not associative: a pixel whose running T
//                           times the next segment's T falls below the threshold stops folding and flags that segment.
//                           Also writes the background for empty tiles.
//   composite_replay_kernel   replays every flagged segment entry by entry with the exact rule for the pixels that
//                           stopped in it -- all flagged segments of the frame in parallel (inside one CTA per tile
//                           these serial replays took 209 us at config 1).  A warp ballot (lane = entry) first finds each
//                           pixel's contributing entries; the sequential rule then walks the set bits only.
// The blend is FAST arithmetic (FMA, ex2.approx): compared with the fp64 oracle under tolerance.
#include "rga_internal.h"

#define CB 256
#ifndef REPLAY_GRID_MULT
#define REPLAY_GRID_MULT 16
#endif
#ifndef SEGMENT_GRID_MULT
#define SEGMENT_GRID_MULT 8
#endif
#define SCAP_SMALL RGA_SORT_SMALL
#define LOG2E_F 1.4426950408889634f

// Ascending-only bitonic network on buf[0..n): every compare-exchange puts the minimum at the lower index, so virtual
// +inf padding above n never moves and n need not be a power of two.  One thread per PAIR (no idle half), and every
// stage whose partner distance is below 64 stays inside one warp's 64-element block and only needs __syncwarp: of the
// 66 stages of a 2,048-entry sort only 15 take a block barrier.
#define SORT_THREADS 512

__device__ __forceinline__ void cmpx(unsigned long long* buf, int i, int p, int n) {
  if (p < n) { const unsigned long long a = buf[i], b = buf[p]; if (b < a) { buf[i] = b; buf[p] = a; } }
}

// stages j = jmax .. 1 (jmax <= 32) of one 64-element block, by one warp; `mirror` makes the first stage i <-> i ^ (2 jmax - 1)
__device__ __forceinline__ void warp_stages(unsigned long long* buf, int base, int n, int jmax, bool mirror, int lane) {
  int j = jmax;
  if (mirror) {
    const int k = 2 * jmax, r = lane & (jmax - 1), blk = lane / jmax;            // pair `lane` of the 32 pairs of this block
    const int i = base + blk * k + r, p = base + blk * k + (k - 1 - r);
    cmpx(buf, i, p, n);
    __syncwarp();
    j >>= 1;
  }
  for (; j > 0; j >>= 1) {
    const int i = base + 2 * lane - (lane & (j - 1));
    cmpx(buf, i, i + j, n);
    __syncwarp();
  }
}

__device__ __forceinline__ void bitonic_sort(unsigned long long* buf, int n) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarps = SORT_THREADS / 32;
  // k = 2 .. 64: each 64-block on its own
  for (int base = warp * 64; base < n; base += nwarps * 64)
    for (int k = 2; k <= 64; k <<= 1) warp_stages(buf, base, n, k >> 1, true, lane);
  __syncthreads();
  for (int k = 128; (k >> 1) < n; k <<= 1) {
    const int half = k >> 1;
    const int npairs = ((n + k - 1) / k) * half;                                  // every k-block that holds an element
    for (int t = threadIdx.x; t < npairs; t += SORT_THREADS) {                    // mirror step: i <-> i ^ (k-1)
      const int blk = t / half, r = t - blk * half;
      cmpx(buf, blk * k + r, blk * k + (k - 1 - r), n);
    }
    __syncthreads();
    for (int j = k >> 2; j >= 64; j >>= 1) {
      for (int t = threadIdx.x; t * 2 < n; t += SORT_THREADS) {
        const int i = 2 * t - (t & (j - 1));
        cmpx(buf, i, i + j, n);
      }
      __syncthreads();
    }
    for (int base = warp * 64; base < n; base += nwarps * 64) warp_stages(buf, base, n, 32, false, lane);
    __syncthreads();
  }
}

__device__ __forceinline__ void sort_tile(int tile, unsigned capacity, int scap, unsigned long long* s_keys,
    const uint2* __restrict__ ranges, const unsigned* __restrict__ seg_off, unsigned long long* __restrict__ lkeys,
    unsigned long long* __restrict__ keys_out, unsigned* __restrict__ vals_out, unsigned* __restrict__ vals_int,
    const int* __restrict__ inv, unsigned* __restrict__ item_tab, uint2* __restrict__ item_desc) {
  uint2 rg = ranges[tile];
  rg.x = min(rg.x, capacity); rg.y = min(rg.y, capacity);
  const int n = (int)(rg.y - rg.x);
  const unsigned so = seg_off[tile];
  for (int j = threadIdx.x; j < (n + RGA_SEG - 1) / RGA_SEG; j += SORT_THREADS) {
    item_tab[so + j] = (unsigned)tile;
    // what the blend needs to know about the item, in one load: first list entry; tile | entries << 24
    item_desc[so + j] = make_uint2(rg.x + (unsigned)j * RGA_SEG, (unsigned)tile | ((unsigned)min(RGA_SEG, n - j * RGA_SEG) << 24));
  }
  unsigned long long* buf = lkeys + rg.x;
  if (n <= scap) {
    for (int i = threadIdx.x; i < n; i += SORT_THREADS) s_keys[i] = buf[i];
    buf = s_keys;
  }
  __syncthreads();
  bitonic_sort(buf, n);
  for (int i = threadIdx.x; i < n; i += SORT_THREADS) {      // the sorted (tile, depth) keys and values (H8 output)
    const unsigned long long k = buf[i];
    keys_out[rg.x + i] = ((unsigned long long)(unsigned)tile << 32) | (k >> 32);
    vals_out[rg.x + i] = (unsigned)k;                               // caller's index (H8 output)
    vals_int[rg.x + i] = (unsigned)inv[(unsigned)k];                // the same Gaussian in library order (what the blend reads)
  }
  __syncthreads();
}

// Tiles with more than SCAP_SMALL entries (none at config 1, lists up to 8,688 at config 4):
// LSD radix sort of the tile's 64-bit keys, 8 bits per pass, by one CTA per tile, ping-ponging between the bucket buffer and
// the tile's own slice of keys_out (both in L2).  The list is cut into one contiguous part per warp; a pass is (1) per-warp
// digit histograms, (2) a scan in (digit, warp) order, (3) a stable scatter in which every warp walks its part in order and
// ranks equal digits inside a 32-key batch with match.any.  A pass whose digit is the same for every key (the upper index
// bytes, the exponent byte of the depth) is skipped after its histogram.  The histograms live in the 16 KB the short tiles
// use for their keys, so one launch sorts every tile (a separate long-list kernel with 192 KB of shared memory came before:
// it had to wait for an empty SM even with nothing to sort, at the end of the chain the blend waits for).
// Keys are distinct (the low word is the Gaussian's index), so the result is THE ascending order, as the bitonic network's.
#define RADIX_WARPS (SORT_THREADS / 32)
#ifndef RADIX_UNROLL
#define RADIX_UNROLL 4
#endif
__device__ __forceinline__ void radix_sort_tile(int tile, unsigned capacity, int idx_bits, unsigned* s_hist /*[RADIX_WARPS][256]*/,
    unsigned* s_base /*[256]*/, int* s_flag, const uint2* __restrict__ ranges, const unsigned* __restrict__ seg_off,
    unsigned long long* __restrict__ lkeys, unsigned long long* __restrict__ keys_out, unsigned* __restrict__ vals_out,
    unsigned* __restrict__ vals_int, const int* __restrict__ inv, unsigned* __restrict__ item_tab, uint2* __restrict__ item_desc) {
  uint2 rg = ranges[tile];
  rg.x = min(rg.x, capacity); rg.y = min(rg.y, capacity);
  const int n = (int)(rg.y - rg.x);
  const unsigned so = seg_off[tile];
  for (int j = threadIdx.x; j < (n + RGA_SEG - 1) / RGA_SEG; j += SORT_THREADS) {
    item_tab[so + j] = (unsigned)tile;
    // what the blend needs to know about the item, in one load: first list entry; tile | entries << 24
    item_desc[so + j] = make_uint2(rg.x + (unsigned)j * RGA_SEG, (unsigned)tile | ((unsigned)min(RGA_SEG, n - j * RGA_SEG) << 24));
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const unsigned lt = (1u << lane) - 1u;
  const int per = (((n + RADIX_WARPS - 1) / RADIX_WARPS) + 31) & ~31;          // whole batches per warp
  const int lo = min(n, warp * per), hi = min(n, lo + per);
  unsigned long long* src = lkeys + rg.x;
  unsigned long long* dst = keys_out + rg.x;
  unsigned* hist = s_hist + warp * 256;
  const int idx_passes = (idx_bits + 7) >> 3;
  for (int pass = 0; pass < idx_passes + 4; ++pass) {
    const int shift = pass < idx_passes ? 8 * pass : 32 + 8 * (pass - idx_passes);
    for (int t = threadIdx.x; t < RADIX_WARPS * 256; t += SORT_THREADS) s_hist[t] = 0u;
    if (threadIdx.x == 0) *s_flag = 0;
    __syncthreads();
    // (1) histogram of my part; RADIX_UNROLL batches are requested before the first is used (the loop is a chain of L2 trips)
    for (int b = lo; b < hi; b += 32 * RADIX_UNROLL) {
      unsigned long long kk[RADIX_UNROLL];
#pragma unroll
      for (int u = 0; u < RADIX_UNROLL; ++u) { const int i = b + 32 * u + lane; kk[u] = i < hi ? src[i] : 0ull; }
#pragma unroll
      for (int u = 0; u < RADIX_UNROLL; ++u) {
        const bool act = b + 32 * u + lane < hi;
        const unsigned am = __ballot_sync(0xffffffffu, act);
        if (act) {
          const unsigned d = (unsigned)(kk[u] >> shift) & 255u;
          const unsigned m = __match_any_sync(am, d);
          if ((m & lt) == 0u) hist[d] += (unsigned)__popc(m);                   // lowest lane of each digit group; one warp per row
        }
        __syncwarp();
      }
    }
    __syncthreads();
    // (2) exclusive scan in (digit, warp) order: s_hist[w][d] <- keys of digit d in warps before w; s_base[d] <- keys of digits < d
    if (threadIdx.x < 256) {
      unsigned run = 0u;
      for (int w = 0; w < RADIX_WARPS; ++w) { const unsigned c = s_hist[w * 256 + threadIdx.x]; s_hist[w * 256 + threadIdx.x] = run; run += c; }
      s_base[threadIdx.x] = run;
      if (run == (unsigned)n) *s_flag = 1;                                       // every key has this digit: nothing to move
    }
    __syncthreads();
    if (*s_flag) { __syncthreads(); continue; }
    if (warp == 0) {
      unsigned v[8], sum = 0u;
#pragma unroll
      for (int e = 0; e < 8; ++e) { v[e] = s_base[lane * 8 + e]; sum += v[e]; }
      unsigned inc = sum;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { const unsigned u = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += u; }
      unsigned ex = inc - sum;
#pragma unroll
      for (int e = 0; e < 8; ++e) { s_base[lane * 8 + e] = ex; ex += v[e]; }
    }
    __syncthreads();
    // (3) stable scatter
    for (int b = lo; b < hi; b += 32 * RADIX_UNROLL) {
      unsigned long long kk[RADIX_UNROLL];
#pragma unroll
      for (int u = 0; u < RADIX_UNROLL; ++u) { const int i = b + 32 * u + lane; kk[u] = i < hi ? src[i] : 0ull; }
#pragma unroll
      for (int u = 0; u < RADIX_UNROLL; ++u) {
        const bool act = b + 32 * u + lane < hi;
        const unsigned am = __ballot_sync(0xffffffffu, act);
        const unsigned long long k = kk[u];
        unsigned d = 0u, m = 0u, off = 0u;
        if (act) {
          d = (unsigned)(k >> shift) & 255u;
          m = __match_any_sync(am, d);
          off = hist[d];
        }
        __syncwarp();
        if (act) {
          if ((m & lt) == 0u) hist[d] = off + (unsigned)__popc(m);
          dst[s_base[d] + off + (unsigned)__popc(m & lt)] = k;
        }
        __syncwarp();
      }
    }
    __syncthreads();
    unsigned long long* t = src; src = dst; dst = t;
  }
  // H8 output from the sorted keys (in place when they ended in the tile's slice of keys_out: one element per thread)
  for (int i = threadIdx.x; i < n; i += SORT_THREADS) {
    const unsigned long long k = src[i];
    keys_out[rg.x + i] = ((unsigned long long)(unsigned)tile << 32) | (k >> 32);
    vals_out[rg.x + i] = (unsigned)k;
    vals_int[rg.x + i] = (unsigned)inv[(unsigned)k];
  }
  __syncthreads();
}

// one CTA per tile: bitonic in shared memory up to SCAP_SMALL entries, the radix sort above beyond
__global__ void __launch_bounds__(SORT_THREADS) tile_sort_kernel(unsigned capacity, int scap, int idx_bits,
    const uint2* __restrict__ ranges, const unsigned* __restrict__ seg_off, unsigned long long* __restrict__ lkeys,
    unsigned long long* __restrict__ keys_out, unsigned* __restrict__ vals_out, unsigned* __restrict__ vals_int,
    const int* __restrict__ inv, unsigned* __restrict__ item_tab, uint2* __restrict__ item_desc) {
  extern __shared__ __align__(16) unsigned long long s_keys[];                   // scap keys, or RADIX_WARPS x 256 counters
  __shared__ unsigned s_base[256];
  __shared__ int s_flag;
  const uint2 rg = ranges[blockIdx.x];
  const unsigned n = min(rg.y, capacity) - min(rg.x, capacity);
  if (n == 0) return;
  if (n > (unsigned)scap)
    radix_sort_tile(blockIdx.x, capacity, idx_bits, reinterpret_cast<unsigned*>(s_keys), s_base, &s_flag, ranges, seg_off, lkeys, keys_out,
                    vals_out, vals_int, inv, item_tab, item_desc);
  else
    sort_tile(blockIdx.x, capacity, scap, s_keys, ranges, seg_off, lkeys, keys_out, vals_out, vals_int, inv, item_tab, item_desc);
}

// Thread -> pixel of the 16x16 tile: a warp owns an 8x4 block of pixels (2 x 4 blocks per tile), so that a Gaussian
// whose footprint misses the block is skipped by the whole warp.
__device__ __forceinline__ int tile_px(unsigned t) { return (int)(((t >> 5) & 1u) * 8u + (t & 7u)); }
__device__ __forceinline__ int tile_py(unsigned t) { return (int)((t >> 6) * 4u + ((t >> 3) & 3u)); }

// shared-memory staging of one segment: centre, conic pre-scaled so that alpha = o * 2^(x(A x + B y) + C y^2), colour,
// and the half-extents of the bounding box of the region where alpha can reach 1/255
struct SegStage { float2 mu[RGA_SEG]; float4 co[RGA_SEG]; float4 col[RGA_SEG]; float2 ext[RGA_SEG]; };

__device__ __forceinline__ float ex2_approx(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

__device__ __forceinline__ void stage_segment(SegStage& st, int m, const unsigned* __restrict__ vals, const float2* __restrict__ mu2d,
                                              const float4* __restrict__ conic_o, const float4* __restrict__ color) {
  if ((int)threadIdx.x < m) {
    const unsigned g = vals[threadIdx.x];
    const float4 c = conic_o[g];
    st.mu[threadIdx.x] = mu2d[g];
    st.co[threadIdx.x] = make_float4(-0.5f * LOG2E_F * c.x, -LOG2E_F * c.y, -0.5f * LOG2E_F * c.z, c.w);
    st.col[threadIdx.x] = color[g];
    // alpha >= 1/255  <=>  d^T Q d <= 2 ln(255 o), Q = conic: an ellipse whose bounding box has half-extents
    // sqrt(2 L (Q^-1)_xx), sqrt(2 L (Q^-1)_yy); padded by 0.1 % + 0.01 px against rounding (such pixels have alpha ~ 1/255)
    const float L2 = 2.0f * __logf(255.0f * c.w), det = c.x * c.z - c.y * c.y;
    float hx = -1.f, hy = -1.f;                                          // opacity below 1/255: never contributes
    if (L2 > 0.f && det > 0.f) { hx = sqrtf(L2 * c.z / det) * 1.001f + 0.01f; hy = sqrtf(L2 * c.x / det) * 1.001f + 0.01f; }
    st.ext[threadIdx.x] = make_float2(hx, hy);
  }
}

// alpha of entry j at pixel centre (fx, fy); 0 when the 3DGS rules skip it (power > 0, alpha < 1/255)
__device__ __forceinline__ float seg_alpha(const SegStage& st, int j, float fx, float fy) {
  const float2 mm = st.mu[j]; const float4 co = st.co[j];
  const float dx = mm.x - fx, dy = mm.y - fy;
  // log2(e) * power; the contraction is written out so that every inlined copy rounds alike (the replay evaluates an alpha twice)
  const float p2 = fmaf(dx, fmaf(co.x, dx, co.y * dy), (co.z * dy) * dy);
  const float al = fminf(0.99f, co.w * ex2_approx(p2));
  return (p2 > 0.f || al < 1.f / 255.f) ? 0.f : al;
}

#ifndef SEG_MINB
#define SEG_MINB 8             // 8 CTAs per SM resident: caps the kernel at 32 registers (33.8 -> 32.9 us)
#endif
__global__ void __launch_bounds__(CB, SEG_MINB) composite_segment_kernel(int W, int H, int TX, const unsigned* __restrict__ num_items,
    const uint2* __restrict__ item_desc,
    const unsigned* __restrict__ vals, const float2* __restrict__ mu2d, const float4* __restrict__ conic_o,
    const float4* __restrict__ color, float4* __restrict__ part, unsigned* __restrict__ part_last, unsigned* __restrict__ counter) {
  __shared__ SegStage st;
  __shared__ unsigned s_bm[CB / 32][RGA_SEG / 32];                  // per 8x4 pixel block (= warp): the entries whose box reaches it
  __shared__ unsigned s_item;
  const unsigned n_items = *num_items;
  // Large frames (more than two items per CTA) draw their items from a counter: an item's cost differs several-fold with the
  // number of entries that reach the tile's blocks, and with a fixed stride the slowest CTAs set the time (config 4: 344 ->
  // 284 us, config 2: 107 -> 92 us).  The next ticket is drawn before the current item is worked on, so the atomic's round trip
  // is hidden; every CTA draws one ticket beyond the items and the last one re-arms the counter.  With one or two items per
  // CTA (config 1) the tickets only cost: 28.6 -> 33.5 us, so small frames keep the fixed stride.
  const bool dynamic = n_items > 2u * gridDim.x;
  unsigned next = blockIdx.x;
  if (dynamic && threadIdx.x == 0) next = atomicAdd(counter, 1u);
  for (;;) {
    unsigned item = next;
    if (dynamic) {
      if (threadIdx.x == 0) s_item = next;
      __syncthreads();                                                // also: the previous item's walk is done with `st`
      item = s_item;
      if (item >= n_items) {
        if (threadIdx.x == 0 && item == n_items + gridDim.x - 1u) *counter = 0u;
        break;
      }
      if (threadIdx.x == 0) next = atomicAdd(counter, 1u);
    } else {
      if (item >= n_items) break;
      next = item + gridDim.x;
      __syncthreads();
    }
    const uint2 desc = item_desc[item];
    const unsigned tile = desc.y & 0xffffffu, b0 = desc.x;
    const int m = (int)(desc.y >> 24);
    stage_segment(st, m, vals + b0, mu2d, conic_o, color);
    // Which entries can reach which of the tile's eight 8x4 pixel blocks: the staging thread of entry j tests its bounding box
    // against the eight block centres (pixel centres lie at +-3.5, +-1.5 around it) and the bits are transposed by ballots
    // into one mask of entries per block.  A warp then walks the set bits of its own block's mask only -- an entry that
    // misses the block costs nothing (it used to cost the test, per warp and entry: 60 % of the entries at config 1).
    if (threadIdx.x < RGA_SEG) {
      unsigned reach = 0u;
      if ((int)threadIdx.x < m) {
        const float2 mm = st.mu[threadIdx.x], ex = st.ext[threadIdx.x];
        const float cx0 = (float)((int)(tile % TX) * RGA_TILE) + 4.0f, cy0 = (float)((int)(tile / TX) * RGA_TILE) + 2.0f;
#pragma unroll
        for (int b = 0; b < CB / 32; ++b) {
          const float bcx = cx0 + 8.0f * (float)(b & 1), bcy = cy0 + 4.0f * (float)(b >> 1);
          if (!(fabsf(mm.x - bcx) > ex.x + 3.5f || fabsf(mm.y - bcy) > ex.y + 1.5f)) reach |= 1u << b;
        }
      }
#pragma unroll
      for (int b = 0; b < CB / 32; ++b) {
        const unsigned bal = __ballot_sync(0xffffffffu, (reach >> b) & 1u);
        if ((threadIdx.x & 31u) == 0u) s_bm[b][threadIdx.x >> 5] = bal;
      }
    }
    __syncthreads();
    const int px = (int)(tile % TX) * RGA_TILE + tile_px(threadIdx.x), py = (int)(tile / TX) * RGA_TILE + tile_py(threadIdx.x);
    const float fx = (float)px + 0.5f, fy = (float)py + 0.5f;        // DESIGN.md A21: sample at the pixel centre
    float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
    unsigned last = 0;
    bool stop = !(px < W && py < H);
#pragma unroll
    for (int h = 0; h < RGA_SEG / 32; ++h) {
      unsigned mk = s_bm[threadIdx.x >> 5][h];
      while (mk != 0u) {
        // two entries per trip: their alphas are independent, the blend is sequential
        const int j0 = h * 32 + __ffs((int)mk) - 1; mk &= mk - 1u;
        const int j1 = mk ? h * 32 + __ffs((int)mk) - 1 : -1; mk &= mk - 1u;
        const float a0 = seg_alpha(st, j0, fx, fy);
        const float a1 = j1 >= 0 ? seg_alpha(st, j1, fx, fy) : 0.f;
        if (!stop && a0 > 0.f) {
          const float test_T = T * (1.f - a0);
          // below the threshold from T = 1 means below it from any start: the resolve pass replays this segment
          if (test_T < 1e-4f) { stop = true; T = 0.f; }
          else {
            const float4 c = st.col[j0];
            const float w = a0 * T;
            C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
            T = test_T; last = (unsigned)(j0 + 1);
          }
        }
        if (!stop && a1 > 0.f) {
          const float test_T = T * (1.f - a1);
          if (test_T < 1e-4f) { stop = true; T = 0.f; }
          else {
            const float4 c = st.col[j1];
            const float w = a1 * T;
            C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
            T = test_T; last = (unsigned)(j1 + 1);
          }
        }
      }
    }
    part[(size_t)item * CB + threadIdx.x] = make_float4(C0, C1, C2, T);
    part_last[(size_t)item * CB + threadIdx.x] = last;
  }
}

// one entry of the exact sequential rule, read straight from global memory (rare continuation path of the replay)
__device__ __forceinline__ float global_alpha(unsigned g, float fx, float fy, const float2* __restrict__ mu2d,
                                              const float4* __restrict__ conic_o) {
  const float2 mm = mu2d[g]; const float4 c = conic_o[g];
  const float dx = mm.x - fx, dy = mm.y - fy;
  const float p2 = dx * ((-0.5f * LOG2E_F * c.x) * dx + (-LOG2E_F * c.y) * dy) + (-0.5f * LOG2E_F * c.z) * dy * dy;
  const float al = fminf(0.99f, c.w * exp2f(p2));
  return (p2 > 0.f || al < 1.f / 255.f) ? 0.f : al;
}

// Folds the segment partials of each pixel in order (no shared memory, no barrier).  A pixel whose running T times the
// next segment's T falls below the stopping threshold stops folding there: its accumulated (C, T, last) are written
// out as they stand, the segment index goes to stop_seg and the work item is flagged for composite_replay_kernel.
__global__ void __launch_bounds__(CB) composite_resolve_kernel(int W, int H, int TX, unsigned capacity,
    const uint2* __restrict__ ranges, const unsigned* __restrict__ seg_off, const float4* __restrict__ part,
    const unsigned* __restrict__ part_last, float3 bg, float* __restrict__ image, float* __restrict__ t_final,
    unsigned* __restrict__ n_contrib, int* __restrict__ stop_seg, unsigned char* __restrict__ item_flag) {
  const int tile = blockIdx.y * TX + blockIdx.x;
  uint2 rg = ranges[tile];
  rg.x = min(rg.x, capacity); rg.y = min(rg.y, capacity);
  const int n = (int)(rg.y - rg.x), nseg = (n + RGA_SEG - 1) / RGA_SEG;
  const unsigned so = seg_off[tile];
  const int px = blockIdx.x * RGA_TILE + tile_px(threadIdx.x), py = blockIdx.y * RGA_TILE + tile_py(threadIdx.x);
  if (!(px < W && py < H)) return;
  float T = 1.f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
  unsigned last = 0;
  int stop = -1;
  const float4* pp = part + (size_t)so * CB + threadIdx.x;
  const unsigned* pl = part_last + (size_t)so * CB + threadIdx.x;
  for (int s0 = 0; s0 < nseg && stop < 0; s0 += 4) {       // four segments per trip: their loads are independent
    float4 p[4]; unsigned l[4];
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (s0 + u < nseg) { p[u] = pp[(size_t)(s0 + u) * CB]; l[u] = pl[(size_t)(s0 + u) * CB]; }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      if (s0 + u < nseg && stop < 0) {
        if (T * p[u].w >= 1.00001e-4f) {                   // the whole segment passes the stopping rule
          C0 = fmaf(T, p[u].x, C0); C1 = fmaf(T, p[u].y, C1); C2 = fmaf(T, p[u].z, C2);
          T *= p[u].w;
          if (l[u]) last = (unsigned)((s0 + u) * RGA_SEG) + l[u];
        } else stop = s0 + u;
      }
    }
  }
  const size_t p = (size_t)py * W + px;
  if (stop >= 0) {                                         // unfinished: background is added by the replay
    image[3 * p] = C0; image[3 * p + 1] = C1; image[3 * p + 2] = C2;
    item_flag[so + stop] = 1;
  } else {
    image[3 * p] = C0 + T * bg.x; image[3 * p + 1] = C1 + T * bg.y; image[3 * p + 2] = C2 + T * bg.z;
  }
  t_final[p] = T; n_contrib[p] = last; stop_seg[p] = stop;
}

// Replays flagged segments entry by entry with the exact 3DGS stopping rule for the pixels that stopped in them, all
// flagged (tile, segment) items of the frame in parallel.
__global__ void __launch_bounds__(CB) composite_replay_kernel(int W, int H, int TX, const unsigned* __restrict__ num_items,
    const unsigned* __restrict__ item_tab, const unsigned* __restrict__ seg_off, const uint2* __restrict__ ranges,
    const unsigned* __restrict__ vals, const float2* __restrict__ mu2d, const float4* __restrict__ conic_o,
    const float4* __restrict__ color, float3 bg, float* __restrict__ image, float* __restrict__ t_final,
    unsigned* __restrict__ n_contrib, const int* __restrict__ stop_seg, unsigned char* __restrict__ item_flag) {
  __shared__ SegStage st;
  __shared__ int s_cnt;
  __shared__ unsigned short s_pix[CB];
  __shared__ unsigned s_mask[CB][RGA_SEG / 32];
  const unsigned n_items = *num_items;
  for (unsigned item = blockIdx.x; item < n_items; item += gridDim.x) {
    if (!item_flag[item]) continue;                        // block-uniform
    __syncthreads();
    if (threadIdx.x == 0) { item_flag[item] = 0; s_cnt = 0; }   // flag re-armed for the next frame
    const unsigned tile = item_tab[item];
    const int seg = (int)(item - seg_off[tile]);
    const uint2 rg = ranges[tile];
    const int n = (int)(rg.y - rg.x);
    const int m = min(RGA_SEG, n - seg * RGA_SEG);
    stage_segment(st, m, vals + rg.x + seg * RGA_SEG, mu2d, conic_o, color);
    __syncthreads();
    // the pixels of the tile that stop in this segment are usually a minority: compact them so that whole warps
    // either replay or leave (7 of 32 lanes were active before)
    {
      const int qx = (int)(tile % TX) * RGA_TILE + tile_px(threadIdx.x), qy = (int)(tile / TX) * RGA_TILE + tile_py(threadIdx.x);
      if (qx < W && qy < H && stop_seg[(size_t)qy * W + qx] == seg) s_pix[atomicAdd(&s_cnt, 1)] = (unsigned short)threadIdx.x;
    }
    __syncthreads();
    // few pixels replay, so latency rules.  Phase 1, all warps: a warp takes one stopping pixel at a time and evaluates the
    // segment's entries one per lane; the ballot of alpha > 0 is the pixel's list of contributing entries (about one in
    // eight).  Phase 2, one thread per pixel: the sequential rule over the set bits only, four alphas per trip (the same
    // seg_alpha on the same operands, so the same values as in phase 1).
    const int cnt = s_cnt;
    const int tx0 = (int)(tile % TX) * RGA_TILE, ty0 = (int)(tile / TX) * RGA_TILE;
    for (int i = (int)(threadIdx.x >> 5); i < cnt; i += CB / 32) {
      const unsigned qq = s_pix[i];
      const float gx = (float)(tx0 + tile_px(qq)) + 0.5f, gy = (float)(ty0 + tile_py(qq)) + 0.5f;
#pragma unroll
      for (int h = 0; h < RGA_SEG / 32; ++h) {
        const int j = h * 32 + (int)(threadIdx.x & 31u);
        const float a = j < m ? seg_alpha(st, j, gx, gy) : 0.f;
        const unsigned mk = __ballot_sync(0xffffffffu, a > 0.f);
        if ((threadIdx.x & 31u) == 0) s_mask[i][h] = mk;
      }
    }
    __syncthreads();
    if ((int)threadIdx.x >= cnt) continue;
    const unsigned q = s_pix[threadIdx.x];
    const int px = tx0 + tile_px(q), py = ty0 + tile_py(q);
    const size_t p = (size_t)py * W + px;
    const float fx = (float)px + 0.5f, fy = (float)py + 0.5f;
    float T = t_final[p], C0 = image[3 * p], C1 = image[3 * p + 1], C2 = image[3 * p + 2];
    unsigned last = n_contrib[p];
    bool done = false;
#pragma unroll
    for (int h = 0; h < RGA_SEG / 32; ++h) {
      unsigned mk = s_mask[threadIdx.x][h];
      while (mk != 0u && !done) {
        int jj[4]; float a[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { jj[u] = mk ? h * 32 + __ffs((int)mk) - 1 : -1; mk &= mk - 1u; }
#pragma unroll
        for (int u = 0; u < 4; ++u) a[u] = jj[u] >= 0 ? seg_alpha(st, jj[u], fx, fy) : 0.f;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          if (!done && a[u] > 0.f) {
            const float test_T = T * (1.f - a[u]);
            if (test_T < 1e-4f) done = true;
            else {
              const float4 c = st.col[jj[u]];
              const float w = a[u] * T;
              C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
              T = test_T; last = (unsigned)(seg * RGA_SEG + jj[u] + 1);
            }
          }
        }
      }
    }
    // the fold's threshold has a 1e-5 relative guard band: a pixel inside it may not stop here after all and walks the
    // rest of its list from global memory (rare)
    for (int i = (seg + 1) * RGA_SEG; i < n && !done; ++i) {
      const unsigned g = vals[rg.x + i];
      const float a = global_alpha(g, fx, fy, mu2d, conic_o);
      if (a > 0.f) {
        const float test_T = T * (1.f - a);
        if (test_T < 1e-4f) { done = true; break; }
        const float4 c = color[g];
        const float w = a * T;
        C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
        T = test_T; last = (unsigned)(i + 1);
      }
    }
    image[3 * p] = C0 + T * bg.x; image[3 * p + 1] = C1 + T * bg.y; image[3 * p + 2] = C2 + T * bg.z;
    t_final[p] = T; n_contrib[p] = last;
  }
}


int rga_composite_init_attributes() {
  return 0;                                                      // no kernel here needs more than the default 48 KB
}

// Attribute maps (PAPER.md:177 albedo map for editing; PAPER.md:239 albedo and normal maps for the metrics): the colour
// that is splatted is the Gaussian's albedo a_g or its posed normal n_gd instead of the shaded colour.
__global__ void attr_color_kernel(int ng, int which, const float4* __restrict__ g_static, const float4* __restrict__ g_nposed,
                                  float4* __restrict__ out) {
  const int g = blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= ng) return;
  const float4 v = which == 1 ? g_static[4 * (size_t)g + 2] : g_nposed[g];
  out[g] = make_float4(v.x, v.y, v.z, 0.f);
}

cudaError_t rga_launch_attr_color(rga_avatar* av, int which, cudaStream_t s) {
  attr_color_kernel<<<(av->n_gauss + 255) / 256, 256, 0, s>>>(av->n_gauss, which, av->g_static, av->g_nposed, av->attr_color);
  rga_prof_mark(av, "attr_color", s);
  av->launches += 1;
  return cudaGetLastError();
}

// H8 second digit: per-tile sort of the binned keys (needs only the projection, not the shading)
cudaError_t rga_launch_tile_sort(rga_avatar* av, const rga_camera* cam, cudaStream_t s) {
  const int TX = (cam->width + RGA_TILE - 1) / RGA_TILE, TY = (cam->height + RGA_TILE - 1) / RGA_TILE;
  const int ntiles = TX * TY;
  static_assert(SCAP_SMALL * 8 >= RADIX_WARPS * 256 * 4, "the radix histograms reuse the key buffer");
  int idx_bits = 1; while (idx_bits < 32 && (1ll << idx_bits) < (long long)av->n_gauss) ++idx_bits;
  tile_sort_kernel<<<ntiles, SORT_THREADS, SCAP_SMALL * 8, s>>>((unsigned)av->max_dup, SCAP_SMALL, idx_bits, av->ranges, av->seg_off, av->keys[0],
                                                           av->keys[1], av->vals[0], av->vals[1], av->g_inv, av->item_tab, av->item_desc);
  rga_prof_mark(av, "tile_sort", s);
  av->launches += 1;
  return cudaGetLastError();
}

// H10: blend (needs the sorted lists and the shaded colours)
cudaError_t rga_launch_composite(rga_avatar* av, const rga_camera* cam, float3 bg, const float4* color, float* out, cudaStream_t s) {
  const int TX = (cam->width + RGA_TILE - 1) / RGA_TILE, TY = (cam->height + RGA_TILE - 1) / RGA_TILE;
  composite_segment_kernel<<<av->num_sms * SEGMENT_GRID_MULT, CB, 0, s>>>(cam->width, cam->height, TX, av->num_items, av->item_desc,
      av->vals[1], av->mu2d, av->conic_o, color, av->part, av->part_last, av->seg_counter);
  rga_prof_mark(av, "composite_segments", s);
  composite_resolve_kernel<<<dim3(TX, TY), CB, 0, s>>>(cam->width, cam->height, TX, (unsigned)av->max_dup, av->ranges, av->seg_off,
      av->part, av->part_last, bg, out, av->t_final, av->n_contrib, av->stop_seg, av->item_flag);
  rga_prof_mark(av, "composite_resolve", s);
  composite_replay_kernel<<<av->num_sms * REPLAY_GRID_MULT, CB, 0, s>>>(cam->width, cam->height, TX, av->num_items, av->item_tab, av->seg_off,
      av->ranges, av->vals[1], av->mu2d, av->conic_o, color, bg, out, av->t_final, av->n_contrib, av->stop_seg, av->item_flag);
  rga_prof_mark(av, "composite_replay", s);
  av->launches += 3;
  return cudaGetLastError();
}
