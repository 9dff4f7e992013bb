// Displacement MLP d(x, theta) ("dx = d(x, theta) ... d is a multilayer perceptron", "four
// layers, each with a width of 256 and activated by ReLU", "Random Fourier Features"; readings A26-A28) -- the
// one dense contraction of the method, so it runs on the 5th-generation tensor cores:
//   tcgen05.mma kind::tf32, M = 128 vertices per CTA, N = 256 = the layer width, K = 8 per instruction, issued by one
//   thread (warp 7, which does nothing else in the main loop).  The activations never leave TENSOR MEMORY: columns
//   [256, 512) hold the A operand (row = lane, K = column; the "TS" form of the instruction), columns [0, 256) the fp32
//   accumulator; the epilogue reads the accumulator with tcgen05.ld, applies bias + ReLU and writes the next layer's A
//   operand back with tcgen05.st.  Shared memory therefore belongs to the weights: six 256 x 32 chunk buffers in the
//   K-major 128-byte-swizzle layout (8-row x 128-byte atoms), filled by cp.async four chunks ahead and released by
//   tcgen05.commit on an mbarrier.
// All four hidden layers and the 256 -> 3 head run in one kernel.  theta is the same for every vertex, so its part of
// layer 1 is folded into that layer's bias once per call (mlp_bias1_kernel).
// FAST file: the result is compared with the fp64 oracle under the TF32 tolerance derived in DESIGN.md.
#include "rga_internal.h"

#define MLP_M 128              // vertices per CTA (UMMA M)
#define MLP_W 256              // layer width (UMMA N)
#define MLP_KC 32              // weight chunk along K (four K = 8 instructions): every chunk costs ~1,000 cycles of
                               // barriers and fences whatever its size, so few large chunks beat many small ones
#define MLP_NBUF 6             // weight chunk buffers: the activations live in tensor memory, so shared memory is all theirs
#define MLP_LAG 2              // a buffer is refilled two chunks after its MMAs were issued
#define MLP_PD (MLP_NBUF - MLP_LAG)   // cp.async prefetch distance in chunks
#define MLP_THREADS 256
#define MLP_SBO 1024u          // 128-byte swizzle, K-major: an atom is 8 rows x 128 bytes (32 tf32), 8-row groups 1 KB apart
#define MLP_CHUNK_BYTES (MLP_W * MLP_KC * 4)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor (K-major, SWIZZLE_128B): start >> 4, leading byte offset (unused: K stays inside one
// atom) >> 4, stride (8-row group) byte offset >> 4, version 1, layout type 2.  The no-swizzle layout is correct too but
// the tensor core then reads its operands at a quarter of the rate (measured: ~550 cycles per 128x256x8 instruction).
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr) {
  return (uint64_t)((saddr >> 4) & 0x3fffu) | ((uint64_t)1 << 16) | ((uint64_t)((MLP_SBO >> 4) & 0x3fffu) << 32) |
         ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done)
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(done) : "r"(bar), "r"(parity) : "memory");
}

// theta is the same for every vertex: its columns of W1 are folded into layer 1's bias once per call, one warp per row
__global__ void __launch_bounds__(256) mlp_bias1_kernel(int K1, int n_pose, const float* __restrict__ W1, const float* __restrict__ b1,
                                                        const float* __restrict__ theta, float* __restrict__ bias1) {
  const int n = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  float acc = 0.f;
  for (int j = lane; j < n_pose; j += 32) acc = fmaf(W1[(size_t)n * (K1 + n_pose) + K1 + j], theta[j], acc);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if (lane == 0) bias1[n] = b1[n] + acc;
}

// 32 consecutive fp32 columns of this thread's TMEM lane -> registers / registers -> TMEM
#define TMEM_LD32(taddr, r)                                                                                                    \
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 "                                                                     \
               "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];" \
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), \
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), \
                 "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), \
                 "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])                                                              \
               : "r"(taddr) : "memory")
#define TMEM_ST32(taddr, r)                                                                                                    \
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "                                                               \
               "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" \
               :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), \
                  "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), \
                  "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), \
                  "r"(r[30]), "r"(r[31]) : "memory")

__global__ void __launch_bounds__(MLP_THREADS, 1) disp_mlp_kernel(int nv, int F, int n_pose, const float4* __restrict__ v_pos,
    const float* __restrict__ rff, const float* __restrict__ bias1, const float* __restrict__ W1,
    const float* __restrict__ Wh, const float* __restrict__ bh, const float* __restrict__ Wo, const float* __restrict__ bo,
    float4* __restrict__ v_disp) {
  extern __shared__ __align__(1024) unsigned char smem[];
  unsigned char* sB = smem;                                           // MLP_NBUF x (256 x 32 tf32, swizzled): 6 x 32 KB
  float* sBias = reinterpret_cast<float*>(sB + (size_t)MLP_NBUF * MLP_CHUNK_BYTES);     // [4][256]
  float* sWo = sBias + 4 * MLP_W;                                     // [3][256]
  float* sRff = sWo + 3 * MLP_W;                                      // [F][3]
  float* sOut = sRff + 3 * 128;                                       // [128][3] partial head sums of the upper column half
  __shared__ __align__(8) unsigned long long bars[MLP_NBUF + 1];      // weight buffers free, accumulator ready
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int K1 = 2 * F, in1 = K1 + n_pose;
  if (warp == 0) {                                                    // all 512 columns: accumulator [0,256), activations [256,512)
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" :: "r"(smem_u32(&tmem_base_s)), "r"(512u));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (tid == 0) {
    for (int i = 0; i <= MLP_NBUF; ++i) asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(&bars[i])), "r"(1u));
    asm volatile("fence.mbarrier_init.release.cluster;");
  }
  // chunk t of the whole network: layer, weight matrix and row stride, first column
  const int nch1 = K1 / MLP_KC, total = nch1 + 3 * (MLP_W / MLP_KC);
  constexpr int nchh = MLP_W / MLP_KC;
  auto stage = [&](int t) {                                           // cp.async: 256 rows x 32 columns, 16 bytes per copy
    const int layer = t < nch1 ? 0 : 1 + (t - nch1) / nchh, c = t < nch1 ? t : (t - nch1) % nchh;
    const float* Wl = layer == 0 ? W1 : Wh + (size_t)(layer - 1) * MLP_W * MLP_W;
    const int ldw = layer == 0 ? in1 : MLP_W;
    unsigned char* buf = sB + (size_t)(t % MLP_NBUF) * MLP_CHUNK_BYTES;
    // 16-byte piece q of the chunk in shared-memory order (destination 16 q: conflict-free): row r = (q >> 3) & 7 of row
    // group g = q >> 6, physical slot q & 7 of the row, which holds K piece (q & 7) ^ r; a warp reads 4 rows x 128 bytes
    // (warps 0..6 stage; warp 7 issues the MMAs and stays off the staging path)
    for (int q = tid; q < MLP_W * MLP_KC / 4 && tid < MLP_THREADS - 32; q += MLP_THREADS - 32) {
      const int r = (q >> 3) & 7, n = ((q >> 6) << 3) | r, kq = (q & 7) ^ r;
      const float* src = Wl + (size_t)n * ldw + c * MLP_KC + 4 * kq;
      const uint32_t dst = smem_u32(buf) + 16u * (uint32_t)q;
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  // biases (layer 1's already holds the pose, mlp_bias1_kernel), head weights, Fourier matrix
  for (int n = tid; n < MLP_W; n += MLP_THREADS) {
    sBias[n] = bias1[n];
    for (int l = 0; l < 3; ++l) sBias[(l + 1) * MLP_W + n] = bh[l * MLP_W + n];
    for (int c = 0; c < 3; ++c) sWo[c * MLP_W + n] = Wo[c * MLP_W + n];
  }
  for (int i = tid; i < 3 * F; i += MLP_THREADS) sRff[i] = rff[i];
  for (int t = 0; t < MLP_PD; ++t) stage(t);                          // the first weight chunks fly during the prologue
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem_base = tmem_base_s;
  // Thread -> TMEM: warp w owns lanes 32 (w & 3) .. +31 (the tile's rows) and the column half w >> 2.
  const int erow = (warp & 3) * 32 + lane, half = warp >> 2;
  const uint32_t tlane = tmem_base + ((uint32_t)((warp & 3) * 32) << 16);
  const int v = blockIdx.x * MLP_M + erow;
  // layer-1 operand: gamma(x) = [sin(2 pi B x), cos(2 pi B x)] of the row's vertex, straight into the activation columns
  {
    float4 x = make_float4(0.f, 0.f, 0.f, 0.f);
    if (v < nv) x = v_pos[v];
    for (int f0 = half * (F / 2); f0 < (half + 1) * (F / 2); f0 += 8) {
      uint32_t sn8[8], cs8[8];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const int f = f0 + j;
        const float p = fmaf(sRff[3 * f + 2], x.z, fmaf(sRff[3 * f + 1], x.y, sRff[3 * f] * x.x));
        // sin / cos of 2 pi p: the period is removed exactly (p - rint(p) is exact in fp32), then the MUFU approximations
        float sn, cs;
        __sincosf(6.283185307179586f * (p - rintf(p)), &sn, &cs);
        sn8[j] = __float_as_uint(sn); cs8[j] = __float_as_uint(cs);
      }
      asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                   :: "r"(tlane + 256u + (uint32_t)f0), "r"(sn8[0]), "r"(sn8[1]), "r"(sn8[2]), "r"(sn8[3]), "r"(sn8[4]), "r"(sn8[5]),
                      "r"(sn8[6]), "r"(sn8[7]) : "memory");
      asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                   :: "r"(tlane + 256u + (uint32_t)(F + f0)), "r"(cs8[0]), "r"(cs8[1]), "r"(cs8[2]), "r"(cs8[3]), "r"(cs8[4]), "r"(cs8[5]),
                      "r"(cs8[6]), "r"(cs8[7]) : "memory");
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  }
  const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(MLP_W >> 3) << 17) | ((uint32_t)(MLP_M >> 4) << 24);
  uint32_t par_acc = 0u;
  float out0 = 0.f, out1 = 0.f, out2 = 0.f;

  for (int t = 0; t < total; ++t) {
    const int layer = t < nch1 ? 0 : 1 + (t - nch1) / nchh, c = t < nch1 ? t : (t - nch1) % nchh;
    const int nchunks = layer == 0 ? nch1 : nchh;
    // chunk t+PD goes into the buffer of chunk t-LAG, whose MMAs were issued LAG iterations ago
    if (t + MLP_PD < total) {
      if (t >= MLP_LAG) mbar_wait(smem_u32(&bars[(t + MLP_PD) % MLP_NBUF]), (uint32_t)(((t - MLP_LAG) / MLP_NBUF) & 1));
      stage(t + MLP_PD);
    } else asm volatile("cp.async.commit_group;" ::: "memory");      // keeps the group count uniform
    asm volatile("cp.async.wait_group %0;" :: "n"(MLP_PD) : "memory");       // chunk t has landed (this thread's copies)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy writes -> the tensor core's async proxy
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (tid == MLP_THREADS - 32) {
      asm volatile("tcgen05.fence::after_thread_sync;");
      const uint32_t buf = smem_u32(sB + (size_t)(t % MLP_NBUF) * MLP_CHUNK_BYTES);
#pragma unroll
      for (int j = 0; j < MLP_KC / 8; ++j) {
        const uint32_t ta = tmem_base + 256u + (uint32_t)(c * MLP_KC + 8 * j);        // A from tensor memory: row = lane, K = column
        const uint64_t db = umma_desc(buf + 32u * j);
        const uint32_t acc = (c > 0 || j > 0) ? 1u : 0u;
        asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
                     :: "r"(tmem_base), "r"(ta), "l"(db), "r"(idesc), "r"(acc) : "memory");
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&bars[t % MLP_NBUF])) : "memory");
      if (c == nchunks - 1)
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(smem_u32(&bars[MLP_NBUF])) : "memory");
    }
    if (c != nchunks - 1) continue;
    // accumulator ready: every MMA of the layer has read its A operand, so the activation columns may be overwritten
    mbar_wait(smem_u32(&bars[MLP_NBUF]), par_acc); par_acc ^= 1u;
    asm volatile("tcgen05.fence::after_thread_sync;");
    const float* bias = sBias + layer * MLP_W;
    for (int c0 = half * (MLP_W / 2); c0 < half * (MLP_W / 2) + MLP_W / 2; c0 += 32) {
      uint32_t r[32];
      TMEM_LD32(tlane + (uint32_t)c0, r);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      if (layer < 3) {
#pragma unroll
        for (int j = 0; j < 32; ++j) r[j] = __float_as_uint(fmaxf(__uint_as_float(r[j]) + bias[c0 + j], 0.f));
        TMEM_ST32(tlane + 256u + (uint32_t)c0, r);                     // the next layer's A operand never leaves tensor memory
      } else {                                                         // head: 256 -> 3, fp32 on the CUDA cores
#pragma unroll
        for (int j = 0; j < 32; ++j) {
          const float h = fmaxf(__uint_as_float(r[j]) + bias[c0 + j], 0.f);
          out0 = fmaf(sWo[c0 + j], h, out0); out1 = fmaf(sWo[MLP_W + c0 + j], h, out1); out2 = fmaf(sWo[2 * MLP_W + c0 + j], h, out2);
        }
      }
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    // (the next chunk's fence + barrier order these TMEM reads and writes before the next layer's MMAs)
  }
  // head: the lower column half adds the upper half's partial sums (fixed order: lower + upper)
  if (warp >= 4) { sOut[3 * erow] = out0; sOut[3 * erow + 1] = out1; sOut[3 * erow + 2] = out2; }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (warp < 4 && v < nv)
    v_disp[v] = make_float4((out0 + sOut[3 * erow]) + bo[0], (out1 + sOut[3 * erow + 1]) + bo[1], (out2 + sOut[3 * erow + 2]) + bo[2], 0.f);
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"(512u));
}

size_t rga_mlp_smem(int F) {
  (void)F;
  return (size_t)MLP_NBUF * MLP_CHUNK_BYTES + (size_t)(4 + 3) * MLP_W * 4 + (size_t)3 * 128 * 4 + (size_t)3 * MLP_M * 4 + 64;
}

int rga_mlp_init_attributes() {
  return (int)cudaFuncSetAttribute(disp_mlp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rga_mlp_smem(128));
}

cudaError_t rga_launch_disp_mlp(rga_avatar* av, const rga_disp_mlp* m, const float* theta, cudaStream_t s) {
  const int grid = (av->n_verts + MLP_M - 1) / MLP_M;
  mlp_bias1_kernel<<<MLP_W / 8, 256, 0, s>>>(2 * m->n_freq, m->n_pose, m->W1, m->b1, theta, av->mlp_bias1);
  rga_prof_mark(av, "mlp_bias1", s);
  disp_mlp_kernel<<<grid, MLP_THREADS, rga_mlp_smem(m->n_freq), s>>>(av->n_verts, m->n_freq, m->n_pose, av->v_pos, m->rff, av->mlp_bias1, m->W1,
                                                               m->Wh, m->bh, m->Wo, m->bo, av->v_disp);
  av->launches += 2;
  rga_prof_mark(av, "disp_mlp", s);
  return cudaGetLastError();
}
