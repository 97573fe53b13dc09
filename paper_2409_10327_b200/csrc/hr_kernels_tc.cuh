// hr_kernels_tc.cuh -- tensor-core (tcgen05 / TMEM) implementation of the fused path for mlp_dtype == HR_F16.
//
// Design: a CTA is 128 threads = the 128 TMEM lanes; thread p owns primary point
// p of the CTA's 128-point tile for the whole frame (direct set, secondary set, and the tertiary set of each of its
// secondary points), so no activation ever crosses threads.  Every 64-wide MLP layer over the tile is ONE
// M=128 x N=64 tcgen05.mma group: each thread packs its row of fp16 activations straight into TMEM (tcgen05.st,
// the A operand is read from TMEM), weights sit in shared memory as K-major SWIZZLE_128B UMMA tiles, the fp32
// accumulator comes back with tcgen05.ld and the bias/ReLU/last-layer dot products run from constant-bank
// operands.  Layer-1 biases ride in the MMA as an extra K step (hi + lo fp16 split => exact to 2^-22).
// Several CTAs per SM overlap one tile's MMA round trip with the others' ALU work.
//
// Precision contract (Q34): tables/weights fp16 (rounded once by the caller's generator), hidden activations
// rounded to fp16 (RNE), accumulation fp32, final-layer outputs / t / x' / the index path / shading fp32.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>

#include <vector>

#include "../../include/hashrender.h"
#include "hr_device.cuh"

namespace hr {
namespace tc {

constexpr int kThreads = 128;
constexpr int kTmemCols = 128;
constexpr int kTileBytes = 64 * 128;          // one 64 x 64 fp16 K-major SW128 weight tile
constexpr int kNumTiles = 4;                  // I.W1f(+b1), B.W1(+b1), I.W2, B.W2
constexpr int kMaxS2 = 16;                    // shared tertiary set staged in smem
// TMEM column map (per CTA): A operand (fp16 pairs) | constant bias K-step | accumulator
constexpr uint32_t kColA = 0, kColOne = 56, kColD = 64;   // a split-precision 64-wide A (cols 0..63) overwrites the bias step

struct __align__(16) TcConst {                // lives in the kernel-parameter constant bank
  float w1w[3][kH];                           // I layer 1, direction columns
  float b2[kH]; float w3[2][kH]; float b3[2]; float pad0[2];
  float Bb2[kH]; float BW3[7][kH]; float Bb3[8];
  uint32_t w3v_h2[kH / 2];                    // fp16x2 pairs of w3[0] (visibility row) for the fast epilogue
};

// ---------------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

__device__ __forceinline__ void mma_f16_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accum)
      : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t mbar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.b32 %0, 1, 0, P1;\n\t}\n"
                 : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
  } while (!done);
}

#define HR_R16(r, o) "=r"(r[o+0]), "=r"(r[o+1]), "=r"(r[o+2]), "=r"(r[o+3]), "=r"(r[o+4]), "=r"(r[o+5]), "=r"(r[o+6]), "=r"(r[o+7]), \
                     "=r"(r[o+8]), "=r"(r[o+9]), "=r"(r[o+10]), "=r"(r[o+11]), "=r"(r[o+12]), "=r"(r[o+13]), "=r"(r[o+14]), "=r"(r[o+15])
#define HR_W16(r, o) "r"(r[o+0]), "r"(r[o+1]), "r"(r[o+2]), "r"(r[o+3]), "r"(r[o+4]), "r"(r[o+5]), "r"(r[o+6]), "r"(r[o+7]), \
                     "r"(r[o+8]), "r"(r[o+9]), "r"(r[o+10]), "r"(r[o+11]), "r"(r[o+12]), "r"(r[o+13]), "r"(r[o+14]), "r"(r[o+15])

// 32 consecutive fp32 columns of this thread's TMEM lane -> registers (no wait)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,"
      "%26,%27,%28,%29,%30,%31}, [%32];"
      : HR_R16(r, 0), HR_R16(r, 16) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&r)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};" ::"r"(taddr), HR_W16(r, 0)
               : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,"
      "%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr), HR_W16(r, 0), HR_W16(r, 16)
      : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t (&r)[8]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]),
               "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
               : "memory");
}

__device__ __forceinline__ void tmem_st1(uint32_t taddr, uint32_t r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x1.b32 [%0], {%1};" ::"r"(taddr), "r"(r) : "memory");
}

// two floats -> packed fp16x2 (lo = a, hi = b), optionally with ReLU fused into the conversion
__device__ __forceinline__ uint32_t pack_relu(float a, float b) {
  uint32_t r;
  asm("cvt.rn.relu.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a));
  return r;
}
__device__ __forceinline__ uint32_t pack_rn(float a, float b) {
  uint32_t r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a));
  return r;
}

// K-major SWIZZLE_128B shared-memory matrix descriptor (sm_100 UMMA): 8-row groups of 128 B rows, SBO = 1024 B.
__device__ __forceinline__ uint64_t make_bdesc(uint32_t smem_addr) {
  uint64_t d = 0;
  d |= (uint64_t)((smem_addr & 0x3FFFF) >> 4);      // start address
  d |= (uint64_t)1 << 16;                           // leading byte offset (ignored for swizzled K-major)
  d |= (uint64_t)(1024 >> 4) << 32;                 // stride byte offset
  d |= (uint64_t)1 << 46;                           // descriptor version (Blackwell)
  d |= (uint64_t)2 << 61;                           // SWIZZLE_128B
  return d;
}
// kind::f16, A/B = F16 K-major, D = F32, M = 128, N = 64
constexpr uint32_t kIdesc = (1u << 4) | ((64u >> 3) << 17) | ((128u >> 4) << 24);

struct Ctx {
  uint32_t tA, tOne, tD;       // TMEM addresses incl. this warp's lane base
  uint32_t tA0, tOne0, tD0;    // lane-0 addresses (MMA operands)
  uint32_t mbar, phase;
  uint32_t tile[kNumTiles];    // smem addresses of the weight tiles
};

// One 128 x 64 layer: D = A[:, 0:16*ksteps] * W^T (+ a bias K-step: A = [1,1,0..] times K-step `bias_kstep` of tile
// `bias_tile`, whose first two columns hold the bias as an fp16 hi/lo pair; bias_tile < 0 = none).
// split: A holds a hi block (columns 0..8*ksteps) and a lo block (the next 8*ksteps columns) of an error-compensated
// fp16 pair; both are multiplied by the same (exact fp16) weights, so the layer input is good to ~2^-22.
// Every thread must have issued its tcgen05.st of A before calling.  Returns when D is readable.
__device__ __forceinline__ void mma_layer(Ctx& c, int tile, int ksteps, int bias_tile, int bias_kstep, bool split = false) {
  wait_st();
  fence_before();
  __syncthreads();
  if (threadIdx.x == 0) {
    fence_after();
    const uint64_t bd = make_bdesc(c.tile[tile]);
    for (int k = 0; k < ksteps; ++k) mma_f16_ts(c.tD0, c.tA0 + 8 * k, bd + 2 * k, kIdesc, k > 0);
    if (split)
      for (int k = 0; k < ksteps; ++k) mma_f16_ts(c.tD0, c.tA0 + 8 * (ksteps + k), bd + 2 * k, kIdesc, 1u);
    if (bias_tile >= 0) mma_f16_ts(c.tD0, c.tOne0, make_bdesc(c.tile[bias_tile]) + 2 * bias_kstep, kIdesc, 1u);
    mma_commit(c.mbar);
  }
  mbar_wait(c.mbar, c.phase);
  c.phase ^= 1u;
  fence_after();
}

// ---------------------------------------------------------------------------------------------------- per-row stages
// residual of an fp16x2 pack: (a - fp16(a), b - fp16(b)) packed again (the "lo" half of a hi/lo split)
__device__ __forceinline__ uint32_t pack_lo(uint32_t hi, float a, float b) {
  const float2 h = __half22float2(*reinterpret_cast<const __half2*>(&hi));
  return pack_rn(a - h.x, b - h.y);
}

// f = H(x) straight into the A operand: level l -> TMEM column l (fp16 pair) and its fp16 residual into column
// 16 + l (split-precision features for the layer-1 partial P, which feeds the t that moves x').  The level loop stays
// rolled (x2) to keep the kernel inside the instruction cache; 16 gathers per thread are in flight.
template <bool F16>
__device__ __forceinline__ void encode_to_A(const GridP& g, const Ctx& c, float x, float y, float z) {
#pragma unroll 2
  for (int l = 0; l < kMaxL; ++l) {
    uint32_t hi = 0u, lo = 0u;
    if (l < (int)g.L) {
      const float2 v = encode_level<F16>(g, l, x, y, z, nullptr, nullptr);
      hi = pack_rn(v.x, v.y);
      lo = pack_lo(hi, v.x, v.y);
    }
    tmem_st1(c.tA + l, hi);
    tmem_st1(c.tA + 16 + l, lo);
  }
}

__device__ __forceinline__ void restore_one(const Ctx& c) {
  uint32_t one[8] = {0x3C003C00u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};     // bias K-step of A: [1, 1, 0, ... 0]
  tmem_st8(c.tOne, one);
}

// Precise epilogue of I (secondary set: z_t becomes t): (z_v, z_t) = b3 + W3 relu(D + b2), all fp32.
__device__ __forceinline__ void irt_epilogue_precise(const Ctx& c, const TcConst& cw, float& zv, float& zt) {
  float z0 = cw.b3[0], z1 = cw.b3[1];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(c.tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const float a = fmaxf(__uint_as_float(r[k]) + cw.b2[32 * h + k], 0.f);
      z0 = fmaf(a, cw.w3[0][32 * h + k], z0);
      z1 = fmaf(a, cw.w3[1][32 * h + k], z1);
    }
  }
  zv = z0; zt = z1;
}

// Fast epilogue of I (direct and tertiary queries need only visibility): b2 already rode in the MMA (bias K-step),
// h2 = relu(D) is rounded to fp16 by the packing conversion, z_v = b3 + w3v . h2 with fp16x2 FMAs into four short
// accumulators summed in fp32.
__device__ __forceinline__ float irt_epilogue_fast(const Ctx& c, const TcConst& cw) {
  __half2 acc[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) acc[q] = __float2half2_rn(0.f);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(c.tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const uint32_t p = pack_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
      const uint32_t w = cw.w3v_h2[16 * h + k];
      acc[k & 3] = __hfma2(*reinterpret_cast<const __half2*>(&p), *reinterpret_cast<const __half2*>(&w), acc[k & 3]);
    }
  }
  float z = cw.b3[0];
#pragma unroll
  for (int q = 0; q < 4; ++q) { const float2 f = __half22float2(acc[q]); z += f.x + f.y; }
  return z;
}

__device__ __forceinline__ float vis_of(const ShadeP& sp, float zv) { return sp.vis_mode ? (zv > 0.f ? 1.f : 0.f) : sigmoidf_(zv); }

// D (= W1 f + b1 of B) -> relu -> fp16 -> A columns 0..31
__device__ __forceinline__ void hidden_to_A(const Ctx& c) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(c.tD + 32 * h, r);
    wait_ld();
    uint32_t p[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) p[k] = pack_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
    tmem_st16(c.tA + 16 * h, p);
  }
}

// B(f) with f already in A[0..15]: layer 1 and layer 2 biases ride in the MMAs, layer 3 in fp32 registers
__device__ __forceinline__ void brdf_from_A(Ctx& c, const TcConst& cw, const ShadeP& sp, float (&b)[7]) {
  mma_layer(c, 1, 2, 1, 2);
  hidden_to_A(c);
  mma_layer(c, 3, 4, 1, 3);
  float o[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) o[q] = cw.Bb3[q];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(c.tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const float a = fmaxf(__uint_as_float(r[k]), 0.f);
#pragma unroll
      for (int q = 0; q < 7; ++q) o[q] = fmaf(a, cw.BW3[q][32 * h + k], o[q]);
    }
  }
  brdf_maps(sp, o, b);
}

// h1 = relu(P + W1w . w) -> A columns 0..31 (P in registers)
__device__ __forceinline__ void h1_from_regs(const Ctx& c, const TcConst& cw, const float (&P)[kH], float wx, float wy, float wz) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t p[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int j = 32 * h + 2 * k;
      float a0 = fmaf(cw.w1w[0][j], wx, P[j]);
      a0 = fmaf(cw.w1w[1][j], wy, a0); a0 = fmaf(cw.w1w[2][j], wz, a0);
      float a1 = fmaf(cw.w1w[0][j + 1], wx, P[j + 1]);
      a1 = fmaf(cw.w1w[1][j + 1], wy, a1); a1 = fmaf(cw.w1w[2][j + 1], wz, a1);
      p[k] = pack_relu(a0, a1);
    }
    tmem_st16(c.tA + 16 * h, p);
  }
}
// split-precision variant for the secondary set (its z_t becomes t and moves x': SURVEY 8(c) conditioning note):
// h1 in fp32 -> hi (columns 0..31) + lo (columns 32..63); P from this thread's shared-memory column
__device__ __forceinline__ void h1_from_smem_split(const Ctx& c, const TcConst& cw, const float* Ps, float wx, float wy, float wz) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t p[16], q[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int j = 32 * h + 2 * k;
      float a0 = fmaf(cw.w1w[0][j], wx, Ps[j * kThreads]);
      a0 = fmaf(cw.w1w[1][j], wy, a0); a0 = fmaxf(fmaf(cw.w1w[2][j], wz, a0), 0.f);
      float a1 = fmaf(cw.w1w[0][j + 1], wx, Ps[(j + 1) * kThreads]);
      a1 = fmaf(cw.w1w[1][j + 1], wy, a1); a1 = fmaxf(fmaf(cw.w1w[2][j + 1], wz, a1), 0.f);
      p[k] = pack_rn(a0, a1);
      q[k] = pack_lo(p[k], a0, a1);
    }
    tmem_st16(c.tA + 16 * h, p);
    tmem_st16(c.tA + 32 + 16 * h, q);
  }
}
// shared direction set: the direction part Q = W1w . w'_k is precomputed per CTA, h1 = relu(P + Q)
__device__ __forceinline__ void h1_from_regs_shared(const Ctx& c, const float (&P)[kH], const float* __restrict__ Q) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t p[16];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const float4 q = reinterpret_cast<const float4*>(Q)[8 * h + k];
      const int j = 32 * h + 4 * k;
      p[2 * k] = pack_relu(P[j] + q.x, P[j + 1] + q.y);
      p[2 * k + 1] = pack_relu(P[j + 2] + q.z, P[j + 3] + q.w);
    }
    tmem_st16(c.tA + 16 * h, p);
  }
}

// D -> registers (64 fp32)
__device__ __forceinline__ void load_D(const Ctx& c, float (&P)[kH]) {
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(c.tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; ++k) P[32 * h + k] = __uint_as_float(r[k]);
  }
}

// ---------------------------------------------------------------------------------------------------- shared setup
struct Smem {
  uint8_t* tiles;      // 4 x 8 KB, 1024-aligned
  float* Ps;           // [64][128]
  float* Qt;           // [kMaxS2][64]
  float* Lt;           // [kMaxS2][4]
  uint64_t* mbar;
  uint32_t* tmem_slot;
};
constexpr size_t kSmemBytes = 1024 + kNumTiles * kTileBytes + kH * kThreads * 4 + kMaxS2 * kH * 4 + kMaxS2 * 4 * 4 + 64;

__device__ __forceinline__ Smem carve(uint8_t* raw) {
  Smem s;
  uint8_t* p = raw + ((1024u - (smem_u32(raw) & 1023u)) & 1023u);      // pointer arithmetic keeps the shared address space
  s.tiles = p; p += kNumTiles * kTileBytes;
  s.Ps = reinterpret_cast<float*>(p); p += kH * kThreads * 4;
  s.Qt = reinterpret_cast<float*>(p); p += kMaxS2 * kH * 4;
  s.Lt = reinterpret_cast<float*>(p); p += kMaxS2 * 4 * 4;
  s.mbar = reinterpret_cast<uint64_t*>(p); p += 16;
  s.tmem_slot = reinterpret_cast<uint32_t*>(p);
  return s;
}

__device__ __forceinline__ void setup(const Smem& s, const uint8_t* __restrict__ wtiles, Ctx& c) {
  const int warp = threadIdx.x >> 5;
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(s.tmem_slot)), "r"((uint32_t)kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (threadIdx.x == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(s.mbar)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const uint4* src = reinterpret_cast<const uint4*>(wtiles);
  uint4* dst = reinterpret_cast<uint4*>(s.tiles);
  for (int i = threadIdx.x; i < kNumTiles * kTileBytes / 16; i += kThreads) dst[i] = __ldg(src + i);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the tensor core
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t base = *s.tmem_slot;
  const uint32_t lane_base = (uint32_t)(warp * 32) << 16;
  c.tA0 = base + kColA; c.tOne0 = base + kColOne; c.tD0 = base + kColD;
  c.tA = c.tA0 + lane_base; c.tOne = c.tOne0 + lane_base; c.tD = c.tD0 + lane_base;
  c.mbar = smem_u32(s.mbar); c.phase = 0;
#pragma unroll
  for (int t = 0; t < kNumTiles; ++t) c.tile[t] = smem_u32(s.tiles + t * kTileBytes);
  restore_one(c);
  wait_st();
}

__device__ __forceinline__ void teardown(const Ctx& c) {
  fence_before();
  __syncthreads();
  if ((threadIdx.x >> 5) == 0) {
    fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(c.tA0), "r"((uint32_t)kTmemCols) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------- kernels
// render_frame (a1-a11), tensor-core path.  The point loop `j` runs -1 (the primary point itself) .. S_i-1 (its
// secondary points) so that encode + layer-1 partial + BRDF decoder exist once in the instruction stream.
template <bool F16>
__global__ void __launch_bounds__(kThreads, 3) k_render_tc(const __grid_constant__ GridP g, EnvP env, ShadeP sp, const __grid_constant__ TcConst cw,
                                                           const uint8_t* __restrict__ wtiles, FrameP fr, float* __restrict__ rgb) {
  extern __shared__ uint8_t smem_raw[];
  const Smem s = carve(smem_raw);
  Ctx c;
  setup(s, wtiles, c);
  const bool indirect = (fr.flags & 4u) && fr.s.S && fr.t.S;
  const bool tshared = fr.t.stride == 0;
  if (indirect && tshared) {                    // shared tertiary set: Q_k = W1w . w'_k, L_k = env(w'_k)
    for (int e = threadIdx.x; e < (int)fr.t.S * kH; e += kThreads) {
      const int k = e / kH, q = e % kH;
      const float* dp = fr.t.dir + 3 * k;
      s.Qt[e] = cw.w1w[0][q] * __ldg(dp) + cw.w1w[1][q] * __ldg(dp + 1) + cw.w1w[2][q] * __ldg(dp + 2);
    }
    for (int k = threadIdx.x; k < (int)fr.t.S; k += kThreads) {
      const float* dp = fr.t.dir + 3 * k;
      float3 L;
      if (fr.t.Lin) L = make_float3(__ldg(fr.t.Lin + 3 * k), __ldg(fr.t.Lin + 3 * k + 1), __ldg(fr.t.Lin + 3 * k + 2));
      else L = env_lookup(env, __ldg(dp), __ldg(dp + 1), __ldg(dp + 2));
      s.Lt[4 * k] = L.x; s.Lt[4 * k + 1] = L.y; s.Lt[4 * k + 2] = L.z;
    }
  }
  __syncthreads();
  float* Ps = s.Ps + threadIdx.x;
  const unsigned long long ntiles = (fr.N + kThreads - 1) / kThreads;
  const int jend = indirect ? (int)fr.s.S : 0;
  for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const unsigned long long i_raw = tile * kThreads + threadIdx.x;
    const bool valid = i_raw < fr.N;
    const unsigned long long i = valid ? i_raw : fr.N - 1;        // idle rows shadow the last point (uniform control flow)
    const bool live = valid && !(fr.mask && !fr.mask[i]);
    const float px = __ldg(fr.x + 3 * i), py = __ldg(fr.x + 3 * i + 1), pz = __ldg(fr.x + 3 * i + 2);
    const float ox = __ldg(fr.wo + 3 * i), oy = __ldg(fr.wo + 3 * i + 1), oz = __ldg(fr.wo + 3 * i + 2);
    float b[7];                                                     // primary BRDF
    float r = 0.f, gch = 0.f, bch = 0.f;                            // direct term of Eq. 1
    float ir = 0.f, ig = 0.f, ib = 0.f;                             // (1 - V) L'_o term of Eq. 2
    for (int j = -1; j < jend; ++j) {
      float ex = px, ey = py, ez = pz, wx = 0.f, wy = 0.f, wz = 0.f, pdf = 0.f, v = 0.f;
      if (j >= 0) {                                                 // a6/a7 along secondary direction j (split precision)
        const float* dp = dir_of(fr.s, i, j);
        wx = __ldg(dp); wy = __ldg(dp + 1); wz = __ldg(dp + 2);
        pdf = pdf_of(fr.s, i, j);
        h1_from_smem_split(c, cw, Ps, wx, wy, wz);
        mma_layer(c, 2, 4, -1, 0, true);
        float zv, zt, t;
        irt_epilogue_precise(c, cw, zv, zt);
        irt_maps(sp, zv, zt, v, t);
        restore_one(c);                                             // the split A block overwrote the bias K-step columns
        ex = sec_hit(px, t, wx); ey = sec_hit(py, t, wy); ez = sec_hit(pz, t, wz);
      }
      // a1-a5 at the point: f -> A, P = W1f f + b1, B(f)
      encode_to_A<F16>(g, c, ex, ey, ez);
      mma_layer(c, 0, 2, 0, 2, true);
      float P[kH];
      load_D(c, P);
      float bb[7];
      if (j < 0 && fr.brdf) {
#pragma unroll
        for (int k = 0; k < 7; ++k) bb[k] = __ldg(fr.brdf + i * 7 + k);
      } else {
        brdf_from_A(c, cw, sp, bb);                                 // A[0..15] still holds f (hi)
      }
      if (j < 0) {
#pragma unroll
        for (int k = 0; k < 7; ++k) b[k] = bb[k];
        if (jend > 0) {
#pragma unroll
          for (int k = 0; k < kH; ++k) Ps[k * kThreads] = P[k];
        }
        if ((fr.flags & 1u) && fr.d.S) {                            // direct term of Eq. 1 over the direct set
          float ar = 0.f, ag = 0.f, ab = 0.f;
          const float* dp = dir_of(fr.d, i, 0);
          float dx = __ldg(dp), dy = __ldg(dp + 1), dz = __ldg(dp + 2), dpdf = pdf_of(fr.d, i, 0);
          for (uint32_t sidx = 0; sidx < fr.d.S; ++sidx) {
            const uint32_t sn = sidx + 1 < fr.d.S ? sidx + 1 : sidx;      // prefetch the next direction
            const float* dn = dir_of(fr.d, i, sn);
            const float nx = __ldg(dn), ny = __ldg(dn + 1), nz = __ldg(dn + 2), npdf = pdf_of(fr.d, i, sn);
            float vd = 1.f;
            if (fr.flags & 2u) {
              h1_from_regs(c, cw, P, dx, dy, dz);
              mma_layer(c, 2, 4, 0, 3);
              vd = vis_of(sp, irt_epilogue_fast(c, cw));
            }
            const float3 gg = brdf_cos_over_pdf(sp, bb, dx, dy, dz, ox, oy, oz, dpdf);
            const float3 L = incoming(env, fr.d, i, sidx, dx, dy, dz);
            ar = fmaf(vd * L.x, gg.x, ar); ag = fmaf(vd * L.y, gg.y, ag); ab = fmaf(vd * L.z, gg.z, ab);
            dx = nx; dy = ny; dz = nz; dpdf = npdf;
          }
          const float inv = 1.f / (float)fr.d.S;
          r = ar * inv; gch = ag * inv; bch = ab * inv;
        }
      } else {                                                      // a8: Eq. 1 at x' over the tertiary set, w_o' = -w_j
        float lr = 0.f, lg = 0.f, lb = 0.f;
        const unsigned long long trow = tshared ? 0ull : i * fr.s.S + j;
        for (uint32_t k = 0; k < fr.t.S; ++k) {
          const float* tp = dir_of(fr.t, trow, k);
          const float tx = __ldg(tp), ty = __ldg(tp + 1), tz = __ldg(tp + 2);
          if (tshared) h1_from_regs_shared(c, P, s.Qt + k * kH);
          else h1_from_regs(c, cw, P, tx, ty, tz);
          mma_layer(c, 2, 4, 0, 3);
          const float v2 = vis_of(sp, irt_epilogue_fast(c, cw));
          const float3 gg = brdf_cos_over_pdf(sp, bb, tx, ty, tz, -wx, -wy, -wz, pdf_of(fr.t, trow, k));
          float3 L;
          if (tshared) L = make_float3(s.Lt[4 * k], s.Lt[4 * k + 1], s.Lt[4 * k + 2]);
          else L = incoming(env, fr.t, trow, k, tx, ty, tz);
          lr = fmaf(v2 * L.x, gg.x, lr); lg = fmaf(v2 * L.y, gg.y, lg); lb = fmaf(v2 * L.z, gg.z, lb);
        }
        const float3 gg = brdf_cos_over_pdf(sp, b, wx, wy, wz, ox, oy, oz, pdf);
        const float m = (1.f - v) / (float)fr.t.S;
        ir = fmaf(m * lr, gg.x, ir); ig = fmaf(m * lg, gg.y, ig); ib = fmaf(m * lb, gg.z, ib);
      }
    }
    if (jend > 0) {
      const float inv = 1.f / (float)jend;
      r = fmaf(ir, inv, r); gch = fmaf(ig, inv, gch); bch = fmaf(ib, inv, bch);
    }
    if (valid) {
      rgb[3 * i] = live ? r : 0.f; rgb[3 * i + 1] = live ? gch : 0.f; rgb[3 * i + 2] = live ? bch : 0.f;
    }
  }
  teardown(c);
}

// trace with the encode fused (a1-a4, a6, a7), tensor-core path (t is an output: precise epilogue).
template <bool F16>
__global__ void __launch_bounds__(kThreads, 3) k_trace_tc(const __grid_constant__ GridP g, ShadeP sp, const __grid_constant__ TcConst cw,
                                                          const uint8_t* __restrict__ wtiles, const float* __restrict__ x,
                                                          unsigned long long N, DirsetP ds, float* __restrict__ vis,
                                                          float* __restrict__ zvo, float* __restrict__ to, float* __restrict__ xsec) {
  extern __shared__ uint8_t smem_raw[];
  const Smem s = carve(smem_raw);
  Ctx c;
  setup(s, wtiles, c);
  const unsigned long long ntiles = (N + kThreads - 1) / kThreads;
  for (unsigned long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
    const unsigned long long i_raw = tile * kThreads + threadIdx.x;
    const bool valid = i_raw < N;
    const unsigned long long i = valid ? i_raw : N - 1;
    const float px = __ldg(x + 3 * i), py = __ldg(x + 3 * i + 1), pz = __ldg(x + 3 * i + 2);
    encode_to_A<F16>(g, c, px, py, pz);
    mma_layer(c, 0, 2, 0, 2, true);
    float P[kH];
    load_D(c, P);
    for (uint32_t sidx = 0; sidx < ds.S; ++sidx) {
      const float* dp = dir_of(ds, i, sidx);
      const float wx = __ldg(dp), wy = __ldg(dp + 1), wz = __ldg(dp + 2);
      h1_from_regs(c, cw, P, wx, wy, wz);
      mma_layer(c, 2, 4, -1, 0);
      float zv, zt, v, t;
      irt_epilogue_precise(c, cw, zv, zt);
      irt_maps(sp, zv, zt, v, t);
      if (valid) {
        const unsigned long long o = i * ds.S + sidx;
        vis[o] = v; to[o] = t;
        if (zvo) zvo[o] = zv;
        if (xsec) { xsec[o * 3] = sec_hit(px, t, wx); xsec[o * 3 + 1] = sec_hit(py, t, wy); xsec[o * 3 + 2] = sec_hit(pz, t, wz); }
      }
    }
  }
  teardown(c);
}

// ---------------------------------------------------------------------------------------------------- host side
struct HostWeights { TcConst cw; };

inline size_t tile_off(int j, int k) { return (size_t)(j / 8) * 1024 + (j % 8) * 128 + (((k / 8) ^ (j % 8)) * 16) + (k % 8) * 2; }

// Blob = [ TcConst | 4 UMMA tiles ].  The TcConst part is passed by value at launch, the tiles stay in HBM/L2.
inline void prepare_weights(const hr_config& cfg, const float* bw, const float* iw, std::vector<uint8_t>& out) {
  const int D = cfg.L * cfg.F, H = kH, Din = D + 3;
  out.assign(sizeof(TcConst) + kNumTiles * kTileBytes, 0);
  TcConst& cw = *reinterpret_cast<TcConst*>(out.data());
  __half* tiles = reinterpret_cast<__half*>(out.data() + sizeof(TcConst));
  auto put = [&](int t, int j, int k, float v) {
    *reinterpret_cast<__half*>(reinterpret_cast<uint8_t*>(tiles) + (size_t)t * kTileBytes + tile_off(j, k)) = __float2half_rn(v);
  };
  auto put_bias = [&](int t, int j, int col, float b) {   // hi + lo split in columns col, col+1 (one bias K-step)
    const __half hi = __float2half_rn(b);
    put(t, j, col, __half2float(hi));
    put(t, j, col + 1, b - __half2float(hi));
  };
  const float* BW1 = bw; const float* Bb1 = BW1 + H * D; const float* BW2 = Bb1 + H; const float* Bb2 = BW2 + H * H;
  const float* BW3 = Bb2 + H; const float* Bb3 = BW3 + 7 * H;
  const float* IW1 = iw; const float* Ib1 = IW1 + H * Din; const float* IW2 = Ib1 + H; const float* Ib2 = IW2 + H * H;
  const float* IW3 = Ib2 + H; const float* Ib3 = IW3 + 2 * H;
  for (int j = 0; j < H; ++j) {
    for (int k = 0; k < D; ++k) { put(0, j, k, IW1[j * Din + k]); put(1, j, k, BW1[j * D + k]); }
    put_bias(0, j, 32, Ib1[j]); put_bias(1, j, 32, Bb1[j]);       // K-step 2: layer-1 biases
    put_bias(0, j, 48, Ib2[j]); put_bias(1, j, 48, Bb2[j]);       // K-step 3: layer-2 biases (spare columns of the K=32 tiles)
    for (int k = 0; k < H; ++k) { put(2, j, k, IW2[j * H + k]); put(3, j, k, BW2[j * H + k]); }
    for (int d = 0; d < 3; ++d) cw.w1w[d][j] = IW1[j * Din + D + d];
    cw.b2[j] = Ib2[j]; cw.w3[0][j] = IW3[j]; cw.w3[1][j] = IW3[H + j];
    cw.Bb2[j] = Bb2[j];
    for (int q = 0; q < 7; ++q) cw.BW3[q][j] = BW3[q * H + j];
  }
  cw.b3[0] = Ib3[0]; cw.b3[1] = Ib3[1];
  for (int k = 0; k < H / 2; ++k) {
    const __half2 w = __floats2half2_rn(IW3[2 * k], IW3[2 * k + 1]);
    cw.w3v_h2[k] = *reinterpret_cast<const uint32_t*>(&w);
  }
  for (int q = 0; q < 8; ++q) cw.Bb3[q] = q < 7 ? Bb3[q] : 0.f;
}

inline cudaError_t set_attributes() {
  cudaError_t e;
  if ((e = cudaFuncSetAttribute(k_render_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes))) return e;
  if ((e = cudaFuncSetAttribute(k_render_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes))) return e;
  if ((e = cudaFuncSetAttribute(k_trace_tc<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes))) return e;
  if ((e = cudaFuncSetAttribute(k_trace_tc<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes))) return e;
  return cudaSuccess;
}

inline bool frame_supported(const FrameP& fr) { return !(fr.flags & 4u) || fr.t.stride != 0 || fr.t.S <= (uint32_t)kMaxS2; }

inline int grid_size(unsigned long long N, int num_sms) {
  const unsigned long long tiles = (N + kThreads - 1) / kThreads;
  const unsigned long long cap = (unsigned long long)num_sms * 3;
  return (int)(tiles < cap ? tiles : cap);
}

// h_blob: host copy of the prepared blob (for the by-value TcConst); d_tiles: device pointer to the tiles
inline cudaError_t launch_render(const GridP& g, const EnvP& env, const ShadeP& sp, const TcConst& cw, const uint8_t* d_tiles,
                                 const FrameP& fr, float* rgb, int num_sms, cudaStream_t st) {
  const int grid = grid_size(fr.N, num_sms);
  if (g.f16) k_render_tc<true><<<grid, kThreads, kSmemBytes, st>>>(g, env, sp, cw, d_tiles, fr, rgb);
  else k_render_tc<false><<<grid, kThreads, kSmemBytes, st>>>(g, env, sp, cw, d_tiles, fr, rgb);
  return cudaGetLastError();
}

inline cudaError_t launch_trace(const GridP& g, const ShadeP& sp, const TcConst& cw, const uint8_t* d_tiles, const float* x,
                                unsigned long long N, const DirsetP& ds, float* vis, float* zv, float* t, float* xsec, int num_sms,
                                cudaStream_t st) {
  const int grid = grid_size(N, num_sms);
  if (g.f16) k_trace_tc<true><<<grid, kThreads, kSmemBytes, st>>>(g, sp, cw, d_tiles, x, N, ds, vis, zv, t, xsec);
  else k_trace_tc<false><<<grid, kThreads, kSmemBytes, st>>>(g, sp, cw, d_tiles, x, N, ds, vis, zv, t, xsec);
  return cudaGetLastError();
}

}  // namespace tc
}  // namespace hr
