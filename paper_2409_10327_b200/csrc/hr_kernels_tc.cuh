// hr_kernels_tc.cuh -- tensor-core (tcgen05 / TMEM) implementation of the fused path for mlp_dtype == HR_F16.
//
// Design: a CTA is 128 threads = the 128 TMEM lanes; thread p owns primary point
// p of the CTA's 128-point tile for the whole frame (direct set, secondary set, and the tertiary set of each of its
// secondary points), so no activation ever crosses threads.  Every 64-wide MLP layer over the tile is ONE
// M=128 x N=64 tcgen05.mma group: each thread packs its row of fp16 activations straight into TMEM (tcgen05.st,
// the A operand is read from TMEM), weights sit in shared memory as K-major SWIZZLE_128B UMMA tiles, the fp32
// accumulator comes back with tcgen05.ld and the bias/ReLU/last-layer dot products run from constant-bank
// operands.  Layer-1 biases ride in the MMA as an extra K step (hi + lo fp16 split => exact to 2^-22).
// The query loops are software-pipelined two deep over two (A, D) TMEM buffer pairs, and the gathers of the next
// secondary point are spread over the tertiary loop of the current one, so a thread's gathers, packing, MMA and
// epilogue overlap; two CTAs per SM cover the remaining serial phases.
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
constexpr int kTmemCols = 256;                // per CTA; two CTAs per SM own the whole TMEM
constexpr int kTileBytes = 64 * 128;          // one 64 x 64 fp16 K-major SW128 weight tile
constexpr int kNumTiles = 4;                  // I.W1f(+b1,b2), B.W1(+b1,b2), I.W2, B.W2  (64 x 64 each)
constexpr int kTile3Bytes = 16 * 128;         // B.W3 zero-padded to 16 x 64 (N = 16 MMA)
constexpr int kAllTileBytes = kNumTiles * kTileBytes + kTile3Bytes;
constexpr int kCtasPerSm = 2;
constexpr int kMaxS2 = 16;                    // shared tertiary set staged in smem
// TMEM column map (per CTA).  Two (A, D) buffer pairs let one query's MMA run under the next query's packing and
// the previous query's epilogue.  A buffer b: columns 64 b .. 64 b + 31 (fp16 pairs); the split-precision layers use
// A0 columns 0..63 (hi | lo).  Columns 32..47 stage the NEXT secondary point's features while the tertiary loop of
// the current one runs.  Columns 96..103 hold the constant bias K-step [1, 1, 0 .. 0].  D buffer b: 128 + 64 b.
constexpr uint32_t kColA = 0, kColNext = 32, kColOne = 96, kColD = 128, kBufStride = 64;

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
// Warp-level variants: the whole (converged) warp executes them and one elected lane issues, so the operands stay in the
// uniform datapath instead of being broadcast lane by lane inside a divergent branch.
__device__ __forceinline__ void mma_f16_ts_elect(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p, e;\n\tsetp.ne.b32 p, %4, 0;\n\telect.sync _|e, 0xffffffff;\n\t"
      "@e tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accum)
      : "memory");
}
// A from shared memory (descriptor), B from shared memory
__device__ __forceinline__ void mma_f16_ss_elect(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p, e;\n\tsetp.ne.b32 p, %4, 0;\n\telect.sync _|e, 0xffffffff;\n\t"
      "@e tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accum)
      : "memory");
}
__device__ __forceinline__ void mma_commit_elect(uint32_t mbar) {
  asm volatile("{\n\t.reg .pred e;\n\telect.sync _|e, 0xffffffff;\n\t"
               "@e tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];\n\t}\n" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mma_commit(uint32_t mbar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile("{\n\t.reg .pred P1;\n\tmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\n\tselp.b32 %0, 1, 0, P1;\n\t}\n"
                 : "=r"(done) : "r"(mbar), "r"(parity) : "memory");
  } while (!__all_sync(0xFFFFFFFFu, done));                 // warp-uniform exit keeps the code after the wait convergent
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
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr) : "memory");
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
constexpr uint32_t kIdescN16 = (1u << 4) | ((16u >> 3) << 17) | ((128u >> 4) << 24);


struct Ctx {
  uint32_t lane;               // this warp's TMEM lane base (bits 31..16)
  uint32_t base;               // TMEM base of the CTA's allocation (lane 0, column 0)
  uint32_t mbar;               // smem address of mbarrier 0 (mbarrier 1 at +8)
  uint32_t phase;              // bit b = parity to wait for on mbarrier b
  uint32_t tile0;              // smem address of weight tile 0 (tile t at + t * kTileBytes)
};
__device__ __forceinline__ uint32_t colA(const Ctx& c, int buf) { return c.base + c.lane + kColA + kBufStride * buf; }
__device__ __forceinline__ uint32_t colD(const Ctx& c, int buf) { return c.base + c.lane + kColD + kBufStride * buf; }
__device__ __forceinline__ uint32_t colNext(const Ctx& c) { return c.base + c.lane + kColNext; }

// Issue one 128 x N layer on buffer pair `buf`: D[buf] = A * W^T where A starts `a_off` columns into the CTA's TMEM
// (lane 0 address), `ksteps` K-steps of 16; optional split lo block right after the hi block; optional bias K-step
// (A = [1,1,0..] times K-step `bias_kstep` of tile `bias_tile`).  Every thread must have issued its tcgen05.st of A.
// Does NOT wait for the MMA: wait_layer(c, buf) does.
__device__ __forceinline__ void issue_layer(Ctx& c, int buf, uint32_t a_off, int tile, int ksteps, int bias_tile, int bias_kstep,
                                            bool split = false, uint32_t idesc = kIdesc) {
  wait_st();
  fence_before();
  __syncthreads();
  if (threadIdx.x == 0) {
    fence_after();
    const uint32_t d = c.base + kColD + kBufStride * buf;
    const uint32_t a = c.base + a_off;
    const uint64_t bd = make_bdesc(c.tile0 + tile * kTileBytes);
    for (int k = 0; k < ksteps; ++k) mma_f16_ts(d, a + 8 * k, bd + 2 * k, idesc, k > 0);
    if (split)
      for (int k = 0; k < ksteps; ++k) mma_f16_ts(d, a + 8 * (ksteps + k), bd + 2 * k, idesc, 1u);
    if (bias_tile >= 0) mma_f16_ts(d, c.base + kColOne, make_bdesc(c.tile0 + bias_tile * kTileBytes) + 2 * bias_kstep, idesc, 1u);
    mma_commit(c.mbar + 8 * buf);
  }
}
__device__ __forceinline__ void wait_layer(Ctx& c, int buf) {
  mbar_wait(c.mbar + 8 * buf, (c.phase >> buf) & 1u);
  c.phase ^= 1u << buf;
  fence_after();
}

// ---------------------------------------------------------------------------------------------------- encode pieces
// residual of an fp16x2 pack: (a - fp16(a), b - fp16(b)) packed again (the "lo" half of a hi/lo split)
__device__ __forceinline__ uint32_t pack_lo(uint32_t hi, float a, float b) {
  const float2 h = __half22float2(*reinterpret_cast<const __half2*>(&hi));
  return pack_rn(a - h.x, b - h.y);
}

// Primary point: f = H(x) in fp32, level l -> A0 column l (fp16 pair) and its fp16 residual -> column 16 + l
// (split-precision features for the layer-1 partial P, which feeds the t that moves x').
template <bool F16>
__device__ __forceinline__ void encode_split_to_A(const GridP& g, const Ctx& c, float x, float y, float z) {
  const uint32_t tA = colA(c, 0);
#pragma unroll 2
  for (int l = 0; l < kMaxL; ++l) {
    uint32_t hi = 0u, lo = 0u;
    if (l < (int)g.L) {
      const float2 v = encode_level<F16>(g, l, x, y, z, nullptr, nullptr);
      hi = pack_rn(v.x, v.y);
      lo = pack_lo(hi, v.x, v.y);
    }
    tmem_st1(tA + l, hi);
    tmem_st1(tA + 16 + l, lo);
  }
}

// Secondary points: the gathers of one level (issued early) and their interpolation (consumed late) are separate so
// the caller can put a whole tertiary query between them.  fp16 tables: the 8 half2 rows are interpolated with fp16x2
// lerps (x, y, z: 7 sub + 7 fma) and the result IS the packed A-operand word.  The cell / index path is fp32 + integer,
// identical to encode_level.
template <bool F16> struct LevelTaps;
template <> struct LevelTaps<true> { __half2 v[8]; __half2 w[3]; };
template <> struct LevelTaps<false> { float2 v[8]; float w[3]; };

template <bool F16>
__device__ __forceinline__ void gather_level(const GridP& g, int l, float x, float y, float z, LevelTaps<F16>& t) {
  const uint32_t N = g.res[l];
  const Cell cl = cell_of_clamped(N, x, y, z);                 // callers pass x' = sec_hit(...), already in [0,1]^3
  uint32_t idx[8];
  corner_indices(cl, N, (g.dense_mask >> l) & 1u, g.log2_T, idx);
  const void* lb = level_base<F16>(g.tables, g.log2_T, l);
  if constexpr (F16) {
#pragma unroll
    for (int k = 0; k < 8; ++k) t.v[k] = gather_h2(lb, idx[k]);
#pragma unroll
    for (int d = 0; d < 3; ++d) t.w[d] = __float2half2_rn(cl.w[d]);
  } else {
#pragma unroll
    for (int k = 0; k < 8; ++k) t.v[k] = gather_f2(lb, idx[k]);
#pragma unroll
    for (int d = 0; d < 3; ++d) t.w[d] = cl.w[d];
  }
}
__device__ __forceinline__ uint32_t lerp_level(const LevelTaps<true>& t) {
  __half2 a[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) a[k] = __hfma2(t.w[0], __hsub2(t.v[2 * k + 1], t.v[2 * k]), t.v[2 * k]);
  const __half2 b0 = __hfma2(t.w[1], __hsub2(a[1], a[0]), a[0]);
  const __half2 b1 = __hfma2(t.w[1], __hsub2(a[3], a[2]), a[2]);
  const __half2 r = __hfma2(t.w[2], __hsub2(b1, b0), b0);
  return *reinterpret_cast<const uint32_t*>(&r);
}
__device__ __forceinline__ uint32_t lerp_level(const LevelTaps<false>& t) {
  float2 a[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    a[k].x = fmaf(t.w[0], t.v[2 * k + 1].x - t.v[2 * k].x, t.v[2 * k].x);
    a[k].y = fmaf(t.w[0], t.v[2 * k + 1].y - t.v[2 * k].y, t.v[2 * k].y);
  }
  const float b0x = fmaf(t.w[1], a[1].x - a[0].x, a[0].x), b0y = fmaf(t.w[1], a[1].y - a[0].y, a[0].y);
  const float b1x = fmaf(t.w[1], a[3].x - a[2].x, a[2].x), b1y = fmaf(t.w[1], a[3].y - a[2].y, a[2].y);
  return pack_rn(fmaf(t.w[2], b1x - b0x, b0x), fmaf(t.w[2], b1y - b0y, b0y));
}

// whole fast encode of one secondary point into the staging columns (used for the first secondary point of a pixel
// and whenever the tertiary loop cannot carry the gathers)
template <bool F16>
__device__ __forceinline__ void encode_next_plain(const GridP& g, const Ctx& c, float x, float y, float z) {
  const uint32_t tN = colNext(c);
#pragma unroll 1
  for (int l0 = 0; l0 < kMaxL; l0 += 2) {
    LevelTaps<F16> t0, t1;
    const bool on0 = l0 < (int)g.L, on1 = l0 + 1 < (int)g.L;
    if (on0) gather_level<F16>(g, l0, x, y, z, t0);
    if (on1) gather_level<F16>(g, l0 + 1, x, y, z, t1);
    tmem_st1(tN + l0, on0 ? lerp_level(t0) : 0u);
    tmem_st1(tN + l0 + 1, on1 ? lerp_level(t1) : 0u);
  }
}

// ---------------------------------------------------------------------------------------------------- per-row stages
// Precise epilogue of I (secondary set: z_t becomes t): (z_v, z_t) = b3 + W3 relu(D + b2), all fp32.
__device__ __forceinline__ void irt_epilogue_precise(const Ctx& c, const TcConst& cw, int buf, float& zv, float& zt) {
  float z0[4] = {cw.b3[0], 0.f, 0.f, 0.f}, z1[4] = {cw.b3[1], 0.f, 0.f, 0.f};
  const uint32_t tD = colD(c, buf);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; ++k) {
      const float a = fmaxf(__uint_as_float(r[k]) + cw.b2[32 * h + k], 0.f);
      z0[k & 3] = fmaf(a, cw.w3[0][32 * h + k], z0[k & 3]);
      z1[k & 3] = fmaf(a, cw.w3[1][32 * h + k], z1[k & 3]);
    }
  }
  zv = (z0[0] + z0[1]) + (z0[2] + z0[3]);
  zt = (z1[0] + z1[1]) + (z1[2] + z1[3]);
}

// Fast epilogue of I (direct and tertiary queries need only visibility): b2 already rode in the MMA (bias K-step),
// h2 = relu(D) is rounded to fp16 by the packing conversion, z_v = b3 + w3v . h2 with fp16x2 FMAs into four short
// accumulators summed in fp32.
__device__ __forceinline__ float irt_epilogue_fast(const Ctx& c, const TcConst& cw, int buf) {
  __half2 acc[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) acc[q] = __float2half2_rn(0.f);
  const uint32_t tD = colD(c, buf);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
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

// D0 -> relu -> fp16 -> A0 columns 0..31
__device__ __forceinline__ void hidden_to_A(const Ctx& c) {
  const uint32_t tD = colD(c, 0), tA = colA(c, 0);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
    uint32_t p[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) p[k] = pack_relu(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
    tmem_st16(tA + 16 * h, p);
  }
}

// B(f) with the fp16 features at column offset f_off: all three layers on the tensor core (layer-1/2 biases ride in
// the MMAs, layer 3 is an N = 16 MMA over the zero-padded 7-row W3; b3 is added in registers).  Buffer pair 0.
__device__ __forceinline__ void brdf_from_A(Ctx& c, const TcConst& cw, const ShadeP& sp, uint32_t f_off, float (&b)[7]) {
  issue_layer(c, 0, f_off, 1, 2, 1, 2);
  wait_layer(c, 0);
  hidden_to_A(c);
  issue_layer(c, 0, kColA, 3, 4, 1, 3);
  wait_layer(c, 0);
  hidden_to_A(c);
  issue_layer(c, 0, kColA, 4, 4, -1, 0, false, kIdescN16);
  wait_layer(c, 0);
  uint32_t r[8];
  tmem_ld8(colD(c, 0), r);
  wait_ld();
  float o[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) o[q] = __uint_as_float(r[q]) + cw.Bb3[q];
  brdf_maps(sp, o, b);
}

// Primary point only (once per pixel): B in split precision.  n = o/||o|| amplifies an absolute error of o by 1/||o||
// and every sample of the pixel sees the same n, so fp16-grade activations here would be a COHERENT pixel error; the
// hi/lo split of f (already in A0[0..31]) and of the hidden layer keeps B's inputs to ~2^-22, layer 3 runs in fp32.
__device__ __forceinline__ void brdf_precise_from_A(Ctx& c, const TcConst& cw, const ShadeP& sp, float (&b)[7]) {
  issue_layer(c, 0, kColA, 1, 2, 1, 2, true);
  wait_layer(c, 0);
  const uint32_t tD = colD(c, 0), tA = colA(c, 0);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
    uint32_t p[16], q[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const float a0 = fmaxf(__uint_as_float(r[2 * k]), 0.f), a1 = fmaxf(__uint_as_float(r[2 * k + 1]), 0.f);
      p[k] = pack_rn(a0, a1);
      q[k] = pack_lo(p[k], a0, a1);
    }
    tmem_st16(tA + 16 * h, p);
    tmem_st16(tA + 32 + 16 * h, q);
  }
  issue_layer(c, 0, kColA, 3, 4, 1, 3, true);
  wait_layer(c, 0);
  float o[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) o[q] = cw.Bb3[q];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
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

// h1 = relu(P + W1w . w) -> A[buf] columns 0..31 (P in registers)
__device__ __forceinline__ void h1_from_regs(const Ctx& c, const TcConst& cw, int buf, const float (&P)[kH], float wx, float wy, float wz) {
  const uint32_t tA = colA(c, buf);
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
    tmem_st16(tA + 16 * h, p);
  }
}
// split-precision variant for the secondary set (its z_t becomes t and moves x': SURVEY 8(c) conditioning note):
// h1 in fp32 -> hi (A0 columns 0..31) + lo (columns 32..63); P from this thread's shared-memory column
__device__ __forceinline__ void h1_from_smem_split(const Ctx& c, const TcConst& cw, const float* Ps, float wx, float wy, float wz) {
  const uint32_t tA = colA(c, 0);
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
    tmem_st16(tA + 16 * h, p);
    tmem_st16(tA + 32 + 16 * h, q);
  }
}
// shared direction set: the direction part Q = W1w . w'_k is precomputed per CTA, h1 = relu(P + Q)
__device__ __forceinline__ void h1_from_regs_shared(const Ctx& c, int buf, const float (&P)[kH], const float* __restrict__ Q) {
  const uint32_t tA = colA(c, buf);
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
    tmem_st16(tA + 16 * h, p);
  }
}

// shared direction set, all-fp16x2 form: P and Q both pre-rounded to fp16 pairs, h1 = fma.relu(P, 1, Q): one
// instruction per pair (the sum is rounded once more: 1.5 ulp of fp16 instead of 0.5 -- tertiary visibility only)
__device__ __forceinline__ void h1_from_h2_shared(const Ctx& c, int buf, const uint32_t (&Ph)[kH / 2], const uint32_t* __restrict__ Qh) {
  const uint32_t tA = colA(c, buf);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t p[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint4 q = reinterpret_cast<const uint4*>(Qh)[4 * h + k];
      const uint32_t qq[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
      for (int e = 0; e < 4; ++e)
        asm("fma.rn.relu.f16x2 %0, %1, %2, %3;" : "=r"(p[4 * k + e]) : "r"(Ph[16 * h + 4 * k + e]), "r"(0x3C003C00u), "r"(qq[e]));
    }
    tmem_st16(tA + 16 * h, p);
  }
}
// D0 -> fp16 pairs (32 registers)
__device__ __forceinline__ void load_D_h2(const Ctx& c, uint32_t (&Ph)[kH / 2]) {
  const uint32_t tD = colD(c, 0);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 16; ++k) Ph[16 * h + k] = pack_rn(__uint_as_float(r[2 * k]), __uint_as_float(r[2 * k + 1]));
  }
}

// D0 -> registers (64 fp32)
__device__ __forceinline__ void load_D(const Ctx& c, float (&P)[kH]) {
  const uint32_t tD = colD(c, 0);
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    uint32_t r[32];
    tmem_ld32(tD + 32 * h, r);
    wait_ld();
#pragma unroll
    for (int k = 0; k < 32; ++k) P[32 * h + k] = __uint_as_float(r[k]);
  }
}

// ---------------------------------------------------------------------------------------------------- shared setup
struct Smem {
  uint8_t* tiles;      // 4 x 8 KB + 2 KB, 1024-aligned
  float* Ps;           // [64][128]
  float* Qt;           // [kMaxS2][64]
  float* Lt;           // [kMaxS2][8]: radiance rgb, pdf, direction xyz, pad
  uint64_t* mbar;      // [2]
  uint32_t* tmem_slot;
};
constexpr size_t kSmemBytes = 1024 + kAllTileBytes + kH * kThreads * 4 + kMaxS2 * kH * 4 + kMaxS2 * 8 * 4 + 64;

__device__ __forceinline__ Smem carve(uint8_t* raw) {
  Smem s;
  uint8_t* p = raw + ((1024u - (smem_u32(raw) & 1023u)) & 1023u);      // pointer arithmetic keeps the shared address space
  s.tiles = p; p += kAllTileBytes;
  s.Ps = reinterpret_cast<float*>(p); p += kH * kThreads * 4;
  s.Qt = reinterpret_cast<float*>(p); p += kMaxS2 * kH * 4;
  s.Lt = reinterpret_cast<float*>(p); p += kMaxS2 * 8 * 4;
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
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(s.mbar + 1)) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const uint4* src = reinterpret_cast<const uint4*>(wtiles);
  uint4* dst = reinterpret_cast<uint4*>(s.tiles);
  for (int i = threadIdx.x; i < kAllTileBytes / 16; i += kThreads) dst[i] = __ldg(src + i);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the tensor core
  fence_before();
  __syncthreads();
  fence_after();
  c.base = *s.tmem_slot;
  c.lane = (uint32_t)(warp * 32) << 16;
  c.mbar = smem_u32(s.mbar); c.phase = 0;
  c.tile0 = smem_u32(s.tiles);
  uint32_t one[8] = {0x3C003C00u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};     // bias K-step of A: [1, 1, 0, ... 0]
  tmem_st8(c.base + c.lane + kColOne, one);
  wait_st();
}

__device__ __forceinline__ void teardown(const Ctx& c) {
  fence_before();
  __syncthreads();
  if ((threadIdx.x >> 5) == 0) {
    fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(c.base), "r"((uint32_t)kTmemCols) : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------- host side
struct HostWeights { TcConst cw; };

inline size_t tile_off(int j, int k) { return (size_t)(j / 8) * 1024 + (j % 8) * 128 + (((k / 8) ^ (j % 8)) * 16) + (k % 8) * 2; }

// Blob = [ TcConst | 4 UMMA tiles ].  The TcConst part is passed by value at launch, the tiles stay in HBM/L2.
inline void prepare_weights(const hr_config& cfg, const float* bw, const float* iw, std::vector<uint8_t>& out) {
  const int D = cfg.L * cfg.F, H = kH, Din = D + 3;
  out.assign(sizeof(TcConst) + kAllTileBytes, 0);
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
    for (int q = 0; q < 7; ++q) { cw.BW3[q][j] = BW3[q * H + j]; put(4, q, j, BW3[q * H + j]); }
  }
  cw.b3[0] = Ib3[0]; cw.b3[1] = Ib3[1];
  for (int k = 0; k < H / 2; ++k) {
    const __half2 w = __floats2half2_rn(IW3[2 * k], IW3[2 * k + 1]);
    cw.w3v_h2[k] = *reinterpret_cast<const uint32_t*>(&w);
  }
  for (int q = 0; q < 8; ++q) cw.Bb3[q] = q < 7 ? Bb3[q] : 0.f;
}

inline bool frame_supported(const FrameP& fr) { return !(fr.flags & 4u) || fr.t.stride != 0 || fr.t.S <= (uint32_t)kMaxS2; }

}  // namespace tc
}  // namespace hr
