// hr_kernels_tc.cuh -- tcgen05 / TMEM building blocks shared by the warpgroup kernels (hr_render_wg.cuh): PTX wrappers
// (tcgen05.mma / ld / st / commit, mbarrier), fp16x2 packing, the K-major SWIZZLE_128B shared-memory descriptor, the
// per-level gather + fp16x2 interpolation of the fast encoder, the constant block passed by value (TcConst) and the host-side
// layout of the UMMA weight tiles.
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

constexpr int kTileBytes = 64 * 128;          // one 64 x 64 fp16 K-major SW128 weight tile
constexpr int kNumTiles = 4;                  // I.W1f(+b1,b2), B.W1(+b1,b2), I.W2, B.W2  (64 x 64 each)
constexpr int kTile3Bytes = 16 * 128;         // B.W3 zero-padded to 16 x 64 (N = 16 MMA)
constexpr int kAllTileBytes = kNumTiles * kTileBytes + kTile3Bytes;
constexpr int kMaxS2 = 16;                    // shared tertiary set staged in smem

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

// The whole (converged) warp executes these and one elected lane issues, so the operands stay in the uniform datapath
// instead of being broadcast lane by lane inside a divergent branch.
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
// A short poll.  (Measured and not kept: try_wait with a long suspend-time hint turns the six-instruction loop -- 6.4 iterations per
// tertiary query, 12 % of the instructions issued -- into one or two instructions, but the warp then wakes later than a poll notices
// the phase flip, and the kernel is bound by exactly that MMA round trip: C2 23.35 -> 23.6 ms, C3 16.7 -> 17.05 ms.)
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
constexpr uint32_t kIdescN128 = (1u << 4) | ((128u >> 3) << 17) | ((128u >> 4) << 24);

// ---------------------------------------------------------------------------------------------------- encode pieces
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
  if constexpr (F16) {
    uint32_t r[8];
    gather8_h2(g, l, cl.c0, r);
#pragma unroll
    for (int k = 0; k < 8; ++k) t.v[k] = *reinterpret_cast<const __half2*>(&r[k]);
#pragma unroll
    for (int d = 0; d < 3; ++d) t.w[d] = __float2half2_rn(cl.w[d]);
  } else {
    gather8_f2(g, l, cl.c0, t.v);
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

__device__ __forceinline__ float vis_of(const ShadeP& sp, float zv) { return sp.vis_mode ? (zv > 0.f ? 1.f : 0.f) : sigmoidf_(zv); }
// ---------------------------------------------------------------------------------------------------- host side

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
